"""Thin ctypes binding of libafqmc (include/afqmc.h): argument marshalling only.

Every step of the path runs inside the library's CUDA kernels; PyTorch is used for device
memory (torch tensors own every buffer) and for the current CUDA stream.  There is no CPU
fallback: if the library is missing or a call fails, an exception is raised.
"""
from __future__ import annotations

import ctypes
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libafqmc.so")
_lib = None

ERRORS = {0: "ok", 1: "invalid argument", 2: "unsupported configuration", 3: "CUDA error", 4: "out of device memory",
          5: "request exceeds the static scratch array of the no-allocation entry point"}


class AfqmcError(RuntimeError):
    def __init__(self, code, where):
        self.code = code
        super().__init__("%s failed: %s (code %d)" % (where, ERRORS.get(code, "?"), code))


class Dims(ctypes.Structure):
    _fields_ = [("g", ctypes.c_int * 3), ("m", ctypes.c_int), ("n", ctypes.c_int), ("nchol", ctypes.c_int),
                ("closed_shell", ctypes.c_int), ("precision", ctypes.c_int), ("max_walkers", ctypes.c_int),
                ("n_dn", ctypes.c_int)]


EXPORTS = ["afqmc_strerror", "afqmc_create", "afqmc_destroy", "afqmc_overlap", "afqmc_green", "afqmc_force_bias",
           "afqmc_vhs", "afqmc_propagate", "afqmc_local_energy", "afqmc_step", "afqmc_step_host",
           "afqmc_launch_count", "afqmc_exchange_flops", "afqmc_force_bias_flops", "afqmc_set_option", "afqmc_stage_times", "afqmc_probe_fp64",
           "afqmc_set_onebody", "afqmc_apply_onebody", "afqmc_hybrid_weight", "afqmc_orthogonalize",
           "afqmc_mixed_estimator", "afqmc_block",
           "afqmc_step_host_begin", "afqmc_step_host_end",
           "afqmc_overlap_noalloc", "afqmc_overlap_noalloc_setup", "afqmc_overlap_noalloc_bytes", "afqmc_overlap_noalloc_max_bytes"]


def lib():
    """Loads libafqmc.so (built in-tree by `paper_2003_09468_b200.build`); raises if it is absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError("libafqmc.so not found at %s: run `python -m paper_2003_09468_b200.build` "
                           "(there is no CPU fallback)" % LIB_PATH)
    L = ctypes.CDLL(LIB_PATH)
    vp, ci, cd = ctypes.c_void_p, ctypes.c_int, ctypes.c_double
    L.afqmc_strerror.restype = ctypes.c_char_p
    L.afqmc_strerror.argtypes = [ci]
    L.afqmc_create.argtypes = [ctypes.POINTER(vp), ctypes.POINTER(Dims), vp, vp, vp, vp]
    L.afqmc_destroy.argtypes = [vp]
    L.afqmc_destroy.restype = None
    L.afqmc_overlap.argtypes = [vp, vp, ci, vp, vp, vp]
    L.afqmc_green.argtypes = [vp, vp, ci, vp, vp, vp, vp]
    L.afqmc_force_bias.argtypes = [vp, vp, ci, vp, vp]
    L.afqmc_vhs.argtypes = [vp, vp, vp, cd, ci, vp, vp]
    L.afqmc_propagate.argtypes = [vp, vp, cd, ci, vp, ci, vp]
    L.afqmc_local_energy.argtypes = [vp, vp, ci, vp, vp]
    L.afqmc_step.argtypes = [vp, vp, vp, cd, ci, ci, vp, vp, vp, vp]
    L.afqmc_step_host.argtypes = [vp, vp, vp, cd, ci, ci, vp, vp, vp, vp]
    L.afqmc_launch_count.argtypes = [vp]
    L.afqmc_launch_count.restype = ctypes.c_longlong
    L.afqmc_exchange_flops.argtypes = [vp, ci]
    L.afqmc_exchange_flops.restype = cd
    L.afqmc_force_bias_flops.argtypes = [vp, ci]
    L.afqmc_force_bias_flops.restype = cd
    L.afqmc_set_option.argtypes = [vp, ctypes.c_char_p, ci]
    L.afqmc_probe_fp64.argtypes = [ci, ci, ctypes.POINTER(cd)]
    L.afqmc_stage_times.argtypes = [vp, ctypes.POINTER(ctypes.c_float)]
    L.afqmc_set_onebody.argtypes = [vp, vp, cd, vp, vp]
    L.afqmc_apply_onebody.argtypes = [vp, vp, ci, vp]
    L.afqmc_hybrid_weight.argtypes = [vp, vp, vp, cd, vp, vp, ci, vp, vp, vp]
    L.afqmc_orthogonalize.argtypes = [vp, vp, ci, vp, vp, vp]
    L.afqmc_mixed_estimator.argtypes = [vp, vp, vp, ci, vp, vp]
    L.afqmc_block.argtypes = [vp, vp, vp, vp, cd, ci, ci, ci, vp, vp, vp, vp, vp]
    L.afqmc_step_host_begin.argtypes = [vp, ci, vp, vp, cd, ci, ci, vp, vp, vp, vp, vp]
    L.afqmc_step_host_end.argtypes = [vp, ci]
    L.afqmc_overlap_noalloc.argtypes = [ctypes.POINTER(Dims), vp, vp, ci, vp, vp, vp]
    L.afqmc_overlap_noalloc_setup.argtypes = []
    L.afqmc_overlap_noalloc_bytes.argtypes = [ctypes.POINTER(Dims), ci]
    L.afqmc_overlap_noalloc_bytes.restype = ctypes.c_size_t
    L.afqmc_overlap_noalloc_max_bytes.argtypes = []
    L.afqmc_overlap_noalloc_max_bytes.restype = ctypes.c_size_t
    for name in EXPORTS:
        if name not in ("afqmc_strerror", "afqmc_destroy", "afqmc_launch_count", "afqmc_exchange_flops", "afqmc_force_bias_flops",
                        "afqmc_overlap_noalloc_bytes", "afqmc_overlap_noalloc_max_bytes"):
            getattr(L, name).restype = ci
    _lib = L
    return L


def _stream():
    return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)


def _ptr(t, dtype=None, optional=False):
    if t is None:
        if optional:
            return ctypes.c_void_p(0)
        raise ValueError("required tensor is None")
    if dtype is not None and t.dtype != dtype:
        raise TypeError("expected %s, got %s" % (dtype, t.dtype))
    if not t.is_contiguous():
        raise ValueError("tensor must be contiguous")
    return ctypes.c_void_p(t.data_ptr())


def _check(code, where):
    if code != 0:
        raise AfqmcError(code, where)


def overlap_noalloc_max_bytes() -> int:
    return int(lib().afqmc_overlap_noalloc_max_bytes())


def overlap_noalloc_bytes(mesh, m, n, nw) -> int:
    d = Dims((ctypes.c_int * 3)(*[int(g) for g in mesh]), int(m), int(n), 0, 1, 0, int(nw), 0)
    return int(lib().afqmc_overlap_noalloc_bytes(ctypes.byref(d), int(nw)))


def overlap_noalloc_setup():
    """Resolves the static scratch array's device address on the current device (e.g. before a graph capture)."""
    _check(lib().afqmc_overlap_noalloc_setup(), "afqmc_overlap_noalloc_setup")


def overlap_noalloc(mesh, m, n, psi_t, phi, logdet, info=None):
    """afqmc_overlap_noalloc: log det of the trial-walker overlaps with NO allocation anywhere (no context; the matrices live
    in the library's static 16 MiB device array).  The caller passes inputs AND outputs: psi_t [Nk][m][n], phi [nw][M][N],
    logdet [nw] complex128 CUDA tensors, info [nw] int32 or None.  Raises AfqmcError (code 5) beyond the scratch limit."""
    nk = int(mesh[0]) * int(mesh[1]) * int(mesh[2])
    nw = int(phi.shape[0])
    for t, shape, dt, name in ((psi_t, (nk, m, n), torch.complex128, "psi_t"), (phi, (nw, nk * m, nk * n), torch.complex128, "phi"),
                               (logdet, (nw,), torch.complex128, "logdet")) + (((info, (nw,), torch.int32, "info"),) if info is not None else ()):
        if not t.is_cuda or t.device != phi.device or tuple(t.shape) != tuple(shape) or t.dtype != dt:
            raise ValueError("%s: expected a %s CUDA tensor of shape %s on %s" % (name, dt, tuple(shape), phi.device))
    d = Dims((ctypes.c_int * 3)(*[int(g) for g in mesh]), int(m), int(n), 0, 1, 0, nw, 0)
    with torch.cuda.device(phi.device):
        _check(lib().afqmc_overlap_noalloc(ctypes.byref(d), _ptr(psi_t), _ptr(phi), nw, _ptr(logdet), _ptr(info, optional=True), _stream()),
               "afqmc_overlap_noalloc")
    return logdet, info


def probe_fp64(kind: int, iters: int = 20000) -> float:
    out = ctypes.c_double(0.0)
    _check(lib().afqmc_probe_fp64(kind, iters, ctypes.byref(out)), "afqmc_probe_fp64")
    return out.value


class Afqmc:
    """Context of one Hamiltonian + trial on the current CUDA device (afqmc_create / afqmc_destroy)."""

    def __init__(self, mesh, m, n, nchol, h1, L, psi_t, max_walkers, closed_shell=1, precision=0, n_dn=0):
        """Open shell (closed_shell=0): `n` is the spin-up and `n_dn` the spin-down occupied count per k-point, `psi_t` is the
        pair (psi_up [Nk][m][n], psi_dn [Nk][m][n_dn]); walkers and Green's functions are then FLAT spin-major tensors (the
        spin-up block of all walkers followed by the spin-down block, include/afqmc.h "Open shell"): see join_spin/split_*."""
        self._h = ctypes.c_void_p(0)
        self.mesh = tuple(int(v) for v in mesh)
        self.nk = self.mesh[0] * self.mesh[1] * self.mesh[2]
        self.m, self.n, self.nchol = int(m), int(n), int(nchol)
        self.M, self.N = self.nk * self.m, self.nk * self.n
        self.open_shell = int(closed_shell) == 0
        self.n_dn = int(n_dn) if self.open_shell else 0
        self.N_dn = self.nk * self.n_dn
        self.max_walkers = int(max_walkers)
        self.precision = int(precision)
        # dtypes at the boundary: complex128/float64, or complex64/float32 with precision = 1 (include/afqmc.h "Precision 1")
        self.cdtype = torch.complex64 if self.precision == 1 else torch.complex128
        self.rdtype = torch.float32 if self.precision == 1 else torch.float64
        d = Dims((ctypes.c_int * 3)(*self.mesh), self.m, self.n, self.nchol, closed_shell, precision, self.max_walkers, self.n_dn)
        if self.open_shell:
            psi_up, psi_dn = psi_t
            if tuple(psi_up.shape) != (self.nk, self.m, self.n) or tuple(psi_dn.shape) != (self.nk, self.m, self.n_dn):
                raise ValueError("open shell: psi_t must be the pair ([Nk][m][n], [Nk][m][n_dn])")
            psi_t = torch.cat([psi_up.contiguous().reshape(-1), psi_dn.contiguous().reshape(-1)])
        for name, t, shape in (("h1", h1, (self.nk, self.m, self.m)),
                               ("L", L, (self.nk, self.nk, self.nchol, self.m, self.m)),
                               ("psi_t", psi_t, (psi_t.numel(),) if self.open_shell else (self.nk, self.m, self.n))):
            if not t.is_cuda or tuple(t.shape) != shape:
                raise ValueError("%s must be a CUDA tensor of shape %s" % (name, shape))
        self.device = h1.device
        for t in (L, psi_t):
            if t.device != self.device:
                raise ValueError("h1, L and psi_t must live on the same CUDA device")
        h = ctypes.c_void_p(0)
        with torch.cuda.device(self.device):       # the library allocates its workspace on the CURRENT device
            code = lib().afqmc_create(ctypes.byref(h), ctypes.byref(d), _ptr(h1, self.cdtype),
                                      _ptr(L, self.cdtype), _ptr(psi_t, self.cdtype), _stream())
        _check(code, "afqmc_create")
        self._h = h

    def close(self):
        if self._h:
            lib().afqmc_destroy(self._h)
            self._h = ctypes.c_void_p(0)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- helpers -------------------------------------------------------------------------
    def _empty(self, shape, dtype=None):
        return torch.empty(shape, dtype=self.cdtype if dtype is None else dtype, device=self.device)

    # ---- open shell: flat spin-major walker / Green's function tensors ----
    def join_spin(self, up, dn):
        """(up [nw][..][..], dn [nw][..][..]) -> the flat spin-major tensor the library takes."""
        return torch.cat([up.contiguous().reshape(-1), dn.contiguous().reshape(-1)])

    def split_phi(self, flat, nw):
        a = nw * self.M * self.N
        return flat[:a].view(nw, self.M, self.N), flat[a:].view(nw, self.M, self.N_dn)

    def split_theta(self, flat, nw):
        a = nw * self.N * self.M
        return flat[:a].view(nw, self.N, self.M), flat[a:].view(nw, self.N_dn, self.M)

    def _phi_shape(self, nw):
        return (nw * self.M * (self.N + self.N_dn),) if self.open_shell else (nw, self.M, self.N)

    def _theta_shape(self, nw):
        return (nw * (self.N + self.N_dn) * self.M,) if self.open_shell else (nw, self.N, self.M)

    def _nw(self, t, name):
        """Batch size of a per-walker tensor; the library would read past `max_walkers` worth of workspace otherwise."""
        nw = int(t.shape[0])
        if self.open_shell and t.dim() == 1 and name in ("phi", "theta", "phi_host"):
            per = self.M * (self.N + self.N_dn)
            if t.numel() % per != 0:
                raise ValueError("%s: flat spin-major tensor of %d elements is not a multiple of M*(N_up+N_dn) = %d" % (name, t.numel(), per))
            nw = t.numel() // per
        if nw > self.max_walkers:
            raise ValueError("%s: %d walkers > max_walkers = %d" % (name, nw, self.max_walkers))
        return nw

    def _dev(self, t, shape, dtype, name, optional=False):
        """Marshals one DEVICE tensor: exact shape, dtype, contiguity and device are checked here, because past this
        point the tensor is a raw pointer (a wrong shape would be a silent out-of-bounds access in a kernel)."""
        if t is None:
            if optional:
                return ctypes.c_void_p(0)
            raise ValueError("%s is required" % name)
        if not t.is_cuda or t.device != self.device:
            raise ValueError("%s must be a CUDA tensor on %s (got %s)" % (name, self.device, t.device))
        if tuple(t.shape) != tuple(shape):
            raise ValueError("%s must have shape %s (got %s)" % (name, tuple(shape), tuple(t.shape)))
        return _ptr(t, dtype)

    def _host(self, t, shape, dtype, name, optional=False):
        if t is None:
            if optional:
                return ctypes.c_void_p(0)
            raise ValueError("%s is required" % name)
        if t.is_cuda:
            raise ValueError("%s must be a host tensor" % name)
        if tuple(t.shape) != tuple(shape):
            raise ValueError("%s must have shape %s (got %s)" % (name, tuple(shape), tuple(t.shape)))
        return _ptr(t, dtype)

    def _call(self, fn, *args):
        with torch.cuda.device(self.device):
            return fn(self._h, *args, _stream())

    def launch_count(self) -> int:
        return int(lib().afqmc_launch_count(self._h))

    def exchange_flops(self, nw) -> float:
        return float(lib().afqmc_exchange_flops(self._h, int(nw)))

    def force_bias_flops(self, nw) -> float:
        return float(lib().afqmc_force_bias_flops(self._h, int(nw)))

    def set_option(self, name: str, value: int):
        _check(lib().afqmc_set_option(self._h, name.encode(), int(value)), "afqmc_set_option")

    STAGES = ("green", "force_bias", "vhs", "propagate", "green2", "force_bias2", "exchange", "finalize")

    def stage_times(self):
        """Per-stage ms of the last step() (needs set_option('timers', 1) and a synchronised stream)."""
        buf = (ctypes.c_float * 8)()
        _check(lib().afqmc_stage_times(self._h, buf), "afqmc_stage_times")
        return dict(zip(self.STAGES, [float(v) for v in buf]))

    # ---- the six step calls ----------------------------------------------------------------
    def overlap(self, phi, logdet=None, info=None):
        nw = self._nw(phi, "phi")
        logdet = self._empty((nw,)) if logdet is None else logdet
        info = self._empty((nw,), torch.int32) if info is None else info
        _check(self._call(lib().afqmc_overlap, self._dev(phi, self._phi_shape(nw), self.cdtype, "phi"), nw,
                          self._dev(logdet, (nw,), self.cdtype, "logdet"), self._dev(info, (nw,), torch.int32, "info")),
               "afqmc_overlap")
        return logdet, info

    def green(self, phi, theta=None, logdet=None, info=None):
        nw = self._nw(phi, "phi")
        theta = self._empty(self._theta_shape(nw)) if theta is None else theta
        logdet = self._empty((nw,)) if logdet is None else logdet
        info = self._empty((nw,), torch.int32) if info is None else info
        _check(self._call(lib().afqmc_green, self._dev(phi, self._phi_shape(nw), self.cdtype, "phi"), nw,
                          self._dev(theta, self._theta_shape(nw), self.cdtype, "theta"),
                          self._dev(logdet, (nw,), self.cdtype, "logdet"), self._dev(info, (nw,), torch.int32, "info")),
               "afqmc_green")
        return theta, logdet, info

    def force_bias(self, theta, vbias=None):
        nw = self._nw(theta, "theta")
        vbias = self._empty((nw, self.nk, self.nchol)) if vbias is None else vbias
        _check(self._call(lib().afqmc_force_bias, self._dev(theta, self._theta_shape(nw), self.cdtype, "theta"), nw,
                          self._dev(vbias, (nw, self.nk, self.nchol), self.cdtype, "vbias")), "afqmc_force_bias")
        return vbias

    def vhs(self, x, vbias, dtau, vhs=None):
        nw = self._nw(x, "x")
        vhs = self._empty((nw, self.M, self.M)) if vhs is None else vhs
        _check(self._call(lib().afqmc_vhs, self._dev(x, (nw, self.nk, self.nchol), self.rdtype, "x"),
                          self._dev(vbias, (nw, self.nk, self.nchol), self.cdtype, "vbias", optional=True),
                          float(dtau), nw, self._dev(vhs, (nw, self.M, self.M), self.cdtype, "vhs")), "afqmc_vhs")
        return vhs

    def propagate(self, vhs, dtau, order, phi):
        nw = self._nw(phi, "phi")
        _check(self._call(lib().afqmc_propagate, self._dev(vhs, (nw, self.M, self.M), self.cdtype, "vhs"), float(dtau),
                          int(order), self._dev(phi, self._phi_shape(nw), self.cdtype, "phi"), nw), "afqmc_propagate")
        return phi

    def local_energy(self, theta, energy=None):
        nw = self._nw(theta, "theta")
        energy = self._empty((nw, 3)) if energy is None else energy
        _check(self._call(lib().afqmc_local_energy, self._dev(theta, self._theta_shape(nw), self.cdtype, "theta"), nw,
                          self._dev(energy, (nw, 3), self.cdtype, "energy")), "afqmc_local_energy")
        return energy

    # ---- the whole step ------------------------------------------------------------------------
    def step(self, phi, x, dtau, order, energy=None, logdet=None, info=None):
        nw = self._nw(phi, "phi")
        energy = self._empty((nw, 3)) if energy is None else energy
        logdet = self._empty((nw,)) if logdet is None else logdet
        info = self._empty((nw,), torch.int32) if info is None else info
        _check(self._call(lib().afqmc_step, self._dev(phi, self._phi_shape(nw), self.cdtype, "phi"),
                          self._dev(x, (nw, self.nk, self.nchol), self.rdtype, "x"), float(dtau), int(order), nw,
                          self._dev(energy, (nw, 3), self.cdtype, "energy"), self._dev(logdet, (nw,), self.cdtype, "logdet"),
                          self._dev(info, (nw,), torch.int32, "info")), "afqmc_step")
        return energy, logdet, info

    def step_host(self, phi_host, x_host, dtau, order, energy_host, logdet_host=None, info_host=None):
        """Host (ideally pinned) tensors in and out; H2D/D2H copies happen inside the call."""
        nw = self._nw(phi_host, "phi_host")
        _check(self._call(lib().afqmc_step_host, self._host(phi_host, self._phi_shape(nw), self.cdtype, "phi_host"),
                          self._host(x_host, (nw, self.nk, self.nchol), self.rdtype, "x_host"), float(dtau), int(order), nw,
                          self._host(energy_host, (nw, 3), self.cdtype, "energy_host"),
                          self._host(logdet_host, (nw,), self.cdtype, "logdet_host", optional=True),
                          self._host(info_host, (nw,), torch.int32, "info_host", optional=True)), "afqmc_step_host")
        return energy_host

    def step_host_begin(self, slot, phi_host, x_host, dtau, order, phi_out_host, energy_host, logdet_host=None, info_host=None):
        """Pipelined host step (two slots): enqueues upload, step and downloads and returns at once; step_host_end(slot) waits."""
        nw = self._nw(phi_host, "phi_host")
        with torch.cuda.device(self.device):
            _check(lib().afqmc_step_host_begin(self._h, int(slot), self._host(phi_host, self._phi_shape(nw), self.cdtype, "phi_host"),
                                               self._host(x_host, (nw, self.nk, self.nchol), self.rdtype, "x_host"), float(dtau),
                                               int(order), nw, self._host(phi_out_host, self._phi_shape(nw), self.cdtype, "phi_out_host"),
                                               self._host(energy_host, (nw, 3), self.cdtype, "energy_host"),
                                               self._host(logdet_host, (nw,), self.cdtype, "logdet_host", optional=True),
                                               self._host(info_host, (nw,), torch.int32, "info_host", optional=True), _stream()),
                   "afqmc_step_host_begin")

    def step_host_end(self, slot):
        with torch.cuda.device(self.device):
            _check(lib().afqmc_step_host_end(self._h, int(slot)), "afqmc_step_host_end")

    # ---- the AFQMC block (include/afqmc.h "The AFQMC block") ----------------------------------------
    def set_onebody(self, h1p, dtau, b1_out=None):
        """B1[k] = exp(-dtau/2 h1p[k]) computed on the device and kept in the context; returns a copy."""
        shp = (self.nk, self.m, self.m)
        b1_out = self._empty(shp) if b1_out is None else b1_out
        _check(self._call(lib().afqmc_set_onebody, self._dev(h1p, shp, torch.complex128, "h1p"), float(dtau),
                          self._dev(b1_out, shp, torch.complex128, "b1_out")), "afqmc_set_onebody")
        return b1_out

    def apply_onebody(self, phi):
        nw = self._nw(phi, "phi")
        _check(self._call(lib().afqmc_apply_onebody, self._dev(phi, self._phi_shape(nw), torch.complex128, "phi"), nw),
               "afqmc_apply_onebody")
        return phi

    def hybrid_weight(self, x, vbias, dtau, logdet_old, logdet_new, weight, log_i=None):
        nw = self._nw(x, "x")
        log_i = self._empty((nw,)) if log_i is None else log_i
        fld = (nw, self.nk, self.nchol)
        _check(self._call(lib().afqmc_hybrid_weight, self._dev(x, fld, torch.float64, "x"),
                          self._dev(vbias, fld, torch.complex128, "vbias"), float(dtau),
                          self._dev(logdet_old, (nw,), torch.complex128, "logdet_old"),
                          self._dev(logdet_new, (nw,), torch.complex128, "logdet_new"), nw,
                          self._dev(weight, (nw,), torch.float64, "weight"), self._dev(log_i, (nw,), torch.complex128, "log_i")),
               "afqmc_hybrid_weight")
        return weight, log_i

    def orthogonalize(self, phi, logdet_r=None, info=None):
        nw = self._nw(phi, "phi")
        logdet_r = self._empty((nw,), torch.float64) if logdet_r is None else logdet_r
        info = self._empty((nw,), torch.int32) if info is None else info
        _check(self._call(lib().afqmc_orthogonalize, self._dev(phi, self._phi_shape(nw), torch.complex128, "phi"), nw,
                          self._dev(logdet_r, (nw,), torch.float64, "logdet_r"), self._dev(info, (nw,), torch.int32, "info")),
               "afqmc_orthogonalize")
        return phi, logdet_r, info

    def mixed_estimator(self, energy, weight, out=None):
        nw = int(energy.shape[0])
        out = self._empty((4,)) if out is None else out
        _check(self._call(lib().afqmc_mixed_estimator, self._dev(energy, (nw, 3), torch.complex128, "energy"),
                          self._dev(weight, (nw,), torch.float64, "weight"), nw, self._dev(out, (4,), torch.complex128, "out")),
               "afqmc_mixed_estimator")
        return out

    def block(self, phi, weight, x, dtau, order, energy=None, emixed=None, logdet_r=None, info=None):
        """x [nsteps][nw][Nk][nchol]; phi and weight are updated in place."""
        nsteps, nw = int(x.shape[0]), self._nw(phi, "phi")
        energy = self._empty((nw, 3)) if energy is None else energy
        emixed = self._empty((4,)) if emixed is None else emixed
        logdet_r = self._empty((nw,), torch.float64) if logdet_r is None else logdet_r
        info = self._empty((nw,), torch.int32) if info is None else info
        _check(self._call(lib().afqmc_block, self._dev(phi, self._phi_shape(nw), torch.complex128, "phi"),
                          self._dev(weight, (nw,), torch.float64, "weight"),
                          self._dev(x, (nsteps, nw, self.nk, self.nchol), torch.float64, "x"), float(dtau), int(order), nsteps, nw,
                          self._dev(energy, (nw, 3), torch.complex128, "energy"), self._dev(emixed, (4,), torch.complex128, "emixed"),
                          self._dev(logdet_r, (nw,), torch.float64, "logdet_r"), self._dev(info, (nw,), torch.int32, "info")),
               "afqmc_block")
        return energy, emixed, logdet_r, info


def from_problem(pb, max_walkers=None, device="cuda", precision=0):
    """Builds a context from a `synth.Problem` (host numpy arrays -> device tensors; complex64 with precision = 1)."""
    cfg = pb.cfg
    dev = torch.device(device)
    cd = torch.complex64 if precision == 1 else torch.complex128
    h1 = torch.from_numpy(pb.h1).to(dev).to(cd)
    L = torch.from_numpy(pb.L).to(dev).to(cd)
    psi_t = torch.from_numpy(pb.psi_t).to(dev).to(cd)
    ctx = Afqmc(cfg.mesh, cfg.m, cfg.n, cfg.nchol, h1, L, psi_t, max_walkers or pb.phi.shape[0], precision=precision)
    del L
    return ctx
