"""CPU-side checks of the boundary: the library builds, loads, and exports every symbol that
include/afqmc.h declares.  No compute calls (no GPU here)."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "afqmc.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(afqmc_[a-z0-9_]+)\s*\(", text)))


def test_library_builds_and_exports_every_declared_symbol():
    from paper_2003_09468_b200 import build, binding
    path = build.build()
    assert os.path.exists(path)
    lib = ctypes.CDLL(path)
    declared = _declared_symbols()
    assert len(declared) >= 12
    for name in declared:
        assert hasattr(lib, name), name
    assert set(binding.EXPORTS) == set(declared)
    assert binding.lib() is not None


def test_strerror_is_callable_without_a_gpu():
    from paper_2003_09468_b200 import binding
    lib = binding.lib()
    assert lib.afqmc_strerror(0) == b"ok"
    assert lib.afqmc_strerror(2) == b"unsupported configuration"
    assert lib.afqmc_strerror(99) == b"unknown error code"
    assert lib.afqmc_launch_count(None) == 0


def test_create_rejects_bad_arguments_before_touching_cuda():
    from paper_2003_09468_b200 import binding
    lib = binding.lib()
    h = ctypes.c_void_p(0)
    d = binding.Dims((ctypes.c_int * 3)(2, 2, 2), 8, 4, 32, 1, 0, 4, 0)
    assert lib.afqmc_create(ctypes.byref(h), ctypes.byref(d), None, None, None, None) == 1
    assert lib.afqmc_create(None, ctypes.byref(d), None, None, None, None) == 1
    lib.afqmc_destroy(None)


def test_pipelined_host_entry_rejects_bad_arguments_before_touching_cuda():
    from paper_2003_09468_b200 import binding
    lib = binding.lib()
    assert lib.afqmc_step_host_end(None, 0) == 1
    assert lib.afqmc_step_host_begin(None, 0, None, None, 0.005, 6, 1, None, None, None, None, None) == 1


def test_product_path_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2003_09468_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle", src, flags=re.M), f
                assert "afqmc_oracle" not in src and "oracle/" not in src and '#include "oracle' not in src, f


def test_synth_real_orbital_inputs_are_real_and_keep_the_pair_identity():
    """synth.make_problem(real_orbitals=True): h1, psi_t, L real (zero imaginary parts), the (Q,-Q) identity holds with
    transposes, walkers stay complex; the default stream is unchanged by the option's existence."""
    import numpy as np
    from paper_2003_09468_b200 import synth
    cfg = synth.tiny_config(mesh=(2, 1, 1), m=4, n=2, nchol=3, nw=2, seed=9)
    pb = synth.make_problem(cfg, real_orbitals=True)
    assert np.all(pb.L.imag == 0) and np.all(pb.psi_t.imag == 0) and np.all(pb.h1.imag == 0)
    assert np.abs(pb.phi.imag).max() > 0
    kminus, neg = synth.kpoint_tables(cfg.mesh)
    for Q in range(cfg.nk):
        for k in range(cfg.nk):
            assert np.array_equal(pb.L[neg[Q], kminus[k, Q]], np.swapaxes(pb.L[Q, k], -1, -2))
    assert np.array_equal(synth.make_problem(cfg).L, synth.make_problem(cfg, real_orbitals=False).L)
