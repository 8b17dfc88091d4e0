// Context creation (a0 setup: half-rotation + repack into DMMA fragment layouts), destruction,
// error strings, options.  Setup is once per simulation and is not timed.
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <vector>
#include "common.cuh"

int afqmc_i_vhs_setup(afqmc_ctx* c, const double2* L, const std::vector<int>& kminus, const std::vector<int>& kneg,
                      cudaStream_t st);   // vhs.cu

AFQMC_API const char* afqmc_strerror(int code) {
    switch (code) {
        case AFQMC_OK: return "ok";
        case AFQMC_INVALID_ARGUMENT: return "invalid argument";
        case AFQMC_UNSUPPORTED: return "unsupported configuration";
        case AFQMC_CUDA_ERROR: return "CUDA error";
        case AFQMC_OUT_OF_MEMORY: return "out of device memory";
        case AFQMC_SCRATCH_LIMIT: return "request exceeds the static scratch array of the no-allocation entry point";
        default: return "unknown error code";
    }
}

// ---------------------------------------------------------------------------------------
// Fragment layouts.  In all three the innermost 32 doubles are one DMMA A-fragment in lane
// order: lane l holds A[row = l>>2][kk = l&3]; the k-step s covers reals 4s..4s+3 of the
// real-embedded K index (complex index j>>1, part j&1 with j = 4s+kk).
//
//  Lx (exchange, a9):   [Q][k][ag][gq][s][lane][i]  two M-tiles i = 0,1 per gamma-quad gq, interleaved
//                        per lane (one LDG.128 feeds both); rows (gl = row>>2, al = row&3):
//                        gamma = 4gq+2i+gl, a = 4ag+al;  K = (r, part) of Lh[Q][k][a][gamma][r]
//                        (+ AFQMC_LX_PAD zero doubles at the end: the kernel's prefetch may run past the last task)
//  (the force-bias operand Lf3, the vHS operand Lv3 and the 3M exchange operands are described and packed in force_bias.cu,
//   vhs.cu and exchange3m.cu)
// Out-of-range rows / K entries are stored as zeros, so kernels never branch on tails.
// ---------------------------------------------------------------------------------------
// Lh[Q][k][a][gam][r] = sum_p conj(A_k[p][a]) L[Q][k][gam][p][r], computed once; natural layout
__global__ void half_rot_L_kernel(Dims d, const double2* __restrict__ L, const double2* __restrict__ psi_t,
                                  double2* __restrict__ Lh, size_t total) {
    for (size_t idx = blockIdx.x * (size_t)blockDim.x + threadIdx.x; idx < total; idx += (size_t)gridDim.x * blockDim.x) {
        size_t t = idx;
        const int r = (int)(t % d.m); t /= d.m;
        const int gam = (int)(t % d.nchol); t /= d.nchol;
        const int a = (int)(t % d.n); t /= d.n;
        const int k = (int)(t % d.Nk);
        const int Q = (int)(t / d.Nk);
        const double2* Lb = L + (((size_t)(Q * d.Nk + k) * d.nchol + gam) * d.m) * d.m + r;
        const double2* Ab = psi_t + (size_t)k * d.m * d.n + a;
        double2 acc = make_double2(0.0, 0.0);
        for (int p = 0; p < d.m; ++p) {
            double2 av = Ab[(size_t)p * d.n];
            av.y = -av.y;
            acc = cfma(av, Lb[(size_t)p * d.m], acc);
        }
        Lh[idx] = acc;
    }
}

__device__ __forceinline__ double2 lh_elem(const double2* __restrict__ Lh, const Dims& d, int Q, int k, int a, int gam, int r) {
    return Lh[((((size_t)Q * d.Nk + k) * d.n + a) * d.nchol + gam) * d.m + r];
}

__global__ void pack_Lx_kernel(Dims d, const double2* __restrict__ Lh, double* __restrict__ Lx, size_t total) {
    for (size_t idx = blockIdx.x * (size_t)blockDim.x + threadIdx.x; idx < total;
         idx += (size_t)gridDim.x * blockDim.x) {
        size_t t = idx;
        int i = (int)(t & 1); t >>= 1;
        int lane = (int)(t & 31); t >>= 5;
        int s = (int)(t % d.KS); t /= d.KS;
        int gq = (int)(t % d.GQ); t /= d.GQ;
        int ag = (int)(t % d.NAG); t /= d.NAG;
        int k = (int)(t % d.Nk);
        int Q = (int)(t / d.Nk);
        int row = lane >> 2, kk = lane & 3;
        int gam = 4 * gq + 2 * i + (row >> 2), a = 4 * ag + (row & 3);
        int j = 4 * s + kk, r = j >> 1, c = j & 1;
        double v = 0.0;
        if (Q < d.Nk && a < d.n && gam < d.nchol && r < d.m) {   // Q >= Nk: the zero pad
            double2 z = lh_elem(Lh, d, Q, k, a, gam, r);
            v = c ? z.y : z.x;
        }
        Lx[idx] = v;
    }
}

// max |Im z| over an array (ordered-int atomic on the bit pattern of a non-negative double: exact, order independent)
__global__ void max_abs_imag_kernel(const double2* __restrict__ p, size_t n, unsigned long long* __restrict__ out) {
    double mx = 0.0;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) mx = fmax(mx, fabs(p[i].y));
    atomicMax(out, (unsigned long long)__double_as_longlong(mx));
}

int afqmc_i_max_abs_imag(afqmc_ctx* c, const double2* p, size_t n, double* out_host, cudaStream_t st) {
    unsigned long long* d = nullptr;
    AFQMC_CUDA_TRY(cudaMalloc((void**)&d, sizeof(unsigned long long)));
    cudaMemsetAsync(d, 0, sizeof(unsigned long long), st);
    max_abs_imag_kernel<<<148 * 8, 256, 0, st>>>(p, n, d);
    c->launches++;
    unsigned long long h = 0;
    cudaError_t e = cudaMemcpyAsync(&h, d, sizeof(h), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    cudaFree(d);
    if (e != cudaSuccess) { (void)cudaGetLastError(); return AFQMC_CUDA_ERROR; }
    memcpy(out_host, &h, 8);
    return AFQMC_OK;
}

__global__ void half_rot_h_kernel(Dims d, const double2* __restrict__ h1, const double2* __restrict__ psi_t,
                                  double2* __restrict__ ht) {
    // ht[k][a][q] = sum_p conj(A_k[p][a]) h_k[p][q]     (first line of Eq. 49)
    int total = d.Nk * d.n * d.m;
    for (int idx = blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += gridDim.x * blockDim.x) {
        int q = idx % d.m, a = (idx / d.m) % d.n, k = idx / (d.m * d.n);
        double2 acc = make_double2(0.0, 0.0);
        for (int p = 0; p < d.m; ++p) {
            double2 av = psi_t[((size_t)k * d.m + p) * d.n + a];
            av.y = -av.y;
            acc = cfma(av, h1[((size_t)k * d.m + p) * d.m + q], acc);
        }
        ht[idx] = acc;
    }
}

// ---------------------------------------------------------------------------------------
static int kidx(const int* g, int a, int b, int c) {
    a = ((a % g[0]) + g[0]) % g[0];
    b = ((b % g[1]) + g[1]) % g[1];
    c = ((c % g[2]) + g[2]) % g[2];
    return (a * g[1] + b) * g[2] + c;
}

template <typename T>
static int dev_alloc(T** p, size_t count) {
    *p = nullptr;
    if (count == 0) count = 1;
    cudaError_t e = cudaMalloc((void**)p, count * sizeof(T));
    if (e != cudaSuccess) {
        (void)cudaGetLastError();
        *p = nullptr;
        return (e == cudaErrorMemoryAllocation) ? AFQMC_OUT_OF_MEMORY : AFQMC_CUDA_ERROR;
    }
    return AFQMC_OK;
}

AFQMC_API void afqmc_destroy(afqmc_ctx* c) {
    if (!c) return;
    for (int slot = 0; slot < 2; ++slot) (void)afqmc_step_host_end(c, slot);      // pipelined host steps still in flight
    if (c->dn) { afqmc_destroy(c->dn); c->dn = nullptr; }
    if (c->is_child) c->b1 = nullptr;        // owned by the spin-up context
    void* ptrs[] = {c->kminus, c->kplus, c->kneg, c->units, c->psi_t, c->ht, c->Lh, c->Lxc, c->Lxr, c->Lx3t, c->Lx, c->LxT, c->LxU, c->Lf, c->Lff, c->Lv3, c->Lv3f, c->vunits,
                    c->ws_O, c->ws_oinvT, c->ws_theta, c->ws_vbias, c->ws_xi, c->ws_vhs, c->ws_T, c->ws_Tx,
                    c->ws_expart, c->ws_fbpart, c->ws_thetaF, c->ws_thetaU, c->ws_vbtot, c->ws_ld_chan, c->ws_info_chan, c->ws_ldr_chan, c->ws_x, c->ws_phi, c->ws_energy, c->ws_logdet, c->ws_info,
                    c->ws_f32, c->b1, c->ws_b1tmp, c->ws_gram, c->ws_rinv, c->ws_logdet2, c->ws_ldr, c->ws_info2};
    for (void* p : ptrs)
        if (p) cudaFree(p);
    for (cudaEvent_t e : c->ev)
        if (e) cudaEventDestroy(e);
    for (cudaEvent_t e : c->ev_copy)
        if (e) cudaEventDestroy(e);
    if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
    if (c->copyin_stream) cudaStreamDestroy(c->copyin_stream);
    for (int s = 0; s < 2; ++s)
        for (cudaEvent_t e : c->ev_pipe[s])
            if (e) cudaEventDestroy(e);
    void* pipe_ptrs[] = {c->pipe_phi, c->pipe_x, c->pipe_energy, c->pipe_logdet, c->pipe_info};
    for (void* p : pipe_ptrs)
        if (p) cudaFree(p);
    delete c;
}

// One spin channel: the whole closed-shell context (n = `n_chan` occupied orbitals per k-point), or one of the two channels
// of an open-shell context (spin_factor 1).  The spin-DOWN channel (`child`) has no vHS operand, no field / vHS workspace
// and no one-body propagator of its own: those are spin independent and live in the spin-up (parent) context.
static int create_channel(afqmc_ctx** out, const afqmc_dims* dims, int n_chan, int n_total, const void* h1, const void* L,
                          const void* psi_t, cudaStream_t st, bool child, bool open_shell) {
    *out = nullptr;
    const long long nk_ll = (long long)dims->g[0] * dims->g[1] * dims->g[2];
    afqmc_ctx* c = new afqmc_ctx();
    memset(c, 0, sizeof(*c));
    Dims& d = c->d;
    for (int i = 0; i < 3; ++i) d.g[i] = dims->g[i];
    d.Nk = (int)nk_ll; d.m = dims->m; d.n = n_chan; d.nchol = dims->nchol;
    d.M = d.Nk * d.m; d.N = d.Nk * d.n;
    d.KS = (2 * d.m + 3) / 4;
    d.NAG = (d.n + 3) / 4;
    d.GP = (d.nchol + 1) / 2;
    d.GQ = (d.nchol + 3) / 4;
    d.PRT = (d.m * d.m + 7) / 8;
    c->max_walkers = dims->max_walkers;
    c->prec32 = dims->precision == 1 ? 1 : 0;
    c->opt_exchange_3m = 1;
    c->opt_real = 1;
    c->opt_exchange_tc = 1;
    c->opt_exchange_regb = 1;
    c->spin_factor = open_shell ? 1.0 : 2.0;
    c->is_child = child ? 1 : 0;
    const int nw = c->max_walkers;

    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { delete c; return AFQMC_CUDA_ERROR; }
    c->device = dev;
    cudaDeviceGetAttribute(&c->smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    cudaDeviceGetAttribute(&c->num_sms, cudaDevAttrMultiProcessorCount, dev);
    cudaDeviceGetAttribute(&c->smem_sm, cudaDevAttrMaxSharedMemoryPerMultiprocessor, dev);

    // ---- k-point tables and exchange work units (host) ----
    const int Nk = d.Nk;
    std::vector<int> kminus(Nk * Nk), kplus(Nk * Nk), kneg(Nk);
    for (int k = 0; k < Nk; ++k) {
        int k1 = k / (d.g[1] * d.g[2]), k2 = (k / d.g[2]) % d.g[1], k3 = k % d.g[2];
        kneg[k] = kidx(d.g, -k1, -k2, -k3);
        for (int Q = 0; Q < Nk; ++Q) {
            int q1 = Q / (d.g[1] * d.g[2]), q2 = (Q / d.g[2]) % d.g[1], q3 = Q % d.g[2];
            kminus[k * Nk + Q] = kidx(d.g, k1 - q1, k2 - q2, k3 - q3);
            kplus[k * Nk + Q] = kidx(d.g, k1 + q1, k2 + q2, k3 + q3);
        }
    }
    // unit (Q,k,k2): T^Q[(k,a),(k2,b),g] contracted with its partner T^{-Q}[(k2,b),(k,a),g];
    // the partner unit is (-Q,k2,k) (an involution), so each unordered pair is computed once.
    std::vector<int> units;
    for (int Q = 0; Q < Nk; ++Q)
        for (int k = 0; k < Nk; ++k)
            for (int k2 = 0; k2 < Nk; ++k2) {
                int Qp = kneg[Q], kp = k2, k2p = k;
                long long me = ((long long)Q * Nk + k) * Nk + k2, pa = ((long long)Qp * Nk + kp) * Nk + k2p;
                if (pa < me) continue;
                units.push_back(Q); units.push_back(k); units.push_back(k2);
                units.push_back(pa == me ? 1 : 2);
            }
    c->nunits = (int)(units.size() / 4);

    int rc = AFQMC_OK;
    auto A = [&](int r) { if (rc == AFQMC_OK) rc = r; };
    const size_t nLh = (size_t)Nk * Nk * d.n * d.nchol * d.m;
    const int LD = d.N | 1;
    A(dev_alloc(&c->kminus, (size_t)Nk * Nk));
    A(dev_alloc(&c->kplus, (size_t)Nk * Nk));
    A(dev_alloc(&c->kneg, (size_t)Nk));
    A(dev_alloc(&c->units, units.size()));
    A(dev_alloc(&c->psi_t, (size_t)Nk * d.m * d.n));
    A(dev_alloc(&c->ht, (size_t)Nk * d.n * d.m));
    A(dev_alloc(&c->Lh, nLh));
    A(dev_alloc(&c->ws_O, (size_t)nw * d.N * LD));
    A(dev_alloc(&c->ws_oinvT, (size_t)nw * d.N * d.N));
    A(dev_alloc(&c->ws_theta, (size_t)nw * (child ? d.N : Nk * n_total) * d.M));     // spin-up context: both channels, spin-major
    A(dev_alloc(&c->ws_vbias, (size_t)nw * Nk * d.nchol));
    if (!child) {
        A(dev_alloc(&c->ws_xi, (afqmc_i_vhs_field_doubles(d, nw) + 1) / 2));   // expanded field fragments (vhs.cu)
        A(dev_alloc(&c->ws_vhs, (size_t)nw * d.M * d.M));
        if (open_shell) A(dev_alloc(&c->ws_vbtot, (size_t)nw * Nk * d.nchol));  // spin-summed force bias
    }
    A(dev_alloc(&c->ws_T, (size_t)2 * nw * d.M * d.N));
    const size_t nTx = (size_t)2 * nw * afqmc_i_taylor_ws_doubles(d);
    A(dev_alloc(&c->ws_Tx, nTx));
    c->ex_parts_max = afqmc_i_exchange3m_parts_max(c);      // exchange partial sums per unit (exchange3m.cu)
    c->ex_parts = 1;
    A(dev_alloc(&c->ws_expart, (size_t)c->nunits * nw * c->ex_parts_max));
    A(dev_alloc(&c->ws_fbpart, (size_t)AFQMC_FB_MAXKC * nw * Nk * d.nchol));
    if (!child) {      // host-entry staging: all channels of a walker batch
        A(dev_alloc(&c->ws_x, (size_t)nw * Nk * d.nchol));
        A(dev_alloc(&c->ws_phi, (size_t)nw * d.M * Nk * n_total));
    }
    A(dev_alloc(&c->ws_energy, (size_t)nw * 3));
    A(dev_alloc(&c->ws_logdet, (size_t)nw));
    A(dev_alloc(&c->ws_info, (size_t)nw));
    if (!child) {
        A(dev_alloc(&c->b1, (size_t)Nk * d.m * d.m));
        A(dev_alloc(&c->ws_b1tmp, (size_t)Nk * 3 * d.m * d.m));
    }
    A(dev_alloc(&c->ws_gram, (size_t)nw * d.N * d.N));
    A(dev_alloc(&c->ws_rinv, (size_t)nw * d.N * d.N));
    A(dev_alloc(&c->ws_logdet2, (size_t)nw));
    A(dev_alloc(&c->ws_ldr, (size_t)2 * nw));
    A(dev_alloc(&c->ws_info2, (size_t)2 * nw));
    A(dev_alloc(&c->ws_ld_chan, (size_t)nw));
    A(dev_alloc(&c->ws_info_chan, (size_t)nw));
    A(dev_alloc(&c->ws_ldr_chan, (size_t)nw));
    if (c->prec32) A(dev_alloc(&c->ws_f32, (size_t)nw * ((size_t)d.M * d.N * 2 + (size_t)Nk * d.nchol + 8)));
    if (rc != AFQMC_OK) { afqmc_destroy(c); return rc; }
    // complex64 boundary: the static inputs are widened once into FP64 temporaries (freed before returning)
    double *h1w = nullptr, *Lw = nullptr, *psiw = nullptr;
    if (c->prec32) {
        A(afqmc32_widen_alloc(c, h1, (size_t)Nk * d.m * d.m * 2, &h1w, st));
        A(afqmc32_widen_alloc(c, L, (size_t)Nk * Nk * d.nchol * d.m * d.m * 2, &Lw, st));
        A(afqmc32_widen_alloc(c, psi_t, (size_t)Nk * d.m * d.n * 2, &psiw, st));
        if (rc != AFQMC_OK) { cudaFree(h1w); cudaFree(Lw); cudaFree(psiw); afqmc_destroy(c); return rc; }
        h1 = h1w; L = Lw; psi_t = psiw;
    }

    auto H2D = [&](void* dst, const void* src, size_t bytes) {
        if (rc == AFQMC_OK && cudaMemcpyAsync(dst, src, bytes, cudaMemcpyHostToDevice, st) != cudaSuccess)
            rc = AFQMC_CUDA_ERROR;
    };
    // the padding tiles of the expanded Taylor buffers are read but never written by the GEMM epilogue
    if (cudaMemsetAsync(c->ws_Tx, 0, nTx * sizeof(double), st) != cudaSuccess) rc = AFQMC_CUDA_ERROR;
    H2D(c->kminus, kminus.data(), kminus.size() * sizeof(int));
    H2D(c->kplus, kplus.data(), kplus.size() * sizeof(int));
    H2D(c->kneg, kneg.data(), kneg.size() * sizeof(int));
    H2D(c->units, units.data(), units.size() * sizeof(int));
    if (rc == AFQMC_OK &&
        cudaMemcpyAsync(c->psi_t, psi_t, (size_t)Nk * d.m * d.n * sizeof(double2), cudaMemcpyDeviceToDevice, st) != cudaSuccess)
        rc = AFQMC_CUDA_ERROR;
    if (rc == AFQMC_OK) {
        const int T = 256;
        auto grid = [&](size_t total) { return (int)((total + T - 1) / T > 148 * 64 ? 148 * 64 : (total + T - 1) / T); };
        half_rot_h_kernel<<<grid((size_t)Nk * d.n * d.m), T, 0, st>>>(d, (const double2*)h1, c->psi_t, c->ht);
        half_rot_L_kernel<<<grid(nLh), T, 0, st>>>(d, (const double2*)L, c->psi_t, c->Lh, nLh);     // the half rotation, once
        c->launches += 2;
        if (cudaGetLastError() != cudaSuccess) rc = AFQMC_CUDA_ERROR;
        // real orbitals?  (exact zeros: a real L half-rotated with a real trial has no imaginary part at all)
        if (rc == AFQMC_OK) {
            double im = 1.0;
            rc = afqmc_i_max_abs_imag(c, c->Lh, nLh, &im, st);
            c->real_lh = (rc == AFQMC_OK && im == 0.0) ? 1 : 0;
        }
        // force-bias operand Lf3 (single-precision storage when precision = 1)
        if (rc == AFQMC_OK) rc = afqmc_i_pack_force_bias_operand(c, st);
        if (rc == AFQMC_OK) rc = afqmc_i_pack_exchange_operand(c, st);
        if (rc == AFQMC_OK && !child) rc = afqmc_i_vhs_setup(c, (const double2*)L, kminus, kneg, st);
    }
    // host vectors must outlive the async copies; the caller may free its arrays after return
    if (cudaStreamSynchronize(st) != cudaSuccess && rc == AFQMC_OK) rc = AFQMC_CUDA_ERROR;
    cudaFree(h1w); cudaFree(Lw); cudaFree(psiw);
    if (rc != AFQMC_OK) { (void)cudaGetLastError(); afqmc_destroy(c); return rc; }
    if (c->prec32 && d.NAG == 1) c->opt_exchange_prec = 1;      // complex64 boundary: 3xTF32 exchange by default (operands packed on first use)
    *out = c;
    return AFQMC_OK;
}

AFQMC_API int afqmc_create(afqmc_ctx** out, const afqmc_dims* dims, const void* h1, const void* L,
                            const void* psi_t, void* stream) {
    if (!out) return AFQMC_INVALID_ARGUMENT;
    *out = nullptr;
    if (!dims || !h1 || !L || !psi_t) return AFQMC_INVALID_ARGUMENT;
    if (dims->g[0] < 1 || dims->g[1] < 1 || dims->g[2] < 1 || dims->m < 1 || dims->n < 1 ||
        dims->n > dims->m || dims->nchol < 1 || dims->max_walkers < 1)
        return AFQMC_INVALID_ARGUMENT;
    const long long nk_ll = (long long)dims->g[0] * dims->g[1] * dims->g[2];
    if (nk_ll > AFQMC_MAX_NK) return AFQMC_INVALID_ARGUMENT;
    if (dims->closed_shell != 0 && dims->closed_shell != 1) return AFQMC_INVALID_ARGUMENT;
    if (dims->precision != 0 && dims->precision != 1) return AFQMC_UNSUPPORTED;
    cudaStream_t st = (cudaStream_t)stream;
    if (dims->closed_shell == 1) return create_channel(out, dims, dims->n, dims->n, h1, L, psi_t, st, false, false);
    // open shell: n = spin-up, n_dn = spin-down occupied orbitals per k-point; psi_t = [Nk][m][n] then [Nk][m][n_dn]
    if (dims->n_dn < 1 || dims->n_dn > dims->m) return AFQMC_INVALID_ARGUMENT;
    if (dims->precision != 0) return AFQMC_UNSUPPORTED;        // the complex64 boundary is closed-shell only
    afqmc_ctx *up = nullptr, *dn = nullptr;
    int rc = create_channel(&up, dims, dims->n, dims->n + dims->n_dn, h1, L, psi_t, st, false, true);
    if (rc != AFQMC_OK) return rc;
    const double2* psi_dn = (const double2*)psi_t + (size_t)nk_ll * dims->m * dims->n;
    rc = create_channel(&dn, dims, dims->n_dn, dims->n + dims->n_dn, h1, L, psi_dn, st, true, true);
    if (rc != AFQMC_OK) { afqmc_destroy(up); return rc; }
    dn->b1 = up->b1;            // shared (owned by the spin-up context)
    up->dn = dn;
    *out = up;
    return AFQMC_OK;
}

// The operands of the two optional exchange kernels are re-layouts of Lh made the first time the option is used
// (they add 1x |Lh| each, so they are not resident unless asked for).
int afqmc_i_ensure_lx(afqmc_ctx* c, cudaStream_t st) {
    if (c->Lx) return AFQMC_OK;
    const Dims& d = c->d;
    const size_t nLx = (size_t)d.Nk * d.Nk * d.NAG * d.GQ * d.KS * 64 + AFQMC_LX_PAD;
    int rc = dev_alloc(&c->Lx, nLx);
    if (rc != AFQMC_OK) return rc;
    const size_t g = (nLx + 255) / 256;
    pack_Lx_kernel<<<(unsigned)(g > 148 * 64 ? 148 * 64 : g), 256, 0, st>>>(d, c->Lh, c->Lx, nLx);
    AFQMC_LAUNCH_CHECK(c);
    return AFQMC_OK;
}

int afqmc_i_ensure_lxt(afqmc_ctx* c, cudaStream_t st) {
    if (c->LxT) return AFQMC_OK;
    if (c->d.NAG != 1) return AFQMC_UNSUPPORTED;
    int rc = dev_alloc(&c->LxT, afqmc_i_lxt_floats(c->d));
    if (rc != AFQMC_OK) return rc;
    return afqmc_i_pack_lxt(c, st);
}

AFQMC_API long long afqmc_launch_count(const afqmc_ctx* c) { return c ? c->launches : 0; }

AFQMC_API double afqmc_exchange_flops(const afqmc_ctx* c, int nw) {
    if (!c) return 0.0;
    if (c->dn) { afqmc_ctx up = *c; up.dn = nullptr; return afqmc_exchange_flops(&up, nw) + afqmc_exchange_flops(c->dn, nw); }
    const Dims& d = c->d;
    // per unit and walker: two complex GEMMs (n x m)(m x n) per gamma, plus the complex contraction 8*n*n*nchol.
    // 4M kernel: 8 real flops per complex multiply-add = 2 * 8*n*n*m*nchol.  3M kernel (exchange3m.cu): 6 real
    // flops per complex multiply-add = 2 * 6*n*n*m*nchol, plus 3 additions per element of both T tensors.
    double per = 16.0 * d.n * d.n * d.m * d.nchol + 8.0 * d.n * d.n * d.nchol;
    if (c->opt_exchange_prec != 0 && c->d.NAG == 1) return (c->opt_exchange_prec == 1 ? 3.0 : 1.0) * per * (double)c->nunits * (double)nw;      // TF32 kernel: the 4M real embedding
    // (counted as pure 3M; the <= 2 tail elements of a row with m mod 4 in {1,2} are really done as 4M: not counted)
    if (c->opt_exchange_3m) per = 12.0 * d.n * d.n * d.m * d.nchol + 6.0 * d.n * d.n * d.nchol + 8.0 * d.n * d.n * d.nchol;
    // real orbitals (two real products per complex product, no additions before the contraction), default prefetch depth only
    if (c->opt_exchange_3m && c->real_lh && c->opt_real && c->opt_exchange_depth != 2)      // (the generic kernel's default depths)
        per = 8.0 * d.n * d.n * d.m * d.nchol + 8.0 * d.n * d.n * d.nchol;
    return per * (double)c->nunits * (double)nw;
}

AFQMC_API int afqmc_set_option(afqmc_ctx* c, const char* name, int value) {
    if (!c || !name) return AFQMC_INVALID_ARGUMENT;
    if (c->dn && strcmp(name, "timers") != 0) {     // tuning options apply to both spin channels
        int rc = afqmc_set_option(c->dn, name, value);
        if (rc != AFQMC_OK) return rc;
    }
    if (strcmp(name, "exchange_warps") == 0) {
        if (value != 0 && value != 2 && value != 4 && value != 5 && value != 6 && value != 8) return AFQMC_INVALID_ARGUMENT;
        c->opt_exchange_wpc = value;
        return AFQMC_OK;
    }
    if (strcmp(name, "exchange_precision") == 0) {
        if (value < 0 || value > 2) return AFQMC_INVALID_ARGUMENT;
        if (value != 0 && c->d.NAG != 1) return AFQMC_UNSUPPORTED;   // the mixed-precision kernels take n <= 4 (operands: first use)
        c->opt_exchange_prec = value;
        return AFQMC_OK;
    }
    if (strcmp(name, "exchange_tc") == 0) {        // 0 = the mma.sync TF32 kernel instead of the tcgen05 one; 2..8 = at most that many ring stages
        if (value < 0 || value > 8) return AFQMC_INVALID_ARGUMENT;
        c->opt_exchange_tc = value;
        return AFQMC_OK;
    }
    if (strcmp(name, "exchange_3m") == 0) {
        if (!value) {
            int rc = afqmc_i_ensure_lx(c, 0);
            if (rc == AFQMC_OK && cudaStreamSynchronize(0) != cudaSuccess) rc = AFQMC_CUDA_ERROR;
            if (rc != AFQMC_OK) return rc;
        }
        c->opt_exchange_3m = value ? 1 : 0;
        return AFQMC_OK;
    }
    if (strcmp(name, "exchange_regb") == 0) {
        if (value < 0 || value > 2) return AFQMC_INVALID_ARGUMENT;
        c->opt_exchange_regb = value;
        return AFQMC_OK;
    }
    if (strcmp(name, "exchange_ctas") == 0) {
        if (value < 0 || value > 16) return AFQMC_INVALID_ARGUMENT;
        c->opt_exchange_ctas = value;
        return AFQMC_OK;
    }
    if (strcmp(name, "exchange_np") == 0) {
        if (value != 0 && value != 1 && value != 2 && value != 4) return AFQMC_INVALID_ARGUMENT;
        c->opt_exchange_np = value;
        return AFQMC_OK;
    }
    if (strcmp(name, "exchange_minblocks") == 0) {
        c->opt_exchange_minb = value ? 1 : 0;
        return AFQMC_OK;
    }
    if (strcmp(name, "exchange_depth") == 0) {
        if (value != 0 && value != 2 && value != 3 && value != 6) return AFQMC_INVALID_ARGUMENT;
        c->opt_exchange_depth = value;
        return AFQMC_OK;
    }
    if (strcmp(name, "taylor_legacy") == 0) {
        c->opt_taylor_legacy = value ? 1 : 0;
        return AFQMC_OK;
    }
    if (strcmp(name, "taylor_warps") == 0) {
        if (value != 0 && (value < 3 || value > 5)) return AFQMC_INVALID_ARGUMENT;
        c->opt_taylor_wpc = value;
        return AFQMC_OK;
    }
    if (strcmp(name, "taylor_groups") == 0) {
        if (value < 0 || value > 64) return AFQMC_INVALID_ARGUMENT;
        c->opt_taylor_groups = value;
        return AFQMC_OK;
    }
    if (strcmp(name, "real_orbitals") == 0) {      // 0 = run the complex kernels even if the inputs were detected as real
        c->opt_real = value ? 1 : 0;
        return AFQMC_OK;
    }
    if (strcmp(name, "taylor_subbatch") == 0) {
        if (value < 0) return AFQMC_INVALID_ARGUMENT;
        c->opt_taylor_subbatch = value;
        return AFQMC_OK;
    }
    if (strcmp(name, "green_cluster") == 0) {
        if (value != 0 && value != 2 && value != 4) return AFQMC_INVALID_ARGUMENT;
        c->opt_green_cs = value;
        return AFQMC_OK;
    }
    if (strcmp(name, "green_legacy") == 0) {
        c->opt_green_legacy = value ? 1 : 0;
        return AFQMC_OK;
    }
    if (strcmp(name, "timers") == 0) {
        if (value && !c->ev[0])
            for (int i = 0; i <= AFQMC_NUM_STAGES; ++i)
                if (cudaEventCreate(&c->ev[i]) != cudaSuccess) return AFQMC_CUDA_ERROR;
        c->opt_timers = value ? 1 : 0;
        c->ev_valid = 0;
        return AFQMC_OK;
    }
    return AFQMC_INVALID_ARGUMENT;
}

AFQMC_API int afqmc_stage_times(afqmc_ctx* c, float* ms) {
    if (!c || !ms || !c->opt_timers || !c->ev_valid) return AFQMC_INVALID_ARGUMENT;
    for (int i = 0; i < AFQMC_NUM_STAGES; ++i)
        if (cudaEventElapsedTime(&ms[i], c->ev[i], c->ev[i + 1]) != cudaSuccess) {
            (void)cudaGetLastError();
            return AFQMC_CUDA_ERROR;
        }
    return AFQMC_OK;
}
