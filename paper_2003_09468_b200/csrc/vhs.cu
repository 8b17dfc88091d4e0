// a5 vHS:  field assembly (reading R7) and the contraction of Eq. 48:
//   vhs_w[(k,p),(k-Q,r)] = sum_g L[Q][k][g][p][r] xi_w[Q][g]
//
// Per (Q,k) this is a real-embedded complex GEMM on the FP64 tensor pipe:
//   rows = (p,r) pairs (8 per DMMA m-tile; packed layout Lv, see context.cu)
//   K    = (gamma, re/im) = 2*nchol reals
//   cols = (walker, re/im), 4 walkers per n-tile
// L (the largest tensor of the problem) is streamed from HBM exactly once per call, as coalesced
// 256-byte fragments in lane order; the tiny B operand (the fields) is pre-expanded by the field
// kernel into fragment order so a B fragment is also one coalesced LDG.64 (L1/L2 resident).
// Every (k,k') block of vhs is written exactly once (Q = k-k'), so no zero fill is needed.
#include "common.cuh"

namespace {

// xi = -i (z - zbar), written directly as DMMA B fragments  Bxi[Q][s][t][lane]:
//   lane: kk = lane&3 -> gamma = 2s + (kk>>1), c = kk&1;  col = lane>>2 -> w = 4t + (col>>1), d = col&1
//   value = d==0 ? (c==0 ? Re xi : -Im xi) : (c==0 ? Im xi : Re xi)
__global__ void fields_kernel(Dims d, int nw, int ntq, const int* __restrict__ kneg, const double* __restrict__ x,
                              const double2* __restrict__ vbias, double sqrt_dtau, double* __restrict__ Bxi) {
    const size_t total = (size_t)d.Nk * d.GP * ntq * 32;
    for (size_t idx = blockIdx.x * (size_t)blockDim.x + threadIdx.x; idx < total;
         idx += (size_t)gridDim.x * blockDim.x) {
        size_t t_ = idx;
        int lane = (int)(t_ & 31); t_ >>= 5;
        int t = (int)(t_ % ntq); t_ /= ntq;
        int s = (int)(t_ % d.GP);
        int Q = (int)(t_ / d.GP);
        int kk = lane & 3, col = lane >> 2;
        int gam = 2 * s + (kk >> 1), c = kk & 1, w = 4 * t + (col >> 1), dd = col & 1;
        double v = 0.0;
        if (gam < d.nchol && w < nw) {
            const int mq = kneg[Q];
            const double xq = x[((size_t)w * d.Nk + Q) * d.nchol + gam];
            double zr, zi;
            if (mq == Q) { zr = xq; zi = 0.0; }
            else {
                const double xm = x[((size_t)w * d.Nk + mq) * d.nchol + gam];
                const double r2 = 0.70710678118654752440;
                if (Q < mq) { zr = xq * r2; zi = xm * r2; }       // z_Q    = (x_Q + i x_{-Q})/sqrt2
                else        { zr = xm * r2; zi = -xq * r2; }      // z_{-Q} = conj(z_Q)
            }
            if (vbias) {   // zbar = -i sqrt(dtau) vbias[-Q]  (Eq. 17)
                double2 vb = vbias[((size_t)w * d.Nk + mq) * d.nchol + gam];
                zr -= sqrt_dtau * vb.y;
                zi += sqrt_dtau * vb.x;
            }
            const double xr = zi, xi = -zr;                        // xi = -i (z - zbar)
            v = dd == 0 ? (c == 0 ? xr : -xi) : (c == 0 ? xi : xr);
        }
        Bxi[idx] = v;
    }
}

constexpr int VHS_WARPS = 8;

template <int MT, int NT>
__global__ void __launch_bounds__(32 * VHS_WARPS) vhs_kernel(
    Dims d, int nw, int ntq, int ngroups, const int* __restrict__ kminus, const double* __restrict__ Lv,
    const double* __restrict__ Bxi, double2* __restrict__ vhs) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const long long task = (long long)blockIdx.x * VHS_WARPS + warp;
    const long long ntasks = (long long)d.Nk * d.Nk * ngroups;
    if (task >= ntasks) return;
    const int grp = (int)(task % ngroups);
    const int qk = (int)(task / ngroups);
    const int Q = qk / d.Nk, k = qk % d.Nk;
    const int prt0 = grp * MT;
    const int t0 = blockIdx.y * NT;

    double acc[MT][NT][2];
#pragma unroll
    for (int i = 0; i < MT; ++i)
#pragma unroll
        for (int j = 0; j < NT; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

    const double* aptr[MT];
    bool aok[MT];
#pragma unroll
    for (int i = 0; i < MT; ++i) {
        aok[i] = prt0 + i < d.PRT;
        aptr[i] = Lv + (((size_t)qk * d.PRT + (aok[i] ? prt0 + i : 0)) * d.GP) * 32 + lane;
    }
    const double* bptr = Bxi + ((size_t)Q * d.GP * ntq + t0) * 32 + lane;
    bool bok[NT];
#pragma unroll
    for (int j = 0; j < NT; ++j) bok[j] = t0 + j < ntq;

#pragma unroll 2
    for (int s = 0; s < d.GP; ++s) {
        double af[MT], bf[NT];
#pragma unroll
        for (int i = 0; i < MT; ++i) af[i] = aok[i] ? __ldg(aptr[i] + (size_t)s * 32) : 0.0;
#pragma unroll
        for (int j = 0; j < NT; ++j) bf[j] = bok[j] ? __ldg(bptr + ((size_t)s * ntq + j) * 32) : 0.0;
#pragma unroll
        for (int i = 0; i < MT; ++i)
#pragma unroll
            for (int j = 0; j < NT; ++j) dmma884(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
    }

    const int kq = kminus[k * d.Nk + Q];
#pragma unroll
    for (int i = 0; i < MT; ++i) {
        const int pr = (prt0 + i) * 8 + (lane >> 2);
        if (prt0 + i >= d.PRT || pr >= d.m * d.m) continue;
        const int p = pr / d.m, r = pr % d.m;
#pragma unroll
        for (int j = 0; j < NT; ++j) {
            const int w = (t0 + j) * 4 + (lane & 3);
            if (w < nw)
                vhs[((size_t)w * d.M + (size_t)k * d.m + p) * d.M + (size_t)kq * d.m + r] =
                    make_double2(acc[i][j][0], acc[i][j][1]);
        }
    }
}

template <int MT, int NT>
void launch_vhs(afqmc_ctx* c, int nw, int ntq, double2* vhs, cudaStream_t st) {
    const Dims& d = c->d;
    const int ngroups = (d.PRT + MT - 1) / MT;
    const long long ntasks = (long long)d.Nk * d.Nk * ngroups;
    dim3 grid((unsigned)((ntasks + VHS_WARPS - 1) / VHS_WARPS), (ntq + NT - 1) / NT);
    vhs_kernel<MT, NT><<<grid, 32 * VHS_WARPS, 0, st>>>(d, nw, ntq, ngroups, c->kminus, c->Lv,
                                                         reinterpret_cast<const double*>(c->ws_xi), vhs);
}

}  // namespace

int afqmc_i_vhs(afqmc_ctx* c, const double* x, const double2* vbias, double dtau, int nw, double2* vhs,
                cudaStream_t st) {
    const Dims& d = c->d;
    const int ntq = (nw + 3) / 4;
    {
        size_t total = (size_t)d.Nk * d.GP * ntq * 32;
        int T = 256, G = (int)((total + T - 1) / T);
        if (G > 148 * 16) G = 148 * 16;
        fields_kernel<<<G, T, 0, st>>>(d, nw, ntq, c->kneg, x, vbias, sqrt(dtau), reinterpret_cast<double*>(c->ws_xi));
        AFQMC_LAUNCH_CHECK(c);
    }
    if (ntq >= 5) launch_vhs<2, 8>(c, nw, ntq, vhs, st);
    else if (ntq >= 3) launch_vhs<4, 4>(c, nw, ntq, vhs, st);
    else if (ntq == 2) launch_vhs<4, 2>(c, nw, ntq, vhs, st);
    else launch_vhs<4, 1>(c, nw, ntq, vhs, st);
    AFQMC_LAUNCH_CHECK(c);
    return AFQMC_OK;
}

AFQMC_API int afqmc_vhs(afqmc_ctx* c, const double* x, const void* vbias, double dtau, int nw, void* vhs,
                         void* stream) {
    if (!c || !x || !vhs || nw < 0 || nw > c->max_walkers || !(dtau >= 0.0)) return AFQMC_INVALID_ARGUMENT;
    if (nw == 0) return AFQMC_OK;
    return afqmc_i_vhs(c, x, (const double2*)vbias, dtau, nw, (double2*)vhs, (cudaStream_t)stream);
}
