// a4 force bias:  vbias[w][Q][g] = 2 sum_k sum_{a,r} Lh[Q][k][a][g][r] theta_w[(k,a),(k-Q,r)]
// (the half-rotated contraction of Eq. 47; = 2 X_g of Eq. 37).
//
// Per Q this is a real-embedded complex GEMM on the FP64 tensor pipe:
//   rows   = gamma (8 per DMMA m-tile, packed layout Lf, see context.cu)
//   K      = (k, a, r, re/im)  = Nk*n*2m reals
//   cols   = (walker, re/im)   = 4 walkers per DMMA n-tile
// CTA = (Q, group of MT gamma-octets, group of NT walker-quads).  The 8 warps split K (the (k,a)
// items), each keeping an MT x NT accumulator tile set in registers; A fragments stream from HBM in
// lane order (one coalesced 256-byte LDG.64 per fragment), B fragments are read straight from theta
// (4 full 32-byte sectors per LDG.64) with the real embedding applied as a component select + sign
// flip.  Lf is read exactly once per call when all walkers fit one walker group.  The K-split
// partial tiles are combined deterministically through shared memory (no atomics).
#include "common.cuh"

namespace {

constexpr int FB_WARPS = 8;

template <int MT, int NT>
__global__ void __launch_bounds__(32 * FB_WARPS) force_bias_kernel(
    Dims d, int nw, const int* __restrict__ kminus, const double* __restrict__ Lf,
    const double2* __restrict__ theta, double2* __restrict__ vbias) {
    __shared__ double red[FB_WARPS / 2][MT * NT * 64];
    const int Q = blockIdx.x, gt0 = blockIdx.y * MT, t0 = blockIdx.z * NT;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int kk = lane & 3, col = lane >> 2;
    const int cpar = kk & 1, dpar = col & 1;
    const int comp = cpar ^ dpar;
    const unsigned smask = (cpar && !dpar) ? 0x80000000u : 0u;
    const int roff = kk >> 1;                  // complex r offset inside a k-step

    double acc[MT][NT][2];
#pragma unroll
    for (int i = 0; i < MT; ++i)
#pragma unroll
        for (int j = 0; j < NT; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

    const int nitems = d.Nk * d.n;
    for (int item = warp; item < nitems; item += FB_WARPS) {
        const int k = item / d.n, a = item % d.n;
        const int kq = kminus[k * d.Nk + Q];
        const double* bptr[NT];
        bool bok[NT];
#pragma unroll
        for (int j = 0; j < NT; ++j) {
            int w = (t0 + j) * 4 + (col >> 1);
            bok[j] = w < nw;
            bptr[j] = reinterpret_cast<const double*>(theta + ((size_t)(bok[j] ? w : 0) * d.N + k * d.n + a) * d.M +
                                                      (size_t)kq * d.m + roff) + comp;
        }
        const double* aptr[MT];
        bool aok[MT];
#pragma unroll
        for (int i = 0; i < MT; ++i) {
            aok[i] = gt0 + i < d.GT;
            aptr[i] = Lf + ((((size_t)Q * d.GT + (aok[i] ? gt0 + i : 0)) * d.Nk + k) * d.n + a) * d.KS * 32 + lane;
        }
#pragma unroll 2
        for (int s = 0; s < d.KS; ++s) {
            double af[MT], bf[NT];
#pragma unroll
            for (int i = 0; i < MT; ++i) af[i] = aok[i] ? __ldg(aptr[i] + s * 32) : 0.0;
            const bool rok = 2 * s + roff < d.m;
#pragma unroll
            for (int j = 0; j < NT; ++j) bf[j] = (bok[j] && rok) ? flip_sign(__ldg(bptr[j] + 4 * s), smask) : 0.0;
#pragma unroll
            for (int i = 0; i < MT; ++i)
#pragma unroll
                for (int j = 0; j < NT; ++j) dmma884(acc[i][j][0], acc[i][j][1], af[i], bf[j]);
        }
    }

    // deterministic tree reduction over the K-split warps
#pragma unroll
    for (int half = FB_WARPS / 2; half >= 1; half >>= 1) {
        if (warp >= half && warp < 2 * half) {
#pragma unroll
            for (int i = 0; i < MT; ++i)
#pragma unroll
                for (int j = 0; j < NT; ++j) {
                    red[warp - half][(i * NT + j) * 64 + lane] = acc[i][j][0];
                    red[warp - half][(i * NT + j) * 64 + 32 + lane] = acc[i][j][1];
                }
        }
        __syncthreads();
        if (warp < half) {
#pragma unroll
            for (int i = 0; i < MT; ++i)
#pragma unroll
                for (int j = 0; j < NT; ++j) {
                    acc[i][j][0] += red[warp][(i * NT + j) * 64 + lane];
                    acc[i][j][1] += red[warp][(i * NT + j) * 64 + 32 + lane];
                }
        }
        __syncthreads();
    }
    if (warp == 0) {
#pragma unroll
        for (int i = 0; i < MT; ++i) {
            int gam = (gt0 + i) * 8 + (lane >> 2);
            if (gt0 + i >= d.GT || gam >= d.nchol) continue;
#pragma unroll
            for (int j = 0; j < NT; ++j) {
                int w = (t0 + j) * 4 + (lane & 3);
                if (w < nw)
                    vbias[((size_t)w * d.Nk + Q) * d.nchol + gam] = make_double2(2.0 * acc[i][j][0], 2.0 * acc[i][j][1]);
            }
        }
    }
}

}  // namespace

int afqmc_i_force_bias(afqmc_ctx* c, const double2* theta, int nw, double2* vbias, cudaStream_t st) {
    const Dims& d = c->d;
    const int ntq = (nw + 3) / 4;   // walker quads
    if (ntq >= 4 || ntq == 3) {
        constexpr int MT = 5, NT = 4;
        dim3 grid(d.Nk, (d.GT + MT - 1) / MT, (ntq + NT - 1) / NT);
        force_bias_kernel<MT, NT><<<grid, 32 * FB_WARPS, 0, st>>>(d, nw, c->kminus, c->Lf, theta, vbias);
    } else if (ntq == 2) {
        constexpr int MT = 5, NT = 2;
        dim3 grid(d.Nk, (d.GT + MT - 1) / MT, 1);
        force_bias_kernel<MT, NT><<<grid, 32 * FB_WARPS, 0, st>>>(d, nw, c->kminus, c->Lf, theta, vbias);
    } else {
        constexpr int MT = 5, NT = 1;
        dim3 grid(d.Nk, (d.GT + MT - 1) / MT, 1);
        force_bias_kernel<MT, NT><<<grid, 32 * FB_WARPS, 0, st>>>(d, nw, c->kminus, c->Lf, theta, vbias);
    }
    AFQMC_LAUNCH_CHECK(c);
    return AFQMC_OK;
}

AFQMC_API int afqmc_force_bias(afqmc_ctx* c, const void* theta, int nw, void* vbias, void* stream) {
    if (!c || !theta || !vbias || nw < 0 || nw > c->max_walkers) return AFQMC_INVALID_ARGUMENT;
    if (nw == 0) return AFQMC_OK;
    return afqmc_i_force_bias(c, (const double2*)theta, nw, (double2*)vbias, (cudaStream_t)stream);
}
