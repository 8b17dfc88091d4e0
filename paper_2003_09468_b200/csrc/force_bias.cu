// a4 force bias:  vbias[w][Q][g] = f_s sum_k sum_{a,r} Lh[Q][k][a][g][r] theta_w[(k,a),(k-Q,r)]      (f_s = 2: closed shell;
// open shell: f_s = 1 per spin channel and the two channels are added, openshell.cu)
// (the half-rotated contraction of Eq. 47; = 2 X_g of Eq. 37).
//
// Per Q this is a real-embedded complex GEMM on the FP64 tensor pipe:
//   rows   = gamma (8 per DMMA m-tile; two m-tiles interleaved per lane in the packed layout Lf, context.cu)
//   K      = (k, a, r, re/im)  = Nk*n*KS k-steps of 4 reals, one contiguous stream per m-tile pair
//   cols   = (walker, re/im)   = 4 walkers per DMMA n-tile
// CTA = (Q, K chunk, walker group, group of m-tile pairs); its 4 warps split the K chunk evenly.  A warp
// keeps an (MP pairs x NT n-tiles) accumulator set in registers and runs both fragment streams D k-steps
// ahead in statically rotated register buffers, with branch-free pointer updates, so the loads of a
// k-step are issued between its DMMAs:
//   A: one coalesced 512-byte LDG.128 per m-tile pair per k-step, straight from HBM (read once per call
//      when all walkers fit one walker group);
//   B: straight from theta (4 full 32-byte sectors per LDG.64, L1/L2 hits: CTAs that differ only in the
//      m-tile group are adjacent in the grid), real embedding = component select + sign flip.
// The K split (warps, then chunks) is combined deterministically: shared-memory tree inside the CTA,
// then a fixed-order sum over chunks in force_bias_reduce_kernel.  No atomics.
#include "common.cuh"

namespace {

constexpr int FB_WARPS = 4;
constexpr int FB_D = 3;   // k-steps of register prefetch (3 CTAs of 4 warps stay resident at 168 registers)

// AT = double2: FP64 storage of the operand; float2: single-precision storage (precision = 1), widened at use
template <int MP, int NT, typename AT>
__global__ void __launch_bounds__(32 * FB_WARPS, (MP * NT > 8 ? 2 : 3)) force_bias_kernel(
    Dims d, int nw, int KC, int nmg, int nwgrp, int pf, const int* __restrict__ kminus, const AT* __restrict__ Lf,
    const double2* __restrict__ theta, double2* __restrict__ out, int out_is_partial, double spin_factor) {
    extern __shared__ __align__(16) double fb_smem[];
    // blockIdx.x = ((Q*KC + kc)*nwgrp + wgrp)*nmg + mg
    int bx = blockIdx.x;
    const int mg = bx % nmg; bx /= nmg;
    const int wgrp = bx % nwgrp; bx /= nwgrp;
    const int kc = bx % KC, Q = bx / KC;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int kk = lane & 3, col = lane >> 2;
    const int cpar = kk & 1, dpar = col & 1;
    const unsigned smask = (cpar && !dpar) ? 0x80000000u : 0u;
    const int roff = kk >> 1;                  // complex r offset inside a k-step
    const int KS = d.KS, nitems = d.Nk * d.n;
    const int S = nitems * KS;                 // k-steps of the whole K range

    // item -> offset (in doubles) of theta[(k,a)][(k-Q)*m] inside one walker; one pad entry
    int* offtab = reinterpret_cast<int*>(fb_smem);
    for (int it = tid; it <= nitems; it += 32 * FB_WARPS) {
        const int item = it < nitems ? it : nitems - 1;
        const int k = item / d.n;
        offtab[it] = 2 * (item * d.M + kminus[k * d.Nk + Q] * d.m);
    }
    double* red = fb_smem + ((nitems + 1 + 1) / 2 + 1) / 2 * 2;     // 16-byte aligned, after the table

    // this warp's K range
    const int c0 = (int)((long long)kc * S / KC), c1 = (int)((long long)(kc + 1) * S / KC);
    const int g_begin = c0 + (int)((long long)warp * (c1 - c0) / FB_WARPS);
    const int g_end = c0 + (int)((long long)(warp + 1) * (c1 - c0) / FB_WARPS);

    const AT* ap[MP];
    bool aok[MP];
#pragma unroll
    for (int i = 0; i < MP; ++i) {
        const int gtp = mg * MP + i;
        aok[i] = gtp < d.GT2;
        ap[i] = Lf + (((size_t)Q * d.GT2 + (aok[i] ? gtp : d.GT2 - 1)) * S + g_begin) * 32 + lane;
    }
    const double* bw[NT];
    bool bok[NT];
#pragma unroll
    for (int j = 0; j < NT; ++j) {
        const int w = (wgrp * NT + j) * 4 + (col >> 1);
        bok[j] = w < nw;
        bw[j] = reinterpret_cast<const double*>(theta + (size_t)(bok[j] ? w : 0) * d.N * d.M) + 2 * roff + (cpar ^ dpar);
    }
    __syncthreads();   // offtab ready

    double acc[2 * MP][NT][2];
#pragma unroll
    for (int i = 0; i < 2 * MP; ++i)
#pragma unroll
        for (int j = 0; j < NT; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

    // loader state (runs FB_D k-steps ahead; stops advancing at g_end, so nothing is read out of range)
    int lg = g_begin, item = g_begin / KS, ls = g_begin - item * KS;
    int boff = offtab[item] + 4 * ls;
    AT fa[FB_D][MP];
    double fb[FB_D][NT];
    auto refill = [&](const int q) {
        const bool rok = 2 * ls + roff < d.m;
#pragma unroll
        for (int i = 0; i < MP; ++i) {
            fa[q][i] = __ldg(ap[i]);
            // pull the HBM stream into L2 `pf` k-steps ahead of the register loads (stays inside this warp's range)
            if (lg + pf < g_end) asm volatile("prefetch.global.L2 [%0];" ::"l"(ap[i] + pf * 32));
        }
#pragma unroll
        for (int j = 0; j < NT; ++j) {
            fb[q][j] = (bok[j] && rok) ? __ldg(bw[j] + boff) : 0.0;   // raw: the sign flip waits until use
        }
        const bool adv = lg + 1 < g_end;
        const bool wrap = ls + 1 == KS;
        lg += adv ? 1 : 0;
#pragma unroll
        for (int i = 0; i < MP; ++i) ap[i] += adv ? 32 : 0;
        ls = adv ? (wrap ? 0 : ls + 1) : ls;
        item += (adv && wrap) ? 1 : 0;
        boff = offtab[item] + 4 * ls;
    };
    auto kstep = [&](const int q) {
        double b[NT];
#pragma unroll
        for (int j = 0; j < NT; ++j) b[j] = flip_sign(fb[q][j], smask);      // real embedding: -Im for (c=1, d=0)
#pragma unroll
        for (int i = 0; i < MP; ++i) {
            const double ax = (double)fa[q][i].x, ay = (double)fa[q][i].y;
#pragma unroll
            for (int j = 0; j < NT; ++j) {
                dmma884(acc[2 * i][j][0], acc[2 * i][j][1], ax, b[j]);
                dmma884(acc[2 * i + 1][j][0], acc[2 * i + 1][j][1], ay, b[j]);
            }
        }
        refill(q);
    };
    const int total = g_end - g_begin;
    if (total > 0) {
#pragma unroll
        for (int q = 0; q < FB_D; ++q) refill(q);     // steps g_begin .. g_begin+D-1 (repeats the last one if total < D)
    }
    const int nfull = total - total % FB_D;
    for (int g0 = 0; g0 < nfull; g0 += FB_D) {
#pragma unroll
        for (int q = 0; q < FB_D; ++q) kstep(q);
    }
#pragma unroll
    for (int q = 0; q < FB_D - 1; ++q)
        if (nfull + q < total) kstep(q);

    // deterministic tree reduction over the K-split warps
    constexpr int TILE = 2 * MP * NT * 64;
#pragma unroll
    for (int half = FB_WARPS / 2; half >= 1; half >>= 1) {
        if (warp >= half && warp < 2 * half) {
#pragma unroll
            for (int i = 0; i < 2 * MP; ++i)
#pragma unroll
                for (int j = 0; j < NT; ++j) {
                    red[(warp - half) * TILE + (i * NT + j) * 64 + lane] = acc[i][j][0];
                    red[(warp - half) * TILE + (i * NT + j) * 64 + 32 + lane] = acc[i][j][1];
                }
        }
        __syncthreads();
        if (warp < half) {
#pragma unroll
            for (int i = 0; i < 2 * MP; ++i)
#pragma unroll
                for (int j = 0; j < NT; ++j) {
                    acc[i][j][0] += red[warp * TILE + (i * NT + j) * 64 + lane];
                    acc[i][j][1] += red[warp * TILE + (i * NT + j) * 64 + 32 + lane];
                }
        }
        __syncthreads();
    }
    if (warp == 0) {
        const double scale = out_is_partial ? 1.0 : spin_factor;      // 2 = both spins of a closed shell, 1 = one channel
        double2* dst = out + (out_is_partial ? (size_t)kc * nw * d.Nk * d.nchol : 0);
#pragma unroll
        for (int i = 0; i < 2 * MP; ++i) {
            const int gam = ((mg * MP + (i >> 1)) * 2 + (i & 1)) * 8 + (lane >> 2);
            if (!aok[i >> 1] || gam >= d.nchol) continue;
#pragma unroll
            for (int j = 0; j < NT; ++j) {
                const int w = (wgrp * NT + j) * 4 + (lane & 3);
                if (w < nw)
                    dst[((size_t)w * d.Nk + Q) * d.nchol + gam] = make_double2(scale * acc[i][j][0], scale * acc[i][j][1]);
            }
        }
    }
}

// vbias = spin_factor * sum over K chunks of the partial results, in chunk order
__global__ void force_bias_reduce_kernel(size_t n, int KC, double spin_factor, const double2* __restrict__ part, double2* __restrict__ vbias) {
    for (size_t e = blockIdx.x * (size_t)blockDim.x + threadIdx.x; e < n; e += (size_t)gridDim.x * blockDim.x) {
        double2 s = part[e];
        for (int c = 1; c < KC; ++c) { const double2 p = part[(size_t)c * n + e]; s.x += p.x; s.y += p.y; }
        vbias[e] = make_double2(spin_factor * s.x, spin_factor * s.y);
    }
}

template <int MP, int NT, typename AT>
int launch_force_bias_t(afqmc_ctx* c, const AT* Lf, const double2* theta, int nw, double2* vbias, cudaStream_t st) {
    const Dims& d = c->d;
    const int ntq = (nw + 3) / 4;
    const int nmg = (d.GT2 + MP - 1) / MP, nwgrp = (ntq + NT - 1) / NT;
    const long long base = (long long)d.Nk * nmg * nwgrp;
    const int S = d.Nk * d.n * d.KS;
    // K chunks: the count (<= AFQMC_FB_MAXKC, every warp keeps >= 8 k-steps) that fills the SMs most evenly
    int KC = 1;
    double best = -1.0;
    for (int kc = 1; kc <= AFQMC_FB_MAXKC; ++kc) {
        if (kc > 1 && S / (kc * FB_WARPS) < 8) break;
        const double n = (double)base * kc, waves = n / c->num_sms;
        const double eff = waves / (double)(long long)(waves + 0.999999) - 0.004 * kc;
        if (eff > best) { best = eff; KC = kc; }
    }
    const size_t smem = (size_t)(((d.Nk * d.n + 2) / 2 + 1) / 2 * 2 + (FB_WARPS / 2) * 2 * MP * NT * 64) * sizeof(double);
    auto kern = force_bias_kernel<MP, NT, AT>;
    if (int rc = afqmc_smem_optin(c, (const void*)kern, smem)) return rc;
    kern<<<(unsigned)(base * KC), 32 * FB_WARPS, smem, st>>>(d, nw, KC, nmg, nwgrp, c->opt_fb_pf, c->kminus, Lf, theta,
                                                             KC > 1 ? c->ws_fbpart : vbias, KC > 1 ? 1 : 0, c->spin_factor);
    AFQMC_LAUNCH_CHECK(c);
    if (KC > 1) {
        const size_t n = (size_t)nw * d.Nk * d.nchol;
        int G = (int)((n + 255) / 256);
        if (G > c->num_sms * 8) G = c->num_sms * 8;
        force_bias_reduce_kernel<<<G, 256, 0, st>>>(n, KC, c->spin_factor, c->ws_fbpart, vbias);
        AFQMC_LAUNCH_CHECK(c);
    }
    return AFQMC_OK;
}

template <int MP, int NT>
int launch_force_bias(afqmc_ctx* c, const double2* theta, int nw, double2* vbias, cudaStream_t st) {
    if (c->Lff) return launch_force_bias_t<MP, NT, float2>(c, reinterpret_cast<const float2*>(c->Lff), theta, nw, vbias, st);
    return launch_force_bias_t<MP, NT, double2>(c, reinterpret_cast<const double2*>(c->Lf), theta, nw, vbias, st);
}

}  // namespace

int afqmc_i_force_bias(afqmc_ctx* c, const double2* theta, int nw, double2* vbias, cudaStream_t st) {
    const int ntq = (nw + 3) / 4;   // walker quads
    // 16 DMMAs per k-step and warp in every shape; all walkers in one group up to 32 walkers
    // > 16 walkers: 2 m-tile pairs x 4 n-tiles per warp (16 walkers per CTA, 2 A loads + 4 B loads per 16 DMMAs) measured
    // fastest with the 3-deep prefetch (C3: 0.1725 ms against 0.1800 ms for 1 x 8 and 0.1964 ms for 2 x 8)
    if (ntq >= 5) return c->opt_fb_tile == 1 ? launch_force_bias<2, 8>(c, theta, nw, vbias, st)
                     : c->opt_fb_tile == 2 ? launch_force_bias<1, 8>(c, theta, nw, vbias, st)
                                           : launch_force_bias<2, 4>(c, theta, nw, vbias, st);
    if (ntq >= 3) return launch_force_bias<2, 4>(c, theta, nw, vbias, st);
    if (ntq == 2) return launch_force_bias<4, 2>(c, theta, nw, vbias, st);
    return launch_force_bias<4, 1>(c, theta, nw, vbias, st);
}

AFQMC_API int afqmc_force_bias(afqmc_ctx* c, const void* theta, int nw, void* vbias, void* stream) {
    if (!c || !theta || !vbias || nw < 0 || nw > c->max_walkers) return AFQMC_INVALID_ARGUMENT;
    if (nw == 0) return AFQMC_OK;
    if (c->prec32) return afqmc32_force_bias(c, theta, nw, vbias, (cudaStream_t)stream);
    if (c->dn) return afqmc_os_force_bias(c, (const double2*)theta, nw, (double2*)vbias, (cudaStream_t)stream);
    return afqmc_i_force_bias(c, (const double2*)theta, nw, (double2*)vbias, (cudaStream_t)stream);
}
