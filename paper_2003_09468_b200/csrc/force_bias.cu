// a4 force bias:  vbias[w][Q][g] = f_s sum_k sum_{a,r} Lh[Q][k][a][g][r] theta_w[(k,a),(k-Q,r)]      (f_s = 2: closed shell;
// open shell: f_s = 1 per spin channel and the two channels are added, openshell.cu)
// (the half-rotated contraction of Eq. 47; = 2 X_g of Eq. 37).
//
// Per Q this is one complex GEMM  C[gamma][walker] = sum_kappa A[gamma][kappa] B[kappa][walker]  with the FLATTENED K index
// kappa = (k*n + a)*m + r  (Kc = Nk*n*m complex numbers, no padding per (k,a) row), on the FP64 tensor pipe (DMMA m8n8k4):
//
//  * 3M complex product (Karatsuba):  Prr = Ar Br,  Pii = Ai Bi,  Pss = (Ar+Ai)(Br+Bi);  Re = Prr - Pii,  Im = Pss - Prr - Pii:
//    three real GEMMs with K = kappa and one real column per walker, 6 real flops per complex multiply-add instead of the 8 of
//    the real embedding (one DADD per fragment on either side).
//  * rows   = gamma: m-tiles of 8; a warp owns MT consecutive m-tiles (MT = 5 when nchol = 200: 25 tiles, no padded tile)
//    cols   = walker: n-tiles of 8; a warp owns NT n-tiles (16 walkers; 8 when nw <= 8)
//    k-step = 4 consecutive kappa: 3 * MT * NT DMMAs per MT + NT operand loads.
//  * Operand Lf3[Q][m-group][k-step][m-tile][lane] (complex; single precision when precision = 1; written once in a0): the A
//    fragments of FB_KPC k-steps of a warp are ONE contiguous block, read from HBM exactly once per call: the WG warps of a CTA
//    that own the same m-group and different walkers share it through a shared-memory ring filled by bulk asynchronous copies
//    (cp.async.bulk + mbarrier, SASS UBLKCP; full/empty barrier pair per stage, FB_S - 1 chunks in flight), so the inner loop
//    has no global load at all and needs no registers for prefetching (a register-prefetched version stalled 16 % of its
//    warp-samples on the A loads at two k-steps of lookahead, which is all that 234 registers allowed; profiles/r02b).
//  * theta is first re-laid out (theta_frag_kernel: one pass over theta, 2 x |theta| bytes, L2 resident) into B fragments
//    thetaF[Q][walker group][k-step][n-tile][..] over the same flattened kappa, so that the B operand of FB_KPC k-steps of a
//    warp is ONE contiguous block.  It reaches the warp through a private ring of bulk asynchronous copies: one copy of
//    FB_KPC * NT * 512 bytes per chunk, and a B fragment is one conflict-free LDS.128 per n-tile.  (A first version copied the rows of theta themselves, <= 416 contiguous bytes each:
//    1.2 M copies per call at C3, and the kernel ran at the TMA unit's issue rate of about one copy per 40-50 cycles and SM,
//    0.162 ms; profiles/r02b.)  No table lookups and no L2 round trips in the inner loop; no CTA-wide barrier anywhere.
//  * STREAM-K work split: the (Q, m-group, walker super-group) tiles times their k-steps form one line of X k-steps that is cut
//    into U equal pieces, U = the number of resident warp groups: every warp gets the same number of DMMAs in ONE wave whatever
//    the shape (the previous kernel lost 19 % to wave quantisation and 11 % to a padded m-tile pair at C3).  A piece that
//    crosses a tile boundary produces two partial tiles; partial tiles are combined in a fixed order by
//    force_bias3_reduce_kernel (no atomics: bitwise reproducible).
#include <type_traits>
#include "common.cuh"

namespace {

constexpr int FB_WARPS = 4;
#ifndef AFQMC_FB_KPC
#define AFQMC_FB_KPC 4
#endif
#ifndef AFQMC_FB_STAGES
#define AFQMC_FB_STAGES 3
#endif
#ifndef AFQMC_FB_MINB
#define AFQMC_FB_MINB 2
#endif
constexpr int FB_KPC = AFQMC_FB_KPC;       // k-steps per ring chunk
constexpr int FB_S = AFQMC_FB_STAGES;      // stages of the rings: FB_S - 1 chunks are in flight while one is computed
constexpr int FB_MAXSLOTS = AFQMC_FB_MAXKC;

// How one call is cut up (host computes it, kernels get it by value)
struct FbPlan {
    int MT, NG, GT;        // m-tiles per warp, m-groups per Q, m-tiles per Q
    int KSf, Kc;           // k-steps and complex length of the flattened K range
    int NT, nwg, WG, wsup; // n-tiles per warp, walker groups, warps that share an A stream, walker super-groups
    long long X;           // k-steps of all tiles
    int U;                 // pieces (warp groups)
};

__host__ __device__ inline long long fb_bound(long long u, long long X, int U) { return u * X / U; }
// the piece that holds k-step x of the line
__host__ __device__ inline int fb_unit_of(long long x, long long X, int U) { return (int)(((x + 1) * U - 1) / X); }

// ---- a0: Lh -> Lf3[Q][g][ks][i < MT][lane]: lane (row = lane>>2, kk = lane&3) of m-tile g*MT + i, kappa = 4 ks + kk ----
template <typename T2>
__global__ void pack_Lf3_kernel(Dims d, int MT, int NG, int KSf, const double2* __restrict__ Lh, T2* __restrict__ Lf3, size_t total) {
    const int Kc = d.Nk * d.n * d.m;
    for (size_t idx = blockIdx.x * (size_t)blockDim.x + threadIdx.x; idx < total; idx += (size_t)gridDim.x * blockDim.x) {
        size_t t = idx;
        const int lane = (int)(t & 31); t >>= 5;
        const int i = (int)(t % MT); t /= MT;
        const int ks = (int)(t % KSf); t /= KSf;
        const int g = (int)(t % NG);
        const size_t Q = t / NG;
        const int gam = 8 * (g * MT + i) + (lane >> 2), kap = 4 * ks + (lane & 3);
        double2 z = make_double2(0.0, 0.0);
        if (gam < d.nchol && kap < Kc) {                  // zeros in the padded tiles of a ragged last group and past Kc
            const int it = kap / d.m, r = kap - it * d.m;
            z = Lh[(((Q * d.Nk + it / d.n) * d.n + it % d.n) * d.nchol + gam) * d.m + r];
        }
        T2 o; o.x = z.x; o.y = z.y;
        Lf3[idx] = o;
    }
}

// theta -> thetaF[Q][wg][ks][j < NT][lane]: B fragment of k-step ks and n-tile j of walker group wg; lane (col = lane>>2,
// kk = lane&3) holds theta_w[(k,a),(k-Q,r)] with w = (wg*NT + j)*8 + col and kappa = 4 ks + kk = (k*n + a)*m + r; zeros past nw
// and past Kc.  One thread per element: 64-byte runs of theta in, fully coalesced stores out.
__global__ void __launch_bounds__(256) theta_frag_kernel(Dims d, int NT, int nwg, int KSf, int nw, const int* __restrict__ kminus,
                                                         const double2* __restrict__ theta, double2* __restrict__ thetaF, size_t total) {
    const int Kc = d.Nk * d.n * d.m;
    for (size_t idx = blockIdx.x * (size_t)blockDim.x + threadIdx.x; idx < total; idx += (size_t)gridDim.x * blockDim.x) {
        size_t t = idx;
        const int lane = (int)(t & 31); t >>= 5;
        const int j = (int)(t % NT); t /= NT;
        const int ks = (int)(t % KSf); t /= KSf;
        const int wg = (int)(t % nwg);
        const int Q = (int)(t / nwg);
        const int w = (wg * NT + j) * 8 + (lane >> 2), kap = 4 * ks + (lane & 3);
        double2 z = make_double2(0.0, 0.0);
        if (w < nw && kap < Kc) {
            const int it = kap / d.m, r = kap - it * d.m;
            z = __ldg(theta + ((size_t)w * d.N + it) * d.M + (size_t)kminus[(it / d.n) * d.Nk + Q] * d.m + r);
        }
        thetaF[idx] = z;
    }
}

// AT = double2: FP64 storage of the operand; float2: single-precision storage (precision = 1), widened at use
// REAL: the operand is real (real orbitals: imaginary parts exactly zero, detected in a0): Re = Ar Br, Im = Ar Bi, two real
// products per complex product and no addition at all
template <int MT, int NT, typename AT, bool REAL>
__global__ void __launch_bounds__(32 * FB_WARPS, AFQMC_FB_MINB) force_bias3_kernel(
    Dims d, FbPlan p, int nw, const AT* __restrict__ Lf3, const double2* __restrict__ thetaF, double2* __restrict__ part) {
    extern __shared__ __align__(128) unsigned char fb_smem[];
    constexpr int STAGE_A = FB_KPC * MT * 32;              // AT elements of one stage of an A ring
    constexpr int STAGE_B = FB_KPC * NT * 32;              // complex numbers of one stage of a B ring
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int row = lane >> 2, kk = lane & 3;
    // shared memory: A rings [units of the CTA][FB_S][STAGE_A] | B rings [warp][FB_S][STAGE_B] | barriers
    const int nunit = FB_WARPS / p.WG, ul = warp / p.WG, sub = warp - ul * p.WG;
    AT* ringA = reinterpret_cast<AT*>(fb_smem) + ul * (FB_S * STAGE_A);
    double2* ringB = reinterpret_cast<double2*>(fb_smem + (size_t)nunit * FB_S * STAGE_A * sizeof(AT)) + warp * (FB_S * STAGE_B);
    uint64_t* bars = reinterpret_cast<uint64_t*>(fb_smem + (size_t)nunit * FB_S * STAGE_A * sizeof(AT) +
                                                 (size_t)FB_WARPS * FB_S * STAGE_B * sizeof(double2));
    uint64_t* fullA = bars + ul * FB_S;                    // [FB_WARPS units at most][FB_S]: the A chunk has landed
    uint64_t* emptyA = bars + (FB_WARPS + ul) * FB_S;      // every warp of the unit has read the A chunk
    uint64_t* fullB = bars + (2 * FB_WARPS + warp) * FB_S; // this warp's B chunk has landed
    if (threadIdx.x == 0) {
        for (int i = 0; i < FB_WARPS * FB_S; ++i) {
            mbar_init(&bars[i], 1);
            mbar_init(&bars[FB_WARPS * FB_S + i], p.WG);
            mbar_init(&bars[2 * FB_WARPS * FB_S + i], 1);
        }
        mbar_fence_init();
    }
    __syncthreads();                                        // the only CTA-wide barrier

    const int u = blockIdx.x * nunit + ul;                  // the piece of this warp group
    if (u >= p.U) return;
    long long x = fb_bound(u, p.X, p.U);
    const long long xe = fb_bound(u + 1, p.X, p.U);
    uint32_t cc0 = 0;                                      // A chunks consumed so far (the same in every warp of the unit)
    uint32_t ccB = 0;                                      // B chunks consumed so far by this warp (none in a tile without walkers)
    const size_t nout = (size_t)nw * d.Nk * d.nchol;

    while (x < xe) {
        const long long tau = x / p.KSf;
        const int ksa = (int)(x - tau * p.KSf);
        const int nks = (int)(((long long)p.KSf - ksa) < (xe - x) ? ((long long)p.KSf - ksa) : (xe - x));
        x += nks;
        const int s = (int)(tau % p.wsup);
        const int g = (int)((tau / p.wsup) % p.NG), Q = (int)(tau / ((long long)p.wsup * p.NG));
        const int wg = s * p.WG + sub;
        const bool idle = wg >= p.nwg;                     // no walkers in this tile (never the unit's first warp)
        const int w0 = wg * 8 * NT;
        const int nch = (nks + FB_KPC - 1) / FB_KPC;
        const AT* asrc = Lf3 + (((size_t)Q * p.NG + g) * p.KSf + ksa) * (MT * 32);
        const double2* bsrc = thetaF + (((size_t)Q * p.nwg + (idle ? 0 : wg)) * p.KSf + ksa) * (NT * 32);

        // chunk c of this segment = FB_KPC k-steps: one bulk copy of A fragments per unit (its first warp), one of B per warp
        auto issue = [&](const int c) {
            if (lane == 0) {
                const uint32_t gc = cc0 + (uint32_t)c;
                const int st = (int)(gc % FB_S);
                const int nk = (nks - c * FB_KPC) < FB_KPC ? (nks - c * FB_KPC) : FB_KPC;
                if (sub == 0) {
                    if (gc >= FB_S) mbar_wait(&emptyA[st], ((gc / FB_S) - 1) & 1);      // the stage's previous chunk was read by all
                    const uint32_t bytes = (uint32_t)(nk * MT * 32 * sizeof(AT));
                    mbar_expect_tx(&fullA[st], bytes);
                    bulk_g2s(ringA + st * STAGE_A, asrc + (size_t)c * STAGE_A, bytes, &fullA[st]);
                }
                if (!idle) {
                    const int sb = (int)((ccB + (uint32_t)c) % FB_S);
                    const uint32_t bytes = (uint32_t)(nk * NT * 32 * sizeof(double2));
                    mbar_expect_tx(&fullB[sb], bytes);
                    bulk_g2s(ringB + sb * STAGE_B, bsrc + (size_t)c * STAGE_B, bytes, &fullB[sb]);
                }
            }
        };
#pragma unroll 1
        for (int c = 0; c < FB_S - 1 && c < nch; ++c) issue(c);

        constexpr int NV = REAL ? 2 : 3;
        double acc[NV][MT][NT][2];
#pragma unroll
        for (int v = 0; v < NV; ++v)
#pragma unroll
            for (int i = 0; i < MT; ++i)
#pragma unroll
                for (int j = 0; j < NT; ++j) acc[v][i][j][0] = acc[v][i][j][1] = 0.0;

        for (int c = 0; c < nch; ++c) {
            const uint32_t gc = cc0 + (uint32_t)c;
            const int st = (int)(gc % FB_S);
            // the stage of chunk c - 1 is free in this warp (and almost surely in its partners): fetch chunk c + FB_S - 1 into it
            __syncwarp();
            if (c + FB_S - 1 < nch) issue(c + FB_S - 1);
            mbar_wait(&fullA[st], (gc / FB_S) & 1);
            if (!idle) {
                const uint32_t gb = ccB + (uint32_t)c;
                const int sb = (int)(gb % FB_S);
                mbar_wait(&fullB[sb], (gb / FB_S) & 1);
                const AT* ra = ringA + st * STAGE_A + lane;                    // A fragment of (k-step kin, m-tile i): + (kin*MT + i)*32
                const double2* rb = ringB + sb * STAGE_B + lane;               // B fragment of (k-step kin, n-tile j): + (kin*NT + j)*32
                auto kstep = [&](const int kin) {          // kin: a constant after unrolling
                    double b[3][NT], a[3][MT];
#pragma unroll
                    for (int j = 0; j < NT; ++j) {
                        const double2 v = rb[(kin * NT + j) * 32];
                        b[0][j] = v.x; b[1][j] = v.y;
                        b[2][j] = REAL ? 0.0 : v.x + v.y;
                    }
#pragma unroll
                    for (int i = 0; i < MT; ++i) {
                        const AT f = ra[(kin * MT + i) * 32];
                        a[0][i] = (double)f.x; a[1][i] = REAL ? a[0][i] : (double)f.y;
#ifdef FB_NOADD      // timing experiment only (wrong results): what the kernel would cost without the additions
                        a[2][i] = a[1][i];
#else
                        a[2][i] = REAL ? 0.0 : a[0][i] + a[1][i];
#endif
                    }
#pragma unroll
                    for (int i = 0; i < MT; ++i)
#pragma unroll
                        for (int j = 0; j < NT; ++j) {
#pragma unroll
                            for (int v = 0; v < NV; ++v) dmma884(acc[v][i][j][0], acc[v][i][j][1], a[v][i], b[v][j]);
                        }
                };
                const int rel0 = c * FB_KPC;
                if (nks - rel0 >= FB_KPC) {
#pragma unroll
                    for (int kin = 0; kin < FB_KPC; ++kin) kstep(kin);
                } else {
#pragma unroll
                    for (int kin = 0; kin < FB_KPC - 1; ++kin)
                        if (rel0 + kin < nks) kstep(kin);
                }
            }
            fence_proxy_async_smem();                       // this chunk's reads before the refill of its stages (common.cuh)
            __syncwarp();                                   // every lane has read the chunk
            if (lane == 0) mbar_arrive(&emptyA[st]);
        }
        cc0 += (uint32_t)nch;
        if (idle) continue;
        ccB += (uint32_t)nch;

        // ---- this segment's partial tile: slot = position of the piece among the pieces that cut the tile ----
        const int slot = u - fb_unit_of(tau * p.KSf, p.X, p.U);
        double2* dst = part + (size_t)slot * nout;
#pragma unroll
        for (int i = 0; i < MT; ++i) {
            const int gam = 8 * (g * MT + i) + row;
            if (gam >= d.nchol) continue;
#pragma unroll
            for (int j = 0; j < NT; ++j)
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const int w = w0 + 8 * j + 2 * kk + e;
                    if (w < nw)
                        dst[((size_t)w * d.Nk + Q) * d.nchol + gam] =
                            REAL ? make_double2(acc[0][i][j][e], acc[1][i][j][e])
                                 : make_double2(acc[0][i][j][e] - acc[1][i][j][e], acc[NV - 1][i][j][e] - acc[0][i][j][e] - acc[1][i][j][e]);
                }
        }
    }
}

// vbias = spin_factor * sum of the partial tiles, in piece order
__global__ void force_bias3_reduce_kernel(Dims d, FbPlan p, int nw, double spin_factor, const double2* __restrict__ part,
                                          double2* __restrict__ vbias) {
    const size_t n = (size_t)nw * d.Nk * d.nchol;
    for (size_t e = blockIdx.x * (size_t)blockDim.x + threadIdx.x; e < n; e += (size_t)gridDim.x * blockDim.x) {
        const int gam = (int)(e % d.nchol);
        const int Q = (int)((e / d.nchol) % d.Nk);
        const int w = (int)(e / ((size_t)d.nchol * d.Nk));
        const int g = (gam >> 3) / p.MT, s = (w / (8 * p.NT)) / p.WG;
        const long long tau = ((long long)Q * p.NG + g) * p.wsup + s;
        const int u0 = fb_unit_of(tau * p.KSf, p.X, p.U), u1 = fb_unit_of((tau + 1) * p.KSf - 1, p.X, p.U);
        double2 sum = part[e];
        for (int sl = 1; sl <= u1 - u0; ++sl) { const double2 v = part[(size_t)sl * n + e]; sum.x += v.x; sum.y += v.y; }
        vbias[e] = make_double2(spin_factor * sum.x, spin_factor * sum.y);
    }
}

int fb_tiles(const Dims& d) { return (d.nchol + 7) / 8; }
int fb_ksteps(const Dims& d) { return (d.Nk * d.n * d.m + 3) / 4; }

FbPlan fb_plan(const afqmc_ctx* c, int nw) {
    const Dims& d = c->d;
    FbPlan p;
    p.GT = fb_tiles(d);
    p.Kc = d.Nk * d.n * d.m;
    p.KSf = fb_ksteps(d);
    // m-tiles per warp: at most 5 (3 * 5 * NT * 2 accumulators), the count in {5,4,3} that pads the fewest tiles
    if (p.GT <= 5) p.MT = p.GT;
    else {
        int best = 5, waste = (p.GT + 4) / 5 * 5 - p.GT;
        for (int mt = 4; mt >= 3; --mt) {
            const int ws = (p.GT + mt - 1) / mt * mt - p.GT;
            if (ws < waste) { waste = ws; best = mt; }
        }
        p.MT = best;
    }
    p.NG = (p.GT + p.MT - 1) / p.MT;
    p.NT = nw <= 8 ? 1 : 2;
    p.nwg = (nw + 8 * p.NT - 1) / (8 * p.NT);
    p.WG = p.nwg == 1 ? 1 : (p.nwg == 2 ? 2 : 4);
    p.wsup = (p.nwg + p.WG - 1) / p.WG;
    p.X = (long long)d.Nk * p.NG * p.wsup * p.KSf;
    p.U = 1;
    return p;
}

// pieces: one per resident warp group; every piece keeps >= 8 k-steps and no tile is cut into more than FB_MAXSLOTS pieces
void fb_set_pieces(FbPlan& p, long long resident_ctas) {
    long long U = resident_ctas * (FB_WARPS / p.WG);
    if (U > p.X / 8) U = p.X / 8;
    if (U < 1) U = 1;
    while (U > 1 && (p.KSf + (p.X / U) - 1) / (p.X / U) + 1 > FB_MAXSLOTS) U = (U + 1) / 2;
    p.U = (int)U;
}

template <int MT, int NT, typename AT, bool REAL>
int launch_fb3(afqmc_ctx* c, FbPlan p, const AT* Lf3, const double2* theta, int nw, double2* vbias, cudaStream_t st) {
    const Dims& d = c->d;
    // theta -> B fragments (workspace sized for max_walkers in a0), unless Green's epilogue has just written them
    if (!(c->fuse_frag && c->frag_nw == nw && theta == c->frag_src)) {
    const size_t ntf = (size_t)d.Nk * p.nwg * p.KSf * NT * 32;
    long long G0 = (long long)((ntf + 255) / 256);
    if (G0 > (long long)c->num_sms * 16) G0 = (long long)c->num_sms * 16;
    theta_frag_kernel<<<(unsigned)G0, 256, 0, st>>>(d, NT, p.nwg, p.KSf, nw, c->kminus, theta, c->ws_thetaF, ntf);
    AFQMC_LAUNCH_CHECK(c);
    }
    const int nunit = FB_WARPS / p.WG;
    const size_t smem = (size_t)nunit * FB_S * FB_KPC * MT * 32 * sizeof(AT) + (size_t)FB_WARPS * FB_S * FB_KPC * NT * 32 * sizeof(double2) +
                        3 * FB_WARPS * FB_S * sizeof(uint64_t);
    auto kern = force_bias3_kernel<MT, NT, AT, REAL>;
    if (int rc = afqmc_smem_optin(c, (const void*)kern, smem)) return rc;
    afqmc_prefer_smem(c, (const void*)kern);
    // resident CTAs (per shared-memory size: it depends on the walker count through WG); remembered in the context
    FuncAttr* f = afqmc_fattr(c, (const void*)kern);
    int occ = (f && f->occ > 0 && f->occ_smem == (int)smem) ? f->occ : -1;
    if (occ < 0) {
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, 32 * FB_WARPS, smem) != cudaSuccess) { (void)cudaGetLastError(); return AFQMC_CUDA_ERROR; }
        if (occ < 1) return AFQMC_UNSUPPORTED;
        if (f) { f->occ = occ; f->occ_smem = (int)smem; }
    }
    fb_set_pieces(p, (long long)occ * c->num_sms);
    const unsigned grid = (unsigned)((p.U + nunit - 1) / nunit);
    kern<<<grid, 32 * FB_WARPS, smem, st>>>(d, p, nw, Lf3, c->ws_thetaF, c->ws_fbpart);
    AFQMC_LAUNCH_CHECK(c);
    const size_t n = (size_t)nw * d.Nk * d.nchol;
    long long G = (long long)((n + 255) / 256);
    if (G > c->num_sms * 8) G = c->num_sms * 8;
    force_bias3_reduce_kernel<<<(unsigned)G, 256, 0, st>>>(d, p, nw, c->spin_factor, c->ws_fbpart, vbias);
    AFQMC_LAUNCH_CHECK(c);
    return AFQMC_OK;
}

template <int MT, typename AT>
int launch_fb3_nt(afqmc_ctx* c, const FbPlan& p, const AT* Lf3, const double2* theta, int nw, double2* vbias, cudaStream_t st) {
    // real orbitals: the two-product kernel (FP64 storage only)
    if (std::is_same<AT, double2>::value && c->real_lh && c->opt_real)
        return p.NT == 1 ? launch_fb3<MT, 1, double2, true>(c, p, reinterpret_cast<const double2*>(Lf3), theta, nw, vbias, st)
                         : launch_fb3<MT, 2, double2, true>(c, p, reinterpret_cast<const double2*>(Lf3), theta, nw, vbias, st);
    return p.NT == 1 ? launch_fb3<MT, 1, AT, false>(c, p, Lf3, theta, nw, vbias, st) : launch_fb3<MT, 2, AT, false>(c, p, Lf3, theta, nw, vbias, st);
}

template <typename AT>
int launch_fb3_mt(afqmc_ctx* c, const AT* Lf3, const double2* theta, int nw, double2* vbias, cudaStream_t st) {
    const FbPlan p = fb_plan(c, nw);
    switch (p.MT) {
        case 1: return launch_fb3_nt<1, AT>(c, p, Lf3, theta, nw, vbias, st);
        case 2: return launch_fb3_nt<2, AT>(c, p, Lf3, theta, nw, vbias, st);
        case 3: return launch_fb3_nt<3, AT>(c, p, Lf3, theta, nw, vbias, st);
        case 4: return launch_fb3_nt<4, AT>(c, p, Lf3, theta, nw, vbias, st);
        default: return launch_fb3_nt<5, AT>(c, p, Lf3, theta, nw, vbias, st);
    }
}

}  // namespace

// a0: allocates and packs the force-bias operand (complex128, or complex64 when precision = 1) from Lh
int afqmc_i_pack_force_bias_operand(afqmc_ctx* c, cudaStream_t st) {
    const Dims& d = c->d;
    const FbPlan pl = fb_plan(c, 1);                 // MT, NG, KSf depend on the problem only
    const int KSf = pl.KSf;
    const size_t total = (size_t)d.Nk * pl.NG * KSf * pl.MT * 32;
    const size_t bytes = total * (c->prec32 ? sizeof(float2) : sizeof(double2));
    void* p = nullptr;
    cudaError_t e = cudaMalloc(&p, bytes);
    if (e != cudaSuccess) { (void)cudaGetLastError(); return e == cudaErrorMemoryAllocation ? AFQMC_OUT_OF_MEMORY : AFQMC_CUDA_ERROR; }
    size_t nb = (total + 255) / 256;
    if (nb > 148 * 64) nb = 148 * 64;
    if (c->prec32) {
        c->Lff = reinterpret_cast<float*>(p);
        pack_Lf3_kernel<float2><<<(unsigned)nb, 256, 0, st>>>(d, pl.MT, pl.NG, KSf, c->Lh, reinterpret_cast<float2*>(p), total);
    } else {
        c->Lf = reinterpret_cast<double*>(p);
        pack_Lf3_kernel<double2><<<(unsigned)nb, 256, 0, st>>>(d, pl.MT, pl.NG, KSf, c->Lh, reinterpret_cast<double2*>(p), total);
    }
    AFQMC_LAUNCH_CHECK(c);
    // workspace of the B fragments: every Q, max_walkers rounded up to whole n-tile groups, kappa padded to k-steps
    const size_t ntf = (size_t)d.Nk * ((c->max_walkers + 15) / 16) * 2 * KSf * 32;
    e = cudaMalloc((void**)&c->ws_thetaF, ntf * sizeof(double2));
    if (e != cudaSuccess) { (void)cudaGetLastError(); c->ws_thetaF = nullptr; return e == cudaErrorMemoryAllocation ? AFQMC_OUT_OF_MEMORY : AFQMC_CUDA_ERROR; }
    // zeroed once: Green's fused epilogue writes the valid entries only (padding: walkers past nw, kappa past Kc)
    if (cudaMemsetAsync(c->ws_thetaF, 0, ntf * sizeof(double2), st) != cudaSuccess) { (void)cudaGetLastError(); return AFQMC_CUDA_ERROR; }
    return AFQMC_OK;
}

void afqmc_i_fb_frag_layout(const afqmc_ctx* c, int nw, int* NT, int* nwg, int* KSf) {
    const FbPlan p = fb_plan(c, nw);
    *NT = p.NT; *nwg = p.nwg; *KSf = p.KSf;
}

// executed real flops of one call (3M: 6 per complex multiply-add)
AFQMC_API double afqmc_force_bias_flops(const afqmc_ctx* c, int nw) {
    if (!c) return 0.0;
    const Dims& d = c->d;
    const double per = (c->real_lh && c->opt_real && !c->prec32) ? 4.0 : 6.0;      // real orbitals: two real products
    double f = per * d.Nk * d.Nk * d.n * (double)d.m * d.nchol * nw;
    if (c->dn) f += per * d.Nk * d.Nk * c->dn->d.n * (double)d.m * d.nchol * nw;
    return f;
}

int afqmc_i_force_bias(afqmc_ctx* c, const double2* theta, int nw, double2* vbias, cudaStream_t st) {
    if (c->Lff) return launch_fb3_mt<float2>(c, reinterpret_cast<const float2*>(c->Lff), theta, nw, vbias, st);
    return launch_fb3_mt<double2>(c, reinterpret_cast<const double2*>(c->Lf), theta, nw, vbias, st);
}

AFQMC_API int afqmc_force_bias(afqmc_ctx* c, const void* theta, int nw, void* vbias, void* stream) {
    if (!c || !theta || !vbias || nw < 0 || nw > c->max_walkers) return AFQMC_INVALID_ARGUMENT;
    if (nw == 0) return AFQMC_OK;
    if (c->prec32) return afqmc32_force_bias(c, theta, nw, vbias, (cudaStream_t)stream);
    if (c->dn) return afqmc_os_force_bias(c, (const double2*)theta, nw, (double2*)vbias, (cudaStream_t)stream);
    return afqmc_i_force_bias(c, (const double2*)theta, nw, (double2*)vbias, (cudaStream_t)stream);
}
