// Batched complex128 GEMM for tall-skinny right-hand sides on the FP64 tensor pipe (DMMA m8n8k4), used by a6
// (Taylor propagation):
//
//   C_b[i][j] = alpha * sum_k A_b[i][k] * B_b[k][j],     A: M x K (big, streamed once),  B: K x N (small)
//
// Design (B200): the big operand A is read straight from its natural row-major layout into DMMA A-fragments, the
// small operand B lives in an EXPANDED fragment-major layout that is staged into shared memory by bulk asynchronous
// copies (cp.async.bulk + mbarrier pipeline, SASS UBLKCP), so the inner loop is LDG.128 (A, prefetched in
// registers) + LDS.64 (B, conflict-free) + DMMA only.
//
//  * 3M complex product (Gauss's form, as in exchange3m.cu and vhs.cu):
//        P0 = (Ar+Ai) Br,  P1 = Ar (Bi-Br),  P2 = Ai (Br+Bi);      Re C = P0 - P2,   Im C = P0 + P1
//    three real GEMMs with K = k and ONE real column per complex column of B: 6 real flops per complex multiply-add
//    instead of the 8 of the real embedding, 22 % fewer DMMAs at N = 108 (14 n-tiles of 8 columns x 3 products
//    against 27 n-tiles of 4 complex columns x 2 k-parities).  Lane (row r, c) gets Re and Im of A[i][4t+c] with ONE
//    16-byte load; Ar+Ai is one DADD per fragment.
//  * Expanded B ("Bx"): [batch][g][t][prod][nt < NTA][32 doubles], g = column group (<= NTA n-tiles of 8 columns),
//    t = group of 4 consecutive k, prod = 0: Br, 1: Bi-Br, 2: Br+Bi; innermost 32 doubles = one DMMA B-fragment in lane
//    order (lane = col*4 + c: column col of the tile, c = k inside the group).  K is padded to a multiple of 4*KC and
//    unused tiles/columns/rows are ZERO, so the kernel has no tails: A loads are clamped (finite * 0).
//  * The epilogue can (a) accumulate alpha*C into a natural-layout D (D += alpha*C), (b) write alpha*C in the
//    expanded layout of the NEXT product's B operand (rows of C become its K index), (c) store alpha*C
//    transposed in natural layout.  With (b) the Taylor chain T_j = (s/j) V T_{j-1} never converts layouts.
//  * CTA = 4 warps x (16 rows x one column group); the warps share the staged B chunks.  Grid = (groups, row
//    blocks, batch): CTAs of the same rows and walker are adjacent, so A is fetched from HBM once and shared
//    through L2 by the column groups.
#pragma once
#include "common.cuh"

namespace tg {

#ifndef AFQMC_TG_KC
#define AFQMC_TG_KC 4
#endif
#ifndef AFQMC_TG_STAGES
#define AFQMC_TG_STAGES 3
#endif
#ifndef AFQMC_TG_D
#define AFQMC_TG_D 2
#endif
constexpr int KC = AFQMC_TG_KC;        // k-groups (of 4 complex k) per shared-memory stage
constexpr int STAGES = AFQMC_TG_STAGES;
constexpr int DEPTH = AFQMC_TG_D;      // k-groups of register prefetch of the A stream (divides KC)
constexpr int NTMAX = 4;     // n-tiles (8 columns) per column group: 3 products x 2 m-tiles x 4 tiles x 2 = 48 accumulators
// warps per CTA (WPC, 16 rows each) is a template parameter chosen per launch: see launch_cfg()

struct Args {
    const double2* A; long long strideA; int lda;      // [batch][M][lda], K contiguous
    const double* Bx; long long strideBx;              // expanded B operand (see above), K = this product's K
    double* Cx; long long strideCx;                    // nullable: alpha*C expanded as the next product's B (its K = M)
    double2* D; long long strideD; int ldd;            // nullable: D[i][j] += alpha*C[i][j]
    double2* Ct; long long strideCt; int ldct;         // nullable: Ct[j][i]  = alpha*C[i][j]
    int M, N, K;
    int G, nt_base, nt_rem;                            // column groups: group g has nt_base + (g < nt_rem) n-tiles
    int NPp;                                           // padded k-groups of this product: roundup(ceil(K/4), KC)
    int NPcp;                                          // padded k-groups of the Cx layout: roundup(ceil(M/4), KC)
    double alpha;
    int wpc;                                           // 0 = automatic, else 3/4/5 warps per CTA (tuning aid)
};

// column-group geometry shared by host and device
struct Groups { int G, nt_base, nt_rem, NTA; };
__host__ __device__ inline int group_tile0(int g, int nt_base, int nt_rem) { return g * nt_base + (g < nt_rem ? g : nt_rem); }
__host__ __device__ inline int group_tiles(int g, int nt_base, int nt_rem) { return nt_base + (g < nt_rem ? 1 : 0); }

// G = 0: the fewest groups (<= NTMAX tiles each); G > 0: that many groups (clamped to what the tile count allows)
static inline Groups make_groups(int N, int G = 0) {
    Groups gr;
    const int nt = (N + 7) / 8;
    const int gmin = (nt + NTMAX - 1) / NTMAX;
    gr.G = G < gmin ? gmin : (G > nt ? nt : G);
    gr.nt_base = nt / gr.G;
    gr.nt_rem = nt % gr.G;
    gr.NTA = gr.nt_base + (gr.nt_rem ? 1 : 0);         // 1..NTMAX; a group with one tile fewer is zero padded
    return gr;
}
constexpr int GROUP_CHOICES = 3;   // pick_groups() considers gmin .. gmin + GROUP_CHOICES - 1 groups
static inline int padded_pairs(int K) { return (((K + 3) / 4 + KC - 1) / KC) * KC; }
// doubles of one batch entry of an expanded operand with K rows and N columns
static inline size_t expanded_doubles(int K, int N, int G = 0) {
    const Groups gr = make_groups(N, G);
    return (size_t)gr.G * padded_pairs(K) * 3 * gr.NTA * 32;
}
// the largest expanded operand over the group counts pick_groups() may choose (workspace sizing)
static inline size_t expanded_doubles_max(int K, int N) {
    const int gmin = make_groups(N).G;
    size_t mx = 0;
    for (int g = gmin; g < gmin + GROUP_CHOICES; ++g) {
        const size_t e = expanded_doubles(K, N, g);
        if (e > mx) mx = e;
    }
    return mx;
}

// ---- natural [K][N] (ldb) -> expanded; also the zero fill of all padding ----
// TRANS: the source is read as B[k][j] = src[j][k] (transposed, K contiguous).
template <bool TRANS>
__global__ void expand_kernel(const double2* __restrict__ src, long long strideS, int lds, double* __restrict__ Bx,
                              long long strideBx, int K, int N, int G, int nt_base, int nt_rem, int NTA, int NPp) {
    const size_t per_in = (size_t)G * NPp * NTA * 32;          // without the product index
    const int b = blockIdx.y;
    const double2* S = src + (size_t)b * strideS;
    double* out = Bx + (size_t)b * strideBx;
    for (size_t idx = blockIdx.x * (size_t)blockDim.x + threadIdx.x; idx < per_in; idx += (size_t)gridDim.x * blockDim.x) {
        size_t t = idx;
        const int l = (int)(t & 31); t >>= 5;
        const int nt = (int)(t % NTA); t /= NTA;
        const int tt = (int)(t % NPp);
        const int g = (int)(t / NPp);
        const int col = l >> 2;
        const int k = 4 * tt + (l & 3);
        const int j = (group_tile0(g, nt_base, nt_rem) + nt) * 8 + col;
        double2 z = make_double2(0.0, 0.0);
        if (k < K && j < N && nt < group_tiles(g, nt_base, nt_rem)) z = TRANS ? S[(size_t)j * lds + k] : S[(size_t)k * lds + j];
        double* f = out + ((((size_t)g * NPp + tt) * 3) * NTA + nt) * 32 + l;
        f[0] = z.x;
        f[(size_t)NTA * 32] = z.y - z.x;
        f[(size_t)2 * NTA * 32] = z.x + z.y;
    }
}

// ---- the GEMM body for a column group of NT (<= NTA) n-tiles ----
template <int NT, int NTA, int D, int WPC>
__device__ __forceinline__ void body(const Args& p, const double* stage0, uint64_t* full, uint64_t* empty, int g, int b) {
    static_assert(KC % D == 0, "A prefetch depth must divide the chunk");
    constexpr uint32_t STAGE_DOUBLES = KC * 3 * NTA * 32, STAGE_BYTES = STAGE_DOUBLES * 8;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int row0 = blockIdx.y * (16 * WPC) + warp * 16;
    const int r = lane >> 2, c = lane & 3;
    const double2* A = p.A + (size_t)b * p.strideA;
    const int i0 = min(row0 + r, p.M - 1), i1 = min(row0 + 8 + r, p.M - 1);   // clamped rows: finite data, discarded
    const double2* pa0 = A + (size_t)i0 * p.lda;
    const double2* pa1 = A + (size_t)i1 * p.lda;
    const int Km1 = p.K - 1;
    double2 fa0[D], fa1[D];
#pragma unroll
    for (int q = 0; q < D; ++q) {
        const int k = min(4 * q + c, Km1);               // clamped k: the matching B rows are zero
        fa0[q] = __ldg(pa0 + k);
        fa1[q] = __ldg(pa1 + k);
    }
    double acc[3][2][NT][2];
#pragma unroll
    for (int pr = 0; pr < 3; ++pr)
#pragma unroll
        for (int mt = 0; mt < 2; ++mt)
#pragma unroll
            for (int nt = 0; nt < NT; ++nt) acc[pr][mt][nt][0] = acc[pr][mt][nt][1] = 0.0;

    const int nchunks = p.NPp / KC;
    const double* Bsrc = p.Bx + (size_t)b * p.strideBx + (size_t)g * p.NPp * 3 * NTA * 32;
    if (tid == 0) {
        for (int c0 = 0; c0 < STAGES - 1 && c0 < nchunks; ++c0) {
            mbar_expect_tx(&full[c0], STAGE_BYTES);
            bulk_g2s(const_cast<double*>(stage0) + (size_t)c0 * STAGE_DOUBLES, Bsrc + (size_t)c0 * STAGE_DOUBLES, STAGE_BYTES, &full[c0]);
        }
    }
    for (int ch = 0; ch < nchunks; ++ch) {
        const int st = ch % STAGES;
        mbar_wait(&full[st], (uint32_t)((ch / STAGES) & 1));
        const double* bs = stage0 + (size_t)st * STAGE_DOUBLES + lane;
#pragma unroll
        for (int q = 0; q < KC; ++q) {
            const int buf = q % D;
            const double a0[3] = {fa0[buf].x + fa0[buf].y, fa0[buf].x, fa0[buf].y};     // Ar+Ai, Ar, Ai
            const double a1[3] = {fa1[buf].x + fa1[buf].y, fa1[buf].x, fa1[buf].y};
#pragma unroll
            for (int pr = 0; pr < 3; ++pr) {
                double bf[NT];
#pragma unroll
                for (int nt = 0; nt < NT; ++nt) bf[nt] = bs[((q * 3 + pr) * NTA + nt) * 32];
#pragma unroll
                for (int nt = 0; nt < NT; ++nt) {
                    dmma884(acc[pr][0][nt][0], acc[pr][0][nt][1], a0[pr], bf[nt]);
                    dmma884(acc[pr][1][nt][0], acc[pr][1][nt][1], a1[pr], bf[nt]);
                }
            }
            {   // refill this register buffer with the k-group D ahead
                const int k = min(4 * (ch * KC + q + D) + c, Km1);
                fa0[buf] = __ldg(pa0 + k);
                fa1[buf] = __ldg(pa1 + k);
            }
            if (q == 1 && tid == 0) {   // producer duty: refill the stage consumed in the previous iteration
                const int nxt = ch + STAGES - 1;
                if (nxt < nchunks) {
                    const int s2 = nxt % STAGES;
                    mbar_wait(&empty[s2], (uint32_t)(((nxt / STAGES) & 1) ^ 1));
                    mbar_expect_tx(&full[s2], STAGE_BYTES);
                    bulk_g2s(const_cast<double*>(stage0) + (size_t)s2 * STAGE_DOUBLES, Bsrc + (size_t)nxt * STAGE_DOUBLES, STAGE_BYTES, &full[s2]);
                }
            }
        }
        fence_proxy_async_smem();       // the stage's reads before its refill by the bulk copy (see common.cuh)
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[st]);
    }

    // ---- epilogue: lane holds rows r, r+8 and columns 8*tile + 2c + e of each 8x8 tile; Re = P0 - P2, Im = P0 + P1 ----
    const int tile0 = group_tile0(g, p.nt_base, p.nt_rem);
    const int ntg = group_tiles(g, p.nt_base, p.nt_rem);
    double2* Dm = p.D ? p.D + (size_t)b * p.strideD : nullptr;
    double2* Ct = p.Ct ? p.Ct + (size_t)b * p.strideCt : nullptr;
    double* Cx = p.Cx ? p.Cx + (size_t)b * p.strideCx + (size_t)g * p.NPcp * 3 * NTA * 32 : nullptr;
#pragma unroll
    for (int mt = 0; mt < 2; ++mt) {
        const int i = row0 + mt * 8 + r;
        const bool iok = i < p.M;
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) {
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int j = (tile0 + nt) * 8 + 2 * c + e;
                double2 v = make_double2(p.alpha * (acc[0][mt][nt][e] - acc[2][mt][nt][e]),
                                         p.alpha * (acc[0][mt][nt][e] + acc[1][mt][nt][e]));
                if (iok && j < p.N && nt < ntg) {
                    if (Dm) {
                        double2 o = Dm[(size_t)i * p.ldd + j];
                        o.x += v.x; o.y += v.y;
                        Dm[(size_t)i * p.ldd + j] = o;
                    }
                    if (Ct) Ct[(size_t)j * p.ldct + i] = v;
                }
                if (Cx && i < 4 * p.NPcp) {
                    if (!iok) v = make_double2(0.0, 0.0);     // K padding of the next product
                    double* f = Cx + (((size_t)(i >> 2) * 3) * NTA + nt) * 32 + (2 * c + e) * 4 + (i & 3);
                    f[0] = v.x;                               // Br
                    f[NTA * 32] = v.y - v.x;                  // Bi - Br
                    f[2 * NTA * 32] = v.x + v.y;              // Br + Bi
                }
            }
        }
    }
}

template <int NTA, int D, int WPC>
__global__ void __launch_bounds__(32 * WPC, 2) tgemm_kernel(Args p) {
    extern __shared__ __align__(128) double tg_smem[];
    uint64_t* full = reinterpret_cast<uint64_t*>(tg_smem + (size_t)STAGES * KC * 3 * NTA * 32);
    uint64_t* empty = full + STAGES;
    if (threadIdx.x == 0) {
        for (int s = 0; s < STAGES; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], WPC); }
        mbar_fence_init();
    }
    __syncthreads();
    const int g = blockIdx.x, b = blockIdx.z;
    if (NTA == 1 || group_tiles(g, p.nt_base, p.nt_rem) == NTA) body<NTA, NTA, D, WPC>(p, tg_smem, full, empty, g, b);
    else body<(NTA > 1 ? NTA - 1 : 1), NTA, D, WPC>(p, tg_smem, full, empty, g, b);
}

template <int NTA, int D, int WPC>
static inline cudaError_t launch_wpc(afqmc_ctx* c, const Args& a, int batch, cudaStream_t st, int* occ_out) {
    auto kern = tgemm_kernel<NTA, D, WPC>;
    const int smem = STAGES * KC * 3 * NTA * 32 * 8 + 2 * STAGES * 8;
    if (afqmc_smem_optin(c, (const void*)kern, smem) != AFQMC_OK) return cudaErrorInvalidValue;
    if (occ_out) {      // query only: resident CTAs per SM, remembered in the context (per device)
        FuncAttr* f = afqmc_fattr(c, (const void*)kern);
        int occ = f ? f->occ : -1;
        if (occ < 0) {
            int o = 0;
            cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&o, kern, 32 * WPC, smem);
            if (e != cudaSuccess) return e;
            occ = o > 0 ? o : 1;
            if (f) f->occ = occ;
        }
        *occ_out = occ;
        return cudaSuccess;
    }
    dim3 grid(a.G, (a.M + 16 * WPC - 1) / (16 * WPC), batch);
    kern<<<grid, 32 * WPC, smem, st>>>(a);
    return cudaGetLastError();
}

// Warps per CTA.  The DMMA pipe is per SM sub-partition, so resident warps must divide evenly over the four
// sub-partitions: measured at C3 (r01c notes, 4M version of this kernel), 2 CTAs x 4 warps ran 6 sub-partition rounds in
// 3.35 ms, while 2 x 5 warps (1.95 waves instead of 2.38, but 3+3+2+2 warps per sub-partition) took 3.90 ms and 3
// warps 4.39 ms.  4 is therefore the default; 3 and 5 stay selectable as a tuning aid (option "taylor_warps").
template <int NTA, int D>
static inline cudaError_t launch_cfg(afqmc_ctx* c, const Args& a, int batch, cudaStream_t st) {
    int best = 4;
    if (a.wpc >= 3 && a.wpc <= 5) best = a.wpc;
    switch (best) {
        case 3: return launch_wpc<NTA, D, 3>(c, a, batch, st, nullptr);
        case 5: return launch_wpc<NTA, D, 5>(c, a, batch, st, nullptr);
        default: return launch_wpc<NTA, D, 4>(c, a, batch, st, nullptr);
    }
}

#define TG_NTA_SWITCH(NTA_VALUE, CALL)                         \
    switch (NTA_VALUE) {                                       \
        case 1: return CALL(1);                                \
        case 2: return CALL(2);                                \
        case 3: return CALL(3);                                \
        default: return CALL(4);                               \
    }

// resident CTAs per SM of the 4-warp kernel instantiated for NTA tiles per group
static inline cudaError_t query_occupancy(afqmc_ctx* c, int NTA, int* occ) {
    Args a = {};
#define TG_CALL(n) launch_wpc<n, DEPTH, 4>(c, a, 1, nullptr, occ)
    TG_NTA_SWITCH(NTA, TG_CALL)
#undef TG_CALL
}

// Number of column groups for a product with M rows, N columns and `batch` entries.  More groups mean narrower
// warp tiles (fewer accumulators, A re-read from L2 by more CTAs) but a finer grid: the cost model is
//   rounds of resident CTAs x resident CTAs per SM x tiles a warp executes per k-step,
// i.e. the DMMA time of one SM (the kernel is tensor-pipe bound), plus 2 % per extra group for the A re-reads.
static inline int pick_groups(afqmc_ctx* c, int M, int N, int batch) {
    const int gmin = make_groups(N).G;
    const int sms = c->num_sms;
    int best = gmin; long long best_cost = -1;
    for (int g = gmin; g < gmin + GROUP_CHOICES; ++g) {
        const Groups gr = make_groups(N, g);
        if (gr.G != g) break;
        int occ = 1;
        if (query_occupancy(c, gr.NTA, &occ) != cudaSuccess) { (void)cudaGetLastError(); continue; }
        const long long ctas = (long long)gr.G * ((M + 63) / 64) * batch;
        const long long slots = (long long)occ * sms;
        const long long rounds = (ctas + slots - 1) / slots;
        const long long cost = rounds * occ * gr.NTA * (100 + 2 * (g - gmin));
        if (best_cost < 0 || cost < best_cost) { best = g; best_cost = cost; }
    }
    return best;
}

// fills the group fields of `a` from N (and the group count G, 0 = fewest) and launches; `a.NPp`/`a.NPcp` are
// derived from K and M.  The expanded operands must have been written with the same G.
static inline cudaError_t launch(afqmc_ctx* c, Args a, int batch, cudaStream_t st, int G = 0) {
    const Groups gr = make_groups(a.N, G);
    a.G = gr.G; a.nt_base = gr.nt_base; a.nt_rem = gr.nt_rem;
    a.NPp = padded_pairs(a.K);
    a.NPcp = padded_pairs(a.M);
#define TG_CALL(n) launch_cfg<n, DEPTH>(c, a, batch, st)
    TG_NTA_SWITCH(gr.NTA, TG_CALL)
#undef TG_CALL
}

template <bool TRANS>
static inline cudaError_t launch_expand(const double2* src, long long strideS, int lds, double* Bx, int K, int N,
                                        int batch, cudaStream_t st, int G = 0) {
    const Groups gr = make_groups(N, G);
    const int NPp = padded_pairs(K);
    const size_t per = (size_t)gr.G * NPp * 3 * gr.NTA * 32;
    int bx = (int)((per / 3 + 255) / 256);
    if (bx > 148 * 8) bx = 148 * 8;
    expand_kernel<TRANS><<<dim3(bx, batch), 256, 0, st>>>(src, strideS, lds, Bx, (long long)per, K, N, gr.G, gr.nt_base,
                                                           gr.nt_rem, gr.NTA, NPp);
    return cudaGetLastError();
}

}  // namespace tg
