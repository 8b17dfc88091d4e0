// a9 exchange energy in MIXED PRECISION on the 5th-generation tensor cores: tcgen05.mma.kind::tf32 with the accumulators in
// tensor memory (TMEM).  Same contraction and same two modes as exchange_tf32.cu (3xTF32 operand split / 1xTF32; PAPER.md:260,
// :306-319, Eq. 49); that file is the legacy mma.sync version and stays as the fallback (option "exchange_tc" = 0).  This is the
// one contraction of the library whose dtype has a tcgen05 kind (FP64 has none).
//
//  unit (Q,k,k2), 16 walkers per CTA (8 when the batch has at most 8), row tiles of 128 rows = 32 gamma x 4 orbitals:
//     D1[(gamma,a)][(w,b,c)] = sum_kappa A1[(gamma,a)][kappa] B1[(w,b,c)][kappa]        T1 = Lh[ Q][k ] theta_w[(k2,b),(k-Q ,r)]
//     D2[(gamma,b)][(w,a,c)] = sum_kappa A2[(gamma,b)][kappa] B2[(w,a,c)][kappa]        T2 = Lh[-Q][k2] theta_w[(k ,a),(k2+Q,s)]
//  real embedding: kappa = (r, re/im of Lh), c = re/im of T;  B[(.,c=0)] = (theta_r, -theta_i), B[(.,c=1)] = (theta_i, theta_r).
//  M = 128, N = 128 (64), K = 2m padded to 8: one tcgen05.mma (UMMA 128x128x8) per k-step and operand-split term, 7 k-steps at m = 26.
//
//  * A operand: packed ONCE in a0 as the shared-memory image itself: K-major with the 128-byte swizzle (UMMA layout type
//    SWIZZLE_128B: K-blocks of 32 floats, rows of 128 bytes, 8-row atoms of 1024 bytes, 16-byte chunk c of row r stored at
//    c ^ (r & 7)), TF32-rounded high and low planes.  A ring stage holds one K-block (32 kappa of the 128 rows, 16 KB) of the
//    images of BOTH T; it arrives by two tensor-map copies (cp.async.bulk.tensor.2d, SASS UTMALDG; the operand is viewed as rows
//    of 256 bytes, box = one K-block, no TMA swizzle: the bytes are already in place).  The ring has as many stages as fit beside
//    the B images (three at 3xTF32, m = 26, 16 walkers; two are nearly as fast: the copies are not the bottleneck).
//  * B operand: the real-embedded, TF32-split images of EVERY theta block (row block, column block, walker group) are built
//    once per call by tc_pack_theta_kernel in the same swizzled layout (each block is used by ~2 Nk units) and arrive like A,
//    K-block by K-block: block kb of the NEXT item is fetched as soon as the last tiles of the current item are through with
//    block kb (the uses of a tile run K-block by K-block), i.e. behind their remaining MMAs.
//  * Warp roles (13 warps): warp 12 lane 0 is the producer (all tensor-map copies, as far ahead as the ring allows).
//    Lane 0 of warps 8-11 issue the MMAs: thread (T, parity) those of T1 or T2 of the even or odd tiles of the item, and commits
//    them to mbarriers (tcgen05.commit).  One issuing thread was the bottleneck of the first version: clock64 around its
//    sections showed ~100 cycles per MMA and ~160 per commit, all serial, 2.5 of 3.4 ms, with the tensor pipe idle whenever that
//    thread committed or waited; with four independent streams (two T x two accumulator buffers) the pipe is shared at ~66 cycles
//    per 128x128x8 MMA (its nominal rate is 68) and the commits and waits of one stream hide behind the MMAs of the others.
//    Warps 0-7 are the epilogue (TMEM lane quarter w & 3, walker half w >> 2): tcgen05.ld of both accumulators in the
//    16-lane x 256-bit shape, which hands a thread the SAME orbital pair (a, b) of T1 of four gammas that it needs, and T2's element
//    with the pair exchanged sits in the lane with two 2-bit fields swapped: one shuffle per value; then the complex contraction
//    sum_{ab} T1[(g,a),(w,b)] T2[(g,b),(w,a)] in FP32 per tile and FP64 across tiles.  TMEM holds two accumulator buffers
//    (2 x (D1, D2) x N columns = all 512 at N = 128), so the epilogue of tile t overlaps the MMAs of tiles t + 1, t + 2.
//  * Results: unit partial sums in ws_expart, exactly like the FP64 kernels (energy_finalize_kernel applies multiplicities);
//    the item's sum over rows is a halving butterfly over lanes and a fixed order over warps: bitwise reproducible; only the
//    epilogue warps synchronise per item (named barrier), the copy and MMA threads run on into the next item.
//  * Measured (C3, afqmc_local_energy incl. the theta pack, force bias and finalize, ~0.2 ms): 3xTF32 2.57 ms, 1xTF32 1.31 ms
//    (mma.sync kernel: 7.37 / 3.86 ms).  The way there (profiles/r02g_ncu_exchange_tc.md, r02h): thread-built B images cost 1.2 ms
//    per call; chains of dependent MMAs into ONE accumulator ran at ~120 cycles per instruction; an instruction took the SAME time
//    at N = 128 as at N = 64, hence 16 walkers per CTA; a first (a,b) transpose by shuffles picked its registers with
//    lane-dependent compares, which the compiler turned into divergent branches; a CTA-wide barrier per item drained the pipe;
//    neither deeper rings nor removing the A copies altogether changed the time, the single issuing thread did (above).
#include <cuda.h>      // CUtensorMap and the encode function's type only: the entry point is fetched through the runtime, no libcuda link
#include "common.cuh"

namespace {

// walkers per CTA: NWC = 16 (N = 128 columns; an MMA instruction costs the same at N = 64, so wider is free) unless the batch
// has at most 8 walkers (NWC = 8: no padded columns)
constexpr int TC_M = 128;                 // rows of a tile: 32 gamma x 4 orbitals
constexpr int TC_EPI_WARPS = 8;           // epilogue warps: TMEM lane quarter w & 3, walker half w >> 2
constexpr int TC_THREADS = 32 * (TC_EPI_WARPS + 5);       // warps 0-7: epilogue, warps 8-11: MMA issue (T, tile parity), warp 12: tensor-map copies
constexpr int TC_KB = TC_M * 32;          // floats of one K-block of an A image: 32 kappa of the 128 rows = 16 KB (one swizzle atom column)
constexpr int TC_MAXKB = 4;               // most K-blocks of an image (2m <= 128)
constexpr int TC_MAXST = 8;               // most ring stages (a stage = the same K-block of the two operand images T1, T2 = 32 KB)
template <bool SPLIT, int NWC> struct TcCfg {
    static constexpr int N = 8 * NWC;                 // columns (w, orbital, re/im)
    static constexpr int TMEM_COLS = 4 * N;           // two accumulator buffers x (D1, D2)
    // instruction descriptor: D = F32 (bits 4-5 = 1), A and B = TF32 (bits 7-9, 10-12 = 2), both K-major, N >> 3 at bit 17, M >> 4 at bit 24
    static constexpr uint32_t IDESC = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(TC_M >> 4) << 24);
};

__device__ __forceinline__ float tc_tf32(float f) {
    unsigned u;
    asm("cvt.rna.tf32.f32 %0, %1;\n" : "=r"(u) : "f"(f));
    return __uint_as_float(u);
}

// float offset of element (row, kappa) in a K-major image with the 128-byte swizzle (UMMA layout type SWIZZLE_128B): K-blocks of
// 32 floats; inside a K-block every row is 128 contiguous bytes, 8 rows form a 1024-byte atom, and the 16-byte chunk c of row r
// is stored at chunk c ^ (r & 7) (conflict-free operand reads by the tensor core; measured 120 cycles per 128x64x8 MMA with the
// unswizzled core-matrix layout, whose floor is 32)
__host__ __device__ inline int tc_off(int rows, int row, int kap) {
    const int kb = kap >> 5, kin = kap & 31;
    return kb * (rows * 32) + row * 32 + ((((kin >> 2) ^ (row & 7)) << 2) | (kin & 3));
}

// a0: Lh -> LxU[Q][k][tile][plane hi/lo][image of 128 x KP floats]
__global__ void pack_LxU_kernel(Dims d, int KP, int NTILE, const double2* __restrict__ Lh, float* __restrict__ LxU, size_t total) {
    const int img = TC_M * KP;
    for (size_t idx = blockIdx.x * (size_t)blockDim.x + threadIdx.x; idx < total; idx += (size_t)gridDim.x * blockDim.x) {
        size_t t_ = idx;
        const int kap = (int)(t_ % KP); t_ /= KP;               // (row, kappa) enumerated, stored at its swizzled offset
        const int row = (int)(t_ % TC_M); t_ /= TC_M;
        const int tile = (int)(t_ % NTILE); t_ /= NTILE;
        const int k = (int)(t_ % d.Nk);
        const int Q = (int)(t_ / d.Nk);
        const int gam = 32 * tile + (row >> 2), a = row & 3, r = kap >> 1, part = kap & 1;
        float hi = 0.f, lo = 0.f;
        if (a < d.n && gam < d.nchol && r < d.m) {
            const double2 z = Lh[((((size_t)Q * d.Nk + k) * d.n + a) * d.nchol + gam) * d.m + r];
            const double x = part ? z.y : z.x;
            hi = tc_tf32((float)x);
            lo = tc_tf32((float)(x - (double)hi));
        }
        const size_t base = ((((size_t)Q * d.Nk + k) * NTILE + tile) * 2) * img;
        const int o = tc_off(TC_M, row, kap);
        LxU[base + o] = hi;
        LxU[base + img + o] = lo;
    }
}

// per call: theta -> ThU[kr][kc][wg][plane hi/lo][image of (8 nwc) x KP floats]: the B operand of every (row block kr, column block kc)
// of theta for walker group wg, real-embedded: column n = 8 wl + 2 b + c, kappa = 2 r + dd;
//   c = 0: (theta_r, -theta_i) at dd = 0, 1;   c = 1: (theta_i, theta_r).   Each block is used by many work units.
__global__ void tc_pack_theta_kernel(Dims d, int KP, int nwc, int nwg, int nw, int npl, const double2* __restrict__ theta,
                                     float* __restrict__ ThU, size_t total) {
    const int ncol = 8 * nwc, img = ncol * KP, rper = KP / 2;
    for (size_t idx = blockIdx.x * (size_t)blockDim.x + threadIdx.x; idx < total; idx += (size_t)gridDim.x * blockDim.x) {
        size_t t_ = idx;
        const int r = (int)(t_ % rper); t_ /= rper;
        const int b = (int)(t_ & 3); t_ >>= 2;
        const int wl = (int)(t_ % nwc); t_ /= nwc;
        const int wg = (int)(t_ % nwg); t_ /= nwg;
        const int kc = (int)(t_ % d.Nk);
        const int kr = (int)(t_ / d.Nk);
        const int w = wg * nwc + wl;
        double2 z = make_double2(0.0, 0.0);
        if (b < d.n && w < nw && r < d.m) z = __ldg(theta + ((size_t)w * d.N + kr * d.n + b) * d.M + (size_t)kc * d.m + r);
        float* im = ThU + ((((size_t)kr * d.Nk + kc) * nwg + wg) * 2) * img;
        const int n0 = 8 * wl + 2 * b;
        const int o0 = tc_off(ncol, n0, 2 * r), o1 = tc_off(ncol, n0 + 1, 2 * r);
        const float xr = tc_tf32((float)z.x), xi = tc_tf32((float)z.y);
        *reinterpret_cast<float2*>(im + o0) = make_float2(xr, -xi);
        *reinterpret_cast<float2*>(im + o1) = make_float2(xi, xr);
        if (npl == 2) {
            const float lr = tc_tf32((float)(z.x - (double)xr)), li = tc_tf32((float)(z.y - (double)xi));
            *reinterpret_cast<float2*>(im + img + o0) = make_float2(lr, -li);
            *reinterpret_cast<float2*>(im + img + o1) = make_float2(li, lr);
        }
    }
}

// ---- tcgen05 / TMEM primitives (inline PTX; only this file uses them) ----
__device__ __forceinline__ void tc_alloc(uint32_t* slot_smem, uint32_t ncols) {       // whole warp
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;\n" ::"r"(smem_u32(slot_smem)), "r"(ncols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;\n" ::: "memory");
}
__device__ __forceinline__ void tc_dealloc(uint32_t taddr, uint32_t ncols) {           // whole warp
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;\n" ::"r"(taddr), "r"(ncols) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;\n" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;\n" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint64_t* bar) {     // arrives on `bar` when every MMA issued so far by this thread is done
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];\n" ::"r"(smem_u32(bar)) : "memory");
}
// D[tmem] (+)= A[smem] * B[smem]^T, TF32 inputs, FP32 accumulation
__device__ __forceinline__ void tc_mma_tf32(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\n"
        "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n}\n" ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
        : "memory");
}
// shared-memory matrix descriptor, K-major, 128-byte swizzle (version 1 = sm_100; layout type 2 at bits 61-63): start address
// (the k-step's 32 bytes inside the swizzle atom are selected by advancing it), LBO = 1 unit (unused with a swizzle), SBO = 1024
// bytes between 8-row groups; all in 16-byte units
__device__ __forceinline__ uint64_t tc_desc(uint32_t smem_addr) {
    return (uint64_t)((smem_addr >> 4) & 0x3FFF) | ((uint64_t)1 << 16) | ((uint64_t)(1024 >> 4) << 32) | ((uint64_t)1 << 46) | ((uint64_t)2 << 61);
}
// one image by one tensor-map copy: box = (64 floats, rows), coordinates (0, first row of 256 bytes)
__device__ __forceinline__ void tc_tma_rows(float* dst, const CUtensorMap* tmap, int row, uint64_t* bar) {
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];\n" ::"r"(smem_u32(dst)),
                 "l"(reinterpret_cast<uint64_t>(tmap)), "r"(0), "r"(row), "r"(smem_u32(bar))
                 : "memory");
}
// 16 TMEM lanes x 256 bits, twice along the columns (16 columns = two walkers): this thread gets, of the lanes l0 + lane/4 (h = 0)
// and l0 + lane/4 + 8 (h = 1), the columns 8 j + 2 (lane % 4) + e:  v[4 j + 2 h + e]
__device__ __forceinline__ void tc_ld16x256x2(uint32_t taddr, float (&v)[8]) {
    uint32_t r[8];
    asm volatile("tcgen05.ld.sync.aligned.16x256b.x2.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];\n"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
                 : "r"(taddr)
                 : "memory");
#pragma unroll
    for (int i = 0; i < 8; ++i) v[i] = __uint_as_float(r[i]);
}
__device__ __forceinline__ void tc_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;\n" ::: "memory"); }


template <bool SPLIT, int NWC>
__global__ void __launch_bounds__(TC_THREADS, 1) exchange_tc_kernel(
    const __grid_constant__ CUtensorMap tmapA, const __grid_constant__ CUtensorMap tmapB, Dims d, int KP, int KS, int NTILE, int nst, int nw,
    int nitems, const int* __restrict__ units, const int* __restrict__ kminus, const int* __restrict__ kplus,
    const int* __restrict__ kneg, double2* __restrict__ partial) {
    extern __shared__ __align__(1024) unsigned char tc_smem[];
    using Cfg = TcCfg<SPLIT, NWC>;
    constexpr int NPL = SPLIT ? 2 : 1, TC_N = Cfg::N, TC_NWC = NWC, TC_NH = NWC / 2;      // NH: walkers of an epilogue warp
    constexpr uint32_t TC_IDESC = Cfg::IDESC;
    const int IMG_A = TC_M * KP, IMG_B = TC_N * KP;        // floats (KP a multiple of 32: whole swizzle atoms)
    const int NKB = KP / 32;                               // K-blocks of an image
    float* A_s = reinterpret_cast<float*>(tc_smem);        // [nst][T1, T2][TC_KB]: ring of K-block pairs
    float* B_s = A_s + (size_t)nst * 2 * TC_KB;            // [T][plane][IMG_B]: the item's B images
    double* red = reinterpret_cast<double*>(B_s + 2 * NPL * IMG_B);    // [2][4 warps][TC_NWC][2]
    uint64_t* bars = reinterpret_cast<uint64_t*>(red + 2 * 4 * TC_NWC * 2);
    uint64_t* fullA = bars;                            // [2][TC_MAXST]: a K-block pair has landed; one barrier ring per tile parity (below)
    uint64_t* stage_free = bars + 2 * TC_MAXST;        // [TC_MAXST]: the MMAs that read the stage are complete (tcgen05.commit)
    uint64_t* mma_done = bars + 3 * TC_MAXST;          // [2]: the MMAs into accumulator buffer b (both T) are complete
    uint64_t* tmem_free = bars + 3 * TC_MAXST + 2;     // [2]: the epilogue has read accumulator buffer b
    uint64_t* fullB = bars + 3 * TC_MAXST + 4;         // [TC_MAXKB]: K-block kb of the item's B images (both T, all planes) has landed
    uint64_t* freeB = bars + 3 * TC_MAXST + 4 + TC_MAXKB;      // [TC_MAXKB]: the item's last MMAs that read K-block kb of B are complete
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 3 * TC_MAXST + 4 + 2 * TC_MAXKB);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) {
        // (completion barriers count 2: the threads of T1 and T2 commit; freeB 4: all four MMA threads)
        for (int i = 0; i < TC_MAXST; ++i) { mbar_init(&fullA[i], 1); mbar_init(&fullA[TC_MAXST + i], 1); mbar_init(&stage_free[i], 2); }
        mbar_init(&mma_done[0], 2); mbar_init(&mma_done[1], 2);
        mbar_init(&tmem_free[0], 32 * TC_EPI_WARPS); mbar_init(&tmem_free[1], 32 * TC_EPI_WARPS);
        for (int i = 0; i < TC_MAXKB; ++i) { mbar_init(&fullB[i], 1); mbar_init(&freeB[i], 4); }
        mbar_fence_init();
    }
    if (warp == TC_EPI_WARPS) tc_alloc(tmem_slot, Cfg::TMEM_COLS);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;

    const int nwg = (nw + TC_NWC - 1) / TC_NWC;
    // One USE = the K-block kb (32 kappa of all 128 rows, 16 KB) of plane pl of BOTH operand images (T1, T2) of tile t, and the MMAs
    // that read the pair.  Plane hi -> Ah Bh (+ Ah Bl), plane lo -> Al Bh.
    //  * Tiles alternate between the two accumulator buffers and between two pairs of issuing threads by the parity of the CTA's
    //    tile count tbase + t (not of t: with an odd number of tiles per item the last tile of an item and the first of the next
    //    would share a buffer, and its epilogue would be exposed); the uses of the item's tiles 2p and 2p + 1 are interleaved in
    //    the ring (position 2 UPT p + 2 u + (t & 1); an unpaired last tile follows), so that the two pairs advance side by side
    //    on a ring of two or three stages.
    //  * Use position pos of the item is the CTA's use g = ubase + pos: ring stage g % nst, phase (g / nst) & 1 of stage_free.
    //    The "landed" barriers are NOT per stage but a ring of nst per tile parity, used in the order of that parity's uses (the
    //    c-th use of a parity: barrier c % nst, phase (c / nst) & 1): with an odd number of stages a stage alternates between the
    //    two pairs of threads, a pair would see only every other phase of a per-stage barrier, and a parity wait that is a whole
    //    phase ahead of its barrier passes at once (copies complete out of order: a wrong energy and a hang once in ~500
    //    launches at C3).  A barrier of the ring is re-armed only after its previous use was consumed: at most nst uses are in flight.
    //  * The n-th use of a buffer (n = (tbase + t) / 2) completes phase n & 1 of mma_done[b] and tmem_free[b].  Items (it): phase
    //    of fullB / freeB, parity of the reduction scratch.
    const int UPT = NPL * NKB;                                           // uses per tile
    const int nuse = NTILE * UPT, npaired = (NTILE / 2) * 2 * UPT;
    uint32_t ubase = 0, tbase = 0, it = 0, cp0 = 0, cp1 = 0;          // cp: uses of the even / odd tiles so far (producer: issued; MMA thread: its own parity)
    for (int item = blockIdx.x; item < nitems; item += gridDim.x, ++it, ubase += (uint32_t)nuse, tbase += (uint32_t)NTILE) {
        const int u = item / nwg, wg = item - u * nwg, w0 = wg * TC_NWC;

        double xr64[TC_NH], xi64[TC_NH];
#pragma unroll
        for (int j = 0; j < TC_NH; ++j) xr64[j] = xi64[j] = 0.0;

        if (warp == TC_EPI_WARPS + 4) {
            // ===== producer: one thread streams the item's B images and the A K-blocks, as far ahead as the ring allows =====
            if (lane == 0) {
                const int Q = units[4 * u], k = units[4 * u + 1], k2 = units[4 * u + 2];
                const int mQ = kneg[Q], kq = kminus[k * d.Nk + Q], k2pq = kplus[k2 * d.Nk + Q];
                // B: T1 from theta[(k2,.),(k-Q,.)], T2 from theta[(k,.),(k2+Q,.)], K-block by K-block (N rows x 32 kappa each): block kb
                // of B_s is free once the previous item's last MMAs that read it are done, i.e. while its last tiles are still being
                // multiplied (uses run K-block by K-block), so these copies are hidden behind those tiles
                for (int kb = 0; kb < NKB; ++kb) {
                    if (it > 0) mbar_wait(&freeB[kb], (it - 1) & 1);
                    mbar_expect_tx(&fullB[kb], 2 * NPL * (uint32_t)(TC_N * 32 * sizeof(float)));
                    for (int T = 0; T < 2; ++T)
                        for (int pl = 0; pl < NPL; ++pl) {
                            const size_t blk = (((size_t)(T == 0 ? k2 : k) * d.Nk + (T == 0 ? kq : k2pq)) * nwg + wg) * 2 + pl;
                            tc_tma_rows(B_s + (size_t)(T * NPL + pl) * IMG_B + (size_t)kb * (TC_N * 32), &tmapB,
                                        (int)(blk * (size_t)(IMG_B / 64) + (size_t)kb * (TC_N / 2)), &fullB[kb]);
                        }
                }
                const size_t blk1 = ((size_t)Q * d.Nk + k) * NTILE, blk2 = ((size_t)mQ * d.Nk + k2) * NTILE;
                uint32_t st = ubase % (uint32_t)nst, ph = (ubase / (uint32_t)nst) & 1;
                for (int pos = 0; pos < nuse; ++pos) {
                    int t, uu;
                    if (pos < npaired) { const int r = pos % (2 * UPT); t = 2 * (pos / (2 * UPT)) + (r & 1); uu = r >> 1; }
                    else { t = NTILE - 1; uu = pos - npaired; }
                    const int kb = uu / NPL, pl = uu - kb * NPL;          // use order of a tile: K-block, then plane
                    if (ubase + (uint32_t)pos >= (uint32_t)nst) mbar_wait(&stage_free[st], ph ^ 1);
                    const int par = (int)((tbase + (uint32_t)t) & 1);
                    const uint32_t c = par ? cp1++ : cp0++;
                    uint64_t* full = &fullA[par * TC_MAXST + (int)(c % (uint32_t)nst)];
                    mbar_expect_tx(full, 2 * TC_KB * (uint32_t)sizeof(float));
                    float* dst = A_s + (size_t)st * 2 * TC_KB;
                    // rows of 256 bytes: image (block + t, plane) starts at row index * IMG_A / 64, its K-block kb 64 rows further per block
                    tc_tma_rows(dst, &tmapA, (int)(((blk1 + t) * 2 + pl) * (size_t)(IMG_A / 64) + (size_t)kb * (TC_KB / 64)), full);
                    tc_tma_rows(dst + TC_KB, &tmapA, (int)(((blk2 + t) * 2 + pl) * (size_t)(IMG_A / 64) + (size_t)kb * (TC_KB / 64)), full);
                    if (++st == (uint32_t)nst) { st = 0; ph ^= 1; }
                }
            }
            __syncwarp();
        } else if (warp >= TC_EPI_WARPS) {
            // ===== MMA issue: four threads, lane 0 of warps 8 .. 11: thread (T, par) issues the MMAs of T (0: T1, 1: T2) of the tiles
            //       t = par, par + 2, ...  An MMA occupies its issuing thread for ~100 cycles and a tcgen05.commit for ~160 (clock64
            //       around them; with ONE issuing thread, 2.5 of the 3.4 ms of the 3xTF32 kernel were that thread's time, and the
            //       tensor pipe idled whenever it committed or waited), so independent streams are issued and committed concurrently:
            //       the two T of a tile, and two tiles with their own accumulator buffers =====
            if (lane == 0) {
                const int T = (warp - TC_EPI_WARPS) & 1, par = (warp - TC_EPI_WARPS) >> 1, t0 = par ^ (int)(tbase & 1);
                const uint32_t a_addr = smem_u32(A_s) + (uint32_t)(T * TC_KB * 4), b_addr = smem_u32(B_s) + (uint32_t)(T * NPL * IMG_B * 4);
                const uint32_t lo_off = (uint32_t)((IMG_B * 4) >> 4);         // hi -> lo plane of a B image (descriptor units of 16 bytes)
                const uint32_t dT = tmem_base + par * (2 * TC_N) + T * TC_N;
                for (int t = t0; t < NTILE; t += 2) {
                    const uint32_t n = (tbase + (uint32_t)t) >> 1;            // how often the buffer was used before
                    if (n >= 1) mbar_wait(&tmem_free[par], (n - 1) & 1);      // the accumulator buffer was read
                    const bool paired = (t | 1) < NTILE;                      // tile t ^ 1 exists: their uses alternate in the ring
                    const int pos0 = paired ? (t >> 1) * 2 * UPT + (t & 1) : npaired, pstep = paired ? 2 : 1;
                    for (int uu = 0; uu < UPT; ++uu) {
                        const int kb = uu / NPL, pl = uu - kb * NPL;
                        const uint32_t st = (ubase + (uint32_t)(pos0 + pstep * uu)) % (uint32_t)nst, c = cp0++;       // (cp0: this thread's own count)
                        if (t == t0 && pl == 0) mbar_wait(&fullB[kb], it & 1);   // first tile: K-block kb of the item's B images has landed
                        mbar_wait(&fullA[par * TC_MAXST + (int)(c % (uint32_t)nst)], (c / (uint32_t)nst) & 1);
                        tc_fence_after();
                        // a k-step is 8 kappa = 32 bytes of every row: slot ks of the K-block's 128-byte rows, i.e. the start-address
                        // field of the descriptor (16-byte units) grows by 2 per k-step
                        uint64_t da = tc_desc(a_addr + (uint32_t)(st * 2 * TC_KB * 4)), db = tc_desc(b_addr + (uint32_t)(kb * TC_N * 128));
                        const int nks = KS - 4 * kb < 4 ? KS - 4 * kb : 4;
                        uint32_t acc = uu == 0 ? 0u : 1u;                     // the first MMA into D_T of a tile overwrites
                        for (int ks = 0; ks < nks; ++ks) {
                            tc_mma_tf32(dT, da, db, TC_IDESC, acc);
                            if (SPLIT && pl == 0) tc_mma_tf32(dT, da, db + lo_off, TC_IDESC, 1);       // plane hi: also Ah Bl
                            acc = 1;
                            da += 2; db += 2;
                        }
                        tc_commit(&stage_free[st]);                           // the stage may be refilled once these MMAs are done
                        if (t + 2 >= NTILE && pl == NPL - 1) tc_commit(&freeB[kb]);   // (last tile of this thread) ... K-block kb of B_s too
                    }
                    tc_commit(&mma_done[par]);                                // the tile's accumulator D_T is complete
                }
                if (t0 >= NTILE)                                              // no tile of this parity: nothing of B_s is read here
                    for (int kb = 0; kb < NKB; ++kb) mbar_arrive(&freeB[kb]);
            }
            __syncwarp();
        } else {
            // ===== epilogue: warps 0-7; warp w reads TMEM lanes 32 (w & 3) .. + 31 = rows (gamma, orbital) and the columns of the
            //       walker half w >> 2 =====
            // The contraction needs  X_w += sum_{a,b} T1[(g,a),(w,b)] * T2[(g,b),(w,a)].  Both accumulators are read with the
            // 16-lane x 256-bit shape: a thread gets, of the rows  l0 + lane/4 (+ 8)  (l0 = 0, 16: two loads), the orbital
            // column  lane % 4  of every walker, i.e. T1[(g, a = (lane/4) % 4), (w, b = lane % 4)] of four gammas, and of T2 the
            // element with the two orbitals exchanged sits in the lane with those two 2-bit fields swapped: ONE shuffle per value
            // (a first version transposed 4 x 4 blocks over adjacent lanes from the one-row-per-lane shape: 4 shuffles + 12 selects).
            const int partner = (lane & 16) | ((lane & 3) << 2) | ((lane >> 2) & 3);
            for (int t = 0; t < NTILE; ++t) {
                const uint32_t buf = (tbase + (uint32_t)t) & 1, n = (tbase + (uint32_t)t) >> 1;
                mbar_wait(&mma_done[buf], n & 1);
                tc_fence_after();
                const uint32_t trow = tmem_base + ((uint32_t)(32 * (warp & 3)) << 16) + buf * (2 * TC_N) + (warp >> 2) * (TC_N / 2);
                // two walkers (16 columns) at a time; the loads of the next pair are in flight while this pair is contracted
                float t1[2][2][8], t2[2][2][8];                         // [parity of the pair][l0][4 walker + 2 (row + 8) + re/im]
#pragma unroll
                for (int l = 0; l < 2; ++l) {
                    tc_ld16x256x2(trow + ((uint32_t)(16 * l) << 16) + TC_N, t2[0][l]);
                    tc_ld16x256x2(trow + ((uint32_t)(16 * l) << 16), t1[0][l]);
                }
#pragma unroll
                for (int q2 = 0; q2 < TC_NH / 2; ++q2) {
                    tc_wait_ld();
                    if (q2 + 1 < TC_NH / 2) {
#pragma unroll
                        for (int l = 0; l < 2; ++l) {
                            tc_ld16x256x2(trow + ((uint32_t)(16 * l) << 16) + TC_N + 16 * (q2 + 1), t2[(q2 + 1) & 1][l]);
                            tc_ld16x256x2(trow + ((uint32_t)(16 * l) << 16) + 16 * (q2 + 1), t1[(q2 + 1) & 1][l]);
                        }
                    } else {                                            // the last columns of the buffer are in registers
                        tc_fence_before();
                        mbar_arrive(&tmem_free[buf]);
                    }
#pragma unroll
                    for (int l = 0; l < 2; ++l)
#pragma unroll
                        for (int i = 0; i < 8; ++i) t2[q2 & 1][l][i] = __shfl_sync(0xffffffffu, t2[q2 & 1][l][i], partner);
#pragma unroll
                    for (int wl = 0; wl < 2; ++wl) {
                        float sr = 0.f, si = 0.f;
#pragma unroll
                        for (int l = 0; l < 2; ++l)
#pragma unroll
                            for (int h = 0; h < 2; ++h) {
                                const float ar = t1[q2 & 1][l][4 * wl + 2 * h], ai = t1[q2 & 1][l][4 * wl + 2 * h + 1];
                                const float pr = t2[q2 & 1][l][4 * wl + 2 * h], pi = t2[q2 & 1][l][4 * wl + 2 * h + 1];
                                sr = fmaf(ar, pr, sr); sr = fmaf(-ai, pi, sr);
                                si = fmaf(ar, pi, si); si = fmaf(ai, pr, si);
                            }
                        xr64[2 * q2 + wl] += (double)sr; xi64[2 * q2 + wl] += (double)si;
                    }
                }
            }
        }

        // ---- the item's result: sum over the 128 rows.  Only the epilogue warps take part (named barrier 1): the producer and the
        //      MMA threads run on into the next item.  Lanes: a butterfly that halves the number of values at every stage (lane l
        //      ends with the total of value l % (2 NH): re of the warp's walker l, im of walker l - NH), then the four warps of a
        //      walker half in a fixed order; the scratch alternates per item, so one barrier per item suffices ----
        if (warp < TC_EPI_WARPS) {
            double* rd = red + (it & 1) * (TC_EPI_WARPS * 2 * TC_NH);
            double v[2 * TC_NH];
#pragma unroll
            for (int j = 0; j < TC_NH; ++j) { v[j] = xr64[j]; v[TC_NH + j] = xi64[j]; }
#pragma unroll
            for (int m = 16; m >= 2 * TC_NH; m >>= 1) {                 // more lanes than values: plain sums first
#pragma unroll
                for (int j = 0; j < 2 * TC_NH; ++j) v[j] += __shfl_xor_sync(0xffffffffu, v[j], m);
            }
#pragma unroll
            for (int m = TC_NH; m >= 1; m >>= 1) {
                const bool hi = lane & m;
#pragma unroll
                for (int i = 0; i < m; ++i) {
                    const double send = hi ? v[i] : v[i + m], keep = hi ? v[i + m] : v[i];
                    v[i] = keep + __shfl_xor_sync(0xffffffffu, send, m);
                }
            }
            if (lane < 2 * TC_NH) rd[warp * (2 * TC_NH) + lane] = v[0];
            asm volatile("bar.sync 1, 256;\n" ::: "memory");
            if (tid < 2 * TC_NWC) {
                const int wl = tid % TC_NWC, c = tid / TC_NWC, hw = wl / TC_NH, j = wl % TC_NH;
                if (w0 + wl < nw) {
                    double r = 0.0;
                    for (int x = 0; x < 4; ++x) r += rd[(4 * hw + x) * (2 * TC_NH) + c * TC_NH + j];
                    reinterpret_cast<double*>(partial)[((size_t)u * nw + w0 + wl) * 2 + c] = r;
                }
            }
        }
    }

    tc_fence_before();
    __syncthreads();
    if (warp == TC_EPI_WARPS) tc_dealloc(tmem_base, Cfg::TMEM_COLS);
}

}  // namespace

static void tc_geom(const Dims& d, int* KP, int* KS, int* NTILE) {
    *KS = (2 * d.m + 7) / 8;                 // k-steps of 8 reals actually multiplied
    *KP = (2 * d.m + 31) / 32 * 32;          // stored K: whole 128-byte swizzle rows
    *NTILE = (d.nchol + 31) / 32;
}

typedef CUresult (*TcEncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                               const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// tensor map of a float array viewed as rows of 64 floats (256 bytes), box = `box_rows` rows (one image)
static bool tc_make_map(void* out128, float* base, size_t floats, int box_rows) {
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (box_rows > 256 || cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn ||
        qres != cudaDriverEntryPointSuccess) {
        (void)cudaGetLastError();
        return false;
    }
    const cuuint64_t gdim[2] = {64, (cuuint64_t)(floats / 64)};
    const cuuint64_t gstride[1] = {256};
    const cuuint32_t box[2] = {64, (cuuint32_t)box_rows};
    const cuuint32_t estr[2] = {1, 1};
    return reinterpret_cast<TcEncodeFn>(fn)(reinterpret_cast<CUtensorMap*>(out128), CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, base, gdim, gstride, box, estr,
                                            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                                            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// packs the operand, allocates the per-call B-image workspace and encodes the tensor maps on first use (two maps of the B
// workspace: images of 8 and of 16 walkers)
int afqmc_i_ensure_lxu(afqmc_ctx* c, cudaStream_t st) {
    if (c->LxU) return AFQMC_OK;
    const Dims& d = c->d;
    if (d.NAG != 1) return AFQMC_UNSUPPORTED;
    int KP, KS, NTILE;
    tc_geom(d, &KP, &KS, &NTILE);
    const size_t total = (size_t)d.Nk * d.Nk * NTILE * TC_M * KP;        // per plane
    const size_t nthu = (size_t)d.Nk * d.Nk * ((c->max_walkers + 15) / 16) * 2 * 128 * KP;     // (>= the 8-walker layout of <= 8 walkers)
    if (cudaMalloc((void**)&c->LxU, 2 * total * sizeof(float)) != cudaSuccess) { (void)cudaGetLastError(); c->LxU = nullptr; return AFQMC_OUT_OF_MEMORY; }
    if (cudaMalloc((void**)&c->ws_thetaU, nthu * sizeof(float)) != cudaSuccess) { (void)cudaGetLastError(); c->ws_thetaU = nullptr; return AFQMC_OUT_OF_MEMORY; }
    size_t g = (total + 255) / 256;
    if (g > 148 * 64) g = 148 * 64;
    pack_LxU_kernel<<<(unsigned)g, 256, 0, st>>>(d, KP, NTILE, c->Lh, c->LxU, total);
    AFQMC_LAUNCH_CHECK(c);
    c->tmap_lxu_ok = (tc_make_map(c->tmap_lxu, c->LxU, 2 * total, TC_KB / 64) && tc_make_map(c->tmap_thu, c->ws_thetaU, nthu, 64 / 2) &&
                      tc_make_map(c->tmap_thu16, c->ws_thetaU, nthu, 128 / 2)) ? 1 : 0;
    return AFQMC_OK;
}

template <bool SPLIT, int NWC>
static int tc_launch(afqmc_ctx* c, int KP, int KS, int NTILE, const double2* theta, int nw, cudaStream_t st) {
    using Cfg = TcCfg<SPLIT, NWC>;
    const Dims& d = c->d;
    constexpr int npl = SPLIT ? 2 : 1;
    // shared memory: the item's B images, the reduction scratch, the barriers, and as many ring stages as fit beside them
    const size_t fixed = (size_t)2 * npl * Cfg::N * KP * sizeof(float) + (size_t)2 * 4 * NWC * 2 * sizeof(double) + (3 * TC_MAXST + 4 + 2 * TC_MAXKB) * sizeof(uint64_t) + 16;
    const size_t stage = (size_t)2 * TC_KB * sizeof(float);
    if (KP / 32 > TC_MAXKB || fixed + 2 * stage > (size_t)c->smem_optin) return AFQMC_UNSUPPORTED;
    int nst = (int)(((size_t)c->smem_optin - fixed) / stage);
    if (nst > TC_MAXST) nst = TC_MAXST;
    if (c->opt_exchange_tc > 1 && c->opt_exchange_tc < nst) nst = c->opt_exchange_tc;       // (experiments: option exchange_tc = stages)
    const size_t smem = fixed + (size_t)nst * stage;
    int rc = afqmc_i_ensure_lxu(c, st);
    if (rc != AFQMC_OK) return rc;
    if (!c->tmap_lxu_ok) return AFQMC_UNSUPPORTED;
    const CUtensorMap tmapA = *reinterpret_cast<const CUtensorMap*>(c->tmap_lxu);
    const CUtensorMap tmapB = *reinterpret_cast<const CUtensorMap*>(NWC == 16 ? c->tmap_thu16 : c->tmap_thu);
    const int nwg = (nw + NWC - 1) / NWC;
    // the B images of every theta block (real embedding, TF32 split) for this call
    {
        const size_t total = (size_t)d.Nk * d.Nk * nwg * NWC * 4 * (KP / 2);
        size_t g = (total + 255) / 256;
        if (g > (size_t)c->num_sms * 32) g = (size_t)c->num_sms * 32;
        tc_pack_theta_kernel<<<(unsigned)g, 256, 0, st>>>(d, KP, NWC, nwg, nw, npl, theta, c->ws_thetaU, total);
        AFQMC_LAUNCH_CHECK(c);
    }
    const long long nitems = (long long)c->nunits * nwg;
    if (nitems > 0x7fffffffLL) return AFQMC_UNSUPPORTED;
    const unsigned grid = (unsigned)(nitems < c->num_sms ? nitems : c->num_sms);
    auto kern = exchange_tc_kernel<SPLIT, NWC>;
    if ((rc = afqmc_smem_optin(c, (const void*)kern, smem)) != AFQMC_OK) return rc;
    kern<<<grid, TC_THREADS, smem, st>>>(tmapA, tmapB, d, KP, KS, NTILE, nst, nw, (int)nitems, c->units, c->kminus, c->kplus, c->kneg, c->ws_expart);
    AFQMC_LAUNCH_CHECK(c);
    c->ex_parts = 1;
    return AFQMC_OK;
}

// Writes the unit partial sums into ws_expart like the FP64 kernels.  AFQMC_UNSUPPORTED for n > 4 or if the tile images do not fit
// shared memory / a tensor-map box (the caller falls back to the mma.sync kernel).
int afqmc_i_exchange_tc(afqmc_ctx* c, const double2* theta, int nw, cudaStream_t st) {
    const Dims& d = c->d;
    if (d.NAG != 1) return AFQMC_UNSUPPORTED;
    int KP, KS, NTILE;
    tc_geom(d, &KP, &KS, &NTILE);
    const bool split = c->opt_exchange_prec == 1;
    if (nw <= 8) return split ? tc_launch<true, 8>(c, KP, KS, NTILE, theta, nw, st) : tc_launch<false, 8>(c, KP, KS, NTILE, theta, nw, st);
    int rc = split ? tc_launch<true, 16>(c, KP, KS, NTILE, theta, nw, st) : tc_launch<false, 16>(c, KP, KS, NTILE, theta, nw, st);
    // (rows too long for the 16-walker images: the 8-walker kernel may still fit)
    if (rc == AFQMC_UNSUPPORTED) rc = split ? tc_launch<true, 8>(c, KP, KS, NTILE, theta, nw, st) : tc_launch<false, 8>(c, KP, KS, NTILE, theta, nw, st);
    return rc;
}
