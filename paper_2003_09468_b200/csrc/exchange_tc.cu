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
//    c ^ (r & 7)), TF32-rounded high and low planes.  An image (32 KB at m = 26) arrives by ONE tensor-map copy
//    (cp.async.bulk.tensor.2d, SASS UTMALDG; the operand is viewed as rows of 256 bytes, box = one image, no TMA swizzle: the
//    bytes are already in place) into a ring of TC_STAGES images.
//  * B operand: the real-embedded, TF32-split images of EVERY theta block (row block, column block, walker group) are built
//    once per call by tc_pack_theta_kernel in the same swizzled layout (each block is used by ~2 Nk units) and arrive like A,
//    four tensor-map copies per work item.
//  * Warp roles: warp 5 lane 0 is the producer (tensor-map copies of the item's B images and of the A images, as far ahead as the
//    ring allows); warp 4 lane 0 issues the MMAs (one thread issues for the CTA) and commits them to mbarriers (tcgen05.commit);
//    warps 0-3 are the epilogue: tcgen05.ld of their 32 TMEM lanes (rows), the (a,b) transpose of the T2 values across the four
//    adjacent lanes of a gamma (two butterfly stages of shuffles), the complex contraction sum_b T1[(g,a),(w,b)] T2[(g,b),(w,a)]
//    in FP32 per tile and FP64 across tiles.  TMEM holds two accumulator buffers (2 x (D1, D2) x N columns = all 512 at N = 128),
//    so the epilogue of tile t overlaps the MMAs of tile t + 1.
//  * Results: unit partial sums in ws_expart, exactly like the FP64 kernels (energy_finalize_kernel applies multiplicities).
//  * Measured (C3, exchange stage incl. the theta pack): 3xTF32 3.98 ms, 1xTF32 1.68 ms (mma.sync kernel: 7.19 / 3.66 ms).  What
//    the versions on the way showed (ablation builds at N = 64, C3; profiles/r02g_ncu_exchange_tc.md): thread-built B images cost
//    1.2 ms per call; chains of dependent 128x64x8 MMAs into ONE accumulator ran at ~120 cycles per instruction (floor 32),
//    alternating the T1 / T2 accumulators brought that to ~90, four chains and the swizzle no further; an instruction took the SAME
//    time at N = 128 as at N = 64 (its cost is the fetch of the A tile), hence 16 walkers per CTA: 6.01 -> 3.98 ms and 2.51 ->
//    1.68 ms.  The first (a,b) transpose by shuffles picked its registers with lane-dependent compares, which the compiler turned
//    into divergent branches (11 ms); the butterfly transpose selects by lane bits only.  With 16 walkers the four B planes of
//    3xTF32 (128 KB at m = 26) leave room for three A stages, so that mode multiplies one image at a time (no T1 / T2 pairs).
#include <cuda.h>      // CUtensorMap and the encode function's type only: the entry point is fetched through the runtime, no libcuda link
#include "common.cuh"

namespace {

// walkers per CTA: NWC = 16 (N = 128 columns; an MMA instruction costs the same at N = 64, so wider is free) unless the batch
// has at most 8 walkers (NWC = 8: no padded columns)
constexpr int TC_M = 128;                 // rows of a tile: 32 gamma x 4 orbitals
constexpr int TC_THREADS = 192;           // warps 0-3: epilogue, warp 4: MMA issue, warp 5: bulk copies of the A images
// ring of A images (one image of one plane of one T per stage): what fits beside the B images (3xTF32, 16 walkers: 4 x 32 KB of
// B at m = 26 leave room for three); with four stages the two T of a plane are multiplied as a PAIR (alternating accumulators)
template <bool SPLIT, int NWC> struct TcCfg {
    static constexpr int STAGES = (SPLIT && NWC == 16) ? 3 : 4;
    static constexpr bool PAIRS = STAGES == 4;
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
// 16 consecutive 32-bit columns of this thread's TMEM lane
__device__ __forceinline__ void tc_ld16(uint32_t taddr, float (&v)[16]) {
    uint32_t r[16];
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];\n"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]), "=r"(r[10]),
          "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
        : "r"(taddr)
        : "memory");
#pragma unroll
    for (int i = 0; i < 16; ++i) v[i] = __uint_as_float(r[i]);
}
// 4 x 4 transpose across the four lanes l & ~3 .. (l & ~3) + 3: afterwards v_b on lane a holds what v_a held on lane b
__device__ __forceinline__ void tc_transpose4(float& v0, float& v1, float& v2, float& v3, int lane) {
    {
        const bool hi = lane & 1;
        const float r0 = __shfl_xor_sync(0xffffffffu, hi ? v0 : v1, 1), r1 = __shfl_xor_sync(0xffffffffu, hi ? v2 : v3, 1);
        v0 = hi ? r0 : v0; v1 = hi ? v1 : r0; v2 = hi ? r1 : v2; v3 = hi ? v3 : r1;
    }
    {
        const bool hi = lane & 2;
        const float r0 = __shfl_xor_sync(0xffffffffu, hi ? v0 : v2, 2), r1 = __shfl_xor_sync(0xffffffffu, hi ? v1 : v3, 2);
        v0 = hi ? r0 : v0; v2 = hi ? v2 : r0; v1 = hi ? r1 : v1; v3 = hi ? v3 : r1;
    }
}
__device__ __forceinline__ void tc_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;\n" ::: "memory"); }


template <bool SPLIT, int NWC>
__global__ void __launch_bounds__(TC_THREADS, 1) exchange_tc_kernel(
    const __grid_constant__ CUtensorMap tmapA, const __grid_constant__ CUtensorMap tmapB, Dims d, int KP, int KS, int NTILE, int nw,
    int nitems, const int* __restrict__ units, const int* __restrict__ kminus, const int* __restrict__ kplus,
    const int* __restrict__ kneg, double2* __restrict__ partial) {
    extern __shared__ __align__(1024) unsigned char tc_smem[];
    using Cfg = TcCfg<SPLIT, NWC>;
    constexpr int NPL = SPLIT ? 2 : 1, TC_STAGES = Cfg::STAGES, TC_N = Cfg::N, TC_NWC = NWC;
    constexpr uint32_t TC_IDESC = Cfg::IDESC;
    constexpr bool PAIRS = Cfg::PAIRS;
    const int IMG_A = TC_M * KP, IMG_B = TC_N * KP;        // floats (KP a multiple of 32: whole swizzle atoms)
    float* A_s = reinterpret_cast<float*>(tc_smem);        // [TC_STAGES][IMG_A]: ring of A images
    float* B_s = A_s + TC_STAGES * IMG_A;                  // [T][plane][IMG_B]: the item's B images
    double* red = reinterpret_cast<double*>(B_s + 2 * NPL * IMG_B);    // [2][4 warps][TC_NWC][2]
    uint64_t* bars = reinterpret_cast<uint64_t*>(red + 2 * 4 * TC_NWC * 2);
    uint64_t* fullA = bars;                        // [TC_STAGES]: the image of the stage has landed
    uint64_t* stage_free = bars + TC_STAGES;       // [TC_STAGES]: the MMAs that read the stage are complete (tcgen05.commit)
    uint64_t* mma_done = bars + 2 * TC_STAGES;     // [2]: the MMAs into accumulator buffer b (both T) are complete
    uint64_t* tmem_free = bars + 2 * TC_STAGES + 2;    // [2]: the epilogue has read accumulator buffer b
    uint64_t* fullB = bars + 2 * TC_STAGES + 4;    // the item's B images have landed
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 2 * TC_STAGES + 5);

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) {
        for (int i = 0; i < TC_STAGES; ++i) { mbar_init(&fullA[i], 1); mbar_init(&stage_free[i], 1); }
        mbar_init(&mma_done[0], 1); mbar_init(&mma_done[1], 1);
        mbar_init(&tmem_free[0], 128); mbar_init(&tmem_free[1], 128);
        mbar_init(fullB, 1);
        mbar_fence_init();
    }
    if (warp == 4) tc_alloc(tmem_slot, Cfg::TMEM_COLS);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;

    const int nwg = (nw + TC_NWC - 1) / TC_NWC;
    // One USE = one A image (tile t, T, plane) and the MMAs that read it: plane hi -> Ah Bh (+ Ah Bl), plane lo -> Al Bh.
    // Use g (counted over the CTA's whole life) lives in ring stage g % TC_STAGES; its copy completes phase g / TC_STAGES of
    // fullA[stage], the MMAs that read it complete that phase of stage_free[stage].  Tiles are counted likewise (tt): accumulator
    // buffer tt & 1, phases of mma_done / tmem_free; items (it): phase of fullB, parity of the reduction scratch.
    constexpr int UPT = 2 * NPL;                                         // uses per tile
    const int nuse = NTILE * UPT;
    uint32_t tt = 0, ubase = 0, it = 0;
    for (int item = blockIdx.x; item < nitems; item += gridDim.x, ++it) {
        const int u = item / nwg, wg = item - u * nwg, w0 = wg * TC_NWC;
        const int Q = units[4 * u], k = units[4 * u + 1], k2 = units[4 * u + 2];

        double xr64[TC_NWC], xi64[TC_NWC];
#pragma unroll
        for (int j = 0; j < TC_NWC; ++j) xr64[j] = xi64[j] = 0.0;

        if (warp == 5) {
            // ===== producer: one thread streams the item's B images and the A images, as far ahead as the rings allow =====
            if (lane == 0) {
                const int mQ = kneg[Q], kq = kminus[k * d.Nk + Q], k2pq = kplus[k2 * d.Nk + Q];
                // B: T1 from theta[(k2,.),(k-Q,.)], T2 from theta[(k,.),(k2+Q,.)]; B_s is free once the previous item's MMAs are done
                if (tt > 0) mbar_wait(&mma_done[(tt - 1) & 1], ((tt - 1) >> 1) & 1);
                const uint32_t bytes_b = (uint32_t)(IMG_B * sizeof(float));
                mbar_expect_tx(fullB, 2 * NPL * bytes_b);
                for (int T = 0; T < 2; ++T)
                    for (int pl = 0; pl < NPL; ++pl) {
                        const size_t blk = (((size_t)(T == 0 ? k2 : k) * d.Nk + (T == 0 ? kq : k2pq)) * nwg + wg) * 2 + pl;
                        tc_tma_rows(B_s + (size_t)(T * NPL + pl) * IMG_B, &tmapB, (int)(blk * (size_t)(IMG_B / 64)), fullB);
                    }
                const size_t blk1 = ((size_t)Q * d.Nk + k) * NTILE, blk2 = ((size_t)mQ * d.Nk + k2) * NTILE;
                const uint32_t bytes_a = (uint32_t)(IMG_A * sizeof(float));
                for (int j = 0; j < nuse; ++j) {
                    const uint32_t g = ubase + (uint32_t)j;
                    const int st = (int)(g % TC_STAGES);
                    if (g >= TC_STAGES) mbar_wait(&stage_free[st], ((g / TC_STAGES) - 1) & 1);
                    // use order inside a tile: pairs -> (plane, T) with T fastest; else (T1 hi, T1 lo, T2 hi, T2 lo), one image at a time
                    const int t = j / UPT, T = PAIRS ? (j & 1) : ((j % UPT) >> 1), pl = PAIRS ? ((j % UPT) >> 1) : (j & 1);
                    mbar_expect_tx(&fullA[st], bytes_a);
                    tc_tma_rows(A_s + (size_t)st * IMG_A, &tmapA, (int)((((T == 0 ? blk1 : blk2) + t) * 2 + pl) * (size_t)(IMG_A / 64)), &fullA[st]);
                }
            }
            ubase += (uint32_t)nuse;
            tt += (uint32_t)NTILE;
            __syncwarp();
        } else if (warp == 4) {
            // ===== MMA issue: one thread for the CTA =====
            if (lane == 0) {
                const uint32_t a_addr = smem_u32(A_s), b_addr = smem_u32(B_s);
                mbar_wait(fullB, it & 1);
                uint32_t buf = tt & 1;
                const uint32_t db_T[2] = {b_addr, b_addr + (uint32_t)(NPL * IMG_B * 4)};                      // hi planes of B1, B2
                const uint64_t lo_off = (uint64_t)((IMG_B * 4) >> 4);                                     // hi -> lo plane of a B image
                // a k-step is 8 kappa = 32 bytes of every row: 32-byte slot ks & 3 of K-block ks >> 2 (rows * 128 bytes each), i.e. the
                // start-address field of a descriptor (16-byte units) grows by 2, or jumps to the next block
                auto step_a = [](const int ks) { return (ks & 3) == 3 ? (uint64_t)((TC_M * 128 - 96) >> 4) : (uint64_t)2; };
                auto step_b = [](const int ks) { return (ks & 3) == 3 ? (uint64_t)((Cfg::N * 128 - 96) >> 4) : (uint64_t)2; };
                if (!PAIRS) {
                    // 3xTF32 at 16 walkers: one image per use (the ring holds three beside the four B planes); plane hi -> Ah Bh + Ah Bl, lo -> Al Bh
                    for (int j = 0; j < nuse; ++j) {
                        const uint32_t g = ubase + (uint32_t)j;
                        const int st = (int)(g % TC_STAGES), T = (j >> 1) & 1, pl = j & 1;
                        if ((j & 3) == 0) {                                   // first use of a tile
                            buf = tt & 1;
                            if (tt >= 2) mbar_wait(&tmem_free[buf], ((tt >> 1) - 1) & 1);       // the accumulator buffer was read
                        }
                        mbar_wait(&fullA[st], (g / TC_STAGES) & 1);
                        tc_fence_after();
                        const uint32_t dT = tmem_base + buf * (2 * TC_N) + T * TC_N;
                        uint64_t da = tc_desc(a_addr + (uint32_t)(st * IMG_A * 4)), db = tc_desc(db_T[T]);
                        uint32_t acc = pl == 0 ? 0u : 1u;                     // the first MMA into D_T of a tile overwrites
                        for (int ks = 0; ks < KS; ++ks) {
                            tc_mma_tf32(dT, da, db, TC_IDESC, acc);
                            if (pl == 0) tc_mma_tf32(dT, da, db + lo_off, TC_IDESC, 1);
                            acc = 1;
                            da += step_a(ks); db += step_b(ks);
                        }
                        tc_commit(&stage_free[st]);                           // the stage may be refilled once these MMAs are done
                        if ((j & 3) == 3) { tc_commit(&mma_done[buf]); ++tt; }    // ... and the tile's accumulators are complete
                    }
                } else {
                    // the two images (T1, T2) of a plane as a PAIR, their MMAs alternating, so that consecutive instructions accumulate
                    // into different TMEM columns (dependent MMAs into one accumulator serialise: ~120 against ~90 cycles each)
                    for (int q = 0; q < nuse / 2; ++q) {
                        const uint32_t g0 = ubase + 2u * (uint32_t)q, g1 = g0 + 1;
                        const int s0 = (int)(g0 % TC_STAGES), s1 = (int)(g1 % TC_STAGES);
                        const int pl = q % NPL;
                        if (pl == 0) {                                        // first pair of a tile
                            buf = tt & 1;
                            if (tt >= 2) mbar_wait(&tmem_free[buf], ((tt >> 1) - 1) & 1);       // the accumulator buffer was read
                        }
                        mbar_wait(&fullA[s0], (g0 / TC_STAGES) & 1);
                        mbar_wait(&fullA[s1], (g1 / TC_STAGES) & 1);
                        tc_fence_after();
                        const uint32_t d0 = tmem_base + buf * (2 * TC_N), d1 = d0 + TC_N;
                        uint64_t da0 = tc_desc(a_addr + (uint32_t)(s0 * IMG_A * 4)), da1 = tc_desc(a_addr + (uint32_t)(s1 * IMG_A * 4));
                        uint64_t db0 = tc_desc(db_T[0]), db1 = tc_desc(db_T[1]);
                        uint32_t acc = pl == 0 ? 0u : 1u;                     // the first MMA into D_T of a tile overwrites
                        for (int ks = 0; ks < KS; ++ks) {
                            tc_mma_tf32(d0, da0, db0, TC_IDESC, acc);
                            tc_mma_tf32(d1, da1, db1, TC_IDESC, acc);
                            if (SPLIT && pl == 0) {                           // plane hi: also Ah Bl
                                tc_mma_tf32(d0, da0, db0 + lo_off, TC_IDESC, 1);
                                tc_mma_tf32(d1, da1, db1 + lo_off, TC_IDESC, 1);
                            }
                            acc = 1;
                            da0 += step_a(ks); da1 += step_a(ks); db0 += step_b(ks); db1 += step_b(ks);
                        }
                        tc_commit(&stage_free[s0]);
                        tc_commit(&stage_free[s1]);
                        if (pl == NPL - 1) { tc_commit(&mma_done[buf]); ++tt; }
                    }
                }
            } else {
                tt += (uint32_t)NTILE;
            }
            ubase += (uint32_t)nuse;
            __syncwarp();
        } else {
            // ===== epilogue: warps 0-3 own TMEM lanes 32 warp .. 32 warp + 31 = rows (gamma, orbital) =====
            for (int t = 0; t < NTILE; ++t, ++tt) {
                const uint32_t buf = tt & 1;
                mbar_wait(&mma_done[buf], (tt >> 1) & 1);
                tc_fence_after();
                const uint32_t trow = tmem_base + ((uint32_t)(32 * warp) << 16) + buf * (2 * TC_N);
                // four walkers (32 columns) of both accumulator rows at a time.  The contraction needs
                //   X_w += sum_b T1[(g,a),(w,b)] * T2[(g,b),(w,a)]:
                // T2[(g,b),(w,a)] sits in lane (g,b), one of the four adjacent lanes of this gamma, at the column of the RECEIVER's
                // orbital a: a 4 x 4 transpose across those lanes (no shared memory)
#pragma unroll
                for (int q4 = 0; q4 < TC_NWC / 4; ++q4) {
                    float t1[32], t2[32];
#pragma unroll
                    for (int q = 0; q < 2; ++q) {
                        float v[16];
                        tc_ld16(trow + TC_N + 32 * q4 + 16 * q, v);
#pragma unroll
                        for (int i = 0; i < 16; ++i) t2[16 * q + i] = v[i];
                        tc_ld16(trow + 32 * q4 + 16 * q, v);
#pragma unroll
                        for (int i = 0; i < 16; ++i) t1[16 * q + i] = v[i];
                    }
                    tc_wait_ld();
                    if (q4 == TC_NWC / 4 - 1) {                       // the last columns of the buffer are in registers
                        tc_fence_before();
                        mbar_arrive(&tmem_free[buf]);
                    }
                    // the T2 values of every walker: 4 x 4 transpose over the four lanes of this gamma (two butterfly stages of
                    // shuffles, register choice by the lane's bits only: no lane-dependent register indexing)
#pragma unroll
                    for (int wl = 0; wl < 4; ++wl) {
#pragma unroll
                        for (int c = 0; c < 2; ++c) tc_transpose4(t2[8 * wl + c], t2[8 * wl + 2 + c], t2[8 * wl + 4 + c], t2[8 * wl + 6 + c], lane);
                        float sr = 0.f, si = 0.f;       // now t2[8 wl + 2 b + c] = T2[(g,b),(w,a)] of this lane's a
#pragma unroll
                        for (int b = 0; b < 4; ++b) {
                            const float ar = t1[8 * wl + 2 * b], ai = t1[8 * wl + 2 * b + 1], pr = t2[8 * wl + 2 * b], pi = t2[8 * wl + 2 * b + 1];
                            sr = fmaf(ar, pr, sr); sr = fmaf(-ai, pi, sr);
                            si = fmaf(ar, pi, si); si = fmaf(ai, pr, si);
                        }
                        xr64[4 * q4 + wl] += (double)sr; xi64[4 * q4 + wl] += (double)si;
                    }
                }
            }
        }

        // ---- the item's result: sum over the 128 rows (lanes, then warps in a fixed order); scratch alternates per item, so one
        //      CTA-wide barrier per item suffices ----
        double* rd = red + (it & 1) * (4 * TC_NWC * 2);
        if (warp < 4) {
#pragma unroll
            for (int wl = 0; wl < TC_NWC; ++wl) {
                const double r = warp_sum(xr64[wl]), i = warp_sum(xi64[wl]);
                if (lane == 0) { rd[(warp * TC_NWC + wl) * 2] = r; rd[(warp * TC_NWC + wl) * 2 + 1] = i; }
            }
        }
        __syncthreads();
        if (tid < TC_NWC && w0 + tid < nw) {
            double r = 0.0, i = 0.0;
            for (int x = 0; x < 4; ++x) { r += rd[(x * TC_NWC + tid) * 2]; i += rd[(x * TC_NWC + tid) * 2 + 1]; }
            partial[(size_t)u * nw + w0 + tid] = make_double2(r, i);
        }
    }

    tc_fence_before();
    __syncthreads();
    if (warp == 4) tc_dealloc(tmem_base, Cfg::TMEM_COLS);
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
    c->tmap_lxu_ok = (tc_make_map(c->tmap_lxu, c->LxU, 2 * total, TC_M * KP / 64) && tc_make_map(c->tmap_thu, c->ws_thetaU, nthu, 64 * KP / 64) &&
                      tc_make_map(c->tmap_thu16, c->ws_thetaU, nthu, 128 * KP / 64)) ? 1 : 0;
    return AFQMC_OK;
}

template <bool SPLIT, int NWC>
static int tc_launch(afqmc_ctx* c, int KP, int KS, int NTILE, const double2* theta, int nw, cudaStream_t st) {
    using Cfg = TcCfg<SPLIT, NWC>;
    const Dims& d = c->d;
    constexpr int npl = SPLIT ? 2 : 1;
    const size_t smem = (size_t)(Cfg::STAGES * TC_M + 2 * npl * Cfg::N) * KP * sizeof(float) + (size_t)2 * 4 * NWC * 2 * sizeof(double) +
                        (2 * Cfg::STAGES + 5) * sizeof(uint64_t) + 16;
    if (smem > (size_t)c->smem_optin) return AFQMC_UNSUPPORTED;
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
    kern<<<grid, TC_THREADS, smem, st>>>(tmapA, tmapB, d, KP, KS, NTILE, nw, (int)nitems, c->units, c->kminus, c->kplus, c->kneg, c->ws_expart);
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
