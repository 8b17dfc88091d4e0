// a9 exchange energy with the 3M complex product (same contraction as energy.cu, Eq. 49):
//
//   T = Lh * theta^T  is a complex GEMM.  energy.cu embeds it in ONE real GEMM with K = (r, re/im) and columns
//   (b, re/im): 8 real flops per complex multiply-add (4 real products).  Here every complex product is formed
//   from THREE real products (Gauss's form of the "3M" product: two additions per result instead of Karatsuba's three,
//   which matters because DADD shares the FP64 units with DMMA):
//       P0 = (Ar+Ai) Br,  P1 = Ar (Bi-Br),  P2 = Ai (Br+Bi);      Re T = P0 - P2,   Im T = P0 + P1
//   i.e. three real GEMMs with K = r and columns b: 6 real flops per complex multiply-add, 25 % fewer DMMAs
//   (19 % at m = 26, where K = 26 pads to 7 k-steps of 4).  The tensor pipe is the bound of this kernel
//   (89 % DMMA issue, r01c profile), so fewer DMMAs is the only lever left.  Rounding: Im T carries the error of
//   (|Ar|+|Ai|)(|Br|+|Bi|) instead of |A||B|: a small constant factor, far inside the 1e-10 tolerance.
//
// Layout of the static operand (written once in afqmc_create):
//   Lx3[Q][k][ag][gq][ks][prod][lane][i]   prod = 0: Re + Im of Lh, 1: Re, 2: Im;  two M-tiles i = 0,1 per gamma-quad
//   rows (gl = row>>2, al = row&3): gamma = 4gq+2i+gl, a = 4ag+al;  K: r = 4ks + (lane&3);  zeros outside.
// A warp task is one gamma-quad: 3*KS3 "micro-steps" (ks-major, product-minor), each ONE coalesced 512-byte LDG.128
// of A, consecutive in memory across micro-steps and tasks.  DMMA columns are (walker of a pair, b): one n-tile
// serves two walkers, a CTA handles 2*NP walkers.  The three products keep separate accumulators; the register
// pipeline is 3 deep and unrolled by 3, so buffer q always belongs to product q (static register indexing).
// At the end of a task the products are combined and contracted in registers.  The partner tile is computed with
// the DMMA operands swapped (theta as A, Lh as B: the two fragment lane layouts coincide), which yields it already
// transposed in (a,b); one shuffle per value (lane bits 4 and 1 exchanged) then aligns gamma and walker.  n <= 4 (one
// a-group) uses the tuned kernel below; larger n the multi-group variant after it (falls back to the 4M kernel only if
// the theta blocks of all a-groups do not fit shared memory).
#include "common.cuh"

namespace {

__global__ void pack_Lx3_kernel(Dims d, int KS3, const double2* __restrict__ L, const double2* __restrict__ psi_t,
                                double* __restrict__ Lx3, size_t total_in /* without the product index */, size_t total_out) {
    for (size_t idx = blockIdx.x * (size_t)blockDim.x + threadIdx.x; idx < total_in; idx += (size_t)gridDim.x * blockDim.x) {
        size_t t = idx;
        const int i = (int)(t & 1); t >>= 1;
        const int lane = (int)(t & 31); t >>= 5;
        const int ks = (int)(t % KS3); t /= KS3;
        const int gq = (int)(t % d.GQ); t /= d.GQ;
        const int ag = (int)(t % d.NAG); t /= d.NAG;
        const int k = (int)(t % d.Nk);
        const int Q = (int)(t / d.Nk);
        const int row = lane >> 2, kk = lane & 3;
        const int gam = 4 * gq + 2 * i + (row >> 2), a = 4 * ag + (row & 3), r = 4 * ks + kk;
        double2 z = make_double2(0.0, 0.0);
        if (a < d.n && gam < d.nchol && r < d.m) {
            // Lh[Q][k][a][gam][r] = sum_p conj(A_k[p][a]) L[Q][k][gam][p][r]
            const double2* Lb = L + (((size_t)(Q * d.Nk + k) * d.nchol + gam) * d.m) * d.m + r;
            const double2* Ab = psi_t + (size_t)k * d.m * d.n + a;
            for (int p = 0; p < d.m; ++p) {
                double2 av = Ab[(size_t)p * d.n];
                av.y = -av.y;
                z = cfma(av, Lb[(size_t)p * d.m], z);
            }
        }
        // [..][ks][prod][lane][i]
        const size_t base = ((((((size_t)Q * d.Nk + k) * d.NAG + ag) * d.GQ + gq) * KS3 + ks) * 3) * 64 + lane * 2 + i;
        Lx3[base] = z.x + z.y;
        Lx3[base + 64] = z.x;
        Lx3[base + 128] = z.y;
    }
    // zero pad after the last block (the kernel's prefetch may run 3 micro-steps past the last task)
    const size_t body = total_in * 3;
    for (size_t idx = body + blockIdx.x * (size_t)blockDim.x + threadIdx.x; idx < total_out; idx += (size_t)gridDim.x * blockDim.x)
        Lx3[idx] = 0.0;
}

}  // namespace

size_t afqmc_i_lx3_doubles(const Dims& d) {
    const int KS3 = (d.m + 3) / 4;
    return (size_t)d.Nk * d.Nk * d.NAG * d.GQ * KS3 * 3 * 64 + AFQMC_LX_PAD;
}

int afqmc_i_pack_lx3(afqmc_ctx* c, const double2* L, cudaStream_t st) {
    const Dims& d = c->d;
    const int KS3 = (d.m + 3) / 4;
    const size_t total_in = (size_t)d.Nk * d.Nk * d.NAG * d.GQ * KS3 * 64;
    const size_t total_out = afqmc_i_lx3_doubles(d);
    size_t g = (total_in + 255) / 256;
    if (g > 148 * 64) g = 148 * 64;
    pack_Lx3_kernel<<<(unsigned)g, 256, 0, st>>>(d, KS3, L, c->psi_t, c->Lx3, total_in, total_out);
    AFQMC_LAUNCH_CHECK(c);
    return AFQMC_OK;
}

namespace {

// CTA = (unit, group of 2*NP walkers), WPC warps; see the header comment.  n <= 4 only (NAG == 1).
// DA = micro-steps of register prefetch of the A (Lx3, L2-resident) stream: 3 or 6; B (shared memory) runs 3 ahead.
template <int NP, int WPC, int MINB, int DA>
__global__ void __launch_bounds__(32 * WPC, MINB) exchange3m_kernel(
    Dims d, int KS3, int nw, const int* __restrict__ units, const int* __restrict__ kminus, const int* __restrict__ kplus,
    const int* __restrict__ kneg, const double* __restrict__ Lx3, const double2* __restrict__ theta,
    double2* __restrict__ partial) {
    extern __shared__ __align__(16) double ex3_smem[];
    constexpr int NWC = 2 * NP;                      // walkers of this CTA
    const int nwg = (nw + NWC - 1) / NWC;            // walker groups of one unit are adjacent in the grid
    const int u = blockIdx.x / nwg, w0 = (blockIdx.x % nwg) * NWC;
    const int Q = units[4 * u], k = units[4 * u + 1], k2 = units[4 * u + 2];
    const int mQ = kneg[Q];
    const int kq = kminus[k * d.Nk + Q];        // k - Q   : column block of theta for T^Q rows k
    const int k2pq = kplus[k2 * d.Nk + Q];      // k2 + Q  : column block of theta for T^{-Q} rows k2
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int GQ = d.GQ, MS = 3 * KS3;              // micro-steps of one task
    // Bs[which][ms][j][lane]: which = 0 -> theta[(k2,b),(k-Q,r)], 1 -> theta[(k,a),(k2+Q,s)]
    constexpr int bs_step = NP * 32;
    const int bs_half = MS * bs_step;

    // ---- this warp's contiguous share of the gamma-quads ----
    const int t_begin = (int)((long long)warp * GQ / WPC), t_end = (int)((long long)(warp + 1) * GQ / WPC);
    const int total = (t_end - t_begin) * MS;                       // micro-steps of this warp (a multiple of 3)
    const size_t task_doubles = (size_t)MS * 64;
    const double2* la1 = reinterpret_cast<const double2*>(Lx3 + (((size_t)Q * d.Nk + k) * GQ + t_begin) * task_doubles) + lane;
    const double2* la2 = reinterpret_cast<const double2*>(Lx3 + (((size_t)mQ * d.Nk + k2) * GQ + t_begin) * task_doubles) + lane;
    const double* lb1 = ex3_smem + lane;
    const double* lb2 = ex3_smem + bs_half + lane;
    int ls = 0;
    auto loader_advance = [&]() {        // A is contiguous across micro-steps and tasks, B wraps every MS micro-steps
        const bool wrap = ++ls == MS;
        const int db = wrap ? -(MS - 1) * bs_step : bs_step;
        lb1 += db; lb2 += db;
        ls = wrap ? 0 : ls;
    };
    static_assert(DA == 3 || DA == 6, "A depth is a multiple of the three products");
    double2 fa1[DA], fa2[DA];
    double fb1[3][NP], fb2[3][NP];
    // A prologue: issued before the staging below, which hides the L2 round trip
#pragma unroll
    for (int q = 0; q < DA; ++q) {
        fa1[q] = fa2[q] = make_double2(0.0, 0.0);
        if (total > 0) { fa1[q] = __ldg(la1 + q * 32); fa2[q] = __ldg(la2 + q * 32); }
    }
    la1 += DA * 32; la2 += DA * 32;

    // ---- stage the B fragments: one thread per complex theta element (b, walker, r) ----
    //   lane of a B fragment = (col << 2) | kk,  col = 4*(w&1) + b,  kk = r & 3;  micro-step = 3*(r>>2) + prod
    {
        const int per_which = 4 * NWC * 4 * KS3;
        for (int e = tid; e < 2 * per_which; e += 32 * WPC) {
            const int which = e / per_which;
            int x = e - which * per_which;
            const int b = x & 3; x >>= 2;
            const int wl = x % NWC, r = x / NWC;                 // r < 4*KS3
            const int w = w0 + wl;
            const int rowblk = which == 0 ? k2 : k, colblk = which == 0 ? kq : k2pq;
            double2 v = make_double2(0.0, 0.0);
            if (b < d.n && w < nw && r < d.m)
                v = __ldg(theta + ((size_t)w * d.N + rowblk * d.n + b) * d.M + (size_t)colblk * d.m + r);
            double* dst = ex3_smem + which * bs_half + ((3 * (r >> 2)) * NP + (wl >> 1)) * 32 + (((wl & 1) * 4 + b) << 2) + (r & 3);
            dst[0] = v.x;
            dst[bs_step] = v.y - v.x;
            dst[2 * bs_step] = v.x + v.y;
        }
    }
    __syncthreads();   // B fragments staged

    // B prologue, and bring the loader state to micro-step 3
#pragma unroll
    for (int q = 0; q < 3; ++q) {
#pragma unroll
        for (int j = 0; j < NP; ++j) { fb1[q][j] = lb1[j * 32]; fb2[q][j] = lb2[j * 32]; }
        loader_advance();
    }

    double er[NP], ei[NP];
#pragma unroll
    for (int j = 0; j < NP; ++j) er[j] = ei[j] = 0.0;
    // lane geometry of the C fragments (row = lane>>2, columns 2c+e with c = lane&3, register e):
    //   T1   : row (gamma of pair g, a),   columns (walker of pair wp = c>>1, b = 2(c&1)+e)
    //   T2^T : row (walker of pair wp, a), columns (gamma of pair g = c>>1,  b = 2(c&1)+e)
    // The contraction sum_{a,b} T1[(g,a),(wp,b)] T2[(g,b),(wp,a)] = sum T1[(g,a),(wp,b)] T2^T[(wp,a),(g,b)] pairs
    // register e of lane (g, a | wp, c&1) with register e of lane (wp, a | g, c&1): lane bits 4 and 1 exchanged.
    const int srcl = (lane & ~0x12) | ((lane & 16) >> 3) | ((lane & 2) << 3);
    double acc1[3][2][NP][2], acc2[3][2][NP][2];
#pragma unroll
    for (int p = 0; p < 3; ++p)
#pragma unroll
        for (int i = 0; i < 2; ++i)
#pragma unroll
            for (int j = 0; j < NP; ++j)
                acc1[p][i][j][0] = acc1[p][i][j][1] = acc2[p][i][j][0] = acc2[p][i][j][1] = 0.0;

    int cs = 0;   // micro-step of the compute state inside its task
    auto mstep = [&](const int qa) {     // A buffer qa; product and B buffer q = qa % 3
        const int q = qa % 3;
#pragma unroll
        for (int j = 0; j < NP; ++j) {
            dmma884(acc1[q][0][j][0], acc1[q][0][j][1], fa1[qa].x, fb1[q][j]);
            dmma884(acc1[q][1][j][0], acc1[q][1][j][1], fa1[qa].y, fb1[q][j]);
        }
        // partner tile with the operands swapped: theta is the A fragment and Lh the B fragment (their lane
        // layouts coincide), so the result is T2^T with rows (walker of pair, a) and columns (gamma of pair, b)
#pragma unroll
        for (int j = 0; j < NP; ++j) {
            dmma884(acc2[q][0][j][0], acc2[q][0][j][1], fb2[q][j], fa2[qa].x);
            dmma884(acc2[q][1][j][0], acc2[q][1][j][1], fb2[q][j], fa2[qa].y);
        }
        // refill the buffers with the micro-steps DA (A) and 3 (B) ahead (may run past the warp's last task:
        // loaded, never used)
        fa1[qa] = __ldg(la1); fa2[qa] = __ldg(la2);
        la1 += 32; la2 += 32;
#pragma unroll
        for (int j = 0; j < NP; ++j) { fb1[q][j] = lb1[j * 32]; fb2[q][j] = lb2[j * 32]; }
        loader_advance();
        if (q == 2) {
            cs += 3;
            if (cs == MS) {
                cs = 0;
#pragma unroll
                for (int i = 0; i < 2; ++i)
#pragma unroll
                    for (int j = 0; j < NP; ++j) {
                        double t1r[2], t1i[2], t2r[2], t2i[2];
#pragma unroll
                        for (int e = 0; e < 2; ++e) {
                            t1r[e] = acc1[0][i][j][e] - acc1[2][i][j][e];
                            t1i[e] = acc1[0][i][j][e] + acc1[1][i][j][e];
                            t2r[e] = acc2[0][i][j][e] - acc2[2][i][j][e];
                            t2i[e] = acc2[0][i][j][e] + acc2[1][i][j][e];
                        }
                        // T1 lane (g, a | wp, bp) pairs with T2^T lane (wp, a | g, bp), same register: swap lane bits 4 and 1
                        const double pr0 = __shfl_sync(0xffffffffu, t2r[0], srcl), pi0 = __shfl_sync(0xffffffffu, t2i[0], srcl);
                        const double pr1 = __shfl_sync(0xffffffffu, t2r[1], srcl), pi1 = __shfl_sync(0xffffffffu, t2i[1], srcl);
                        er[j] = fma(t1r[0], pr0, er[j]); er[j] = fma(-t1i[0], pi0, er[j]);
                        ei[j] = fma(t1r[0], pi0, ei[j]); ei[j] = fma(t1i[0], pr0, ei[j]);
                        er[j] = fma(t1r[1], pr1, er[j]); er[j] = fma(-t1i[1], pi1, er[j]);
                        ei[j] = fma(t1r[1], pi1, ei[j]); ei[j] = fma(t1i[1], pr1, ei[j]);
#pragma unroll
                        for (int p = 0; p < 3; ++p)
                            acc1[p][i][j][0] = acc1[p][i][j][1] = acc2[p][i][j][0] = acc2[p][i][j][1] = 0.0;
                    }
            }
        }
    };
    for (int g0 = 0; g0 < total; g0 += 3) {
        mstep(0); mstep(1); mstep(2);
        if (DA == 6) {
            if (g0 + 3 >= total) break;
            g0 += 3;
            mstep(DA - 3); mstep(DA - 2); mstep(DA - 1);
        }
    }

    // ---- reduce over the lanes of each walker-in-pair (lane bit 1), then over warps (deterministic) ----
    __syncthreads();
    double* red = ex3_smem;   // reuse: [warp][NWC][2]
#pragma unroll
    for (int j = 0; j < NP; ++j) {
        double r = er[j], i = ei[j];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            if (o == 2) continue;
            r += __shfl_xor_sync(0xffffffffu, r, o);
            i += __shfl_xor_sync(0xffffffffu, i, o);
        }
        if (lane == 0 || lane == 2) {
            const int wl = 2 * j + (lane >> 1);
            red[(warp * NWC + wl) * 2] = r; red[(warp * NWC + wl) * 2 + 1] = i;
        }
    }
    __syncthreads();
    if (tid < NWC && w0 + tid < nw) {
        double r = 0.0, i = 0.0;
        for (int x = 0; x < WPC; ++x) { r += red[(x * NWC + tid) * 2]; i += red[(x * NWC + tid) * 2 + 1]; }
        partial[(size_t)u * nw + w0 + tid] = make_double2(r, i);
    }
}

// ---------------------------------------------------------------------------------------------------------------
// The same kernel for MORE THAN FOUR occupied orbitals per k-point (NAG = ceil(n/4) > 1 a-groups).  The (ag, bg)
// pairs of a-groups are processed one after the other; inside a pair everything is as above (linear A streams of the
// rows ag of Lh[Q][k] and bg of Lh[-Q][k2], B fragments of the theta rows bg of k2 and ag of k).  The theta blocks of
// ALL groups are staged once per CTA: Bs[which][grp][ms][j][lane].
// ---------------------------------------------------------------------------------------------------------------
template <int NP, int WPC, int MINB>
__global__ void __launch_bounds__(32 * WPC, MINB) exchange3m_multi_kernel(
    Dims d, int KS3, int nw, const int* __restrict__ units, const int* __restrict__ kminus, const int* __restrict__ kplus,
    const int* __restrict__ kneg, const double* __restrict__ Lx3, const double2* __restrict__ theta,
    double2* __restrict__ partial) {
    extern __shared__ __align__(16) double ex3_smem[];
    constexpr int NWC = 2 * NP;
    const int nwg = (nw + NWC - 1) / NWC;
    const int u = blockIdx.x / nwg, w0 = (blockIdx.x % nwg) * NWC;
    const int Q = units[4 * u], k = units[4 * u + 1], k2 = units[4 * u + 2];
    const int mQ = kneg[Q];
    const int kq = kminus[k * d.Nk + Q];
    const int k2pq = kplus[k2 * d.Nk + Q];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int GQ = d.GQ, NAG = d.NAG, MS = 3 * KS3;
    constexpr int bs_step = NP * 32;
    const int bs_grp = MS * bs_step, bs_half = NAG * bs_grp;
    const size_t task_doubles = (size_t)MS * 64;

    // ---- stage the B fragments of every a-group: one thread per complex theta element (orbital, walker, r) ----
    {
        const int per_which = NAG * 4 * NWC * 4 * KS3;
        for (int e = tid; e < 2 * per_which; e += 32 * WPC) {
            const int which = e / per_which;
            int x = e - which * per_which;
            const int b = x & 3; x >>= 2;
            const int wl = x % NWC; x /= NWC;
            const int grp = x % NAG, r = x / NAG;                // r < 4*KS3
            const int orb = 4 * grp + b, w = w0 + wl;
            const int rowblk = which == 0 ? k2 : k, colblk = which == 0 ? kq : k2pq;
            double2 v = make_double2(0.0, 0.0);
            if (orb < d.n && w < nw && r < d.m)
                v = __ldg(theta + ((size_t)w * d.N + rowblk * d.n + orb) * d.M + (size_t)colblk * d.m + r);
            double* dst = ex3_smem + which * bs_half + grp * bs_grp + ((3 * (r >> 2)) * NP + (wl >> 1)) * 32 +
                          (((wl & 1) * 4 + b) << 2) + (r & 3);
            dst[0] = v.x;
            dst[bs_step] = v.y - v.x;
            dst[2 * bs_step] = v.x + v.y;
        }
    }
    __syncthreads();

    const int t_begin = (int)((long long)warp * GQ / WPC), t_end = (int)((long long)(warp + 1) * GQ / WPC);
    const int total = (t_end - t_begin) * MS;
    const int srcl = (lane & ~0x12) | ((lane & 16) >> 3) | ((lane & 2) << 3);
    double er[NP], ei[NP];
#pragma unroll
    for (int j = 0; j < NP; ++j) er[j] = ei[j] = 0.0;

    for (int ab = 0; ab < NAG * NAG; ++ab) {
        const int ag = ab / NAG, bg = ab % NAG;
        const double2* la1 = reinterpret_cast<const double2*>(Lx3 + ((((size_t)Q * d.Nk + k) * NAG + ag) * GQ + t_begin) * task_doubles) + lane;
        const double2* la2 = reinterpret_cast<const double2*>(Lx3 + ((((size_t)mQ * d.Nk + k2) * NAG + bg) * GQ + t_begin) * task_doubles) + lane;
        const double* lb1 = ex3_smem + bg * bs_grp + lane;                 // theta rows bg of k2
        const double* lb2 = ex3_smem + bs_half + ag * bs_grp + lane;       // theta rows ag of k
        int ls = 0;
        auto loader_advance = [&]() {
            const bool wrap = ++ls == MS;
            const int db = wrap ? -(MS - 1) * bs_step : bs_step;
            lb1 += db; lb2 += db;
            ls = wrap ? 0 : ls;
        };
        double2 fa1[3], fa2[3];
        double fb1[3][NP], fb2[3][NP];
#pragma unroll
        for (int q = 0; q < 3; ++q) {
            fa1[q] = fa2[q] = make_double2(0.0, 0.0);
            if (total > 0) { fa1[q] = __ldg(la1 + q * 32); fa2[q] = __ldg(la2 + q * 32); }
#pragma unroll
            for (int j = 0; j < NP; ++j) { fb1[q][j] = lb1[j * 32]; fb2[q][j] = lb2[j * 32]; }
            loader_advance();
        }
        la1 += 96; la2 += 96;
        double acc1[3][2][NP][2], acc2[3][2][NP][2];
#pragma unroll
        for (int p = 0; p < 3; ++p)
#pragma unroll
            for (int i = 0; i < 2; ++i)
#pragma unroll
                for (int j = 0; j < NP; ++j)
                    acc1[p][i][j][0] = acc1[p][i][j][1] = acc2[p][i][j][0] = acc2[p][i][j][1] = 0.0;
        int cs = 0;
        auto mstep = [&](const int q) {
#pragma unroll
            for (int j = 0; j < NP; ++j) {
                dmma884(acc1[q][0][j][0], acc1[q][0][j][1], fa1[q].x, fb1[q][j]);
                dmma884(acc1[q][1][j][0], acc1[q][1][j][1], fa1[q].y, fb1[q][j]);
            }
#pragma unroll
            for (int j = 0; j < NP; ++j) {
                dmma884(acc2[q][0][j][0], acc2[q][0][j][1], fb2[q][j], fa2[q].x);
                dmma884(acc2[q][1][j][0], acc2[q][1][j][1], fb2[q][j], fa2[q].y);
            }
            fa1[q] = __ldg(la1); fa2[q] = __ldg(la2);      // may run up to 3 micro-steps past this pair's last task
            la1 += 32; la2 += 32;
#pragma unroll
            for (int j = 0; j < NP; ++j) { fb1[q][j] = lb1[j * 32]; fb2[q][j] = lb2[j * 32]; }
            loader_advance();
            if (q == 2) {
                cs += 3;
                if (cs == MS) {
                    cs = 0;
#pragma unroll
                    for (int i = 0; i < 2; ++i)
#pragma unroll
                        for (int j = 0; j < NP; ++j) {
                            double t1r[2], t1i[2], t2r[2], t2i[2];
#pragma unroll
                            for (int e = 0; e < 2; ++e) {
                                t1r[e] = acc1[0][i][j][e] - acc1[2][i][j][e];
                                t1i[e] = acc1[0][i][j][e] + acc1[1][i][j][e];
                                t2r[e] = acc2[0][i][j][e] - acc2[2][i][j][e];
                                t2i[e] = acc2[0][i][j][e] + acc2[1][i][j][e];
                            }
                            const double pr0 = __shfl_sync(0xffffffffu, t2r[0], srcl), pi0 = __shfl_sync(0xffffffffu, t2i[0], srcl);
                            const double pr1 = __shfl_sync(0xffffffffu, t2r[1], srcl), pi1 = __shfl_sync(0xffffffffu, t2i[1], srcl);
                            er[j] = fma(t1r[0], pr0, er[j]); er[j] = fma(-t1i[0], pi0, er[j]);
                            ei[j] = fma(t1r[0], pi0, ei[j]); ei[j] = fma(t1i[0], pr0, ei[j]);
                            er[j] = fma(t1r[1], pr1, er[j]); er[j] = fma(-t1i[1], pi1, er[j]);
                            ei[j] = fma(t1r[1], pi1, ei[j]); ei[j] = fma(t1i[1], pr1, ei[j]);
#pragma unroll
                            for (int p = 0; p < 3; ++p)
                                acc1[p][i][j][0] = acc1[p][i][j][1] = acc2[p][i][j][0] = acc2[p][i][j][1] = 0.0;
                        }
                }
            }
        };
        for (int g0 = 0; g0 < total; g0 += 3) { mstep(0); mstep(1); mstep(2); }
    }

    __syncthreads();
    double* red = ex3_smem;
#pragma unroll
    for (int j = 0; j < NP; ++j) {
        double r = er[j], i = ei[j];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            if (o == 2) continue;
            r += __shfl_xor_sync(0xffffffffu, r, o);
            i += __shfl_xor_sync(0xffffffffu, i, o);
        }
        if (lane == 0 || lane == 2) {
            const int wl = 2 * j + (lane >> 1);
            red[(warp * NWC + wl) * 2] = r; red[(warp * NWC + wl) * 2 + 1] = i;
        }
    }
    __syncthreads();
    if (tid < NWC && w0 + tid < nw) {
        double r = 0.0, i = 0.0;
        for (int x = 0; x < WPC; ++x) { r += red[(x * NWC + tid) * 2]; i += red[(x * NWC + tid) * 2 + 1]; }
        partial[(size_t)u * nw + w0 + tid] = make_double2(r, i);
    }
}

// ---------------------------------------------------------------------------------------------------------------
// The variant for LARGE blocks (the theta blocks of all a-groups of a unit do not fit shared memory: many occupied
// orbitals and/or bands per k-point, e.g. the dense Gamma-point supercell shape of SURVEY.md 8(f) NEXT-4).  The pair
// (ag, bg) of a-groups and a chunk of the gamma-quads move from loops inside the CTA into the grid: a CTA stages only
// the theta rows of its two groups, and a unit contributes NAG^2 * nchunk partial sums (summed by the finalisation).
// ---------------------------------------------------------------------------------------------------------------
template <int NP, int WPC, int MINB>
__global__ void __launch_bounds__(32 * WPC, MINB) exchange3m_big_kernel(
    Dims d, int KS3, int nchunk, int nw, const int* __restrict__ units, const int* __restrict__ kminus, const int* __restrict__ kplus,
    const int* __restrict__ kneg, const double* __restrict__ Lx3, const double2* __restrict__ theta,
    double2* __restrict__ partial) {
    extern __shared__ __align__(16) double ex3_smem[];
    constexpr int NWC = 2 * NP;
    const int nwg = (nw + NWC - 1) / NWC;
    const int npairs = d.NAG * d.NAG;
    // blockIdx.x = ((u * nwg + walker group) * npairs + ab) * nchunk + chunk
    int bx = blockIdx.x;
    const int chunk = bx % nchunk; bx /= nchunk;
    const int ab = bx % npairs; bx /= npairs;
    const int w0 = (bx % nwg) * NWC, u = bx / nwg;
    const int ag = ab / d.NAG, bg = ab % d.NAG;
    // A unit that is its own partner under (Q,k,k2) -> (-Q,k2,k) (multiplicity 1; every unit at the Gamma point) has
    // T2 = T1, so the contributions of the pairs (ag,bg) and (bg,ag) are equal: compute ag <= bg only, twice for ag < bg.
    const bool self_unit = units[4 * u + 3] == 1;
    if (self_unit && ag > bg) {
        if (threadIdx.x < 2 * NP && w0 + (int)threadIdx.x < nw)
            partial[(((size_t)u * npairs + ab) * nchunk + chunk) * nw + w0 + threadIdx.x] = make_double2(0.0, 0.0);
        return;
    }
    const double pair_weight = (self_unit && ag < bg) ? 2.0 : 1.0;
    const int Q = units[4 * u], k = units[4 * u + 1], k2 = units[4 * u + 2];
    const int mQ = kneg[Q];
    const int kq = kminus[k * d.Nk + Q];
    const int k2pq = kplus[k2 * d.Nk + Q];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int GQ = d.GQ, NAG = d.NAG, MS = 3 * KS3;
    (void)NAG;
    constexpr int bs_step = NP * 32;
    const int bs_half = MS * bs_step;
    const size_t task_doubles = (size_t)MS * 64;

    // ---- stage the B fragments of the two a-groups of this CTA: theta rows bg of k2 and rows ag of k ----
    {
        const int per_which = 4 * NWC * 4 * KS3;
        for (int e = tid; e < 2 * per_which; e += 32 * WPC) {
            const int which = e / per_which;
            int x = e - which * per_which;
            const int b = x & 3; x >>= 2;
            const int wl = x % NWC, r = x / NWC;                 // r < 4*KS3
            const int orb = 4 * (which == 0 ? bg : ag) + b, w = w0 + wl;
            const int rowblk = which == 0 ? k2 : k, colblk = which == 0 ? kq : k2pq;
            double2 v = make_double2(0.0, 0.0);
            if (orb < d.n && w < nw && r < d.m)
                v = __ldg(theta + ((size_t)w * d.N + rowblk * d.n + orb) * d.M + (size_t)colblk * d.m + r);
            double* dst = ex3_smem + which * bs_half + ((3 * (r >> 2)) * NP + (wl >> 1)) * 32 + (((wl & 1) * 4 + b) << 2) + (r & 3);
            dst[0] = v.x;
            dst[bs_step] = v.y - v.x;
            dst[2 * bs_step] = v.x + v.y;
        }
    }
    __syncthreads();

    const int q_begin = (int)((long long)chunk * GQ / nchunk), q_end = (int)((long long)(chunk + 1) * GQ / nchunk);
    const int t_begin = q_begin + (int)((long long)warp * (q_end - q_begin) / WPC);
    const int t_end = q_begin + (int)((long long)(warp + 1) * (q_end - q_begin) / WPC);
    const int total = (t_end - t_begin) * MS;
    const int srcl = (lane & ~0x12) | ((lane & 16) >> 3) | ((lane & 2) << 3);
    double er[NP], ei[NP];
#pragma unroll
    for (int j = 0; j < NP; ++j) er[j] = ei[j] = 0.0;

    {
        const double2* la1 = reinterpret_cast<const double2*>(Lx3 + ((((size_t)Q * d.Nk + k) * NAG + ag) * GQ + t_begin) * task_doubles) + lane;
        const double2* la2 = reinterpret_cast<const double2*>(Lx3 + ((((size_t)mQ * d.Nk + k2) * NAG + bg) * GQ + t_begin) * task_doubles) + lane;
        const double* lb1 = ex3_smem + lane;                 // theta rows bg of k2
        const double* lb2 = ex3_smem + bs_half + lane;       // theta rows ag of k
        int ls = 0;
        auto loader_advance = [&]() {
            const bool wrap = ++ls == MS;
            const int db = wrap ? -(MS - 1) * bs_step : bs_step;
            lb1 += db; lb2 += db;
            ls = wrap ? 0 : ls;
        };
        double2 fa1[3], fa2[3];
        double fb1[3][NP], fb2[3][NP];
#pragma unroll
        for (int q = 0; q < 3; ++q) {
            fa1[q] = fa2[q] = make_double2(0.0, 0.0);
            if (total > 0) { fa1[q] = __ldg(la1 + q * 32); fa2[q] = __ldg(la2 + q * 32); }
#pragma unroll
            for (int j = 0; j < NP; ++j) { fb1[q][j] = lb1[j * 32]; fb2[q][j] = lb2[j * 32]; }
            loader_advance();
        }
        la1 += 96; la2 += 96;
        double acc1[3][2][NP][2], acc2[3][2][NP][2];
#pragma unroll
        for (int p = 0; p < 3; ++p)
#pragma unroll
            for (int i = 0; i < 2; ++i)
#pragma unroll
                for (int j = 0; j < NP; ++j)
                    acc1[p][i][j][0] = acc1[p][i][j][1] = acc2[p][i][j][0] = acc2[p][i][j][1] = 0.0;
        int cs = 0;
        auto mstep = [&](const int q) {
#pragma unroll
            for (int j = 0; j < NP; ++j) {
                dmma884(acc1[q][0][j][0], acc1[q][0][j][1], fa1[q].x, fb1[q][j]);
                dmma884(acc1[q][1][j][0], acc1[q][1][j][1], fa1[q].y, fb1[q][j]);
            }
#pragma unroll
            for (int j = 0; j < NP; ++j) {
                dmma884(acc2[q][0][j][0], acc2[q][0][j][1], fb2[q][j], fa2[q].x);
                dmma884(acc2[q][1][j][0], acc2[q][1][j][1], fb2[q][j], fa2[q].y);
            }
            fa1[q] = __ldg(la1); fa2[q] = __ldg(la2);      // may run up to 3 micro-steps past this pair's last task
            la1 += 32; la2 += 32;
#pragma unroll
            for (int j = 0; j < NP; ++j) { fb1[q][j] = lb1[j * 32]; fb2[q][j] = lb2[j * 32]; }
            loader_advance();
            if (q == 2) {
                cs += 3;
                if (cs == MS) {
                    cs = 0;
#pragma unroll
                    for (int i = 0; i < 2; ++i)
#pragma unroll
                        for (int j = 0; j < NP; ++j) {
                            double t1r[2], t1i[2], t2r[2], t2i[2];
#pragma unroll
                            for (int e = 0; e < 2; ++e) {
                                t1r[e] = acc1[0][i][j][e] - acc1[2][i][j][e];
                                t1i[e] = acc1[0][i][j][e] + acc1[1][i][j][e];
                                t2r[e] = acc2[0][i][j][e] - acc2[2][i][j][e];
                                t2i[e] = acc2[0][i][j][e] + acc2[1][i][j][e];
                            }
                            const double pr0 = __shfl_sync(0xffffffffu, t2r[0], srcl), pi0 = __shfl_sync(0xffffffffu, t2i[0], srcl);
                            const double pr1 = __shfl_sync(0xffffffffu, t2r[1], srcl), pi1 = __shfl_sync(0xffffffffu, t2i[1], srcl);
                            er[j] = fma(t1r[0], pr0, er[j]); er[j] = fma(-t1i[0], pi0, er[j]);
                            ei[j] = fma(t1r[0], pi0, ei[j]); ei[j] = fma(t1i[0], pr0, ei[j]);
                            er[j] = fma(t1r[1], pr1, er[j]); er[j] = fma(-t1i[1], pi1, er[j]);
                            ei[j] = fma(t1r[1], pi1, ei[j]); ei[j] = fma(t1i[1], pr1, ei[j]);
#pragma unroll
                            for (int p = 0; p < 3; ++p)
                                acc1[p][i][j][0] = acc1[p][i][j][1] = acc2[p][i][j][0] = acc2[p][i][j][1] = 0.0;
                        }
                }
            }
        };
        for (int g0 = 0; g0 < total; g0 += 3) { mstep(0); mstep(1); mstep(2); }
    }

    __syncthreads();
    double* red = ex3_smem;
#pragma unroll
    for (int j = 0; j < NP; ++j) {
        double r = er[j], i = ei[j];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            if (o == 2) continue;
            r += __shfl_xor_sync(0xffffffffu, r, o);
            i += __shfl_xor_sync(0xffffffffu, i, o);
        }
        if (lane == 0 || lane == 2) {
            const int wl = 2 * j + (lane >> 1);
            red[(warp * NWC + wl) * 2] = r; red[(warp * NWC + wl) * 2 + 1] = i;
        }
    }
    __syncthreads();
    if (tid < NWC && w0 + tid < nw) {
        double r = 0.0, i = 0.0;
        for (int x = 0; x < WPC; ++x) { r += red[(x * NWC + tid) * 2]; i += red[(x * NWC + tid) * 2 + 1]; }
        partial[(((size_t)u * npairs + ab) * nchunk + chunk) * nw + w0 + tid] = make_double2(pair_weight * r, pair_weight * i);
    }
}

template <int NP, int WPC>
int launch_exchange3m_big(afqmc_ctx* c, const double2* theta, int nw, cudaStream_t st) {
    const Dims& d = c->d;
    const int KS3 = (d.m + 3) / 4;
    size_t smem = (size_t)2 * 3 * KS3 * NP * 32 * sizeof(double);
    if (smem < (size_t)WPC * 2 * NP * 2 * sizeof(double)) smem = (size_t)WPC * 2 * NP * 2 * sizeof(double);
    if (smem > (size_t)c->smem_optin) return AFQMC_UNSUPPORTED;
    auto kern = exchange3m_big_kernel<NP, WPC, 1>;
    if (int rc = afqmc_smem_optin(c, (const void*)kern, smem)) return rc;
    const int nwg = (nw + 2 * NP - 1) / (2 * NP), npairs = d.NAG * d.NAG;
    // chunks of gamma-quads: enough CTAs for ~4 waves, every warp keeps at least 2 quads, at most ex_parts_max parts per unit
    int nchunk = (int)((4LL * c->num_sms + (long long)c->nunits * nwg * npairs - 1) / ((long long)c->nunits * nwg * npairs));
    if (nchunk > d.GQ / (2 * WPC)) nchunk = d.GQ / (2 * WPC);
    if (nchunk * npairs > c->ex_parts_max) nchunk = c->ex_parts_max / npairs;
    if (nchunk < 1) nchunk = 1;
    if (npairs * nchunk > c->ex_parts_max) return AFQMC_UNSUPPORTED;
    const long long nblocks = (long long)c->nunits * nwg * npairs * nchunk;
    if (nblocks > 0x7fffffffLL) return AFQMC_UNSUPPORTED;
    kern<<<(unsigned)nblocks, 32 * WPC, smem, st>>>(d, KS3, nchunk, nw, c->units, c->kminus, c->kplus, c->kneg, c->Lx3, theta, c->ws_expart);
    AFQMC_LAUNCH_CHECK(c);
    c->ex_parts = npairs * nchunk;
    return AFQMC_OK;
}

template <int NP, int WPC, int MINB>
int launch_exchange3m_multi(afqmc_ctx* c, const double2* theta, int nw, cudaStream_t st) {
    const Dims& d = c->d;
    const int KS3 = (d.m + 3) / 4;
    size_t smem = (size_t)2 * d.NAG * 3 * KS3 * NP * 32 * sizeof(double);
    if (smem < (size_t)WPC * 2 * NP * 2 * sizeof(double)) smem = (size_t)WPC * 2 * NP * 2 * sizeof(double);
    if (smem > (size_t)c->smem_optin) return AFQMC_UNSUPPORTED;
    auto kern = exchange3m_multi_kernel<NP, WPC, MINB>;
    if (int rc = afqmc_smem_optin(c, (const void*)kern, smem)) return rc;
    const long long nblocks = (long long)((nw + 2 * NP - 1) / (2 * NP)) * c->nunits;
    if (nblocks > 0x7fffffffLL) return AFQMC_UNSUPPORTED;
    kern<<<(unsigned)nblocks, 32 * WPC, smem, st>>>(d, KS3, nw, c->units, c->kminus, c->kplus, c->kneg, c->Lx3, theta, c->ws_expart);
    AFQMC_LAUNCH_CHECK(c);
    return AFQMC_OK;
}

template <int NP, int WPC, int MINB, int DA>
int launch_exchange3m_cfg(afqmc_ctx* c, const double2* theta, int nw, cudaStream_t st) {
    const Dims& d = c->d;
    const int KS3 = (d.m + 3) / 4;
    size_t smem = (size_t)2 * 3 * KS3 * NP * 32 * sizeof(double);
    if (smem < (size_t)WPC * 2 * NP * 2 * sizeof(double)) smem = (size_t)WPC * 2 * NP * 2 * sizeof(double);
    auto kern = exchange3m_kernel<NP, WPC, MINB, DA>;
    if (int rc = afqmc_smem_optin(c, (const void*)kern, smem)) return rc;
    const long long nblocks = (long long)((nw + 2 * NP - 1) / (2 * NP)) * c->nunits;
    if (nblocks > 0x7fffffffLL) return AFQMC_UNSUPPORTED;
    kern<<<(unsigned)nblocks, 32 * WPC, smem, st>>>(d, KS3, nw, c->units, c->kminus, c->kplus, c->kneg, c->Lx3, theta, c->ws_expart);
    AFQMC_LAUNCH_CHECK(c);
    return AFQMC_OK;
}

}  // namespace

// Writes the unit partial sums into ws_expart like the 4M kernel.  Returns AFQMC_UNSUPPORTED (caller falls back to the 4M
// kernel) only if the staged theta blocks do not fit shared memory.
int afqmc_i_exchange3m(afqmc_ctx* c, const double2* theta, int nw, cudaStream_t st) {
    const Dims& d = c->d;
    if (!c->Lx3) return AFQMC_UNSUPPORTED;
    c->ex_parts = 1;
    if (d.NAG != 1) {    // more than four occupied orbitals per k-point
        int rc = nw >= 3 ? launch_exchange3m_multi<2, 2, 6>(c, theta, nw, st) : launch_exchange3m_multi<1, 2, 6>(c, theta, nw, st);
        if (rc == AFQMC_UNSUPPORTED && c->ex_parts_max > 1) {       // blocks too large for one CTA's shared memory
            rc = nw >= 3 ? launch_exchange3m_big<2, 8>(c, theta, nw, st) : AFQMC_UNSUPPORTED;
            if (rc == AFQMC_UNSUPPORTED) rc = launch_exchange3m_big<1, 8>(c, theta, nw, st);
        }
        return rc;
    }
    const int wpc = c->opt_exchange_wpc == 4 ? 4 : 2;
    const bool deep = c->opt_exchange_depth == 6;
    if (nw >= 3) {
        if (deep) return wpc == 4 ? launch_exchange3m_cfg<2, 4, 2, 6>(c, theta, nw, st) : launch_exchange3m_cfg<2, 2, 4, 6>(c, theta, nw, st);
        return wpc == 4 ? launch_exchange3m_cfg<2, 4, 3, 3>(c, theta, nw, st) : launch_exchange3m_cfg<2, 2, 6, 3>(c, theta, nw, st);
    }
    return wpc == 4 ? launch_exchange3m_cfg<1, 4, 3, 3>(c, theta, nw, st) : launch_exchange3m_cfg<1, 2, 6, 3>(c, theta, nw, st);
}
