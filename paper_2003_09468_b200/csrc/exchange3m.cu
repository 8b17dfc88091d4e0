// a9 exchange energy, the default kernel (same contraction as energy.cu; Eq. 49):
//
//     EX = - sum_units mult * X(unit),    unit = (Q,k,k2) ~ (-Q,k2,k)   (SURVEY.md P6 / DESIGN.md R6)
//     X   = sum_{gamma,a,b} T1[(gamma,a),(w,b)] * T2[(gamma,b),(w,a)]
//     T1  = sum_r Lh[ Q][k ][a][gamma][r] * theta_w[(k2,b),(k-Q ,r)]        (the paper's step 2(a))
//     T2  = sum_s Lh[-Q][k2][b][gamma][s] * theta_w[(k ,a),(k2+Q,s)]        (step 2(b), Lbar read from Lh: R4)
//
// Both T's are complex GEMMs  (gamma,orbital) x r  times  r x (walker,orbital)  on the FP64 tensor pipe (DMMA m8n8k4); they never
// leave the SM (the paper keeps them in a user-sized global buffer).  What this kernel does about the pipe:
//
//  * 3M complex product (Gauss):  P0 = (Ar+Ai) Br,  P1 = Ar (Bi-Br),  P2 = Ai (Br+Bi);  Re = P0 - P2,  Im = P0 + P1:
//    three real GEMMs with K = r, 6 real flops per complex multiply-add instead of the 8 of the real embedding.
//  * TAIL in the real embedding.  K = m is covered by k-steps of 4; when m mod 4 is 1 or 2 (m = 26: two left-over r) the last
//    k-step of each product would be at least half padding (3 DMMA k-steps for <= 2 complex r).  Those <= 2 tail elements are
//    instead done as 4M with K = (r, re/im) = 4 reals: ONE A fragment [Ar,Ai,Ar',Ai'] against B = [Br,-Bi,Br',-Bi'] (accumulated
//    into P0: adds Re t) and against B = [Bi-Br, Br+Bi, ...] (into P1: adds Im t - Re t), i.e. 2 k-steps instead of 3 and
//    Re = P0 - P2, Im = P0 + P1 still hold.  m = 26: 20 DMMA k-steps per task and tile pair instead of 21 (26 of 26.67 useful).
//  * The static operand is stored COMPLEX (Re, Im per lane; Ar+Ai is one DADD per fragment, as in tgemm.cuh): 2/3 of the bytes
//    and of the load wavefronts of a layout that stores the three A variants, so the register prefetch ring holds DA whole
//    k-steps (3 products each) and covers the L2 latency of the stream (the r01 kernel ran 1 k-step ahead and lost 14 % of its
//    issue slots to that, profiles/r01g).
//  * A warp computes ONE of T1 / T2 (role h = warp & 1); the two warps of a pair meet once per task (gamma-quad): each hands
//    one of its two m-tiles to the partner through shared memory (which also does the (a,b) transpose) and contracts the
//    other one.  Half the accumulators per warp (3 products x 2 m-tiles x NP n-tiles) of a kernel that keeps T1 and T2 in
//    one warp: more resident warps per scheduler, or NP = 4 (eight walkers per CTA: every A fragment feeds four n-tiles).
//
// Operand layout (written once in afqmc_create from Lh, see pack_Lxc_kernel):
//   Lxc[Q][k][ag][gq][ks < KSPT][lane][4]   lane = (row << 2) | kk;  tile i rows: gamma = 4 gq + 2 i + (row >> 2), a = 4 ag + (row & 3)
//     full k-step ks < KSF:  r = 4 ks + kk;  doubles = (Re, Im of tile 0, Re, Im of tile 1)
//     tail k-step ks = KSF:  r = 4 KSF + (kk >> 1), part = kk & 1;  doubles = (part of tile 0, part of tile 1, 0, 0)
//   one coalesced 1 KB access per k-step and warp, consecutive in memory across k-steps and tasks; zeros outside.
// theta blocks are staged once per CTA in shared memory in B-fragment order, already expanded into the three B variants.
#include <type_traits>
#include "common.cuh"

namespace {

struct X3Geom { int KSF, TAIL, KSPT, MSPT; };
// k-steps of a task: KSF full ones (3 micro-steps = products each) + TAIL (0/1) real-embedded one (2 micro-steps)
__host__ __device__ inline X3Geom x3_geom(int m) {
    X3Geom g;
    const int mr = m & 3;
    g.TAIL = (mr == 1 || mr == 2) ? 1 : 0;
    g.KSF = g.TAIL ? m / 4 : (m + 3) / 4;
    g.KSPT = g.KSF + g.TAIL;
    g.MSPT = 3 * g.KSF + 2 * g.TAIL;
    return g;
}

__global__ void pack_Lxc_kernel(Dims d, X3Geom g, const double2* __restrict__ Lh, double* __restrict__ Lxc, size_t total_in,
                                size_t total_out) {
    // one thread per (.., ks, lane, tile i)
    for (size_t idx = blockIdx.x * (size_t)blockDim.x + threadIdx.x; idx < total_in; idx += (size_t)gridDim.x * blockDim.x) {
        size_t t = idx;
        const int i = (int)(t & 1); t >>= 1;
        const int lane = (int)(t & 31); t >>= 5;
        const int ks = (int)(t % g.KSPT); t /= g.KSPT;
        const int gq = (int)(t % d.GQ); t /= d.GQ;
        const int ag = (int)(t % d.NAG); t /= d.NAG;
        const int k = (int)(t % d.Nk);
        const int Q = (int)(t / d.Nk);
        const int row = lane >> 2, kk = lane & 3;
        const int gam = 4 * gq + 2 * i + (row >> 2), a = 4 * ag + (row & 3);
        const bool full = ks < g.KSF;
        const int r = full ? 4 * ks + kk : 4 * g.KSF + (kk >> 1);
        double2 z = make_double2(0.0, 0.0);
        if (a < d.n && gam < d.nchol && r < d.m) z = Lh[((((size_t)Q * d.Nk + k) * d.n + a) * d.nchol + gam) * d.m + r];
        double* out = Lxc + (idx >> 6) * 128 + lane * 4;        // (idx >> 6) = the k-step's linear index
        if (full) {
            out[2 * i] = z.x;
            out[2 * i + 1] = z.y;
        } else {
            out[i] = (kk & 1) ? z.y : z.x;
            out[2 + i] = 0.0;
        }
    }
    // zero pad after the last block (the register prefetch runs up to DA k-steps past a warp's last task)
    const size_t body = total_in * 2;
    for (size_t idx = body + blockIdx.x * (size_t)blockDim.x + threadIdx.x; idx < total_out; idx += (size_t)gridDim.x * blockDim.x)
        Lxc[idx] = 0.0;
}

}  // namespace

size_t afqmc_i_lxc_doubles(const Dims& d) {
    const X3Geom g = x3_geom(d.m);
    return (size_t)d.Nk * d.Nk * d.NAG * d.GQ * g.KSPT * 128 + AFQMC_LX_PAD;
}

int afqmc_i_pack_lxc(afqmc_ctx* c, cudaStream_t st) {
    const Dims& d = c->d;
    const X3Geom g = x3_geom(d.m);
    const size_t total_in = (size_t)d.Nk * d.Nk * d.NAG * d.GQ * g.KSPT * 64;
    size_t nb = (total_in + 255) / 256;
    if (nb > 148 * 64) nb = 148 * 64;
    pack_Lxc_kernel<<<(unsigned)nb, 256, 0, st>>>(d, g, c->Lh, c->Lxc, total_in, afqmc_i_lxc_doubles(d));
    AFQMC_LAUNCH_CHECK(c);
    return AFQMC_OK;
}

namespace {

// B fragments of NP n-tiles for one lane and micro-step sit next to each other: [ms][jp][lane][W], W = min(NP,2) doubles
template <int NP> struct BVec { static constexpr int W = NP >= 2 ? 2 : 1, NPH = NP / W; };

// CTA = (unit, group of 2*NP walkers[, pair of a-groups, chunk of gamma-quads]); 2*NPAIR warps; see the header comment.
//   GRIDPAIRS = false: the theta blocks of ALL a-groups are staged and the CTA loops over the (ag,bg) pairs (n <= 4: one pair);
//   GRIDPAIRS = true : the (ag,bg) pair and a chunk of the gamma-quads come from the grid and only the theta rows of those two
//                      groups are staged (blocks too large for shared memory: many orbitals / bands per k-point, e.g. the
//                      Gamma-point supercell shape); a unit then contributes NAG^2 * nchunk partial sums.
// DA = k-steps of register prefetch of the Lxc stream (L2 resident); the B fragments (shared memory) run one k-step ahead.
template <int NP, int NPAIR, int DA, int MINB, bool GRIDPAIRS>
__global__ void __launch_bounds__(64 * NPAIR, MINB) exchange3m_kernel(
    Dims d, X3Geom g, int nchunk, int nw, const int* __restrict__ units, const int* __restrict__ kminus,
    const int* __restrict__ kplus, const int* __restrict__ kneg, const double* __restrict__ Lxc,
    const double2* __restrict__ theta, double2* __restrict__ partial) {
    extern __shared__ __align__(16) double x3_smem[];
    constexpr int NWC = 2 * NP, NWARP = 2 * NPAIR, NBUF = 2;
    constexpr int W = BVec<NP>::W, NPH = BVec<NP>::NPH;
    const int nwg = (nw + NWC - 1) / NWC;            // walker groups of one unit are adjacent in the grid
    const int NAG = d.NAG, GQ = d.GQ, npairs = NAG * NAG;
    int bx = blockIdx.x, chunk = 0, ab0 = 0, ab1 = npairs;
    if (GRIDPAIRS) {                                  // blockIdx.x = ((u * nwg + walker group) * npairs + ab) * nchunk + chunk
        chunk = bx % nchunk; bx /= nchunk;
        ab0 = bx % npairs; bx /= npairs;
        ab1 = ab0 + 1;
    }
    const int w0 = (bx % nwg) * NWC, u = bx / nwg;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, pair = warp >> 1, h = warp & 1;
    double pair_weight = 1.0;
    if (GRIDPAIRS) {
        // A unit that is its own partner under (Q,k,k2) -> (-Q,k2,k) (multiplicity 1; every unit at the Gamma point) has
        // T2 = T1, so the pairs (ag,bg) and (bg,ag) contribute equally: compute ag <= bg only, twice for ag < bg.
        const int ag = ab0 / NAG, bg = ab0 % NAG;
        const bool self_unit = units[4 * u + 3] == 1;
        if (self_unit && ag > bg) {
            if (tid < NWC && w0 + tid < nw)
                partial[(((size_t)u * npairs + ab0) * nchunk + chunk) * nw + w0 + tid] = make_double2(0.0, 0.0);
            return;
        }
        if (self_unit && ag < bg) pair_weight = 2.0;
    }
    const int Q = units[4 * u], k = units[4 * u + 1], k2 = units[4 * u + 2];
    const int mQ = kneg[Q];
    const int kq = kminus[k * d.Nk + Q];        // k - Q   : column block of theta for T1
    const int k2pq = kplus[k2 * d.Nk + Q];      // k2 + Q  : column block of theta for T2
    const int NGS = GRIDPAIRS ? 1 : NAG;        // a-group slots staged per theta block
    constexpr int bs_step = 32 * NP;            // doubles of one micro-step
    const int bs_grp = (g.MSPT + 1) * bs_step;  // +1: the k-step before a tail prefetches a third micro-step that does not exist
    const int bs_half = NGS * bs_grp;
    double* Bs = x3_smem;                       // Bs[which][slot][ms][jp][lane][W]: which 0 -> theta[(k2,b),(k-Q,r)], 1 -> theta[(k,a),(k2+Q,s)]
    double2* xbuf = reinterpret_cast<double2*>(x3_smem + 2 * bs_half);      // [pair][role][NBUF][NP][64] hand-over tiles

    // ---- this warp's share of the gamma-quads (both warps of a pair walk the same tasks) ----
    const int q_begin = (int)((long long)chunk * GQ / nchunk), q_end = (int)((long long)(chunk + 1) * GQ / nchunk);
    const int t_begin = q_begin + (int)((long long)pair * (q_end - q_begin) / NPAIR);
    const int t_end = q_begin + (int)((long long)(pair + 1) * (q_end - q_begin) / NPAIR);
    const int total = (t_end - t_begin) * g.KSPT;                 // k-steps of this warp per (ag,bg) pair
    const size_t blk = h == 0 ? (size_t)Q * d.Nk + k : (size_t)mQ * d.Nk + k2;
    auto stream_ptr = [&](int grp) {            // 2 double2 per lane and k-step; k-step stride 64 double2
        return reinterpret_cast<const double2*>(Lxc + (((blk * NAG + grp) * GQ + t_begin) * (size_t)g.KSPT) * 128) + lane * 2;
    };
    double2 fa[DA][2];
    const double2* pa = stream_ptr(h == 0 ? ab0 / NAG : ab0 % NAG);
    // prologue of the first pair's A stream: issued before the staging below, which hides the L2 round trip
#pragma unroll
    for (int q = 0; q < DA; ++q) {
        fa[q][0] = fa[q][1] = make_double2(0.0, 0.0);
        if (total > 0) { fa[q][0] = __ldg(pa + q * 64); fa[q][1] = __ldg(pa + q * 64 + 1); }
    }

    // ---- stage the B fragments: one thread per complex theta element (orbital, walker, r) ----
    //   lane of a B fragment = (col << 2) | kk,  col = 4*(w&1) + orbital;  n-tile j = walker >> 1
    {
        const int RP = 4 * g.KSF + 2 * g.TAIL;
        const int per_which = NGS * 4 * NWC * RP;
        for (int e = tid; e < 2 * per_which; e += 64 * NPAIR) {
            const int which = e / per_which;
            int x = e - which * per_which;
            const int b = x & 3; x >>= 2;
            const int wl = x % NWC; x /= NWC;
            const int gs = x % NGS, r = x / NGS;
            const int grp = GRIDPAIRS ? (which == 0 ? ab0 % NAG : ab0 / NAG) : gs;
            const int orb = 4 * grp + b, w = w0 + wl;
            const int rowblk = which == 0 ? k2 : k, colblk = which == 0 ? kq : k2pq;
            double2 v = make_double2(0.0, 0.0);
            if (orb < d.n && w < nw && r < d.m)
                v = __ldg(theta + ((size_t)w * d.N + rowblk * d.n + orb) * d.M + (size_t)colblk * d.m + r);
            const int j = wl >> 1, col = (wl & 1) * 4 + b;
            double* base = Bs + which * bs_half + gs * bs_grp + (j / W) * (32 * W) + (j % W);    // + ms * bs_step + lane * W
            if (r < 4 * g.KSF) {
                double* dst = base + 3 * (r >> 2) * bs_step + ((col << 2) | (r & 3)) * W;
                dst[0] = v.x;                       // Br
                dst[bs_step] = v.y - v.x;           // Bi - Br
                dst[2 * bs_step] = v.x + v.y;       // Br + Bi
            } else {                                // tail: real embedding, lanes kk = 2t (times Ar) and 2t+1 (times Ai)
                double* dst = base + 3 * g.KSF * bs_step + ((col << 2) | (2 * (r - 4 * g.KSF))) * W;
                dst[0] = v.x;  dst[W] = -v.y;                               // -> P0:  Ar Br - Ai Bi
                dst[bs_step] = v.y - v.x;  dst[bs_step + W] = v.x + v.y;    // -> P1:  Ar (Bi-Br) + Ai (Br+Bi)
            }
        }
    }
    __syncthreads();   // B fragments staged

    // lane geometry of a C fragment (row = lane>>2, columns 2c+e, c = lane&3, register e):
    //   rows (gl = row>>2: gamma of the tile's pair, orow = row&3: this warp's ROW orbital), columns (wp = c>>1: walker of the
    //   pair, ocol = 2(c&1)+e: the COLUMN orbital).  T1: orow = a, ocol = b;  T2: orow = b, ocol = a.
    const int gl = lane >> 4, orow = (lane >> 2) & 3, wp = (lane >> 1) & 1, cb = lane & 1;
    const int idx_w = gl * 32 + orow * 8 + wp * 4 + 2 * cb;       // hand-over slot of (this lane, e = 0); e = 1 is the next one
    const int idx_r = gl * 32 + (2 * cb) * 8 + wp * 4 + orow;     // partner element [(gamma, ocol), (w, orow)] for e = 0; e = 1: + 8
    double er[NP], ei[NP];
#pragma unroll
    for (int j = 0; j < NP; ++j) er[j] = ei[j] = 0.0;
    int buf = 0;

    for (int ab = ab0; ab < ab1; ++ab) {
        const int ag = ab / NAG, bg = ab % NAG;
        if (ab != ab0) {                         // next pair of a-groups: restart the A stream
            pa = stream_ptr(h == 0 ? ag : bg);
#pragma unroll
            for (int q = 0; q < DA; ++q)
                if (total > 0) { fa[q][0] = __ldg(pa + q * 64); fa[q][1] = __ldg(pa + q * 64 + 1); }
        }
        pa += DA * 64;
        // T1 needs theta rows bg of k2 (which 0), T2 theta rows ag of k (which 1)
        const double* pb = Bs + h * bs_half + (GRIDPAIRS ? 0 : (h == 0 ? bg : ag)) * bs_grp + lane * W;
        double fb[3][NP];
        auto load_b = [&](const int p, const int ms0) {       // B fragments of micro-step ms0 + p into buffer p
            const double* src = pb + (ms0 + p) * bs_step;
#pragma unroll
            for (int jp = 0; jp < NPH; ++jp) {
                if (W == 2) {
                    const double2 v = *reinterpret_cast<const double2*>(src + jp * 64);
                    fb[p][2 * jp] = v.x; fb[p][2 * jp + (NP > 1 ? 1 : 0)] = v.y;
                } else {
                    fb[p][jp] = src[jp * 32];
                }
            }
        };
        load_b(0, 0); load_b(1, 0); load_b(2, 0);
        double acc[3][2][NP][2];
#pragma unroll
        for (int p = 0; p < 3; ++p)
#pragma unroll
            for (int i = 0; i < 2; ++i)
#pragma unroll
                for (int j = 0; j < NP; ++j) acc[p][i][j][0] = acc[p][i][j][1] = 0.0;

        // end of a task: combine the three products, hand tile GIVE to the partner warp, contract tile KEEP
        auto finish_task = [&](auto KEEP_) {
            constexpr int KEEP = decltype(KEEP_)::value, GIVE = 1 - KEEP;
            double2* xw = xbuf + (((pair * 2 + h) * NBUF + buf) * NP) * 64 + idx_w;
#pragma unroll
            for (int j = 0; j < NP; ++j) {
                xw[j * 64] = make_double2(acc[0][GIVE][j][0] - acc[2][GIVE][j][0], acc[0][GIVE][j][0] + acc[1][GIVE][j][0]);
                xw[j * 64 + 1] = make_double2(acc[0][GIVE][j][1] - acc[2][GIVE][j][1], acc[0][GIVE][j][1] + acc[1][GIVE][j][1]);
            }
            asm volatile("bar.sync %0, 64;" ::"r"(pair + 1) : "memory");       // the two warps of the pair
            const double2* xr = xbuf + (((pair * 2 + (h ^ 1)) * NBUF + buf) * NP) * 64 + idx_r;
#pragma unroll
            for (int j = 0; j < NP; ++j)
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const double tr = acc[0][KEEP][j][e] - acc[2][KEEP][j][e], ti = acc[0][KEEP][j][e] + acc[1][KEEP][j][e];
                    const double2 p = xr[j * 64 + e * 8];
                    er[j] = fma(tr, p.x, er[j]); er[j] = fma(-ti, p.y, er[j]);
                    ei[j] = fma(tr, p.y, ei[j]); ei[j] = fma(ti, p.x, ei[j]);
                }
#pragma unroll
            for (int p = 0; p < 3; ++p)
#pragma unroll
                for (int i = 0; i < 2; ++i)
#pragma unroll
                    for (int j = 0; j < NP; ++j) acc[p][i][j][0] = acc[p][i][j][1] = 0.0;
            buf ^= 1;      // two hand-over buffers: the partner may still read this one while the next task is written
        };

        int cs = 0;   // k-step of the compute state inside its task
        auto kstep = [&](auto Q_) {
            constexpr int q = decltype(Q_)::value;
            const double2 x0 = fa[q][0], x1 = fa[q][1];
            const int nxt = (cs + 1 == g.KSPT) ? 0 : 3 * (cs + 1);      // first micro-step of the next k-step (wraps at the task end)
            if (cs < g.KSF) {
                const double s0 = x0.x + x0.y, s1 = x1.x + x1.y;        // Ar + Ai
#pragma unroll
                for (int j = 0; j < NP; ++j) {
                    dmma884(acc[0][0][j][0], acc[0][0][j][1], s0, fb[0][j]);
                    dmma884(acc[0][1][j][0], acc[0][1][j][1], s1, fb[0][j]);
                }
                load_b(0, nxt);
#pragma unroll
                for (int j = 0; j < NP; ++j) {
                    dmma884(acc[1][0][j][0], acc[1][0][j][1], x0.x, fb[1][j]);
                    dmma884(acc[1][1][j][0], acc[1][1][j][1], x1.x, fb[1][j]);
                }
                load_b(1, nxt);
#pragma unroll
                for (int j = 0; j < NP; ++j) {
                    dmma884(acc[2][0][j][0], acc[2][0][j][1], x0.y, fb[2][j]);
                    dmma884(acc[2][1][j][0], acc[2][1][j][1], x1.y, fb[2][j]);
                }
                load_b(2, nxt);
            } else {                                                     // tail k-step: x0 = (tile 0, tile 1) real-embedded
#pragma unroll
                for (int j = 0; j < NP; ++j) {
                    dmma884(acc[0][0][j][0], acc[0][0][j][1], x0.x, fb[0][j]);
                    dmma884(acc[0][1][j][0], acc[0][1][j][1], x0.y, fb[0][j]);
                }
                load_b(0, nxt);
#pragma unroll
                for (int j = 0; j < NP; ++j) {
                    dmma884(acc[1][0][j][0], acc[1][0][j][1], x0.x, fb[1][j]);
                    dmma884(acc[1][1][j][0], acc[1][1][j][1], x0.y, fb[1][j]);
                }
                load_b(1, nxt);
                load_b(2, nxt);
            }
            // refill this ring slot with the k-step DA ahead (may run past the warp's last task: loaded, never used)
            fa[q][0] = __ldg(pa); fa[q][1] = __ldg(pa + 1);
            pa += 64;
            if (++cs == g.KSPT) {
                cs = 0;
                if (h == 0) finish_task(std::integral_constant<int, 0>());
                else finish_task(std::integral_constant<int, 1>());
            }
        };
        const int nfull = total - total % DA;
        for (int g0 = 0; g0 < nfull; g0 += DA) {
            kstep(std::integral_constant<int, 0>());
            if (DA > 1) kstep(std::integral_constant<int, 1 % DA>());
            if (DA > 2) kstep(std::integral_constant<int, 2 % DA>());
            if (DA > 3) kstep(std::integral_constant<int, 3 % DA>());
        }
        if (nfull + 0 < total) kstep(std::integral_constant<int, 0>());
        if (DA > 2 && nfull + 1 < total) kstep(std::integral_constant<int, 1 % DA>());
        if (DA > 3 && nfull + 2 < total) kstep(std::integral_constant<int, 2 % DA>());
    }

    // ---- reduce over the lanes of each walker-in-pair (lane bit 1 = wp), then over warps (deterministic) ----
    __syncthreads();
    double* red = x3_smem;   // reuse: [warp][NWC][2]
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
        for (int x = 0; x < NWARP; ++x) { r += red[(x * NWC + tid) * 2]; i += red[(x * NWC + tid) * 2 + 1]; }
        const size_t slot = GRIDPAIRS ? ((size_t)u * npairs + ab0) * nchunk + chunk : (size_t)u;
        partial[slot * nw + w0 + tid] = make_double2(pair_weight * r, pair_weight * i);
    }
}

template <int NP>
size_t x3_smem_bytes(const X3Geom& g, int NGS, int NPAIR) {
    const size_t bs = (size_t)2 * NGS * (g.MSPT + 1) * 32 * NP * sizeof(double);
    const size_t xb = (size_t)NPAIR * 2 * 2 * NP * 64 * sizeof(double2);
    return bs + xb;
}

template <int NP, int NPAIR, int DA, int MINB, bool GRIDPAIRS>
int launch_x3(afqmc_ctx* c, const double2* theta, int nw, cudaStream_t st) {
    const Dims& d = c->d;
    const X3Geom g = x3_geom(d.m);
    const size_t smem = x3_smem_bytes<NP>(g, GRIDPAIRS ? 1 : d.NAG, NPAIR);
    auto kern = exchange3m_kernel<NP, NPAIR, DA, MINB, GRIDPAIRS>;
    if (int rc = afqmc_smem_optin(c, (const void*)kern, smem)) return rc;
    const int nwg = (nw + 2 * NP - 1) / (2 * NP), npairs = d.NAG * d.NAG;
    int nchunk = 1;
    long long nblocks = (long long)c->nunits * nwg;
    if (GRIDPAIRS) {
        // chunks of gamma-quads: enough CTAs for ~4 waves, every warp pair keeps at least 2 quads, at most ex_parts_max parts per unit
        nchunk = (int)((4LL * c->num_sms + nblocks * npairs - 1) / (nblocks * npairs));
        if (nchunk > d.GQ / (2 * NPAIR)) nchunk = d.GQ / (2 * NPAIR);
        if (nchunk * npairs > c->ex_parts_max) nchunk = c->ex_parts_max / npairs;
        if (nchunk < 1) nchunk = 1;
        if (npairs * nchunk > c->ex_parts_max) return AFQMC_UNSUPPORTED;
        nblocks *= (long long)npairs * nchunk;
    }
    if (nblocks > 0x7fffffffLL) return AFQMC_UNSUPPORTED;
    kern<<<(unsigned)nblocks, 64 * NPAIR, smem, st>>>(d, g, nchunk, nw, c->units, c->kminus, c->kplus, c->kneg, c->Lxc, theta, c->ws_expart);
    AFQMC_LAUNCH_CHECK(c);
    c->ex_parts = GRIDPAIRS ? npairs * nchunk : 1;
    return AFQMC_OK;
}

// n-tiles per warp: 2 (four walkers per CTA) unless there are at most two walkers; 4 (eight walkers per CTA) on request
template <int NPAIR, int DA, bool GRIDPAIRS>
int launch_x3_np(afqmc_ctx* c, const double2* theta, int nw, cudaStream_t st) {
    int np = c->opt_exchange_np;
    if (np == 0) np = nw <= 2 ? 1 : 2;
    // resident CTAs asked of the compiler: the register budget per thread is 65536 / (MINB * 64 * NPAIR)
    if (np == 1) return launch_x3<1, NPAIR, DA, (NPAIR == 1 ? 8 : 4), GRIDPAIRS>(c, theta, nw, st);
    if (np == 4) return launch_x3<4, NPAIR, (DA > 2 ? 2 : DA), (NPAIR == 1 ? 5 : 2), GRIDPAIRS>(c, theta, nw, st);
    return launch_x3<2, NPAIR, DA, (NPAIR == 1 ? 7 : 3), GRIDPAIRS>(c, theta, nw, st);
}

template <bool GRIDPAIRS>
int launch_x3_cfg(afqmc_ctx* c, const double2* theta, int nw, cudaStream_t st) {
    const bool two_pairs = GRIDPAIRS || c->opt_exchange_wpc == 4;         // option "exchange_warps" = 4: two warp pairs per CTA
    const int da = c->opt_exchange_depth == 2 ? 2 : 3;                     // option "exchange_depth": k-steps of A prefetch
    if (two_pairs) return da == 2 ? launch_x3_np<2, 2, GRIDPAIRS>(c, theta, nw, st) : launch_x3_np<2, 3, GRIDPAIRS>(c, theta, nw, st);
    return da == 2 ? launch_x3_np<1, 2, GRIDPAIRS>(c, theta, nw, st) : launch_x3_np<1, 3, GRIDPAIRS>(c, theta, nw, st);
}

}  // namespace

// Partial sums per unit that ws_expart must hold: 1, or NAG^2 * (up to 8 chunks) when the theta blocks of all a-groups do not
// fit one CTA's shared memory (then the (ag,bg) pairs and chunks of gamma-quads are spread over the grid).
int afqmc_i_exchange3m_parts_max(const afqmc_ctx* c) {
    const Dims& d = c->d;
    if (d.NAG == 1) return 1;
    return x3_smem_bytes<2>(x3_geom(d.m), d.NAG, 1) > (size_t)c->smem_optin ? d.NAG * d.NAG * 8 : 1;
}

// Writes the unit partial sums into ws_expart (ex_parts per unit) for energy_finalize_kernel.  Returns AFQMC_UNSUPPORTED only
// if even the theta rows of two a-groups do not fit shared memory.
int afqmc_i_exchange3m(afqmc_ctx* c, const double2* theta, int nw, cudaStream_t st) {
    c->ex_parts = 1;
    int rc = launch_x3_cfg<false>(c, theta, nw, st);
    if (rc == AFQMC_UNSUPPORTED && c->d.NAG > 1 && c->ex_parts_max > 1) rc = launch_x3_cfg<true>(c, theta, nw, st);
    return rc;
}
