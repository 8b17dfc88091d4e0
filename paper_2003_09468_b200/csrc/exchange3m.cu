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
//  * m <= 28 (exchange3m_reg_kernel): a warp's theta block is only MSPT * NP <= 42 fragments per lane, so it is read from shared
//    memory ONCE per (CTA, a-group pair) and stays in REGISTERS for all gamma-quads; the task (KSF, TAIL are template parameters)
//    is fully unrolled, and the inner loop is LDG.128 (A) + DADD + DMMA only: no shared-memory traffic per micro-step (the
//    generic kernel's B loads were 29 % of its LSU wavefronts, LSU 70 % busy in an ncu capture of this round).
#include <type_traits>
#include "common.cuh"


namespace {

struct X3Geom { int KSF, TAIL, KSPT, MSPT, PV; };      // PV = real products (micro-steps) per full k-step: 3, or 2 for a real operand
// k-steps of a task: KSF full ones (3 micro-steps = products each) + TAIL (0/1) real-embedded one (2 micro-steps)
__host__ __device__ inline X3Geom x3_geom(int m) {
    X3Geom g;
    const int mr = m & 3;
    g.TAIL = (mr == 1 || mr == 2) ? 1 : 0;
    g.KSF = g.TAIL ? m / 4 : (m + 3) / 4;
    g.KSPT = g.KSF + g.TAIL;
    g.MSPT = 3 * g.KSF + 2 * g.TAIL;
    g.PV = 3;
    return g;
}
// real operand (real orbitals): K = r in k-steps of 4, no tail trick, two products per k-step (Ar Br, Ar Bi)
__host__ __device__ inline X3Geom x3_geom_real(int m) {
    X3Geom g;
    g.TAIL = 0; g.KSF = (m + 3) / 4; g.KSPT = g.KSF; g.MSPT = 2 * g.KSF; g.PV = 2;
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

static int pack_lxc(afqmc_ctx* c, cudaStream_t st) {
    const Dims& d = c->d;
    const X3Geom g = x3_geom(d.m);
    const size_t total_in = (size_t)d.Nk * d.Nk * d.NAG * d.GQ * g.KSPT * 64;
    size_t nb = (total_in + 255) / 256;
    if (nb > 148 * 64) nb = 148 * 64;
    pack_Lxc_kernel<<<(unsigned)nb, 256, 0, st>>>(d, g, c->Lh, c->Lxc, total_in, afqmc_i_lxc_doubles(d));
    AFQMC_LAUNCH_CHECK(c);
    return AFQMC_OK;
}

// Lxr (real orbitals, generic kernel): the REAL parts only,  Lxr[Q][k][ag][gq][ks < ceil(m/4)][lane][2] = (tile 0, tile 1) at
// r = 4 ks + kk: half the bytes of Lxc, one LDG.128 per k-step and lane
namespace {
__global__ void pack_Lxr_kernel(Dims d, int KSF, const double2* __restrict__ Lh, double* __restrict__ Lxr, size_t total_in, size_t total_out) {
    for (size_t idx = blockIdx.x * (size_t)blockDim.x + threadIdx.x; idx < total_in; idx += (size_t)gridDim.x * blockDim.x) {
        size_t t = idx;
        const int i = (int)(t & 1); t >>= 1;
        const int lane = (int)(t & 31); t >>= 5;
        const int ks = (int)(t % KSF); t /= KSF;
        const int gq = (int)(t % d.GQ); t /= d.GQ;
        const int ag = (int)(t % d.NAG); t /= d.NAG;
        const int k = (int)(t % d.Nk);
        const int Q = (int)(t / d.Nk);
        const int row = lane >> 2, r = 4 * ks + (lane & 3);
        const int gam = 4 * gq + 2 * i + (row >> 2), a = 4 * ag + (row & 3);
        Lxr[idx] = (a < d.n && gam < d.nchol && r < d.m) ? Lh[((((size_t)Q * d.Nk + k) * d.n + a) * d.nchol + gam) * d.m + r].x : 0.0;
    }
    for (size_t idx = total_in + blockIdx.x * (size_t)blockDim.x + threadIdx.x; idx < total_out; idx += (size_t)gridDim.x * blockDim.x) Lxr[idx] = 0.0;
}
}  // namespace

static int ensure_lxr(afqmc_ctx* c, cudaStream_t st) {
    if (c->Lxr) return AFQMC_OK;
    const Dims& d = c->d;
    const X3Geom g = x3_geom_real(d.m);
    const size_t total_in = (size_t)d.Nk * d.Nk * d.NAG * d.GQ * g.KSF * 64, total_out = total_in + AFQMC_LX_PAD;
    if (cudaMalloc((void**)&c->Lxr, total_out * sizeof(double)) != cudaSuccess) { (void)cudaGetLastError(); c->Lxr = nullptr; return AFQMC_OUT_OF_MEMORY; }
    size_t nb = (total_in + 255) / 256;
    if (nb > 148 * 64) nb = 148 * 64;
    pack_Lxr_kernel<<<(unsigned)nb, 256, 0, st>>>(d, g.KSF, c->Lh, c->Lxr, total_in, total_out);
    AFQMC_LAUNCH_CHECK(c);
    return AFQMC_OK;
}

// Lx3t (m <= 28, exchange3m_reg_kernel): the three A variants STORED, so that the inner loop has no DADD (one FP64 add between
// DMMAs costs the pipe 7-8 cycles, measured: profiles/r02b_ncu_force_bias.md, profiles/r02c_ncu_exchange.md):
//   Lx3t[Q][k][ag][gq][ml < 3 KSF + TAIL][lane][2]   ml = 3 ks + p: variant p (0: Re+Im, 1: Re, 2: Im) of tiles 0,1 at r = 4 ks + kk;
//   ml = 3 KSF (tail): the real-embedded fragment of tiles 0,1 (as in Lxc).  One coalesced 512-byte LDG.128 per micro-step.
namespace {
__global__ void pack_Lx3t_kernel(Dims d, X3Geom g, const double2* __restrict__ Lh, double* __restrict__ Lx3t, size_t total_in,
                                 size_t total_out) {
    const int MST = 3 * g.KSF + g.TAIL;
    for (size_t idx = blockIdx.x * (size_t)blockDim.x + threadIdx.x; idx < total_in; idx += (size_t)gridDim.x * blockDim.x) {
        size_t t = idx;
        const int i = (int)(t & 1); t >>= 1;
        const int lane = (int)(t & 31); t >>= 5;
        const int ml = (int)(t % MST); t /= MST;
        const int gq = (int)(t % d.GQ); t /= d.GQ;
        const int ag = (int)(t % d.NAG); t /= d.NAG;
        const int k = (int)(t % d.Nk);
        const int Q = (int)(t / d.Nk);
        const int row = lane >> 2, kk = lane & 3;
        const int gam = 4 * gq + 2 * i + (row >> 2), a = 4 * ag + (row & 3);
        const bool full = ml < 3 * g.KSF;
        const int r = full ? 4 * (ml / 3) + kk : 4 * g.KSF + (kk >> 1);
        double2 z = make_double2(0.0, 0.0);
        if (a < d.n && gam < d.nchol && r < d.m) z = Lh[((((size_t)Q * d.Nk + k) * d.n + a) * d.nchol + gam) * d.m + r];
        const int p = ml % 3;
        Lx3t[idx] = full ? (p == 0 ? z.x + z.y : (p == 1 ? z.x : z.y)) : ((kk & 1) ? z.y : z.x);
    }
    for (size_t idx = total_in + blockIdx.x * (size_t)blockDim.x + threadIdx.x; idx < total_out; idx += (size_t)gridDim.x * blockDim.x)
        Lx3t[idx] = 0.0;
}
}  // namespace

static size_t lx3t_doubles(const Dims& d) {
    const X3Geom g = x3_geom(d.m);
    return (size_t)d.Nk * d.Nk * d.NAG * d.GQ * (3 * g.KSF + g.TAIL) * 64 + AFQMC_LX_PAD;
}

static int pack_lx3t(afqmc_ctx* c, cudaStream_t st) {
    const Dims& d = c->d;
    const X3Geom g = x3_geom(d.m);
    const size_t total_out = lx3t_doubles(d), total_in = total_out - AFQMC_LX_PAD;
    size_t nb = (total_in + 255) / 256;
    if (nb > 148 * 64) nb = 148 * 64;
    pack_Lx3t_kernel<<<(unsigned)nb, 256, 0, st>>>(d, g, c->Lh, c->Lx3t, total_in, total_out);
    AFQMC_LAUNCH_CHECK(c);
    return AFQMC_OK;
}

// Which operand the default path streams: Lx3t when a warp's theta block fits registers (m <= 28), else Lxc.  The other one is
// packed from Lh the first time an option or a shape (too many orbitals for the staging buffers) asks for its kernel.
static bool x3_prefers_reg(const Dims& d) { return x3_geom(d.m).MSPT <= 21; }

static int ensure_operand(afqmc_ctx* c, bool reg, cudaStream_t st) {
    if (reg) {
        if (c->Lx3t) return AFQMC_OK;
        if (cudaMalloc((void**)&c->Lx3t, lx3t_doubles(c->d) * sizeof(double)) != cudaSuccess) { (void)cudaGetLastError(); c->Lx3t = nullptr; return AFQMC_OUT_OF_MEMORY; }
        return pack_lx3t(c, st);
    }
    if (c->Lxc) return AFQMC_OK;
    if (cudaMalloc((void**)&c->Lxc, afqmc_i_lxc_doubles(c->d) * sizeof(double)) != cudaSuccess) { (void)cudaGetLastError(); c->Lxc = nullptr; return AFQMC_OUT_OF_MEMORY; }
    return pack_lxc(c, st);
}

// a0: the operand of the default exchange kernel (called once from afqmc_create)
int afqmc_i_pack_exchange_operand(afqmc_ctx* c, cudaStream_t st) { return ensure_operand(c, x3_prefers_reg(c->d), st); }

namespace {

// B fragments of NP n-tiles for one lane and micro-step sit next to each other: [ms][jp][lane][W], W = min(NP,2) doubles
template <int NP> struct BVec { static constexpr int W = NP >= 2 ? 2 : 1, NPH = NP / W; };

// ---------------------------------------------------------------------------------------------------------------------
// Pieces shared by the two kernels below
// ---------------------------------------------------------------------------------------------------------------------
struct X3Cta {
    int u, w0, chunk, ab0, ab1;       // unit, first walker, gamma-quad chunk, range of (ag,bg) pairs
    int Q, k, k2, mQ, kq, k2pq;       // kq = k - Q: column block of theta for T1;  k2pq = k2 + Q: column block for T2
    double pair_weight;
};

// Decodes blockIdx.x; returns false if this CTA has nothing to compute (its partial sums are then already written).
template <int NP, bool GRIDPAIRS>
__device__ __forceinline__ bool x3_decode(X3Cta& t, const Dims& d, int nchunk, int nw, const int* __restrict__ units,
                                          const int* __restrict__ kminus, const int* __restrict__ kplus,
                                          const int* __restrict__ kneg, double2* __restrict__ partial) {
    constexpr int NWC = 2 * NP;
    const int nwg = (nw + NWC - 1) / NWC;            // walker groups of one unit are adjacent in the grid
    const int npairs = d.NAG * d.NAG;
    int bx = blockIdx.x;
    t.chunk = 0; t.ab0 = 0; t.ab1 = npairs;
    if (GRIDPAIRS) {                                  // blockIdx.x = ((u * nwg + walker group) * npairs + ab) * nchunk + chunk
        t.chunk = bx % nchunk; bx /= nchunk;
        t.ab0 = bx % npairs; bx /= npairs;
        t.ab1 = t.ab0 + 1;
    }
    t.w0 = (bx % nwg) * NWC; t.u = bx / nwg;
    t.pair_weight = 1.0;
    if (GRIDPAIRS) {
        // A unit that is its own partner under (Q,k,k2) -> (-Q,k2,k) (multiplicity 1; every unit at the Gamma point) has
        // T2 = T1, so the pairs (ag,bg) and (bg,ag) contribute equally: compute ag <= bg only, twice for ag < bg.
        const int ag = t.ab0 / d.NAG, bg = t.ab0 % d.NAG;
        const bool self_unit = units[4 * t.u + 3] == 1;
        if (self_unit && ag > bg) {
            if (threadIdx.x < NWC && t.w0 + (int)threadIdx.x < nw)
                partial[(((size_t)t.u * npairs + t.ab0) * nchunk + t.chunk) * nw + t.w0 + threadIdx.x] = make_double2(0.0, 0.0);
            return false;
        }
        if (self_unit && ag < bg) t.pair_weight = 2.0;
    }
    t.Q = units[4 * t.u]; t.k = units[4 * t.u + 1]; t.k2 = units[4 * t.u + 2];
    t.mQ = kneg[t.Q];
    t.kq = kminus[t.k * d.Nk + t.Q];
    t.k2pq = kplus[t.k2 * d.Nk + t.Q];
    return true;
}

// Stages the two theta blocks of the unit as B fragments, expanded into the B variants of every micro-step:
//   Bs[which][slot][ms][jp][lane][W]   which 0 -> theta[(k2,b),(k-Q,r)] (T1), 1 -> theta[(k,a),(k2+Q,s)] (T2)
//   lane of a B fragment = (col << 2) | kk,  col = 4*(walker & 1) + orbital,  n-tile j = walker >> 1
// One thread per complex theta element; the thread order (r mod 4, orbital mod 2, j fastest) makes the 64-byte runs of
// theta coalesce and the 8-byte shared-memory stores of a half-warp fall into 16 different bank pairs.
template <int NP, int NTHR, bool GRIDPAIRS>
__device__ __forceinline__ void x3_stage_theta(double* __restrict__ Bs, const Dims& d, const X3Geom& g, const X3Cta& t, int nw,
                                               const double2* __restrict__ theta) {
    constexpr int NWC = 2 * NP, W = BVec<NP>::W, bs_step = 32 * NP;
    const int NGS = GRIDPAIRS ? 1 : d.NAG;
    const int bs_grp = (g.MSPT + 1) * bs_step, bs_half = NGS * bs_grp;
    const int per_which = (g.KSF + g.TAIL) * NGS * 4 * NWC * 4;
    for (int e = threadIdx.x; e < 2 * per_which; e += NTHR) {
        const int which = e / per_which;
        int x = e - which * per_which;
        const int r_lo = x & 3; x >>= 2;
        const int b_lo = x & 1; x >>= 1;
        const int j = x % NP; x /= NP;
        const int b = b_lo | ((x & 1) << 1); x >>= 1;
        const int w_lo = x & 1; x >>= 1;
        const int gs = x % NGS, r_hi = x / NGS;
        if (r_hi == g.KSF && r_lo >= 2) continue;          // the tail quad holds two elements
        const int r = 4 * r_hi + r_lo, wl = 2 * j + w_lo;
        const int grp = GRIDPAIRS ? (which == 0 ? t.ab0 % d.NAG : t.ab0 / d.NAG) : gs;
        const int orb = 4 * grp + b, w = t.w0 + wl;
        const int rowblk = which == 0 ? t.k2 : t.k, colblk = which == 0 ? t.kq : t.k2pq;
        double2 v = make_double2(0.0, 0.0);
        if (orb < d.n && w < nw && r < d.m)
            v = __ldg(theta + ((size_t)w * d.N + rowblk * d.n + orb) * d.M + (size_t)colblk * d.m + r);
        const int col = w_lo * 4 + b;
        double* base = Bs + which * bs_half + gs * bs_grp + (j / W) * (32 * W) + (j % W);    // + ms * bs_step + lane * W
        if (g.PV == 2) {                        // real operand: the two B sides are Re and Im themselves
            double* dst = base + 2 * r_hi * bs_step + ((col << 2) | r_lo) * W;
            dst[0] = v.x;
            dst[bs_step] = v.y;
        } else if (r_hi < g.KSF) {
            double* dst = base + 3 * r_hi * bs_step + ((col << 2) | r_lo) * W;
            dst[0] = v.x;                       // Br
            dst[bs_step] = v.y - v.x;           // Bi - Br
            dst[2 * bs_step] = v.x + v.y;       // Br + Bi
        } else {                                // tail: real embedding, lanes kk = 2t (times Ar) and 2t+1 (times Ai)
            double* dst = base + 3 * g.KSF * bs_step + ((col << 2) | (2 * r_lo)) * W;
            dst[0] = v.x;  dst[W] = -v.y;                               // -> P0:  Ar Br - Ai Bi
            dst[bs_step] = v.y - v.x;  dst[bs_step + W] = v.x + v.y;    // -> P1:  Ar (Bi-Br) + Ai (Br+Bi)
        }
    }
}

// Slot (in complex numbers) of element [(gamma gl, orbA), (walker wp, orbB)] of a hand-over tile.  The low three bits are
// chosen so that both the writer's and the reader's quarter-warps (which differ in which orbital bits vary) touch eight
// different 16-byte slots modulo 8: conflict-free STS.128 and LDS.128.
__device__ __forceinline__ int x3_slot(int gl, int orbA, int wp, int orbB) {
    return gl * 32 + ((orbA >> 1) * 2 + (orbB >> 1)) * 8 + ((((orbA ^ (orbA >> 1)) & 1) << 2) | (wp << 1) | ((orbB ^ (orbB >> 1)) & 1));
}

// Lane geometry of a C fragment (row = lane>>2, columns 2c+e, c = lane&3, register e): rows (gl = row>>2: gamma of the tile's
// pair, orow = row&3: this warp's ROW orbital), columns (wp = c>>1: walker of the pair, ocol = 2(c&1)+e: the COLUMN orbital).
// T1: orow = a, ocol = b;  T2: orow = b, ocol = a.  The partner of own element [(g,orow),(w,ocol)] is [(g,ocol),(w,orow)].
struct X3Lane { int sw[2], sr[2]; };
__device__ __forceinline__ X3Lane x3_lane(int lane) {
    const int gl = lane >> 4, orow = (lane >> 2) & 3, wp = (lane >> 1) & 1, cb = lane & 1;
    X3Lane L;
#pragma unroll
    for (int e = 0; e < 2; ++e) {
        L.sw[e] = x3_slot(gl, orow, wp, 2 * cb + e);
        L.sr[e] = x3_slot(gl, 2 * cb + e, wp, orow);
    }
    return L;
}

// End of a task (gamma-quad): combine the three products (Re = P0 - P2, Im = P0 + P1), hand m-tile 1-KEEP to the partner warp
// of the pair through `xw`, take the partner's tile KEEP from `xr` (this is also the (a,b) transpose) and contract it with the
// own tile KEEP; the accumulators are cleared.
// (REAL: two products, Re = P0 = Ar Br, Im = P1 = Ar Bi)
template <int NP, int KEEP, bool REAL = false>
__device__ __forceinline__ void x3_finish_task(double (&acc)[3][2][NP][2], double2* __restrict__ xw, const double2* __restrict__ xr,
                                               int bar_id, const X3Lane& L, double (&er)[NP], double (&ei)[NP]) {
    constexpr int GIVE = 1 - KEEP;
#pragma unroll
    for (int j = 0; j < NP; ++j)
#pragma unroll
        for (int e = 0; e < 2; ++e)
            xw[j * 64 + L.sw[e]] = REAL ? make_double2(acc[0][GIVE][j][e], acc[1][GIVE][j][e])
                                        : make_double2(acc[0][GIVE][j][e] - acc[2][GIVE][j][e], acc[0][GIVE][j][e] + acc[1][GIVE][j][e]);
    // the two warps of the pair (an immediate id where possible: a register id makes ptxas reserve all 16 named barriers)
    if (bar_id == 1) asm volatile("bar.sync 1, 64;" ::: "memory");
    else asm volatile("bar.sync 2, 64;" ::: "memory");        // (at most two warp pairs per CTA)
#pragma unroll
    for (int j = 0; j < NP; ++j)
#pragma unroll
        for (int e = 0; e < 2; ++e) {
            const double tr = REAL ? acc[0][KEEP][j][e] : acc[0][KEEP][j][e] - acc[2][KEEP][j][e];
            const double ti = REAL ? acc[1][KEEP][j][e] : acc[0][KEEP][j][e] + acc[1][KEEP][j][e];
            const double2 p = xr[j * 64 + L.sr[e]];
            er[j] = fma(tr, p.x, er[j]); er[j] = fma(-ti, p.y, er[j]);
            ei[j] = fma(tr, p.y, ei[j]); ei[j] = fma(ti, p.x, ei[j]);
        }
#pragma unroll
    for (int p = 0; p < 3; ++p)
#pragma unroll
        for (int i = 0; i < 2; ++i)
#pragma unroll
            for (int j = 0; j < NP; ++j) acc[p][i][j][0] = acc[p][i][j][1] = 0.0;
}

// ---- pieces of the DEFERRED hand-over (exchange3m_reg_kernel, ASYNC): the tile a warp gives to its partner is published with
// a non-blocking bar.arrive and collected by the partner one task LATER with bar.sync, so neither warp ever waits for the other
// at a task end (the blocking version lost 6.5 % of its warp-samples there, profiles/r02c).  Named barrier 1 + 2 h + buf: "the
// tile of role h in hand-over buffer buf is written" (32 arriving + 32 waiting threads); immediates, see x3_finish_task.
__device__ __forceinline__ void x3_bar_arrive(int h, int buf) {
    switch (2 * h + buf) {
        case 0: asm volatile("bar.arrive 1, 64;" ::: "memory"); break;
        case 1: asm volatile("bar.arrive 2, 64;" ::: "memory"); break;
        case 2: asm volatile("bar.arrive 3, 64;" ::: "memory"); break;
        default: asm volatile("bar.arrive 4, 64;" ::: "memory"); break;
    }
}
__device__ __forceinline__ void x3_bar_wait(int h, int buf) {
    switch (2 * h + buf) {
        case 0: asm volatile("bar.sync 1, 64;" ::: "memory"); break;
        case 1: asm volatile("bar.sync 2, 64;" ::: "memory"); break;
        case 2: asm volatile("bar.sync 3, 64;" ::: "memory"); break;
        default: asm volatile("bar.sync 4, 64;" ::: "memory"); break;
    }
}
// contracts the kept tile of the PREVIOUS task with the partner's tile of that task (in `xr`, hand-over buffer `buf`)
template <int NP>
__device__ __forceinline__ void x3_collect(const double2 (&keep)[NP][2], const double2* __restrict__ xr, int h, int buf, const X3Lane& L,
                                           double (&er)[NP], double (&ei)[NP]) {
    x3_bar_wait(h ^ 1, buf);
#pragma unroll
    for (int j = 0; j < NP; ++j)
#pragma unroll
        for (int e = 0; e < 2; ++e) {
            const double2 p = xr[j * 64 + L.sr[e]];
            er[j] = fma(keep[j][e].x, p.x, er[j]); er[j] = fma(-keep[j][e].y, p.y, er[j]);
            ei[j] = fma(keep[j][e].x, p.y, ei[j]); ei[j] = fma(keep[j][e].y, p.x, ei[j]);
        }
}
// end of a task: combine the three products, publish m-tile 1-KEEP in `xw` (buffer `buf`), keep m-tile KEEP, clear
// PHASED: acc[0] and acc[1] already hold Re and Im (see task_async: the products were accumulated in two phases), nothing to combine
template <int NP, int KEEP, bool PHASED = false>
__device__ __forceinline__ void x3_publish(double (&acc)[3][2][NP][2], double2 (&keep)[NP][2], double2* __restrict__ xw, int h, int buf,
                                           const X3Lane& L) {
    constexpr int GIVE = 1 - KEEP;
#pragma unroll
    for (int j = 0; j < NP; ++j)
#pragma unroll
        for (int e = 0; e < 2; ++e) {
            if (PHASED) {
                xw[j * 64 + L.sw[e]] = make_double2(acc[0][GIVE][j][e], acc[1][GIVE][j][e]);
                keep[j][e] = make_double2(acc[0][KEEP][j][e], acc[1][KEEP][j][e]);
            } else {
                xw[j * 64 + L.sw[e]] = make_double2(acc[0][GIVE][j][e] - acc[2][GIVE][j][e], acc[0][GIVE][j][e] + acc[1][GIVE][j][e]);
                keep[j][e] = make_double2(acc[0][KEEP][j][e] - acc[2][KEEP][j][e], acc[0][KEEP][j][e] + acc[1][KEEP][j][e]);
            }
        }
    x3_bar_arrive(h, buf);
#pragma unroll
    for (int p = 0; p < 3; ++p)
#pragma unroll
        for (int i = 0; i < 2; ++i)
#pragma unroll
            for (int j = 0; j < NP; ++j) acc[p][i][j][0] = acc[p][i][j][1] = 0.0;
}
__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;\n" ::"r"(smem_u32(smem)), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }

// Sum over the lanes of each walker-in-pair (lane bit 1 = wp), then over the warps in a fixed order (deterministic).
template <int NP, int NWARP, bool GRIDPAIRS>
__device__ __forceinline__ void x3_reduce_store(double* red /* shared, [warp][NWC][2] */, const double (&er)[NP], const double (&ei)[NP],
                                                const X3Cta& t, const Dims& d, int nchunk, int nw, double2* __restrict__ partial) {
    constexpr int NWC = 2 * NP;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    __syncthreads();      // every warp is done with the shared memory that `red` reuses
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
    if (tid < NWC && t.w0 + tid < nw) {
        double r = 0.0, i = 0.0;
        for (int x = 0; x < NWARP; ++x) { r += red[(x * NWC + tid) * 2]; i += red[(x * NWC + tid) * 2 + 1]; }
        const size_t slot = GRIDPAIRS ? ((size_t)t.u * d.NAG * d.NAG + t.ab0) * nchunk + t.chunk : (size_t)t.u;
        partial[slot * nw + t.w0 + tid] = make_double2(t.pair_weight * r, t.pair_weight * i);
    }
}

// ---------------------------------------------------------------------------------------------------------------------
// Generic kernel: any m; the B fragments are read from shared memory every micro-step.
// CTA = (unit, group of 2*NP walkers[, pair of a-groups, chunk of gamma-quads]); 2*NPAIR warps; see the header comment.
//   GRIDPAIRS = false: the theta blocks of ALL a-groups are staged and the CTA loops over the (ag,bg) pairs (n <= 4: one pair);
//   GRIDPAIRS = true : the (ag,bg) pair and a chunk of the gamma-quads come from the grid and only the theta rows of those two
//                      groups are staged (blocks too large for shared memory: many orbitals / bands per k-point, e.g. the
//                      Gamma-point supercell shape); a unit then contributes NAG^2 * nchunk partial sums.
// DA = k-steps of register prefetch of the Lxc stream (L2 resident); the B fragments (shared memory) run one k-step ahead.
// ---------------------------------------------------------------------------------------------------------------------
// REAL = the half-rotated tensor is real (real orbitals, detected in a0): T = Lh theta needs two real products per complex one
// (Re = Ar Br, Im = Ar Bi, no addition anywhere); the operand is the real-parts-only layout Lxr (half the bytes, one LDG.128 per
// k-step), the geometry x3_geom_real (no tail trick) and the staged theta blocks hold two B sides per k-step (2/3 of the bytes).
template <int NP, int NPAIR, int DA, int MINB, bool GRIDPAIRS, bool REAL>
__global__ void __launch_bounds__(64 * NPAIR, MINB) exchange3m_kernel(
    Dims d, X3Geom g, int nchunk, int nw, const int* __restrict__ units, const int* __restrict__ kminus,
    const int* __restrict__ kplus, const int* __restrict__ kneg, const double* __restrict__ Lxc,
    const double2* __restrict__ theta, double2* __restrict__ partial) {
    extern __shared__ __align__(16) double x3_smem[];
    constexpr int NWARP = 2 * NPAIR, NBUF = 2;
    constexpr int W = BVec<NP>::W, NPH = BVec<NP>::NPH;
    X3Cta t;
    if (!x3_decode<NP, GRIDPAIRS>(t, d, nchunk, nw, units, kminus, kplus, kneg, partial)) return;
    const int NAG = d.NAG, GQ = d.GQ;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, pair = warp >> 1, h = warp & 1;
    const int NGS = GRIDPAIRS ? 1 : NAG;        // a-group slots staged per theta block
    constexpr int bs_step = 32 * NP;            // doubles of one micro-step
    const int bs_grp = (g.MSPT + 1) * bs_step;  // +1: the k-step before a tail prefetches a third micro-step that does not exist
    const int bs_half = NGS * bs_grp;
    double* Bs = x3_smem;
    double2* xbuf = reinterpret_cast<double2*>(x3_smem + 2 * bs_half);      // [pair][role][NBUF][NP][64] hand-over tiles

    // ---- this warp's share of the gamma-quads (both warps of a pair walk the same tasks) ----
    const int q_begin = (int)((long long)t.chunk * GQ / nchunk), q_end = (int)((long long)(t.chunk + 1) * GQ / nchunk);
    const int t_begin = q_begin + (int)((long long)pair * (q_end - q_begin) / NPAIR);
    const int t_end = q_begin + (int)((long long)(pair + 1) * (q_end - q_begin) / NPAIR);
    const int total = (t_end - t_begin) * g.KSPT;                 // k-steps of this warp per (ag,bg) pair
    const size_t blk = h == 0 ? (size_t)t.Q * d.Nk + t.k : (size_t)t.mQ * d.Nk + t.k2;
    constexpr int AST = REAL ? 32 : 64;         // k-step stride of a lane's A stream in double2
    auto stream_ptr = [&](int grp) {            // 2 double2 per lane and k-step (REAL: one = the real parts of both tiles)
        return REAL ? reinterpret_cast<const double2*>(Lxc + (((blk * NAG + grp) * GQ + t_begin) * (size_t)g.KSPT) * 64) + lane
                    : reinterpret_cast<const double2*>(Lxc + (((blk * NAG + grp) * GQ + t_begin) * (size_t)g.KSPT) * 128) + lane * 2;
    };
    double2 fa[DA][2];
    const double2* pa = stream_ptr(h == 0 ? t.ab0 / NAG : t.ab0 % NAG);
    // prologue of the first pair's A stream: issued before the staging below, which hides the L2 round trip
#pragma unroll
    for (int q = 0; q < DA; ++q) {
        fa[q][0] = fa[q][1] = make_double2(0.0, 0.0);
        if (total > 0) { fa[q][0] = __ldg(pa + q * AST); if (!REAL) fa[q][1] = __ldg(pa + q * AST + 1); }
    }
    x3_stage_theta<NP, 64 * NPAIR, GRIDPAIRS>(Bs, d, g, t, nw, theta);
    __syncthreads();   // B fragments staged

    const X3Lane L = x3_lane(lane);
    double er[NP], ei[NP];
#pragma unroll
    for (int j = 0; j < NP; ++j) er[j] = ei[j] = 0.0;
    int buf = 0;

    for (int ab = t.ab0; ab < t.ab1; ++ab) {
        const int ag = ab / NAG, bg = ab % NAG;
        if (ab != t.ab0) {                       // next pair of a-groups: restart the A stream
            pa = stream_ptr(h == 0 ? ag : bg);
#pragma unroll
            for (int q = 0; q < DA; ++q)
                if (total > 0) { fa[q][0] = __ldg(pa + q * AST); if (!REAL) fa[q][1] = __ldg(pa + q * AST + 1); }
        }
        pa += DA * AST;
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
        constexpr int PV = REAL ? 2 : 3;
        load_b(0, 0); load_b(1, 0);
        if (!REAL) load_b(2, 0);
        double acc[3][2][NP][2];
#pragma unroll
        for (int p = 0; p < 3; ++p)
#pragma unroll
            for (int i = 0; i < 2; ++i)
#pragma unroll
                for (int j = 0; j < NP; ++j) acc[p][i][j][0] = acc[p][i][j][1] = 0.0;

        int cs = 0;   // k-step of the compute state inside its task
        auto kstep = [&](auto Q_) {
            constexpr int q = decltype(Q_)::value;
            const double2 x0 = REAL ? make_double2(fa[q][0].x, 0.0) : fa[q][0], x1 = REAL ? make_double2(fa[q][0].y, 0.0) : fa[q][1];
            const int nxt = (cs + 1 == g.KSPT) ? 0 : PV * (cs + 1);     // first micro-step of the next k-step (wraps at the task end)
            if (REAL || cs < g.KSF) {
                const double s0 = REAL ? x0.x : x0.x + x0.y, s1 = REAL ? x1.x : x1.x + x1.y;        // Ar + Ai
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
                if (!REAL) {
#pragma unroll
                    for (int j = 0; j < NP; ++j) {
                        dmma884(acc[2][0][j][0], acc[2][0][j][1], x0.y, fb[2][j]);
                        dmma884(acc[2][1][j][0], acc[2][1][j][1], x1.y, fb[2][j]);
                    }
                    load_b(2, nxt);
                }
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
                if (!REAL) load_b(2, nxt);
            }
            // refill this ring slot with the k-step DA ahead (may run past the warp's last task: loaded, never used)
            fa[q][0] = __ldg(pa);
            if (!REAL) fa[q][1] = __ldg(pa + 1);
            pa += AST;
            if (++cs == g.KSPT) {
                cs = 0;
                // two hand-over buffers: the partner may still read one while the next task is written into the other
                double2* xw = xbuf + (((pair * 2 + h) * NBUF + buf) * NP) * 64;
                const double2* xr = xbuf + (((pair * 2 + (h ^ 1)) * NBUF + buf) * NP) * 64;
                if (h == 0) x3_finish_task<NP, 0, REAL>(acc, xw, xr, pair + 1, L, er, ei);
                else x3_finish_task<NP, 1, REAL>(acc, xw, xr, pair + 1, L, er, ei);
                buf ^= 1;
            }
        };
        const int nfull = total - total % DA;
        for (int g0 = 0; g0 < nfull; g0 += DA) {
            kstep(std::integral_constant<int, 0>());
            if (DA > 1) kstep(std::integral_constant<int, 1 % DA>());
            if (DA > 2) kstep(std::integral_constant<int, 2 % DA>());
            if (DA > 3) kstep(std::integral_constant<int, 3 % DA>());
            if (DA > 4) kstep(std::integral_constant<int, 4 % DA>());
            if (DA > 5) kstep(std::integral_constant<int, 5 % DA>());
        }
        if (nfull + 0 < total) kstep(std::integral_constant<int, 0>());
        if (DA > 2 && nfull + 1 < total) kstep(std::integral_constant<int, 1 % DA>());
        if (DA > 3 && nfull + 2 < total) kstep(std::integral_constant<int, 2 % DA>());
        if (DA > 4 && nfull + 3 < total) kstep(std::integral_constant<int, 3 % DA>());
        if (DA > 5 && nfull + 4 < total) kstep(std::integral_constant<int, 4 % DA>());
    }
    x3_reduce_store<NP, NWARP, GRIDPAIRS>(x3_smem, er, ei, t, d, nchunk, nw, partial);
}

// ---------------------------------------------------------------------------------------------------------------------
// Register-resident B, persistent CTAs: m <= 28 (MSPT = 3 KSF + 2 TAIL <= 21 micro-steps per task).
//
// One warp pair per CTA (role h = warp: T1 / T2); the grid is as many CTAs as stay resident, and a CTA walks the work items
// (unit, walker group) blockIdx.x, + gridDim.x, ...: walker groups of a unit are adjacent, so the CTAs that run together share
// the unit's Lh blocks in L2.  Per item and warp:
//   1. the warp's theta block arrives RAW (rows (walker, orbital) of m complex numbers) by bulk asynchronous copies
//      (cp.async.bulk + mbarrier, issued one item ahead into the other half of a double buffer: the TMA engine stages while the
//      warp computes, no thread waits on an L2 round trip and there is no CTA-wide barrier);
//   2. the warp expands it into the three B variants straight into MSPT * NP REGISTERS (once per a-group pair);
//   3. every gamma-quad of the unit runs against those registers: the task is fully unrolled (KSF, TAIL are template
//      parameters) and the A stream (Lx3t: the three variants stored) reaches the warp
//        ASYNC (default): through a shared-memory ring that holds exactly ONE task (MST micro-loads of 512 bytes per warp,
//          lane-private 16-byte slots): slot = micro-load index, so every address is a constant; a slot is refilled by the
//          lane's own cp.async (SASS LDGSTS.E.128) with the same micro-load of the NEXT task right after it was read, one
//          commit group per k-step, `cp.async.wait_group KSPT-1` before a k-step: a full task of lookahead at no register cost
//          (222 registers, no spills; the register ring below allowed two k-steps at 255 registers and 6 % of the warp samples
//          sat on DMMAs waiting for an A fragment from L2);
//        !ASYNC (option exchange_regb = 2): prefetched DA k-steps ahead in a register ring whose slot of a task's first k-step
//          (BASE) rotates by KSPT mod DA from task to task (DA copies of the task body behind a warp-uniform switch);
//      either way the stream runs on across tasks, a-group pairs and ITEMS (the last task of an item prefetches the next item's
//      stream): the inner loop is LDS.128 / LDG.128 + DMMA only;
//   4. at the end of each task the two warps swap one m-tile through shared memory and contract: ASYNC publishes its tile with
//      bar.arrive and collects the partner's tile of the PREVIOUS task (x3_publish / x3_collect), so no warp waits at a task
//      end; !ASYNC meets at a blocking bar.sync per task (x3_finish_task).
// ---------------------------------------------------------------------------------------------------------------------
template <int KSF, int TAIL, int NP, int MAXREG, bool ASYNC>
__global__ void __launch_bounds__(64) __maxnreg__(MAXREG) exchange3m_reg_kernel(
    Dims d, int nw, int nitems, const int* __restrict__ units, const int* __restrict__ kminus, const int* __restrict__ kplus,
    const int* __restrict__ kneg, const double* __restrict__ Lx3t, const double2* __restrict__ theta,
    double2* __restrict__ partial) {
    extern __shared__ __align__(16) double x3_smem[];
    constexpr int KSPT = KSF + TAIL, MSPT = 3 * KSF + 2 * TAIL, MST = 3 * KSF + TAIL, NBUF = 2, NWC = 2 * NP;
    constexpr int DA = KSPT >= 2 ? 2 : 1;            // k-steps of A prefetch into registers (<= KSPT)
    constexpr int TASK = MST * 32;                   // double2 per task and lane stream (one double2 per lane and micro-load)
    const int NAG = d.NAG, GQ = d.GQ, npairs = NAG * NAG;
    const int lane = threadIdx.x & 31, h = threadIdx.x >> 5;
    const int nwg = (nw + NWC - 1) / NWC;
    const int raw_len = NWC * d.n * d.m;             // complex numbers of one raw theta block
    // shared memory: raw[role][buf][raw_len] | xbuf[role][NBUF][NP][64] | red[2][NWC] (all double2) | mbar[role][buf]
    double2* raw = reinterpret_cast<double2*>(x3_smem);
    double2* xbuf = raw + 4 * raw_len;
    double2* red = xbuf + 2 * NBUF * NP * 64;
    double2* aring = red + 2 * NWC;                  // ASYNC: [role][MST][32] one task of the A stream per warp, lane-private slots
    uint64_t* mbar = reinterpret_cast<uint64_t*>(aring + (ASYNC ? 2 * MST * 32 : 0));
    if (threadIdx.x == 0) {
        for (int i = 0; i < 4; ++i) mbar_init(&mbar[i], 1);
        mbar_fence_init();
    }
    __syncthreads();

    // ---- per-item state of this warp ----
    struct Item { int u, w0, rowblk, colblk; size_t blk; };
    auto decode = [&](int item) {
        Item it;
        it.u = item / nwg; it.w0 = (item % nwg) * NWC;
        const int Q = units[4 * it.u], k = units[4 * it.u + 1], k2 = units[4 * it.u + 2];
        if (h == 0) {       // T1: Lh[Q][k] against theta[(k2,b),(k-Q,r)]
            it.blk = (size_t)Q * d.Nk + k; it.rowblk = k2; it.colblk = kminus[k * d.Nk + Q];
        } else {            // T2: Lh[-Q][k2] against theta[(k,a),(k2+Q,s)]
            it.blk = (size_t)kneg[Q] * d.Nk + k2; it.rowblk = k; it.colblk = kplus[k2 * d.Nk + Q];
        }
        return it;
    };
    auto stream_ptr = [&](const Item& it, int grp) {
        return reinterpret_cast<const double2*>(Lx3t) + ((it.blk * NAG + grp) * GQ) * (size_t)TASK + lane;
    };
    // bulk copies of this warp's raw theta block of `it` into buffer `b` (rows of padded walkers are not fetched)
    // Theta (38.8 MB at C3) is re-read in full once per Q pair while the 393 MB operand stream passes through L2 between two
    // visits; evict_last keeps its lines ahead of the stream's dead blocks (DRAM read per launch at C3: 985 -> 909 MB,
    // profiles/r02i_exchange_dram.md; no change in time, the kernel is bound by the FP64 pipe)
    const uint64_t theta_policy = l2_policy_evict_last();
    auto issue_theta = [&](const Item& it, int b) {
        const int nvalid = min(NWC, nw - it.w0) * d.n;
        uint64_t* bar = &mbar[h * 2 + b];
        if (lane == 0) mbar_expect_tx(bar, (uint32_t)(nvalid * d.m * 16));
        __syncwarp();
        double2* dst = raw + (h * 2 + b) * raw_len;
        for (int row = lane; row < nvalid; row += 32) {
            const int wl = row / d.n, orb = row - wl * d.n;
            bulk_g2s_hint(dst + (size_t)row * d.m,
                          theta + ((size_t)(it.w0 + wl) * d.N + it.rowblk * d.n + orb) * d.M + (size_t)it.colblk * d.m,
                          (uint32_t)(d.m * 16), bar, theta_policy);
        }
    };

    int item = blockIdx.x;
    if (item >= nitems) return;
    Item cur = decode(item);
    issue_theta(cur, 0);
    int bufsel = 0, phase = 0;          // phase: bit b = parity to wait for on buffer b
    // A ring: fa[slot][p] = micro-load p of the k-step in that slot; prologue = the first DA k-steps of the first item
    // (ASYNC: the ring is one whole task in shared memory, filled by per-lane cp.async, one commit group per k-step; slot =
    // micro-load index, so every address is a constant and the lookahead is a full task)
    double2 fa[ASYNC ? 1 : DA][3];
    const double2* pa = stream_ptr(cur, 0);
    double2* ar = aring + h * (MST * 32) + lane;
    if (ASYNC) {      // the first task, in the group order of task_async: A_0 .. A_{KSF-1}, B_0 .. B_{KSF-1}, tail
#pragma unroll
        for (int ks = 0; ks < KSF; ++ks) { cp_async16(ar + (3 * ks) * 32, pa + (3 * ks) * 32); cp_async_commit(); }
#pragma unroll
        for (int ks = 0; ks < KSF; ++ks) {
            cp_async16(ar + (3 * ks + 1) * 32, pa + (3 * ks + 1) * 32);
            cp_async16(ar + (3 * ks + 2) * 32, pa + (3 * ks + 2) * 32);
            cp_async_commit();
        }
        if (TAIL) { cp_async16(ar + (3 * KSF) * 32, pa + (3 * KSF) * 32); cp_async_commit(); }
    } else {
#pragma unroll
        for (int q = 0; q < DA; ++q) {
#pragma unroll
            for (int p = 0; p < 3; ++p) fa[q][p] = make_double2(0.0, 0.0);
            if (q < KSF) {
#pragma unroll
                for (int p = 0; p < 3; ++p) fa[q][p] = __ldg(pa + (3 * q + p) * 32);
            } else {
                fa[q][0] = __ldg(pa + (3 * KSF) * 32);
            }
        }
    }
    int base = 0;                       // ring slot of the next task's first k-step
    const X3Lane L = x3_lane(lane);
    double er[NP], ei[NP];
#pragma unroll
    for (int j = 0; j < NP; ++j) er[j] = ei[j] = 0.0;
    int buf = 0, par = 0;
    double2 keep[NP][2];                // ASYNC: the kept m-tile of the previous task (contracted one task later)
#pragma unroll
    for (int j = 0; j < NP; ++j) keep[j][0] = keep[j][1] = make_double2(0.0, 0.0);
    double acc[3][2][NP][2];
#pragma unroll
    for (int p = 0; p < 3; ++p)
#pragma unroll
        for (int i = 0; i < 2; ++i)
#pragma unroll
            for (int j = 0; j < NP; ++j) acc[p][i][j][0] = acc[p][i][j][1] = 0.0;

    while (true) {
        const int nxt = item + gridDim.x;
        const bool has_next = nxt < nitems;
        Item nx = cur;
        if (has_next) nx = decode(nxt);
        mbar_wait(&mbar[h * 2 + bufsel], (phase >> bufsel) & 1);        // this item's raw theta block has landed
        phase ^= 1 << bufsel;
        const double2* rw = raw + (h * 2 + bufsel) * raw_len;
        for (int ab = 0; ab < npairs; ++ab) {
            const int ag = ab / NAG, bg = ab % NAG;
            // ---- theta rows of this warp's a-group -> B registers (T1: rows bg of k2; T2: rows ag of k) ----
            double B[MSPT][NP];
            {
                const int kk = lane & 3, col = lane >> 2, b = col & 3, wlo = col >> 2;
                const int orb = 4 * (h == 0 ? bg : ag) + b;
#pragma unroll
                for (int j = 0; j < NP; ++j) {
                    const int wl = 2 * j + wlo;
                    const bool ok = orb < d.n && cur.w0 + wl < nw;
                    const double2* src = rw + (size_t)(wl * d.n + (ok ? orb : 0)) * d.m;
#pragma unroll
                    for (int ks = 0; ks < KSF; ++ks) {
                        const int r = 4 * ks + kk;
                        double2 v = make_double2(0.0, 0.0);
                        if (ok && r < d.m) v = src[r];
                        // ASYNC (phased accumulation, see task_async): the third side is negated, so that its product is
                        // SUBTRACTED from the accumulator that already holds P0: Re = P0 - P2 without an addition
                        B[3 * ks][j] = v.x; B[3 * ks + 1][j] = v.y - v.x; B[3 * ks + 2][j] = ASYNC ? -(v.x + v.y) : v.x + v.y;
                    }
                    if (TAIL) {       // real embedding: lanes kk = 2t (times Ar) and 2t+1 (times Ai)
                        const int r = 4 * KSF + (kk >> 1);
                        double2 v = make_double2(0.0, 0.0);
                        if (ok && r < d.m) v = src[r];
                        B[3 * KSF][j] = (kk & 1) ? -v.y : v.x;                               // -> P0 / Re:  Ar Br - Ai Bi
                        if (ASYNC) B[3 * KSF + (TAIL ? 1 : 0)][j] = (kk & 1) ? v.x : v.y;      // -> Im:  Ar Bi + Ai Br
                        else B[3 * KSF + (TAIL ? 1 : 0)][j] = (kk & 1) ? v.x + v.y : v.y - v.x;     // -> P1:  Ar (Bi-Br) + Ai (Br+Bi)
                    }
                }
            }
            const bool last_pair = ab == npairs - 1;
            if (last_pair) {          // the raw buffer of the previous item is free: fetch the next item's block into it
                fence_proxy_async_smem();       // (its reads before the bulk copies that refill it, common.cuh)
                __syncwarp();
                if (has_next) issue_theta(nx, bufsel ^ 1);
            }
            const int grpA = h == 0 ? ag : bg;
            pa = stream_ptr(cur, grpA);
            // where the stream continues after this pair: the next pair of this item, or the first pair of the next item
            const double2* pcont = last_pair ? (has_next ? stream_ptr(nx, 0) : pa)
                                             : stream_ptr(cur, h == 0 ? (ab + 1) / NAG : (ab + 1) % NAG);

            // one gamma-quad; the ring holds its k-steps 0..DA-1 in slots BASE, BASE+1, .. (mod DA); k-steps >= KSPT come from `pn`
            auto task = [&](auto BASE_, const double2* pn) {
                constexpr int BASE = decltype(BASE_)::value;
#pragma unroll
                for (int ks = 0; ks < KSPT; ++ks) {
                    const int q = (BASE + ks) % DA;                     // a constant after unrolling
                    if (ks < KSF) {
#pragma unroll
                        for (int p = 0; p < 3; ++p)
#pragma unroll
                            for (int j = 0; j < NP; ++j) {
                                dmma884(acc[p][0][j][0], acc[p][0][j][1], fa[q][p].x, B[3 * ks + p][j]);
                                dmma884(acc[p][1][j][0], acc[p][1][j][1], fa[q][p].y, B[3 * ks + p][j]);
                            }
                    } else {                                             // tail k-step
#pragma unroll
                        for (int p = 0; p < 2; ++p)
#pragma unroll
                            for (int j = 0; j < NP; ++j) {
                                dmma884(acc[p][0][j][0], acc[p][0][j][1], fa[q][0].x, B[3 * KSF + (TAIL ? p : 0)][j]);
                                dmma884(acc[p][1][j][0], acc[p][1][j][1], fa[q][0].y, B[3 * KSF + (TAIL ? p : 0)][j]);
                            }
                    }
                    // refill the slot with the k-step DA ahead in execution order
                    const int kn = ks + DA;                             // constants after unrolling
                    const double2* src = kn < KSPT ? pa : pn;
                    const int kr = kn < KSPT ? kn : kn - KSPT;
                    if (kr < KSF) {
#pragma unroll
                        for (int p = 0; p < 3; ++p) fa[q][p] = __ldg(src + (3 * kr + p) * 32);
                    } else {
                        fa[q][0] = __ldg(src + (3 * KSF) * 32);
                    }
                }
                double2* xw = xbuf + ((h * NBUF + buf) * NP) * 64;
                const double2* xr = xbuf + (((h ^ 1) * NBUF + buf) * NP) * 64;
                if (h == 0) x3_finish_task<NP, 0>(acc, xw, xr, 1, L, er, ei);
                else x3_finish_task<NP, 1>(acc, xw, xr, 1, L, er, ei);
                buf ^= 1;
            };
            // ASYNC: the same gamma-quad with the A fragments read from the shared-memory ring (slot = micro-load index) and the
            // slot refilled at once with the same micro-load of the NEXT task (cp.async from `pn`); the partner's tile of the
            // previous task is collected first, this task's tile is published without waiting
            auto task_async = [&](const double2* pn, const bool have_prev) {
                if (have_prev) x3_collect<NP>(keep, xbuf + (((h ^ 1) * NBUF + (buf ^ 1)) * NP) * 64, h, buf ^ 1, L, er, ei);
                // PHASED accumulation: Re = P0 - P2 and Im = P0 + P1 come out of the accumulators themselves.  Phase A runs the
                // P0 micro-steps of every k-step into acc[0]; acc[1] starts as a copy of it (register moves, not FP64
                // instructions); phase B subtracts P2 from acc[0] (negated B side) and adds P1 to acc[1], and the real-embedded
                // tail adds its Re and Im parts directly.  The 16 DADDs per task of the combination are gone (they cost the FP64
                // pipe 7-8 cycles each among DMMAs, profiles/r02c).  Commit groups follow the order of use: A_ks = the (Re+Im)
                // micro-load of k-step ks, then B_ks = its Re and Im micro-loads, then the tail: NGRP groups per task.
                constexpr int NGRP = 2 * KSF + TAIL;
#pragma unroll
                for (int ks = 0; ks < KSF; ++ks) {
                    cp_async_wait<NGRP - 1>();                          // group A_ks of this task has landed
                    const double2 f = ar[(3 * ks) * 32];
#pragma unroll
                    for (int j = 0; j < NP; ++j) {
                        dmma884(acc[0][0][j][0], acc[0][0][j][1], f.x, B[3 * ks][j]);
                        dmma884(acc[0][1][j][0], acc[0][1][j][1], f.y, B[3 * ks][j]);
                    }
                    cp_async16(ar + (3 * ks) * 32, pn + (3 * ks) * 32);
                    cp_async_commit();
                }
#pragma unroll
                for (int i = 0; i < 2; ++i)
#pragma unroll
                    for (int j = 0; j < NP; ++j) { acc[1][i][j][0] = acc[0][i][j][0]; acc[1][i][j][1] = acc[0][i][j][1]; }
#pragma unroll
                for (int ks = 0; ks < KSF; ++ks) {
                    cp_async_wait<NGRP - 1>();                          // group B_ks
                    const double2 f1 = ar[(3 * ks + 1) * 32], f2 = ar[(3 * ks + 2) * 32];
#pragma unroll
                    for (int j = 0; j < NP; ++j) {
                        dmma884(acc[1][0][j][0], acc[1][0][j][1], f1.x, B[3 * ks + 1][j]);      // Im += Ar (Bi - Br)
                        dmma884(acc[1][1][j][0], acc[1][1][j][1], f1.y, B[3 * ks + 1][j]);
                        dmma884(acc[0][0][j][0], acc[0][0][j][1], f2.x, B[3 * ks + 2][j]);      // Re -= Ai (Br + Bi)
                        dmma884(acc[0][1][j][0], acc[0][1][j][1], f2.y, B[3 * ks + 2][j]);
                    }
                    cp_async16(ar + (3 * ks + 1) * 32, pn + (3 * ks + 1) * 32);
                    cp_async16(ar + (3 * ks + 2) * 32, pn + (3 * ks + 2) * 32);
                    cp_async_commit();
                }
                if (TAIL) {
                    cp_async_wait<NGRP - 1>();
                    const double2 f = ar[(3 * KSF) * 32];
#pragma unroll
                    for (int p = 0; p < 2; ++p)
#pragma unroll
                        for (int j = 0; j < NP; ++j) {
                            dmma884(acc[p][0][j][0], acc[p][0][j][1], f.x, B[3 * KSF + (TAIL ? p : 0)][j]);
                            dmma884(acc[p][1][j][0], acc[p][1][j][1], f.y, B[3 * KSF + (TAIL ? p : 0)][j]);
                        }
                    cp_async16(ar + (3 * KSF) * 32, pn + (3 * KSF) * 32);
                    cp_async_commit();
                }
                double2* xw = xbuf + ((h * NBUF + buf) * NP) * 64;
                if (h == 0) x3_publish<NP, 0, true>(acc, keep, xw, h, buf, L);
                else x3_publish<NP, 1, true>(acc, keep, xw, h, buf, L);
                buf ^= 1;
            };
            for (int tq = 0; tq < GQ; ++tq) {
                const double2* pn = tq + 1 < GQ ? pa + TASK : pcont;
                if (ASYNC) task_async(pn, ab > 0 || tq > 0);
                else if (DA == 1 || base == 0) task(std::integral_constant<int, 0>(), pn);
                else task(std::integral_constant<int, 1 % DA>(), pn);
                base = (base + KSPT) % DA;
                pa += TASK;
            }
        }
        if (ASYNC) x3_collect<NP>(keep, xbuf + (((h ^ 1) * NBUF + (buf ^ 1)) * NP) * 64, h, buf ^ 1, L, er, ei);      // the item's last tile
        // ---- the item's result: lanes of each walker-in-pair (lane bit 1), then the two warps (fixed order) ----
#pragma unroll
        for (int j = 0; j < NP; ++j) {
            double r = er[j], i = ei[j];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                if (o == 2) continue;
                r += __shfl_xor_sync(0xffffffffu, r, o);
                i += __shfl_xor_sync(0xffffffffu, i, o);
            }
            er[j] = r; ei[j] = i;
        }
        if (h == 1 && (lane == 0 || lane == 2)) {
#pragma unroll
            for (int j = 0; j < NP; ++j) red[par * NWC + 2 * j + (lane >> 1)] = make_double2(er[j], ei[j]);
        }
        if (ASYNC) asm volatile("bar.sync 5, 64;" ::: "memory");      // (1..4 are the hand-over barriers)
        else asm volatile("bar.sync 1, 64;" ::: "memory");
        if (h == 0 && (lane == 0 || lane == 2)) {
#pragma unroll
            for (int j = 0; j < NP; ++j) {
                const int wl = 2 * j + (lane >> 1);
                const double2 o = red[par * NWC + wl];
                if (cur.w0 + wl < nw) partial[(size_t)cur.u * nw + cur.w0 + wl] = make_double2(er[j] + o.x, ei[j] + o.y);
            }
        }
        par ^= 1;
#pragma unroll
        for (int j = 0; j < NP; ++j) er[j] = ei[j] = 0.0;
        if (!has_next) break;
        item = nxt; cur = nx; bufsel ^= 1;
    }
    if (ASYNC) cp_async_wait<0>();      // (the last task refilled the ring once more: loaded, never used)
}

template <int NP>
size_t x3_smem_bytes(const X3Geom& g, int NGS, int NPAIR) {
    const size_t bs = (size_t)2 * NGS * (g.MSPT + 1) * 32 * NP * sizeof(double);
    const size_t xb = (size_t)NPAIR * 2 * 2 * NP * 64 * sizeof(double2);
    return bs + xb;
}

template <int NP, int NPAIR, int DA, int MINB, bool GRIDPAIRS, bool REAL>
int launch_x3_r(afqmc_ctx* c, const double2* theta, int nw, cudaStream_t st) {
    const Dims& d = c->d;
    const X3Geom g = REAL ? x3_geom_real(d.m) : x3_geom(d.m);
    const size_t smem = x3_smem_bytes<NP>(g, GRIDPAIRS ? 1 : d.NAG, NPAIR);
    auto kern = exchange3m_kernel<NP, NPAIR, DA, MINB, GRIDPAIRS, REAL>;
    if (int rc = afqmc_smem_optin(c, (const void*)kern, smem)) return rc;
    afqmc_prefer_smem(c, (const void*)kern);
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
    kern<<<(unsigned)nblocks, 64 * NPAIR, smem, st>>>(d, g, nchunk, nw, c->units, c->kminus, c->kplus, c->kneg, REAL ? c->Lxr : c->Lxc, theta, c->ws_expart);
    AFQMC_LAUNCH_CHECK(c);
    c->ex_parts = GRIDPAIRS ? npairs * nchunk : 1;
    return AFQMC_OK;
}

// real orbitals: the two-product variant (instantiated for the default prefetch depth only)
template <int NP, int NPAIR, int DA, int MINB, bool GRIDPAIRS>
int launch_x3(afqmc_ctx* c, const double2* theta, int nw, cudaStream_t st) {
    if ((DA == 3 || DA == 6) && c->real_lh && c->opt_real) return launch_x3_r<NP, NPAIR, DA, MINB, GRIDPAIRS, (DA == 3 || DA == 6)>(c, theta, nw, st);
    return launch_x3_r<NP, NPAIR, DA, MINB, GRIDPAIRS, false>(c, theta, nw, st);
}

// n-tiles per warp: 2 (four walkers per CTA) unless there are at most two walkers; 4 (eight walkers per CTA) on request
template <int NPAIR, int DA, bool GRIDPAIRS>
int launch_x3_np(afqmc_ctx* c, const double2* theta, int nw, cudaStream_t st) {
    int np = c->opt_exchange_np;
    if (np == 0) {
        np = nw <= 2 ? 1 : 2;
        // long rows (the Gamma-point supercell shape, m = 208): the staged theta blocks of four walkers leave room for one CTA
        // per SM only (160 KB); two walkers per CTA keep two CTAs resident (G1: exchange 1.95 -> 1.59 ms)
        const X3Geom g = (c->real_lh && c->opt_real) ? x3_geom_real(c->d.m) : x3_geom(c->d.m);
        const int ngs = GRIDPAIRS ? 1 : c->d.NAG;
        if (np == 2 && 2 * x3_smem_bytes<2>(g, ngs, NPAIR) > (size_t)c->smem_sm && 2 * x3_smem_bytes<1>(g, ngs, NPAIR) <= (size_t)c->smem_sm) np = 1;
    }
    // resident CTAs asked of the compiler: the register budget per thread is 65536 / (MINB * 64 * NPAIR)
    // two walkers per CTA: a k-step is only six DMMAs, so the A stream runs six k-steps ahead in registers (three left 43 % of
    // the warp samples of the Gamma-point shape G1 waiting for A fragments: DMMA pipe 41 % busy)
    if (np == 1) return launch_x3<1, NPAIR, (DA == 3 ? 6 : DA), (NPAIR == 1 ? 8 : 4), GRIDPAIRS>(c, theta, nw, st);
    if (np == 4) return launch_x3<4, NPAIR, (DA > 2 ? 2 : DA), (NPAIR == 1 ? 5 : 2), GRIDPAIRS>(c, theta, nw, st);
    return launch_x3<2, NPAIR, DA, (NPAIR == 1 ? 7 : 3), GRIDPAIRS>(c, theta, nw, st);
}

template <bool GRIDPAIRS>
int launch_x3_cfg(afqmc_ctx* c, const double2* theta, int nw, cudaStream_t st) {
    // Warp pairs per CTA: one (64 threads) while seven such CTAs fit an SM's shared memory (the register budget of the
    // two-walker-pair tile); when the staged theta blocks are larger than that (m = 52 at C4: 45 KB per CTA) two pairs share one
    // staging, which keeps 12 warps resident instead of 10 and halves the theta traffic (C4: 25.5 -> 20.6 ms; round 1's kernel:
    // 23.0 ms).  Option "exchange_warps" = 4 forces two pairs, = 2 one.
    const size_t smem1 = x3_smem_bytes<2>((c->real_lh && c->opt_real) ? x3_geom_real(c->d.m) : x3_geom(c->d.m), GRIDPAIRS ? 1 : c->d.NAG, 1);
    const bool two_pairs = GRIDPAIRS || c->opt_exchange_wpc == 4 || (c->opt_exchange_wpc == 0 && smem1 * 7 > (size_t)c->smem_sm);
    const int da = c->opt_exchange_depth == 2 ? 2 : 3;                     // option "exchange_depth": k-steps of A prefetch
    if (two_pairs) return da == 2 ? launch_x3_np<2, 2, GRIDPAIRS>(c, theta, nw, st) : launch_x3_np<2, 3, GRIDPAIRS>(c, theta, nw, st);
    return da == 2 ? launch_x3_np<1, 2, GRIDPAIRS>(c, theta, nw, st) : launch_x3_np<1, 3, GRIDPAIRS>(c, theta, nw, st);
}

template <int NP>
size_t x3_reg_smem_bytes(const Dims& d, bool async) {
    const size_t raw = (size_t)4 * 2 * NP * d.n * d.m * sizeof(double2);
    const X3Geom g = x3_geom(d.m);
    const size_t aring = async ? (size_t)2 * (3 * g.KSF + g.TAIL) * 32 * sizeof(double2) : 0;
    return raw + (size_t)2 * 2 * NP * 64 * sizeof(double2) + (size_t)2 * 2 * NP * sizeof(double2) + aring + 4 * sizeof(uint64_t);
}

template <int KSF, int TAIL, int NP, bool ASYNC>
int launch_x3_reg(afqmc_ctx* c, const double2* theta, int nw, cudaStream_t st) {
    // registers: MSPT * NP B fragments + 12 NP accumulators (doubles) + the A ring; 200 registers = five resident CTAs,
    // 168 = six, 128 = eight
    constexpr int MS = 3 * KSF + 2 * TAIL;
    constexpr int MAXREG = NP == 1 ? 168 : 255;
    const Dims& d = c->d;
    size_t smem = x3_reg_smem_bytes<NP>(d, ASYNC);
    // tuning aid "exchange_ctas": at most that many CTAs per SM (the shared-memory request is padded so that no more fit)
    if (c->opt_exchange_ctas > 0) {
        const size_t pad = ((size_t)c->smem_sm / c->opt_exchange_ctas - 1024) & ~(size_t)127;
        if (pad > smem && pad <= (size_t)c->smem_optin) smem = pad;
    }
    auto kern = exchange3m_reg_kernel<KSF, TAIL, NP, MAXREG, ASYNC>;
    if (int rc = afqmc_smem_optin(c, (const void*)kern, smem)) return rc;
    afqmc_prefer_smem(c, (const void*)kern);
    const long long nitems = (long long)c->nunits * ((nw + 2 * NP - 1) / (2 * NP));
    if (nitems > 0x7fffffffLL) return AFQMC_UNSUPPORTED;
    // persistent grid: as many CTAs as are resident (remembered per context)
    FuncAttr* f = afqmc_fattr(c, (const void*)kern);
    int occ = (f && f->occ_smem == (int)smem) ? f->occ : -1;
    if (occ < 0) {
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, 64, smem) != cudaSuccess) { (void)cudaGetLastError(); return AFQMC_CUDA_ERROR; }
        if (occ < 1) return AFQMC_UNSUPPORTED;
        if (f) { f->occ = occ; f->occ_smem = (int)smem; }
    }
    long long grid = (long long)occ * c->num_sms;
    if (grid > nitems) grid = nitems;
    kern<<<(unsigned)grid, 64, smem, st>>>(d, nw, (int)nitems, c->units, c->kminus, c->kplus, c->kneg, c->Lx3t, theta, c->ws_expart);
    AFQMC_LAUNCH_CHECK(c);
    c->ex_parts = 1;
    return AFQMC_OK;
}

template <int KSF, int TAIL>
int launch_x3_reg_np(afqmc_ctx* c, const double2* theta, int nw, cudaStream_t st) {
    // option exchange_regb: 1 = A stream by cp.async through a shared-memory ring + deferred hand-over (default), 2 = A stream
    // prefetched in registers + blocking hand-over
    const bool async = c->opt_exchange_regb != 2;
    if (nw <= 2 || c->opt_exchange_np == 1)      // two walkers per CTA
        return async ? launch_x3_reg<KSF, TAIL, 1, true>(c, theta, nw, st) : launch_x3_reg<KSF, TAIL, 1, false>(c, theta, nw, st);
    return async ? launch_x3_reg<KSF, TAIL, 2, true>(c, theta, nw, st) : launch_x3_reg<KSF, TAIL, 2, false>(c, theta, nw, st);
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
    const X3Geom g = x3_geom(c->d.m);
    // m <= 28: the theta block of a warp lives in registers (unless the tuning options ask for the generic kernel)
    // (real orbitals: the generic kernel has the two-product variant)
    if (c->opt_exchange_regb && x3_prefers_reg(c->d) && c->opt_exchange_np <= 1 && c->opt_exchange_wpc != 4 && !(c->real_lh && c->opt_real)) {
        int rc = ensure_operand(c, true, st);
        if (rc != AFQMC_OK) return rc;
        rc = AFQMC_UNSUPPORTED;
        switch (g.KSF * 2 + g.TAIL) {
#define X3_CASE(KSF_, TAIL_) case (KSF_) * 2 + (TAIL_): rc = launch_x3_reg_np<KSF_, TAIL_>(c, theta, nw, st); break;
            X3_CASE(0, 1) X3_CASE(1, 0) X3_CASE(1, 1) X3_CASE(2, 0) X3_CASE(2, 1) X3_CASE(3, 0) X3_CASE(3, 1)
            X3_CASE(4, 0) X3_CASE(4, 1) X3_CASE(5, 0) X3_CASE(5, 1) X3_CASE(6, 0) X3_CASE(6, 1) X3_CASE(7, 0)
#undef X3_CASE
            default: break;
        }
        if (rc != AFQMC_UNSUPPORTED) return rc;      // else: the raw theta blocks of all orbitals exceed shared memory
    }
    int rc = (c->real_lh && c->opt_real && c->opt_exchange_depth != 2) ? ensure_lxr(c, st) : ensure_operand(c, false, st);
    if (rc != AFQMC_OK) return rc;
    rc = launch_x3_cfg<false>(c, theta, nw, st);
    if (rc == AFQMC_UNSUPPORTED && c->d.NAG > 1 && c->ex_parts_max > 1) rc = launch_x3_cfg<true>(c, theta, nw, st);
    return rc;
}
