// a7 one-body, a8 Coulomb, a9 exchange energy (Eq. 49; recipe PAPER.md:306-319).
//
// Exchange.  With T^Q[(k,a),(k2,b),g] = sum_r Lh[Q][k][a][g][r] theta[(k2,b),(k-Q,r)] the paper's
// T1(Q,k,k')[b,a,g] is T^Q[(k,a),(k'-Q,b),g] and T2(Q,k,k')[a,b,g] is T^{-Q}[(k'-Q,b),(k,a),g]
// (it uses Lh[-Q][k'-Q], which is Lbar of Eq. 40 under the (Q,-Q) identity of PAPER.md:216), so
//     EX = - sum_{Q,k,k2} X(Q,k,k2),   X = sum_{a,b,g} T^Q[(k,a),(k2,b),g] T^{-Q}[(k2,b),(k,a),g]
// and X(Q,k,k2) = X(-Q,k2,k): the map is an involution, so only one unit of each pair is computed
// (weight 2; fixed points weight 1).  The T tensors never leave the SM: a work unit forms both
// n x n x gamma blocks with DMMA (rows = (gamma pair, a), cols = (b, re/im), K = (r, re/im)),
// transposes one of them across lanes with a shuffle, and contracts in registers.  This replaces
// the paper's T1/T2 global buffers and its separate contraction kernel.
#include "common.cuh"

namespace {


// lane' holding the (a,b)-transposed element inside a 16-lane group of a C fragment
__device__ __forceinline__ int transpose_lane(int lane) { return (lane & 16) | ((lane & 3) << 2) | ((lane >> 2) & 3); }

// ---------------------------------------------------------------------------------------------
// Exchange kernel.  CTA = (unit, group of NT walkers), WPC warps.
//  * B fragments (the two theta blocks of the unit, real-embedded) are staged once per CTA in
//    shared memory in fragment order.
//  * A fragments (Lx) are a LINEAR stream per warp: a warp task is one gamma-quad (two DMMA m-tiles,
//    rows (gamma pair, a)) and the layout Lx[Q][k][ag][gq][s][lane][2] makes every k-step of a task one
//    coalesced 512-byte LDG.128 per operand; consecutive tasks of a warp are consecutive in memory.
//  * Both fragment streams run D k-steps ahead of the DMMAs in statically rotated register buffers
//    (the loop over the warp's flattened (task, k-step) sequence is unrolled by D), so neither the L2
//    round trip of A nor the shared-memory latency of B is exposed, also across task boundaries.
//    With n <= 4 (LINEAR) the refill is branch-free pointer arithmetic, so the loads of a k-step are
//    scheduled between its DMMAs; the refill may run up to D k-steps past the warp's last task, into
//    the next block or the zero pad after Lx (loaded, never used).
//  * The host picks WPC so that the tasks divide evenly over the warps; walker groups of one unit are
//    adjacent in the grid so that the Lx blocks of a unit are fetched from HBM once and shared in L2.
// ---------------------------------------------------------------------------------------------
template <int NT, int WPC, int D, bool LINEAR, int MINB>
__global__ void __launch_bounds__(32 * WPC, MINB) exchange_kernel(
    Dims d, int nw, const int* __restrict__ units, const int* __restrict__ kminus, const int* __restrict__ kplus,
    const int* __restrict__ kneg, const double* __restrict__ Lx, const double2* __restrict__ theta,
    double2* __restrict__ partial) {
    extern __shared__ __align__(16) double ex_smem[];
    const int nwg = (nw + NT - 1) / NT;             // walker groups of one unit are adjacent in the grid
    const int u = blockIdx.x / nwg, w0 = (blockIdx.x % nwg) * NT;
    const int Q = units[4 * u], k = units[4 * u + 1], k2 = units[4 * u + 2];
    const int mQ = kneg[Q];
    const int kq = kminus[k * d.Nk + Q];        // k - Q   : column block of theta for T^Q rows k
    const int k2pq = kplus[k2 * d.Nk + Q];      // k2 + Q  : column block of theta for T^{-Q} rows k2
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int KS = d.KS, NAG = d.NAG, GQ = d.GQ;
    // Bs[which][grp][s][j][lane]: which = 0 -> theta[(k2,b),(k-Q,r)], 1 -> theta[(k,a),(k2+Q,s)]
    const int bs_step = NT * 32, bs_grp = KS * bs_step, bs_half = NAG * bs_grp;

    // ---- this warp's contiguous share of the CTA's tasks t = (ag*NAG + bg)*GQ + gq ----
    const int ntask = NAG * NAG * GQ;
    const int t_begin = (int)((long long)warp * ntask / WPC), t_end = (int)((long long)(warp + 1) * ntask / WPC);
    const int total = (t_end - t_begin) * KS;                       // k-steps of this warp
    const size_t blk1 = ((size_t)Q * d.Nk + k) * NAG, blk2 = ((size_t)mQ * d.Nk + k2) * NAG;
    const size_t task_doubles = (size_t)KS * 64;
    // loader state: runs D k-steps ahead of the compute state
    int lt = t_begin, ls = 0, lg = 0;
    const double2 *la1, *la2;
    const double *lb1, *lb2;
    auto task_ptrs = [&](int t) {
        const int gq = t % GQ, ab = t / GQ, bg = ab % NAG, ag = ab / NAG;
        la1 = reinterpret_cast<const double2*>(Lx + ((blk1 + ag) * GQ + gq) * task_doubles) + lane;
        la2 = reinterpret_cast<const double2*>(Lx + ((blk2 + bg) * GQ + gq) * task_doubles) + lane;
        lb1 = ex_smem + bg * bs_grp + lane;
        lb2 = ex_smem + bs_half + ag * bs_grp + lane;
    };
    auto loader_advance = [&]() {
        if (LINEAR) {                    // one (ag,bg): A is contiguous across tasks, B wraps every KS steps
            la1 += 32; la2 += 32;
            const bool wrap = ++ls == KS;
            const int db = wrap ? -(KS - 1) * bs_step : bs_step;
            lb1 += db; lb2 += db;
            ls = wrap ? 0 : ls;
        } else {
            ++lg;
            if (++ls == KS) {
                ls = 0; ++lt;
                if (lg < total) task_ptrs(lt);
            } else {
                la1 += 32; la2 += 32; lb1 += bs_step; lb2 += bs_step;
            }
        }
    };
    double2 fa1[D], fa2[D];
    double fb1[D][NT], fb2[D][NT];
    task_ptrs(total > 0 ? lt : 0);
    // A prologue: the global loads are issued before the staging below, which hides their latency
#pragma unroll
    for (int q = 0; q < D; ++q) {
        fa1[q] = fa2[q] = make_double2(0.0, 0.0);
        if (LINEAR) {
            if (total > 0) { fa1[q] = __ldg(la1 + q * 32); fa2[q] = __ldg(la2 + q * 32); }
        } else if (q < total) {         // D <= KS is guaranteed by the host, so the prologue stays in task lt
            fa1[q] = __ldg(la1 + q * 32); fa2[q] = __ldg(la2 + q * 32);
        }
    }

    // ---- stage B fragments.  One thread per complex theta element (b, r): all loads of the CTA are
    // independent (one L2 round trip in total), and each element feeds the four fragment entries
    //   (kk = 2(r&1)+c, col = 2(b&3)+d):  d=0: (re, -im) for c = 0,1;  d=1: (im, re).
    {
        const int per_which = NAG * 4 * NT * 2 * KS;             // padded (orb, walker, r) space
        for (int e = tid; e < 2 * per_which; e += 32 * WPC) {
            const int which = e / per_which;
            int x = e - which * per_which;
            const int bl = x & 3; x >>= 2;                       // orbital inside its group of 4
            const int jw = x % NT; x /= NT;
            const int grp = x % NAG, r = x / NAG;                // r < 2*KS
            const int orb = 4 * grp + bl, w = w0 + jw;
            const int rowblk = which == 0 ? k2 : k, colblk = which == 0 ? kq : k2pq;
            double2 v = make_double2(0.0, 0.0);
            if (orb < d.n && w < nw && r < d.m)
                v = __ldg(theta + ((size_t)w * d.N + rowblk * d.n + orb) * d.M + (size_t)colblk * d.m + r);
            double* dst = ex_smem + which * bs_half + ((grp * KS + (r >> 1)) * NT + jw) * 32 + bl * 8 + 2 * (r & 1);
            *reinterpret_cast<double2*>(dst) = make_double2(v.x, -v.y);       // d = 0: lanes (kk = 2(r&1)+{0,1}, col = 2bl)
            *reinterpret_cast<double2*>(dst + 4) = make_double2(v.y, v.x);    // d = 1: col = 2bl+1
        }
    }
    __syncthreads();   // B fragments staged

    // B prologue, and bring the loader state to step D
#pragma unroll
    for (int q = 0; q < D; ++q) {
        if (LINEAR || q < total) {
#pragma unroll
            for (int j = 0; j < NT; ++j) { fb1[q][j] = lb1[j * 32]; fb2[q][j] = lb2[j * 32]; }
            loader_advance();
        } else {
#pragma unroll
            for (int j = 0; j < NT; ++j) fb1[q][j] = fb2[q][j] = 0.0;
        }
    }

    double er[NT], ei[NT];
#pragma unroll
    for (int j = 0; j < NT; ++j) er[j] = ei[j] = 0.0;
    const int srcl = transpose_lane(lane);
    double acc1[2][NT][2], acc2[2][NT][2];
#pragma unroll
    for (int i = 0; i < 2; ++i)
#pragma unroll
        for (int j = 0; j < NT; ++j) acc1[i][j][0] = acc1[i][j][1] = acc2[i][j][0] = acc2[i][j][1] = 0.0;

    int cs = 0;   // k-step of the compute state inside its task
    // one k-step on register buffer q: 4*NT DMMAs, refill of the buffer, contraction at the end of a task
    auto kstep = [&](const int q) {
#pragma unroll
        for (int j = 0; j < NT; ++j) {
            dmma884(acc1[0][j][0], acc1[0][j][1], fa1[q].x, fb1[q][j]);
            dmma884(acc1[1][j][0], acc1[1][j][1], fa1[q].y, fb1[q][j]);
        }
#pragma unroll
        for (int j = 0; j < NT; ++j) {
            dmma884(acc2[0][j][0], acc2[0][j][1], fa2[q].x, fb2[q][j]);
            dmma884(acc2[1][j][0], acc2[1][j][1], fa2[q].y, fb2[q][j]);
        }
        if (LINEAR || lg < total) {      // refill buffer q with the k-step D ahead
            fa1[q] = __ldg(la1); fa2[q] = __ldg(la2);
#pragma unroll
            for (int j = 0; j < NT; ++j) { fb1[q][j] = lb1[j * 32]; fb2[q][j] = lb2[j * 32]; }
            loader_advance();
        }
        if (++cs == KS) {
            cs = 0;
            // contract: lane holds T1[(g,a),(b)]; fetch T2[(g,b),(a)] from the transposed lane
#pragma unroll
            for (int i = 0; i < 2; ++i)
#pragma unroll
                for (int j = 0; j < NT; ++j) {
                    double t2r = __shfl_sync(0xffffffffu, acc2[i][j][0], srcl);
                    double t2i = __shfl_sync(0xffffffffu, acc2[i][j][1], srcl);
                    er[j] = fma(acc1[i][j][0], t2r, er[j]);
                    er[j] = fma(-acc1[i][j][1], t2i, er[j]);
                    ei[j] = fma(acc1[i][j][0], t2i, ei[j]);
                    ei[j] = fma(acc1[i][j][1], t2r, ei[j]);
                    acc1[i][j][0] = acc1[i][j][1] = acc2[i][j][0] = acc2[i][j][1] = 0.0;
                }
        }
    };
    const int nfull = total - total % D;
    for (int g0 = 0; g0 < nfull; g0 += D) {
#pragma unroll
        for (int q = 0; q < D; ++q) kstep(q);
    }
#pragma unroll
    for (int q = 0; q < D - 1; ++q)
        if (nfull + q < total) kstep(q);

    // ---- reduce over lanes and warps (deterministic) ----
    __syncthreads();
    double* red = ex_smem;   // reuse: [warp][NT][2]
#pragma unroll
    for (int j = 0; j < NT; ++j) {
        double r = warp_sum(er[j]), i = warp_sum(ei[j]);
        if (lane == 0) { red[(warp * NT + j) * 2] = r; red[(warp * NT + j) * 2 + 1] = i; }
    }
    __syncthreads();
    if (tid < NT && w0 + tid < nw) {
        double r = 0.0, i = 0.0;
        for (int x = 0; x < WPC; ++x) { r += red[(x * NT + tid) * 2]; i += red[(x * NT + tid) * 2 + 1]; }
        partial[(size_t)u * nw + w0 + tid] = make_double2(r, i);
    }
}

// ---------------------------------------------------------------------------------------------
// Final reduction: one CTA per walker.  E1 (a7), EC from the force bias (a8), EX from the unit partials.
// ---------------------------------------------------------------------------------------------
__device__ double2 block_sum2(double2 v, double* scratch /* >= 64 doubles */) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
    v.x = warp_sum(v.x); v.y = warp_sum(v.y);
    __syncthreads();
    if (lane == 0) { scratch[warp] = v.x; scratch[32 + warp] = v.y; }
    __syncthreads();
    double2 r = make_double2(0.0, 0.0);
    for (int x = 0; x < nwarps; ++x) { r.x += scratch[x]; r.y += scratch[32 + x]; }
    return r;
}

// One spin channel's inputs of the final reduction
struct FinChan {
    int n, N, nunits, parts;
    const int* units;
    const double2 *ht, *theta, *vbias, *partial;      // vbias: this channel's force bias including its spin factor
};

// sf = spin factor (2: closed shell, one channel for both spins; 1: open shell, two channels):
//   E1 = sf sum_ch sum ht theta;   EC = 1/2 sum_Q sum_g v[Q][g] v[-Q][g], v = sum_ch vbias_ch;   EX = -(sf/2) sum_ch sum_units mult X
__global__ void __launch_bounds__(1024) energy_finalize_kernel(
    Dims d, int nw, int nchan, double sf, FinChan c0, FinChan c1, const int* __restrict__ kneg, double2* __restrict__ energy) {
    __shared__ double scratch[64];
    const int w = blockIdx.x, tid = threadIdx.x;
    double2 e1 = make_double2(0.0, 0.0), ex = make_double2(0.0, 0.0);
    for (int ch = 0; ch < nchan; ++ch) {
        const FinChan& c = ch == 0 ? c0 : c1;
        // E1 = sum_k sum_{a,q} ht[k][a][q] theta[(k,a),(k,q)]
        for (int e = tid; e < d.Nk * c.n * d.m; e += blockDim.x) {
            int q = e % d.m, ka = e / d.m, k = ka / c.n;
            e1 = cfma(c.ht[e], c.theta[((size_t)w * c.N + ka) * d.M + (size_t)k * d.m + q], e1);
        }
        // EX = - sum_units mult * X(unit); `parts` partial sums per unit (1 except for large blocks)
        for (int idx = tid; idx < c.nunits * c.parts; idx += blockDim.x) {
            double mult = (double)c.units[4 * (idx / c.parts) + 3];
            double2 p = c.partial[(size_t)idx * nw + w];
            ex.x += mult * p.x; ex.y += mult * p.y;
        }
    }
    e1 = block_sum2(e1, scratch);
    ex = block_sum2(ex, scratch);
    // EC = 1/2 sum_Q sum_g v[Q][g] v[-Q][g]
    double2 ec = make_double2(0.0, 0.0);
    for (int e = tid; e < d.Nk * d.nchol; e += blockDim.x) {
        int g = e % d.nchol, Q = e / d.nchol;
        const size_t i0 = ((size_t)w * d.Nk + Q) * d.nchol + g, i1 = ((size_t)w * d.Nk + kneg[Q]) * d.nchol + g;
        double2 a = c0.vbias[i0], b = c0.vbias[i1];
        if (nchan > 1) { const double2 a1 = c1.vbias[i0], b1 = c1.vbias[i1]; a.x += a1.x; a.y += a1.y; b.x += b1.x; b.y += b1.y; }
        ec = cfma(a, b, ec);
    }
    ec = block_sum2(ec, scratch);
    if (tid == 0) {
        energy[w * 3 + 0] = make_double2(sf * e1.x, sf * e1.y);
        energy[w * 3 + 1] = make_double2(0.5 * ec.x, 0.5 * ec.y);
        energy[w * 3 + 2] = make_double2(-0.5 * sf * ex.x, -0.5 * sf * ex.y);
    }
}

template <int NT, int WPC, int D, bool LINEAR, int MINB>
int launch_exchange_cfg(afqmc_ctx* c, const double2* theta, int nw, cudaStream_t st) {
    const Dims& d = c->d;
    size_t smem = (size_t)2 * d.NAG * d.KS * NT * 32 * sizeof(double);
    if (smem < (size_t)WPC * NT * 2 * sizeof(double)) smem = (size_t)WPC * NT * 2 * sizeof(double);
    auto kern = exchange_kernel<NT, WPC, D, LINEAR, MINB>;
    if (int rc = afqmc_smem_optin(c, (const void*)kern, smem)) return rc;
    const long long nblocks = (long long)((nw + NT - 1) / NT) * c->nunits;   // x only: y/z are capped at 65535
    if (nblocks > 0x7fffffffLL) return AFQMC_UNSUPPORTED;
    dim3 grid((unsigned)nblocks);
    kern<<<grid, 32 * WPC, smem, st>>>(d, nw, c->units, c->kminus, c->kplus, c->kneg, c->Lx, theta, c->ws_expart);
    AFQMC_LAUNCH_CHECK(c);
    return AFQMC_OK;
}

template <int NT, int WPC, int MINB>
int launch_exchange_wm(afqmc_ctx* c, const double2* theta, int nw, cudaStream_t st) {
    const bool linear = c->d.NAG == 1;
    const int depth = (c->opt_exchange_depth == 3 && c->d.KS >= 3) ? 3 : (c->d.KS >= 2 ? 2 : 1);
    if (depth == 3) return linear ? launch_exchange_cfg<NT, WPC, 3, true, MINB>(c, theta, nw, st)
                                  : launch_exchange_cfg<NT, WPC, 3, false, MINB>(c, theta, nw, st);
    if (depth == 2) return linear ? launch_exchange_cfg<NT, WPC, 2, true, MINB>(c, theta, nw, st)
                                  : launch_exchange_cfg<NT, WPC, 2, false, MINB>(c, theta, nw, st);
    return launch_exchange_cfg<NT, WPC, 1, false, MINB>(c, theta, nw, st);     // m = 1: a single k-step per task
}

template <int NT, int WPC>
int launch_exchange_w(afqmc_ctx* c, const double2* theta, int nw, cudaStream_t st) {
    constexpr int MB0 = WPC == 2 ? 4 : (WPC > 6 ? 1 : 2), MB1 = WPC == 2 ? 6 : (WPC == 4 ? 3 : MB0);
    if (c->opt_exchange_minb == 1) return launch_exchange_wm<NT, WPC, MB1>(c, theta, nw, st);
    return launch_exchange_wm<NT, WPC, MB0>(c, theta, nw, st);
}

// Warps per CTA: the count in {2,4,6} that keeps the most warps resident per SM (up to 12 = 3 per
// scheduler; limited by the staged theta blocks in shared memory and by ~160 registers per thread),
// then the one that deals the tasks out most evenly, then the smallest (small CTAs drift out of
// lockstep, so their prologues overlap other CTAs' DMMAs).
template <int NT>
int launch_exchange(afqmc_ctx* c, const double2* theta, int nw, cudaStream_t st) {
    const Dims& d = c->d;
    const int ntask = d.NAG * d.NAG * d.GQ;
    int best = c->opt_exchange_wpc;
    if (best == 0) {
        const size_t smem = (size_t)2 * d.NAG * d.KS * NT * 32 * sizeof(double) + 1024;
        double bests = -1.0;
        const int cand[3] = {2, 4, 6};
        for (int w : cand) {
            const int by_smem = (int)((size_t)c->smem_sm / smem), by_regs = 65536 / (160 * 32 * w);
            const int warps = (by_smem < by_regs ? by_smem : by_regs) * w;
            const double cost = (double)((ntask + w - 1) / w) * w / ntask;   // >= 1, 1 = perfectly even
            const double score = (warps < 12 ? warps : 12) / cost;
            if (score > bests + 1e-9) { bests = score; best = w; }
        }
    }
    switch (best) {
        case 2: return launch_exchange_w<NT, 2>(c, theta, nw, st);
        case 4: return launch_exchange_w<NT, 4>(c, theta, nw, st);
        case 5: return launch_exchange_w<NT, 5>(c, theta, nw, st);
        case 8: return launch_exchange_w<NT, 8>(c, theta, nw, st);
        default: return launch_exchange_w<NT, 6>(c, theta, nw, st);
    }
}

}  // namespace

// force bias (the traces of steps 2(d)) and exchange partial sums of ONE spin channel, left in its workspace
static int channel_energy_parts(afqmc_ctx* c, afqmc_ctx* timers, const double2* theta, int nw, cudaStream_t st) {
    int rc = afqmc_i_force_bias(c, theta, nw, c->ws_vbias, st);     // steps 2(d): the traces are the force bias
    if (rc != AFQMC_OK) return rc;
    if (timers) afqmc_mark(timers, 6, st);
    c->ex_parts = 1;
    if (c->opt_exchange_prec != 0) {       // mixed precision: tcgen05 kernel, else (or if it cannot take the shape) the mma.sync one
        rc = c->opt_exchange_tc ? afqmc_i_exchange_tc(c, theta, nw, st) : AFQMC_UNSUPPORTED;
        if (rc == AFQMC_UNSUPPORTED && (rc = afqmc_i_ensure_lxt(c, st)) == AFQMC_OK) rc = afqmc_i_exchange_tf32(c, theta, nw, st);
    } else {
        rc = c->opt_exchange_3m ? afqmc_i_exchange3m(c, theta, nw, st) : AFQMC_UNSUPPORTED;
    }
    if (rc == AFQMC_UNSUPPORTED) {          // the 4M kernel was asked for (or the TF32 option with n > 4)
        if ((rc = afqmc_i_ensure_lx(c, st)) != AFQMC_OK) return rc;
        if (nw >= 3) rc = launch_exchange<4>(c, theta, nw, st);
        else rc = launch_exchange<2>(c, theta, nw, st);
    }
    return rc;
}

static FinChan fin_chan(const afqmc_ctx* c, const double2* theta) {
    FinChan f;
    f.n = c->d.n; f.N = c->d.N; f.nunits = c->nunits; f.parts = c->ex_parts;
    f.units = c->units; f.ht = c->ht; f.theta = theta; f.vbias = c->ws_vbias; f.partial = c->ws_expart;
    return f;
}

// theta: [nw][N][M]; open shell: the spin-up block followed by the spin-down block [nw][N_dn][M]
int afqmc_i_local_energy(afqmc_ctx* c, const double2* theta, int nw, double2* energy, cudaStream_t st) {
    const Dims& d = c->d;
    int rc = channel_energy_parts(c, c->dn ? nullptr : c, theta, nw, st);
    if (rc != AFQMC_OK) return rc;
    const double2* theta_dn = theta + (size_t)nw * d.N * d.M;
    if (c->dn) {
        if ((rc = channel_energy_parts(c->dn, nullptr, theta_dn, nw, st)) != AFQMC_OK) return rc;
        afqmc_mark(c, 6, st);
    }
    afqmc_mark(c, 7, st);
    const FinChan f0 = fin_chan(c, theta), f1 = c->dn ? fin_chan(c->dn, theta_dn) : f0;
    energy_finalize_kernel<<<nw, 1024, 0, st>>>(d, nw, c->dn ? 2 : 1, c->spin_factor, f0, f1, c->kneg, energy);
    AFQMC_LAUNCH_CHECK(c);
    return AFQMC_OK;
}

AFQMC_API int afqmc_local_energy(afqmc_ctx* c, const void* theta, int nw, void* energy, void* stream) {
    if (!c || !theta || !energy || nw < 0 || nw > c->max_walkers) return AFQMC_INVALID_ARGUMENT;
    if (nw == 0) return AFQMC_OK;
    if (c->prec32) return afqmc32_local_energy(c, theta, nw, energy, (cudaStream_t)stream);
    return afqmc_i_local_energy(c, (const double2*)theta, nw, (double2*)energy, (cudaStream_t)stream);
}
