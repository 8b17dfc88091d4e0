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
// Variant 1 ("simple"): B fragments (theta blocks, real-embedded) staged once per CTA in shared
// memory; A fragments (Lx tiles) loaded straight from global/L2 in lane order, software-pipelined
// one k-step ahead ACROSS tasks so that no task starts with an exposed L2 round trip.
// CTA = (unit, group of NT walkers), WPC warps.  A warp task is a group of MT gamma-pair tiles; the
// host picks WPC so that the tasks divide evenly over the warps (no tail at the final barrier).
// Walker groups of one unit are adjacent in the grid so that the Lx blocks of a unit are fetched
// from HBM once and shared through L2.
// ---------------------------------------------------------------------------------------------
template <int MT, int NT, int WPC>
__global__ void __launch_bounds__(32 * WPC, 16 / WPC) exchange_simple_kernel(
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
    const int KS = d.KS, NAG = d.NAG;
    // Bs[which][grp][s][j][lane]: which = 0 -> theta[(k2,b),(k-Q,r)], 1 -> theta[(k,a),(k2+Q,s)]
    const size_t bs_half = (size_t)NAG * KS * NT * 32;

    // ---- stage B fragments: one (which, grp, walker) fragment column per warp pass, lane = fragment lane ----
    {
        const int kkk = lane & 3, col = lane >> 2;
        const int dd = col & 1, cc = kkk & 1;
        const bool neg = cc && !dd;
        for (int c = warp; c < 2 * NAG * NT; c += WPC) {
            const int jw = c % NT, grp = (c / NT) % NAG, which = c / (NT * NAG);
            const int orb = 4 * grp + (col >> 1), w = w0 + jw;
            const int rowblk = which == 0 ? k2 : k, colblk = which == 0 ? kq : k2pq;
            const bool ok = orb < d.n && w < nw;
            const double* src = reinterpret_cast<const double*>(
                theta + ((size_t)(ok ? w : 0) * d.N + rowblk * d.n + (ok ? orb : 0)) * d.M + (size_t)colblk * d.m + (kkk >> 1)) + (cc ^ dd);
            double* dst = ex_smem + which * bs_half + ((size_t)grp * KS * NT + jw) * 32 + lane;
            for (int s = 0; s < KS; ++s) {
                double v = 0.0;
                if (ok && 2 * s + (kkk >> 1) < d.m) v = __ldg(src + 4 * s);
                dst[(size_t)s * NT * 32] = neg ? -v : v;
            }
        }
    }

    double er[NT], ei[NT];
#pragma unroll
    for (int j = 0; j < NT; ++j) er[j] = ei[j] = 0.0;
    const int srcl = transpose_lane(lane);
    const int ngrp = (d.GP + MT - 1) / MT;
    const size_t tile = (size_t)KS * 32;
    // flattened task list of this warp: t = warp, warp+WPC, ... < NAG*NAG*ngrp ; t -> (ag, bg, mg)
    const int ntask = NAG * NAG * ngrp;
    auto task_ptrs = [&](int t, const double*& a1, const double*& a2, int& ag, int& bg, int& mg) {
        mg = t % ngrp;
        const int ab = t / ngrp;
        bg = ab % NAG; ag = ab / NAG;
        a1 = Lx + ((((size_t)Q * d.Nk + k) * NAG + ag) * d.GP + (size_t)mg * MT) * tile + lane;
        a2 = Lx + ((((size_t)mQ * d.Nk + k2) * NAG + bg) * d.GP + (size_t)mg * MT) * tile + lane;
    };
    const double *a1 = nullptr, *a2 = nullptr;
    int ag = 0, bg = 0, mg = 0;
    double fa1[MT], fa2[MT];
    int t = warp;
    if (t < ntask) {
        task_ptrs(t, a1, a2, ag, bg, mg);
#pragma unroll
        for (int i = 0; i < MT; ++i) {
            const bool ok = mg * MT + i < d.GP;
            fa1[i] = ok ? __ldg(a1 + i * tile) : 0.0;
            fa2[i] = ok ? __ldg(a2 + i * tile) : 0.0;
        }
    }
    __syncthreads();   // B fragments staged

    for (; t < ntask; t += WPC) {
        const double* b1 = ex_smem + (size_t)bg * KS * NT * 32 + lane;
        const double* b2 = ex_smem + bs_half + (size_t)ag * KS * NT * 32 + lane;
        // pointers of the next task (for the cross-task prefetch at the last k-step)
        const double *n1 = a1, *n2 = a2;
        int nag = ag, nbg = bg, nmg = mg;
        const bool has_next = t + WPC < ntask;
        if (has_next) task_ptrs(t + WPC, n1, n2, nag, nbg, nmg);
        double acc1[MT][NT][2], acc2[MT][NT][2];
#pragma unroll
        for (int i = 0; i < MT; ++i)
#pragma unroll
            for (int j = 0; j < NT; ++j) acc1[i][j][0] = acc1[i][j][1] = acc2[i][j][0] = acc2[i][j][1] = 0.0;
        for (int s = 0; s < KS; ++s) {
            double ca1[MT], ca2[MT];
#pragma unroll
            for (int i = 0; i < MT; ++i) { ca1[i] = fa1[i]; ca2[i] = fa2[i]; }
            if (s + 1 < KS) {
#pragma unroll
                for (int i = 0; i < MT; ++i) {
                    const bool ok = mg * MT + i < d.GP;
                    fa1[i] = ok ? __ldg(a1 + i * tile + (s + 1) * 32) : 0.0;
                    fa2[i] = ok ? __ldg(a2 + i * tile + (s + 1) * 32) : 0.0;
                }
            } else if (has_next) {
#pragma unroll
                for (int i = 0; i < MT; ++i) {
                    const bool ok = nmg * MT + i < d.GP;
                    fa1[i] = ok ? __ldg(n1 + i * tile) : 0.0;
                    fa2[i] = ok ? __ldg(n2 + i * tile) : 0.0;
                }
            }
            double fb1[NT], fb2[NT];
#pragma unroll
            for (int j = 0; j < NT; ++j) {
                fb1[j] = b1[((size_t)s * NT + j) * 32];
                fb2[j] = b2[((size_t)s * NT + j) * 32];
            }
#pragma unroll
            for (int i = 0; i < MT; ++i)
#pragma unroll
                for (int j = 0; j < NT; ++j) dmma884(acc1[i][j][0], acc1[i][j][1], ca1[i], fb1[j]);
#pragma unroll
            for (int i = 0; i < MT; ++i)
#pragma unroll
                for (int j = 0; j < NT; ++j) dmma884(acc2[i][j][0], acc2[i][j][1], ca2[i], fb2[j]);
        }
        // contract: lane holds T1[(g,a),(b)]; fetch T2[(g,b),(a)] from the transposed lane
#pragma unroll
        for (int i = 0; i < MT; ++i)
#pragma unroll
            for (int j = 0; j < NT; ++j) {
                double t2r = __shfl_sync(0xffffffffu, acc2[i][j][0], srcl);
                double t2i = __shfl_sync(0xffffffffu, acc2[i][j][1], srcl);
                er[j] = fma(acc1[i][j][0], t2r, er[j]);
                er[j] = fma(-acc1[i][j][1], t2i, er[j]);
                ei[j] = fma(acc1[i][j][0], t2i, ei[j]);
                ei[j] = fma(acc1[i][j][1], t2r, ei[j]);
            }
        a1 = n1; a2 = n2; ag = nag; bg = nbg; mg = nmg;
    }

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

__global__ void __launch_bounds__(256) energy_finalize_kernel(
    Dims d, int nw, int nunits, const int* __restrict__ units, const int* __restrict__ kneg,
    const double2* __restrict__ ht, const double2* __restrict__ theta, const double2* __restrict__ vbias,
    const double2* __restrict__ partial, double2* __restrict__ energy) {
    __shared__ double scratch[64];
    const int w = blockIdx.x, tid = threadIdx.x;
    // E1 = 2 sum_k sum_{a,q} ht[k][a][q] theta[(k,a),(k,q)]
    double2 e1 = make_double2(0.0, 0.0);
    for (int e = tid; e < d.Nk * d.n * d.m; e += blockDim.x) {
        int q = e % d.m, ka = e / d.m, k = ka / d.n;
        e1 = cfma(ht[e], theta[((size_t)w * d.N + ka) * d.M + (size_t)k * d.m + q], e1);
    }
    e1 = block_sum2(e1, scratch);
    // EC = 1/2 sum_Q sum_g v[Q][g] v[-Q][g]
    double2 ec = make_double2(0.0, 0.0);
    for (int e = tid; e < d.Nk * d.nchol; e += blockDim.x) {
        int g = e % d.nchol, Q = e / d.nchol;
        ec = cfma(vbias[((size_t)w * d.Nk + Q) * d.nchol + g], vbias[((size_t)w * d.Nk + kneg[Q]) * d.nchol + g], ec);
    }
    ec = block_sum2(ec, scratch);
    // EX = - sum_units mult * X(unit)
    double2 ex = make_double2(0.0, 0.0);
    for (int u = tid; u < nunits; u += blockDim.x) {
        double mult = (double)units[4 * u + 3];
        double2 p = partial[(size_t)u * nw + w];
        ex.x += mult * p.x; ex.y += mult * p.y;
    }
    ex = block_sum2(ex, scratch);
    if (tid == 0) {
        energy[w * 3 + 0] = make_double2(2.0 * e1.x, 2.0 * e1.y);
        energy[w * 3 + 1] = make_double2(0.5 * ec.x, 0.5 * ec.y);
        energy[w * 3 + 2] = make_double2(-ex.x, -ex.y);
    }
}

template <int MT, int NT, int WPC>
int launch_exchange_simple_w(afqmc_ctx* c, const double2* theta, int nw, cudaStream_t st) {
    const Dims& d = c->d;
    size_t smem = (size_t)2 * d.NAG * d.KS * NT * 32 * sizeof(double);
    if (smem < (size_t)WPC * NT * 2 * sizeof(double)) smem = (size_t)WPC * NT * 2 * sizeof(double);
    auto kern = exchange_simple_kernel<MT, NT, WPC>;
    static size_t attr_set = 0;
    if (smem > 48 * 1024 && smem > attr_set) {
        if (smem > (size_t)c->smem_optin) return AFQMC_UNSUPPORTED;
        if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
            return AFQMC_CUDA_ERROR;
        attr_set = smem;
    }
    const long long nblocks = (long long)((nw + NT - 1) / NT) * c->nunits;   // x only: y/z are capped at 65535
    if (nblocks > 0x7fffffffLL) return AFQMC_UNSUPPORTED;
    dim3 grid((unsigned)nblocks);
    kern<<<grid, 32 * WPC, smem, st>>>(d, nw, c->units, c->kminus, c->kplus, c->kneg, c->Lx, theta, c->ws_expart);
    AFQMC_LAUNCH_CHECK(c);
    return AFQMC_OK;
}

// warps per CTA in {4,5,6,8}: the count that leaves the smallest tail when the tasks are dealt out
template <int MT, int NT>
int launch_exchange_simple(afqmc_ctx* c, const double2* theta, int nw, cudaStream_t st) {
    const Dims& d = c->d;
    const int ntask = d.NAG * d.NAG * ((d.GP + MT - 1) / MT);
    int best = 8;
    double bestc = 1e30;
    const int cand[4] = {8, 6, 5, 4};
    for (int w : cand) {
        double cost = (double)((ntask + w - 1) / w) * w / ntask;   // >= 1, 1 = perfectly even
        if (cost < bestc - 1e-9) { bestc = cost; best = w; }
    }
    switch (best) {
        case 4: return launch_exchange_simple_w<MT, NT, 4>(c, theta, nw, st);
        case 5: return launch_exchange_simple_w<MT, NT, 5>(c, theta, nw, st);
        case 6: return launch_exchange_simple_w<MT, NT, 6>(c, theta, nw, st);
        default: return launch_exchange_simple_w<MT, NT, 8>(c, theta, nw, st);
    }
}

}  // namespace

int afqmc_i_local_energy(afqmc_ctx* c, const double2* theta, int nw, double2* energy, cudaStream_t st) {
    const Dims& d = c->d;
    int rc = afqmc_i_force_bias(c, theta, nw, c->ws_vbias, st);     // steps 2(d): the traces are the force bias
    if (rc != AFQMC_OK) return rc;
    afqmc_mark(c, 6, st);
    if (nw >= 3) rc = launch_exchange_simple<2, 4>(c, theta, nw, st);
    else rc = launch_exchange_simple<2, 2>(c, theta, nw, st);
    if (rc != AFQMC_OK) return rc;
    afqmc_mark(c, 7, st);
    energy_finalize_kernel<<<nw, 256, 0, st>>>(d, nw, c->nunits, c->units, c->kneg, c->ht, theta, c->ws_vbias,
                                              c->ws_expart, energy);
    AFQMC_LAUNCH_CHECK(c);
    return AFQMC_OK;
}

AFQMC_API int afqmc_local_energy(afqmc_ctx* c, const void* theta, int nw, void* energy, void* stream) {
    if (!c || !theta || !energy || nw < 0 || nw > c->max_walkers) return AFQMC_INVALID_ARGUMENT;
    if (nw == 0) return AFQMC_OK;
    return afqmc_i_local_energy(c, (const double2*)theta, nw, (double2*)energy, (cudaStream_t)stream);
}
