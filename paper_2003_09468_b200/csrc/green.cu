// a1 overlap, a2 elimination (log-det, inverse), a3 half-rotated Green's function.
//
// One CTA per walker: O = A^dagger Phi (N x N, Eq. 27-28; assembled as Nk row
// blocks because the trial is block diagonal) is built in shared memory when it
// fits (N <= 118), otherwise in a context-owned global workspace, and inverted in place by
// Gauss-Jordan elimination with partial (row) pivoting -- the same pivot sequence as an LU with
// partial pivoting, so det O = sign * prod(pivots).  The transposed inverse goes to workspace and
// Theta = (Phi O^{-1})^T = O^{-T} Phi^T (Eq. 30) is one batched DMMA GEMM.
#include <type_traits>
#include <cooperative_groups.h>
#include <math_constants.h>
#include "zgemm.cuh"

namespace {

constexpr int GJ_THREADS = 1024;

struct GJShared {
    double best_val[32];
    double red2[32];
    int best_idx[32];
    int piv_row;
    int info;
    int nswaps;
    int pad_;
};

// shared-memory carve-up (bytes, every section 16-byte aligned):
//   rowbuf[N], colbuf[N], pivs[N] (double2) | prow[N], qperm[N] (int) | GJShared | matrix N x LD (double2)
__host__ __device__ inline size_t gj_off_ints(int N) { return (size_t)3 * N * 16; }
__host__ __device__ inline size_t gj_off_sh(int N) { return gj_off_ints(N) + (((size_t)2 * N * 4 + 15) / 16) * 16; }
__host__ __device__ inline size_t gj_off_mat(int N) { return gj_off_sh(N) + ((sizeof(GJShared) + 15) / 16) * 16; }

// O and the elimination live at `a` (leading dimension LD), in shared or global memory.
__global__ void __launch_bounds__(GJ_THREADS) overlap_inverse_kernel(
    Dims d, int LD, int use_smem, const double2* __restrict__ psi_t, const double2* __restrict__ phi,
    double2* __restrict__ ws_O, double2* __restrict__ oinvT /*nullable*/, double2* __restrict__ logdet /*nullable*/,
    int* __restrict__ info /*nullable*/) {
    extern __shared__ __align__(16) unsigned char gj_smem_raw[];
    const int N = d.N, w = blockIdx.x, tid = threadIdx.x, nthr = blockDim.x;
    double2* rowbuf = reinterpret_cast<double2*>(gj_smem_raw);
    double2* colbuf = rowbuf + N;
    double2* pivs = colbuf + N;
    int* prow = reinterpret_cast<int*>(gj_smem_raw + gj_off_ints(N));
    int* qperm = prow + N;
    GJShared* sh = reinterpret_cast<GJShared*>(gj_smem_raw + gj_off_sh(N));
    double2* a = use_smem ? reinterpret_cast<double2*>(gj_smem_raw + gj_off_mat(N)) : ws_O + (size_t)w * N * LD;
    const double2* ph = phi + (size_t)w * d.M * d.N;

    // ---- a1: O[(k,a)][j] = sum_p conj(A_k[p][a]) Phi[(k,p)][j] ----
    for (int e = tid; e < N * N; e += nthr) {
        int j = e % N, i = e / N, k = i / d.n, aa = i % d.n;
        const double2* Ab = psi_t + (size_t)k * d.m * d.n + aa;
        const double2* Pb = ph + (size_t)k * d.m * N + j;
        double2 acc = make_double2(0.0, 0.0);
        for (int p = 0; p < d.m; ++p) {
            double2 av = Ab[p * d.n];
            av.y = -av.y;
            acc = cfma(av, Pb[(size_t)p * N], acc);
        }
        a[i * LD + j] = acc;
    }
    if (tid == 0) { sh->info = 0; sh->nswaps = 0; }
    __syncthreads();

    // ---- a2: in-place Gauss-Jordan inversion with partial pivoting ----
    const int lane = tid & 31, warp = tid >> 5;
    for (int j = 0; j < N; ++j) {
        // pivot search over rows j..N-1 of column j (largest modulus, smallest index on ties)
        {
            double bv = -1.0;
            int bi = 0x7fffffff;
            for (int i = j + tid; i < N; i += nthr) {
                double2 v = a[i * LD + j];
                double mag = v.x * v.x + v.y * v.y;
                if (mag > bv) { bv = mag; bi = i; }
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                double ov = __shfl_xor_sync(0xffffffffu, bv, o);
                int oi = __shfl_xor_sync(0xffffffffu, bi, o);
                if (ov > bv || (ov == bv && oi < bi)) { bv = ov; bi = oi; }
            }
            if (lane == 0) { sh->best_val[warp] = bv; sh->best_idx[warp] = bi; }
            __syncthreads();
            if (warp == 0) {
                int nwarps = nthr >> 5;
                bv = lane < nwarps ? sh->best_val[lane] : -1.0;
                bi = lane < nwarps ? sh->best_idx[lane] : 0x7fffffff;
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) {
                    double ov = __shfl_xor_sync(0xffffffffu, bv, o);
                    int oi = __shfl_xor_sync(0xffffffffu, bi, o);
                    if (ov > bv || (ov == bv && oi < bi)) { bv = ov; bi = oi; }
                }
                if (lane == 0) {
                    if (bi == 0x7fffffff) bi = j;   // column of NaNs: keep indices in range, flag below
                    sh->piv_row = bi;
                    prow[j] = bi;
                    if (!(bv > 0.0) && sh->info == 0) sh->info = j + 1;   // exactly-zero (or NaN) pivot
                    if (bi != j) sh->nswaps++;
                }
            }
            __syncthreads();
        }
        const int p = sh->piv_row;
        const double2 pv = a[p * LD + j];
        pivs[j] = pv;   // every thread writes the same value
        // 1/pivot
        double den = pv.x * pv.x + pv.y * pv.y;
        double2 ip = (den > 0.0) ? make_double2(pv.x / den, -pv.y / den) : make_double2(0.0, 0.0);
        __syncthreads();   // all threads have read a[p][j] before the row swap overwrites it
        // swap rows j <-> p, build the scaled pivot row
        for (int c = tid; c < N; c += nthr) {
            double2 rj = a[p * LD + c];
            if (p != j) a[p * LD + c] = a[j * LD + c];
            rowbuf[c] = (c == j) ? ip : cmul(rj, ip);
        }
        __syncthreads();
        for (int i = tid; i < N; i += nthr) colbuf[i] = (i == j) ? make_double2(0.0, 0.0) : a[i * LD + j];
        __syncthreads();
        // rank-1 update of the whole matrix
        for (int e = tid; e < N * N; e += nthr) {
            int c = e % N, i = e / N;
            double2 r = rowbuf[c];
            if (i == j) {
                a[i * LD + c] = r;
            } else {
                double2 f = colbuf[i];
                double2 cur = (c == j) ? make_double2(0.0, 0.0) : a[i * LD + c];
                f.x = -f.x; f.y = -f.y;
                a[i * LD + c] = cfma(f, r, cur);
            }
        }
        __syncthreads();
    }

    // ---- log det O = sum log(pivot) + i*pi*(#swaps odd) ----
    if (logdet) {
        double lr = 0.0, li = 0.0;
        for (int j = tid; j < N; j += nthr) {
            double2 pv = pivs[j];
            lr += log(hypot(pv.x, pv.y));
            li += atan2(pv.y, pv.x);
        }
        lr = warp_sum(lr);
        li = warp_sum(li);
        __syncthreads();
        if (lane == 0) { sh->best_val[warp] = lr; sh->red2[warp] = li; }
        __syncthreads();
        if (tid == 0) {
            double sr = 0.0, si = 0.0;
            for (int x = 0; x < (nthr >> 5); ++x) { sr += sh->best_val[x]; si += sh->red2[x]; }
            if (sh->nswaps & 1) si += CUDART_PI;
            // wrap to (-pi, pi]
            si = si - 2.0 * CUDART_PI * ceil((si - CUDART_PI) / (2.0 * CUDART_PI));
            logdet[w] = make_double2(sr, si);
        }
    }
    if (info && tid == 0) info[w] = sh->info;

    // ---- undo the row swaps as a column permutation and write O^{-T} ----
    if (oinvT) {
        __syncthreads();
        if (tid == 0) {
            for (int c = 0; c < N; ++c) qperm[c] = c;
            for (int j = N - 1; j >= 0; --j) {
                int pj = prow[j];
                if (pj != j) { int t = qperm[j]; qperm[j] = qperm[pj]; qperm[pj] = t; }
            }
        }
        __syncthreads();
        double2* out = oinvT + (size_t)w * N * N;
        for (int e = tid; e < N * N; e += nthr) {
            int i = e % N, c = e / N;            // out[c][i] = Oinv[i][c] = a[i][q[c]]
            out[(size_t)c * N + i] = a[i * LD + qperm[c]];
        }
    }
}

// ---------------------------------------------------------------------------------------------
// Register-resident elimination (N <= 32*RT rows, N <= CS*NWARP*CT columns).
//
// The whole N x N overlap lives in registers: lane l of every warp owns rows {l, l+32, ...} (RT of
// them), warp gw (numbered across the CS CTAs of a thread-block cluster) owns columns
// [gw*CT, gw*CT+CT).  Gauss-Jordan with IMPLICIT partial pivoting: rows are never swapped; step j
// picks the largest |a[i][j]| among the rows not yet used as pivots (the same pivot values as LU
// with partial pivoting up to the row labelling), so the stored matrix ends as
//     stored[sigma(i)][c] = (Pi O)^{-1}[i][c],   sigma(j) = pivot row of step j
//     =>  O^{-1}[i][c] = stored[sigma(i)][sigma^{-1}(c)],   det O = sign(sigma) * prod_j pivot_j.
// Per step only ONE warp (the owner of column j) searches the pivot (warp shuffles) and publishes
// {pivot row, 1/pivot, the column of multipliers} to the shared memory of every CTA of the cluster
// (double-buffered by step parity); after ONE barrier (CTA or cluster) every warp fetches the pivot
// row segment of its own columns by shuffles from the lane that owns it and applies the rank-1 update
// to its registers.  No matrix traffic through shared or global memory at all.
// ---------------------------------------------------------------------------------------------
namespace cg = cooperative_groups;

template <int RT, int CT>
struct GJRegShared {
    double2 f[2][32 * RT];      // multipliers (column j before the update), by step parity
    double2 ipiv[2];
    double2 piv[2];
    int prow_cur[2];
    int zero[2];
    double2 pivs[32 * RT];      // pivots, for log det
    int prow[32 * RT];          // sigma
    int sinv[32 * RT];          // sigma^{-1}
    double red[3][32];
    int info;
};

template <int RT, int CT, int NWARP, int CS>
__global__ void __launch_bounds__(32 * NWARP, 1) overlap_inverse_reg_kernel(
    Dims d, const double2* __restrict__ psi_t, const double2* __restrict__ phi, double2* __restrict__ oinvT /*nullable*/,
    double2* __restrict__ logdet /*nullable*/, int* __restrict__ info /*nullable*/) {
    __shared__ GJRegShared<RT, CT> sh;
    const int N = d.N, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int w = blockIdx.x / CS;
    unsigned rank = 0;
    if (CS > 1) rank = cg::this_cluster().block_rank();
    const int gw = (int)rank * NWARP + warp;          // global warp = column group
    const int c0 = gw * CT;
    const double2* ph = phi + (size_t)w * d.M * N;

    // ---- a1: O[(k,a)][c] = sum_p conj(A_k[p][a]) Phi[(k,p)][c] for my rows x my columns ----
    double2 a[RT][CT];
    if (RT * CT <= 8) {
        // few elements per thread (wide clusters): the RT row slots advance together, so that the loads of one p for all of
        // them are in flight at once (the phase is latency-bound: one row slot after the other took a quarter of the kernel at C3)
        const double2* Ab[RT];
        const double2* Pb[RT];
        bool ok[RT];
#pragma unroll
        for (int t = 0; t < RT; ++t) {
#pragma unroll
            for (int cc = 0; cc < CT; ++cc) a[t][cc] = make_double2(0.0, 0.0);
            const int i = lane + 32 * t;
            ok[t] = i < N && c0 < N;
            const int k = ok[t] ? i / d.n : 0, aa = ok[t] ? i - k * d.n : 0;
            Ab[t] = psi_t + (size_t)k * d.m * d.n + aa;
            Pb[t] = ph + (size_t)k * d.m * N + (c0 < N ? c0 : 0);
        }
#pragma unroll 2
        for (int p = 0; p < d.m; ++p) {
#pragma unroll
            for (int t = 0; t < RT; ++t) {
                if (!ok[t]) continue;
                double2 av = __ldg(Ab[t] + (size_t)p * d.n);
                av.y = -av.y;
#pragma unroll
                for (int cc = 0; cc < CT; ++cc)
                    if (c0 + cc < N) a[t][cc] = cfma(av, __ldg(Pb[t] + (size_t)p * N + cc), a[t][cc]);
            }
        }
    } else {
#pragma unroll
    for (int t = 0; t < RT; ++t) {
#pragma unroll
        for (int cc = 0; cc < CT; ++cc) a[t][cc] = make_double2(0.0, 0.0);
        const int i = lane + 32 * t;
        if (i < N && c0 < N) {
            const int k = i / d.n, aa = i - k * d.n;
            const double2* Ab = psi_t + (size_t)k * d.m * d.n + aa;
            const double2* Pb = ph + (size_t)k * d.m * N + c0;
#pragma unroll 2
            for (int p = 0; p < d.m; ++p) {
                double2 av = __ldg(Ab + (size_t)p * d.n);
                av.y = -av.y;
#pragma unroll
                for (int cc = 0; cc < CT; ++cc)
                    if (c0 + cc < N) a[t][cc] = cfma(av, __ldg(Pb + (size_t)p * N + cc), a[t][cc]);
            }
        }
    }
    }
    if (tid == 0) sh.info = 0;
    unsigned used = 0;                                 // bit t: my row lane+32t has been a pivot row
    if (CS > 1) cg::this_cluster().sync(); else __syncthreads();

    // ---- a2: N elimination steps ----
    for (int j = 0; j < N; ++j) {
        const int buf = j & 1;
        const int jw = j / CT, tj = j - jw * CT;       // owner warp and its local column
        if (gw == jw) {
            // column j of my rows
            double2 col[RT];
#pragma unroll
            for (int t = 0; t < RT; ++t) {
                col[t] = a[t][0];
#pragma unroll
                for (int cc = 1; cc < CT; ++cc) if (cc == tj) col[t] = a[t][cc];
            }
            double bv = -2.0;
            int bi = 0x7fffffff;
#pragma unroll
            for (int t = 0; t < RT; ++t) {
                const int i = lane + 32 * t;
                if (i < N && !((used >> t) & 1u)) {
                    double mag = col[t].x * col[t].x + col[t].y * col[t].y;
                    if (!(mag >= 0.0)) mag = -1.0;                 // NaN: never preferred, still a valid row
                    if (mag > bv) { bv = mag; bi = i; }
                }
            }
            // largest modulus over the warp, smallest row index on ties -- the same choice as a butterfly of (value, index)
            // pairs, in three warp reductions on 32-bit keys: non-negative doubles order like their (high, low) words; a lane
            // whose rows are all NaN has bv = -1 (class 1, below every number), a lane without candidate rows class 0
            const unsigned hi = bv >= 0.0 ? (unsigned)__double2hiint(bv) + 2u : (bv == -1.0 ? 1u : 0u);
            const unsigned mh = __reduce_max_sync(0xffffffffu, hi);
            const bool c1 = hi == mh;
            const unsigned lo = (unsigned)__double2loint(bv);
            const unsigned ml = __reduce_max_sync(0xffffffffu, c1 ? lo : 0u);
            const bool c2 = c1 && lo == ml;
            bi = (int)__reduce_min_sync(0xffffffffu, c2 ? (unsigned)bi : 0x7fffffffu);
            const int p = bi, pl = p & 31, pt = p >> 5;
            double2 pvl = col[0];
#pragma unroll
            for (int t = 1; t < RT; ++t) if (t == pt) pvl = col[t];
            double2 pv;
            pv.x = __shfl_sync(0xffffffffu, pvl.x, pl);
            pv.y = __shfl_sync(0xffffffffu, pvl.y, pl);
            const double den = pv.x * pv.x + pv.y * pv.y;
            const bool ok = den > 0.0;
            const double rden = 1.0 / den;
            const double2 ip = ok ? make_double2(pv.x * rden, -pv.y * rden) : make_double2(0.0, 0.0);
            // what the update multiplies the scaled pivot row with: minus the column, and 0 in the pivot row itself (whose new
            // value is the scaled pivot row: the update below computes 0 * r + r there)
#pragma unroll
            for (int t = 0; t < RT; ++t) {
                const bool isp = (lane == pl) && (t == pt);
                col[t].x = isp ? 0.0 : -col[t].x;
                col[t].y = isp ? 0.0 : -col[t].y;
            }
            // publish to every CTA of the cluster
#pragma unroll(CS <= 4 ? CS : 1)
            for (int q = 0; q < CS; ++q) {
                GJRegShared<RT, CT>* dst = &sh;
                if (CS > 1) dst = cg::this_cluster().map_shared_rank(&sh, q);
#pragma unroll
                for (int t = 0; t < RT; ++t) dst->f[buf][lane + 32 * t] = col[t];
                if (lane == 0) { dst->ipiv[buf] = ip; dst->piv[buf] = pv; dst->prow_cur[buf] = p; dst->zero[buf] = ok ? 0 : 1; }
            }
        }
        if (CS > 1) cg::this_cluster().sync(); else __syncthreads();

        const int p = sh.prow_cur[buf], pl = p & 31, pt = p >> 5;
        const double2 ip = sh.ipiv[buf];
        if (tid == 0) {
            sh.prow[j] = p;
            sh.pivs[j] = sh.piv[buf];
            if (sh.zero[buf] && sh.info == 0) sh.info = j + 1;
        }
        if (lane == pl) used |= 1u << pt;
        // scaled pivot row for my columns: r[cc] = a[p][c] / pivot  (column j itself -> 1/pivot).  The register slot pt of the
        // pivot row is the same for every thread, so the slot is picked by a branch (no per-slot selects), and the lane that
        // owns the pivot row takes r as its new row there (its multiplier was published as 0)
        double2 r[CT];
        const bool own_col = gw == jw;
        auto pivot_row = [&](auto tc) {
            constexpr int t = decltype(tc)::value;
            if constexpr (t < RT) {
#pragma unroll
                for (int cc = 0; cc < CT; ++cc) {
                    double2 v;
                    v.x = __shfl_sync(0xffffffffu, a[t][cc].x, pl);
                    v.y = __shfl_sync(0xffffffffu, a[t][cc].y, pl);
                    r[cc] = cmul(v, ip);
                    if (own_col && cc == tj) r[cc] = ip;
                    if (lane == pl) a[t][cc] = r[cc];
                }
            }
        };
        if (own_col) {
#pragma unroll
            for (int cc = 0; cc < CT; ++cc)
                if (cc == tj) {
#pragma unroll
                    for (int t = 0; t < RT; ++t) a[t][cc] = make_double2(0.0, 0.0);
                }
        }
        switch (pt) {
            case 0: pivot_row(std::integral_constant<int, 0>()); break;
            case 1: pivot_row(std::integral_constant<int, 1>()); break;
            case 2: pivot_row(std::integral_constant<int, 2>()); break;
            case 3: pivot_row(std::integral_constant<int, 3>()); break;
            case 4: pivot_row(std::integral_constant<int, 4>()); break;
            case 5: pivot_row(std::integral_constant<int, 5>()); break;
            case 6: pivot_row(std::integral_constant<int, 6>()); break;
            default: pivot_row(std::integral_constant<int, 7>()); break;
        }
#pragma unroll
        for (int t = 0; t < RT; ++t) {
            const double2 f = sh.f[buf][lane + 32 * t];
#pragma unroll
            for (int cc = 0; cc < CT; ++cc) a[t][cc] = cfma(f, r[cc], a[t][cc]);
        }
    }
    if (CS > 1) cg::this_cluster().sync(); else __syncthreads();

    // ---- sigma^{-1}, log det O = sum log(pivot) + i*pi*(sigma odd), info ----
    for (int j = tid; j < N; j += 32 * NWARP) sh.sinv[sh.prow[j]] = j;
    if (rank == 0) {
        double lr = 0.0, li = 0.0, inv = 0.0;
        for (int j = tid; j < N; j += 32 * NWARP) {
            const double2 pv = sh.pivs[j];
            lr += log(hypot(pv.x, pv.y));
            li += atan2(pv.y, pv.x);
            const int sj = sh.prow[j];
            int cnt = 0;
            for (int i = 0; i < j; ++i) cnt += sh.prow[i] > sj;      // inversions of sigma
            inv += (double)cnt;
        }
        lr = warp_sum(lr); li = warp_sum(li); inv = warp_sum(inv);
        if (lane == 0) { sh.red[0][warp] = lr; sh.red[1][warp] = li; sh.red[2][warp] = inv; }
    }
    __syncthreads();
    if (rank == 0 && tid == 0) {
        double sr = 0.0, si = 0.0, sv = 0.0;
        for (int x = 0; x < NWARP; ++x) { sr += sh.red[0][x]; si += sh.red[1][x]; sv += sh.red[2][x]; }
        if (((long long)sv) & 1LL) si += CUDART_PI;
        si = si - 2.0 * CUDART_PI * ceil((si - CUDART_PI) / (2.0 * CUDART_PI));     // wrap to (-pi, pi]
        if (logdet) logdet[w] = make_double2(sr, si);
        if (info) info[w] = sh.info;
    }
    // ---- O^{-T}[sigma(k)][sigma^{-1}(rho)] = stored[rho][k] ----
    if (oinvT) {
        double2* out = oinvT + (size_t)w * N * N;
#pragma unroll
        for (int cc = 0; cc < CT; ++cc) {
            const int k = c0 + cc;
            if (k < N) {
                const size_t rowoff = (size_t)sh.prow[k] * N;
#pragma unroll
                for (int t = 0; t < RT; ++t) {
                    const int rho = lane + 32 * t;
                    if (rho < N) out[rowoff + sh.sinv[rho]] = a[t][cc];
                }
            }
        }
    }
}

template <int RT, int CT, int NWARP, int CS>
int launch_gj_reg(afqmc_ctx* c, const double2* phi, int nw, double2* oinvT, double2* logdet, int* info, cudaStream_t st) {
    auto kern = overlap_inverse_reg_kernel<RT, CT, NWARP, CS>;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(nw * CS));
    cfg.blockDim = dim3(32 * NWARP);
    cfg.dynamicSmemBytes = 0;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = CS; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    if (cudaLaunchKernelEx(&cfg, kern, c->d, (const double2*)c->psi_t, phi, oinvT, logdet, info) != cudaSuccess) {
        (void)cudaGetLastError();
        return AFQMC_CUDA_ERROR;
    }
    AFQMC_LAUNCH_CHECK(c);
    return AFQMC_OK;
}

size_t gj_fixed_smem(int N) { return gj_off_mat(N); }

int run_overlap_inverse(afqmc_ctx* c, const double2* phi, int nw, double2* oinvT, double2* logdet, int* info,
                        cudaStream_t st) {
    const Dims& d = c->d;
    if (!c->opt_green_legacy) {
        // register-resident elimination: one CTA for N <= 64, a cluster of two for N <= 128, of eight for N <= 256
        if (d.N <= 32) return launch_gj_reg<1, 2, 16, 1>(c, phi, nw, oinvT, logdet, info, st);
        if (d.N <= 64) return launch_gj_reg<2, 4, 16, 1>(c, phi, nw, oinvT, logdet, info, st);
        if (d.N <= 128) {
            // four CTAs per walker when they all fit one wave (the update is instruction-bound on the SMs that hold a
            // walker: C3 0.388 -> 0.355 ms), else two
            const bool four = c->opt_green_cs == 4 || (c->opt_green_cs == 0 && 4 * nw <= c->num_sms);
            return four ? launch_gj_reg<4, 2, 16, 4>(c, phi, nw, oinvT, logdet, info, st)
                        : launch_gj_reg<4, 4, 16, 2>(c, phi, nw, oinvT, logdet, info, st);
        }
        if (d.N <= 256) return launch_gj_reg<8, 2, 16, 8>(c, phi, nw, oinvT, logdet, info, st);
    }
    const int LD = d.N | 1;
    size_t fixed = gj_fixed_smem(d.N);
    size_t mat = (size_t)d.N * LD * sizeof(double2);
    int use_smem = (fixed + mat <= (size_t)c->smem_optin) ? 1 : 0;
    size_t smem = fixed + (use_smem ? mat : 0);
    if (int rc = afqmc_smem_optin(c, (const void*)overlap_inverse_kernel, smem)) return rc;
    int threads = GJ_THREADS;
    if (d.N * d.N < 4096) threads = 256;
    overlap_inverse_kernel<<<nw, threads, smem, st>>>(d, LD, use_smem, c->psi_t, phi, c->ws_O, oinvT, logdet, info);
    AFQMC_LAUNCH_CHECK(c);
    return AFQMC_OK;
}

}  // namespace

int afqmc_i_green(afqmc_ctx* c, const double2* phi, int nw, double2* theta, double2* logdet, int* info,
                  cudaStream_t st) {
    const Dims& d = c->d;
    int rc = run_overlap_inverse(c, phi, nw, theta ? c->ws_oinvT : nullptr, logdet, info, st);
    if (rc != AFQMC_OK || !theta) return rc;
    // Theta[i][q] = sum_j OinvT[i][j] * Phi[q][j]   (B is K-contiguous: element (k=j, col=q) at phi[q*N + j])
    zg::Args a = {};
    a.A = c->ws_oinvT; a.strideA = (long long)d.N * d.N; a.lda = d.N;
    a.B = phi; a.strideB = (long long)d.M * d.N; a.ldb = d.N;
    a.C = theta; a.strideC = (long long)d.N * d.M; a.ldc = d.M;
    a.D = nullptr; a.strideD = 0; a.ldd = 0;
    a.M = d.N; a.N = d.M; a.K = d.N; a.alpha = 1.0;
    c->frag_nw = 0; c->frag_src = nullptr;
    if (c->fuse_frag) {      // inside afqmc_step / afqmc_block: the epilogue also writes the force-bias B fragments of this Theta
        a.frag.F = c->ws_thetaF; a.frag.ktab = c->kminus; a.frag.m = d.m; a.frag.n = d.n; a.frag.Nk = d.Nk;
        afqmc_i_fb_frag_layout(c, nw, &a.frag.NT, &a.frag.nwg, &a.frag.KSf);
        c->frag_nw = nw; c->frag_src = theta;
    }
    if (zg::launch<true>(c, a, nw, st) != cudaSuccess) return AFQMC_CUDA_ERROR;
    c->launches++;
    return AFQMC_OK;
}

AFQMC_API int afqmc_overlap(afqmc_ctx* c, const void* phi, int nw, void* logdet, int* info, void* stream) {
    if (!c || !phi || !logdet || nw < 0 || nw > c->max_walkers) return AFQMC_INVALID_ARGUMENT;
    if (nw == 0) return AFQMC_OK;
    if (c->prec32) return afqmc32_green(c, phi, nw, nullptr, logdet, info, (cudaStream_t)stream);
    return afqmc_x_green(c, (const double2*)phi, nw, nullptr, (double2*)logdet, info, (cudaStream_t)stream);
}

AFQMC_API int afqmc_green(afqmc_ctx* c, const void* phi, int nw, void* theta, void* logdet, int* info,
                           void* stream) {
    if (!c || !phi || !theta || nw < 0 || nw > c->max_walkers) return AFQMC_INVALID_ARGUMENT;
    if (nw == 0) return AFQMC_OK;
    if (c->prec32) return afqmc32_green(c, phi, nw, theta, logdet, info, (cudaStream_t)stream);
    return afqmc_x_green(c, (const double2*)phi, nw, (double2*)theta, (double2*)logdet, info, (cudaStream_t)stream);
}
