// The AFQMC block around the step (include/afqmc.h "The AFQMC block"):
//   one-body half steps  exp(-dtau/2 H1')            Eq. 7, 13
//   hybrid importance function, phaseless weights     Eq. 16-19
//   walker orthogonalisation (thin QR)
//   mixed estimator                                   Eq. 34-35
//   block = nsteps hybrid propagation steps + energy + orthogonalisation
// None of these is a hot spot (the step's GEMMs are: r01 profiles), so they are plain FP64 ALU kernels sized to
// fill the SMs, except the Q = phi R^{-1} product of the orthogonalisation, which reuses the DMMA zgemm.
#include <math.h>
#include "zgemm.cuh"

namespace {

// ------------------------------------------------------------------------------------------------
// B1[k] = exp(scale * h1p[k]),  scale = -dtau/2: scaling and squaring of an order-18 Taylor series.
// One CTA per k-point; the m x m matrices live in global scratch (L1/L2 resident, m <= a few dozen).
//   X = scale*h / 2^s with ||X||_inf <= 1/2;   P = sum_{j<=18} X^j/j!  (remainder < 2e-23);   P <- P^2, s times.
// ------------------------------------------------------------------------------------------------
constexpr int EXPM_THREADS = 256;
constexpr int EXPM_ORDER = 18;

__device__ void small_matmul(int m, double f, const double2* A, const double2* B, double2* C) {
    for (int e = threadIdx.x; e < m * m; e += blockDim.x) {      // C = f * A * B
        const int i = e / m, j = e % m;
        double2 s = make_double2(0.0, 0.0);
        for (int k = 0; k < m; ++k) s = cfma(A[i * m + k], B[k * m + j], s);
        C[e] = make_double2(f * s.x, f * s.y);
    }
}

__global__ void __launch_bounds__(EXPM_THREADS) expm_kernel(int m, double scale, const double2* __restrict__ h,
                                                            double2* __restrict__ b1, double2* __restrict__ tmp) {
    __shared__ double red[EXPM_THREADS];
    __shared__ int s_sq;
    const int k = blockIdx.x;
    const double2* H = h + (size_t)k * m * m;
    double2* P = b1 + (size_t)k * m * m;
    double2* X = tmp + (size_t)k * 3 * m * m;
    double2* T = X + m * m;
    double2* T2 = T + m * m;
    // infinity norm of scale*H
    double mx = 0.0;
    for (int i = threadIdx.x; i < m; i += blockDim.x) {
        double rs = 0.0;
        for (int j = 0; j < m; ++j) rs += hypot(H[i * m + j].x, H[i * m + j].y);
        mx = fmax(mx, rs * fabs(scale));
    }
    red[threadIdx.x] = mx;
    __syncthreads();
    for (int o = EXPM_THREADS / 2; o > 0; o >>= 1) {
        if (threadIdx.x < o) red[threadIdx.x] = fmax(red[threadIdx.x], red[threadIdx.x + o]);
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        int s = 0;
        double nrm = red[0];
        while (nrm > 0.5 && s < 60) { nrm *= 0.5; ++s; }
        s_sq = s;
    }
    __syncthreads();
    const int nsq = s_sq;
    const double f = scale * exp2(-(double)nsq);
    for (int e = threadIdx.x; e < m * m; e += blockDim.x) {
        const double2 x = make_double2(f * H[e].x, f * H[e].y);
        X[e] = x;
        T[e] = x;
        const bool diag = (e / m) == (e % m);
        P[e] = make_double2(x.x + (diag ? 1.0 : 0.0), x.y);
    }
    __syncthreads();
    for (int j = 2; j <= EXPM_ORDER; ++j) {
        small_matmul(m, 1.0 / (double)j, X, T, T2);          // T2 = X T / j
        __syncthreads();
        for (int e = threadIdx.x; e < m * m; e += blockDim.x) {
            P[e].x += T2[e].x;
            P[e].y += T2[e].y;
        }
        double2* sw = T; T = T2; T2 = sw;
        __syncthreads();
    }
    for (int q = 0; q < nsq; ++q) {
        small_matmul(m, 1.0, P, P, T);
        __syncthreads();
        for (int e = threadIdx.x; e < m * m; e += blockDim.x) P[e] = T[e];
        __syncthreads();
    }
}

// ------------------------------------------------------------------------------------------------
// phi_w[(k,p), j] <- sum_r B1[k][p][r] phi_w[(k,r), j].   CTA = (column tile, k, walker): the m x CT block of
// phi and B1[k] are staged in shared memory, so the update is in place (a CTA owns its rows and columns).
// ------------------------------------------------------------------------------------------------
constexpr int OB_THREADS = 256;

__global__ void __launch_bounds__(OB_THREADS) onebody_kernel(Dims d, int CT, const double2* __restrict__ b1,
                                                             double2* __restrict__ phi) {
    extern __shared__ __align__(16) double2 ob_smem[];
    double2* Bs = ob_smem;                 // [m][m]
    double2* Xs = ob_smem + d.m * d.m;     // [m][CT]
    const int j0 = blockIdx.x * CT, k = blockIdx.y, w = blockIdx.z;
    const int ct = min(CT, d.N - j0);
    double2* X = phi + ((size_t)w * d.M + (size_t)k * d.m) * d.N + j0;
    for (int e = threadIdx.x; e < d.m * d.m; e += OB_THREADS) Bs[e] = b1[(size_t)k * d.m * d.m + e];
    for (int e = threadIdx.x; e < d.m * ct; e += OB_THREADS) {
        const int r = e / ct, j = e % ct;
        Xs[r * CT + j] = X[(size_t)r * d.N + j];
    }
    __syncthreads();
    // a thread computes 4 rows of one column: every element of the staged block feeds 4 complex FMAs per load
    const int npg = (d.m + 3) / 4;
    for (int e = threadIdx.x; e < npg * ct; e += OB_THREADS) {
        const int pg = e / ct, j = e % ct;
        const int p0 = 4 * pg;
        double2 s[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) s[i] = make_double2(0.0, 0.0);
        for (int r = 0; r < d.m; ++r) {
            const double2 xv = Xs[r * CT + j];
#pragma unroll
            for (int i = 0; i < 4; ++i) s[i] = cfma(Bs[min(p0 + i, d.m - 1) * d.m + r], xv, s[i]);
        }
#pragma unroll
        for (int i = 0; i < 4; ++i)
            if (p0 + i < d.m) X[(size_t)(p0 + i) * d.N + j] = s[i];
    }
}

}  // namespace

int afqmc_i_apply_onebody(afqmc_ctx* c, double2* phi, int nw, cudaStream_t st) {
    const Dims& d = c->d;
    if (!c->b1_set) return AFQMC_INVALID_ARGUMENT;
    // column tile: B1 + block within ~96 KB of shared memory, and enough CTAs to fill the SMs
    int CT = d.N;
    const size_t budget = 96 * 1024;
    const size_t fixed = (size_t)d.m * d.m * sizeof(double2);
    if (fixed + (size_t)d.m * 8 * sizeof(double2) > (size_t)c->smem_optin) {
        // B1[k] does not fit one CTA's shared memory (m above ~116, e.g. the Gamma-point supercell shape): one batched DMMA
        // GEMM per k-point, out of place into the Taylor workspace, then copied back
        const size_t per = (size_t)d.M * d.N;
        for (int k = 0; k < d.Nk; ++k) {
            zg::Args a = {};
            a.A = c->b1 + (size_t)k * d.m * d.m; a.strideA = 0; a.lda = d.m;
            a.B = phi + (size_t)k * d.m * d.N; a.strideB = (long long)per; a.ldb = d.N;
            a.C = c->ws_T + (size_t)k * d.m * d.N; a.strideC = (long long)per; a.ldc = d.N;
            a.D = nullptr; a.strideD = 0; a.ldd = 0;
            a.M = d.m; a.N = d.N; a.K = d.m; a.alpha = 1.0;
            if (zg::launch<false>(c, a, nw, st) != cudaSuccess) return AFQMC_CUDA_ERROR;
            c->launches++;
        }
        AFQMC_CUDA_TRY(cudaMemcpyAsync(phi, c->ws_T, (size_t)nw * per * sizeof(double2), cudaMemcpyDeviceToDevice, st));
        return AFQMC_OK;
    }
    while (CT > 8 && (fixed + (size_t)d.m * CT * sizeof(double2) > budget || (long long)nw * d.Nk * ceil_div(d.N, CT) < 2LL * c->num_sms))
        CT = (CT + 1) / 2;
    const size_t smem = fixed + (size_t)d.m * CT * sizeof(double2);
    if (int rc = afqmc_smem_optin(c, (const void*)onebody_kernel, smem)) return rc;
    onebody_kernel<<<dim3(ceil_div(d.N, CT), d.Nk, nw), OB_THREADS, smem, st>>>(d, CT, c->b1, phi);
    AFQMC_LAUNCH_CHECK(c);
    return AFQMC_OK;
}

AFQMC_API int afqmc_set_onebody(afqmc_ctx* c, const void* h1p, double dtau, void* b1_out, void* stream) {
    if (c && c->prec32) return AFQMC_UNSUPPORTED;      // the block calls are FP64-only (boundary32.cu)
    if (!c || !h1p || !(dtau >= 0.0)) return AFQMC_INVALID_ARGUMENT;
    const Dims& d = c->d;
    cudaStream_t st = (cudaStream_t)stream;
    expm_kernel<<<d.Nk, EXPM_THREADS, 0, st>>>(d.m, -0.5 * dtau, (const double2*)h1p, c->b1, c->ws_b1tmp);
    AFQMC_LAUNCH_CHECK(c);
    c->b1_set = 1;
    if (b1_out)
        AFQMC_CUDA_TRY(cudaMemcpyAsync(b1_out, c->b1, (size_t)d.Nk * d.m * d.m * sizeof(double2), cudaMemcpyDeviceToDevice, st));
    return AFQMC_OK;
}

AFQMC_API int afqmc_apply_onebody(afqmc_ctx* c, void* phi, int nw, void* stream) {
    if (c && c->prec32) return AFQMC_UNSUPPORTED;      // the block calls are FP64-only (boundary32.cu)
    if (!c || !phi || nw < 0 || nw > c->max_walkers) return AFQMC_INVALID_ARGUMENT;
    if (nw == 0) return AFQMC_OK;
    return afqmc_x_apply_onebody(c, (double2*)phi, nw, (cudaStream_t)stream);
}

// ------------------------------------------------------------------------------------------------
// Hybrid importance function and phaseless weight update (Eq. 16, 18, 19).
// One CTA per walker; fixed thread -> (Q,gamma) assignment and a fixed-shape tree: deterministic.
// ------------------------------------------------------------------------------------------------
namespace {

constexpr int HW_THREADS = 256;

__global__ void __launch_bounds__(HW_THREADS) hybrid_weight_kernel(
    Dims d, const int* __restrict__ kneg, const double* __restrict__ x, const double2* __restrict__ vbias,
    double sqrt_dtau, double spin_factor, const double2* __restrict__ ld_old, const double2* __restrict__ ld_new,
    const int* __restrict__ info /* nullable: status of the two overlap factorisations */,
    double* __restrict__ weight, double2* __restrict__ log_i) {
    __shared__ double red[4][HW_THREADS];
    const int w = blockIdx.x;
    const double* xw = x + (size_t)w * d.Nk * d.nchol;
    const double2* vw = vbias + (size_t)w * d.Nk * d.nchol;
    double s_xxb_r = 0.0, s_xxb_i = 0.0, s_bb_r = 0.0, s_bb_i = 0.0;
    for (int e = threadIdx.x; e < d.Nk * d.nchol; e += HW_THREADS) {
        const int Q = e / d.nchol, g = e % d.nchol;
        const int mq = kneg[Q];
        // z_Q as in fields_kernel (vhs.cu)
        const double xq = xw[Q * d.nchol + g];
        double zr, zi;
        if (mq == Q) { zr = xq; zi = 0.0; }
        else {
            const double xm = xw[mq * d.nchol + g];
            const double r2 = 0.70710678118654752440;
            if (Q < mq) { zr = xq * r2; zi = xm * r2; }
            else        { zr = xm * r2; zi = -xq * r2; }
        }
        // zbar_{-Q} = -i sqrt(dtau) vbias[Q],   zbar_Q = -i sqrt(dtau) vbias[-Q]
        const double2 vQ = vw[Q * d.nchol + g], vm = vw[mq * d.nchol + g];
        const double2 zb_m = make_double2(sqrt_dtau * vQ.y, -sqrt_dtau * vQ.x);
        const double2 zb_q = make_double2(sqrt_dtau * vm.y, -sqrt_dtau * vm.x);
        const double2 a = cmul(make_double2(zr, zi), zb_m);       // z_Q zbar_{-Q}
        const double2 b = cmul(zb_q, zb_m);                       // zbar_Q zbar_{-Q}
        s_xxb_r += a.x; s_xxb_i += a.y; s_bb_r += b.x; s_bb_i += b.y;
    }
    red[0][threadIdx.x] = s_xxb_r; red[1][threadIdx.x] = s_xxb_i;
    red[2][threadIdx.x] = s_bb_r;  red[3][threadIdx.x] = s_bb_i;
    __syncthreads();
    for (int o = HW_THREADS / 2; o > 0; o >>= 1) {
        if (threadIdx.x < o)
            for (int q = 0; q < 4; ++q) red[q][threadIdx.x] += red[q][threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        // closed shell: both spins share the walker (ratio squared); open shell: logdet already is the sum over channels
        const double lr_r = spin_factor * (ld_new[w].x - ld_old[w].x), lr_i = spin_factor * (ld_new[w].y - ld_old[w].y);
        const double li_r = lr_r + red[0][0] - 0.5 * red[2][0];
        const double li_i = lr_i + red[1][0] - 0.5 * red[3][0];
        const double twopi = 6.283185307179586476925287, pi = 3.141592653589793238462643;
        double dth = fmod(lr_i + pi, twopi);
        if (dth < 0.0) dth += twopi;
        dth -= pi;
        if (dth == -pi) dth = pi;
        const double c = cos(dth);
        // A walker that is already dead stays dead, and a walker whose overlap is singular or not finite (log det
        // undefined, include/afqmc.h) is killed: 0 * inf or a NaN phase never reaches the weight.
        const double w_old = weight[w];
        const bool bad = (info && info[w] != 0) || !isfinite(lr_r) || !isfinite(lr_i) || !isfinite(li_r);
        const double f = exp(li_r) * (c > 0.0 ? c : 0.0);
        weight[w] = (w_old == 0.0 || bad || !isfinite(f)) ? 0.0 : w_old * f;
        if (log_i) log_i[w] = make_double2(li_r, li_i);
    }
}

// Eq. 35: out[0..2] = sum_w weight_w E_w[0..2], out[3] = sum_w weight_w, in walker order (one thread per output)
__global__ void mixed_estimator_kernel(int nw, const double2* __restrict__ energy, const double* __restrict__ weight,
                                       double2* __restrict__ out) {
    const int c = threadIdx.x;
    if (c >= 4) return;
    double2 s = make_double2(0.0, 0.0);
    for (int w = 0; w < nw; ++w) {
        // dead walkers (weight 0) and walkers without a finite local energy do not enter either sum of Eq. 35
        const double wt = weight[w];
        bool ok = wt != 0.0 && isfinite(wt);
        for (int q = 0; q < 3; ++q) ok = ok && isfinite(energy[w * 3 + q].x) && isfinite(energy[w * 3 + q].y);
        if (!ok) continue;
        if (c < 3) { s.x += wt * energy[w * 3 + c].x; s.y += wt * energy[w * 3 + c].y; }
        else s.x += wt;
    }
    out[c] = s;
}

}  // namespace

static int hybrid_weight_i(afqmc_ctx* c, const double* x, const double2* vbias, double dtau, const double2* ld_old,
                           const double2* ld_new, const int* info, int nw, double* weight, double2* log_i, cudaStream_t st) {
    hybrid_weight_kernel<<<nw, HW_THREADS, 0, st>>>(c->d, c->kneg, x, vbias, sqrt(dtau), c->spin_factor, ld_old, ld_new, info, weight, log_i);
    AFQMC_LAUNCH_CHECK(c);
    return AFQMC_OK;
}

AFQMC_API int afqmc_hybrid_weight(afqmc_ctx* c, const double* x, const void* vbias, double dtau, const void* logdet_old,
                                   const void* logdet_new, int nw, double* weight, void* log_i, void* stream) {
    if (c && c->prec32) return AFQMC_UNSUPPORTED;      // the block calls are FP64-only (boundary32.cu)
    if (!c || !x || !vbias || !logdet_old || !logdet_new || !weight || nw < 0 || nw > c->max_walkers || !(dtau >= 0.0))
        return AFQMC_INVALID_ARGUMENT;
    if (nw == 0) return AFQMC_OK;
    return hybrid_weight_i(c, x, (const double2*)vbias, dtau, (const double2*)logdet_old, (const double2*)logdet_new, nullptr, nw,
                           weight, (double2*)log_i, (cudaStream_t)stream);
}

AFQMC_API int afqmc_mixed_estimator(afqmc_ctx* c, const void* energy, const double* weight, int nw, void* out,
                                     void* stream) {
    if (c && c->prec32) return AFQMC_UNSUPPORTED;      // the block calls are FP64-only (boundary32.cu)
    if (!c || !energy || !weight || !out || nw < 0) return AFQMC_INVALID_ARGUMENT;
    mixed_estimator_kernel<<<1, 32, 0, (cudaStream_t)stream>>>(nw, (const double2*)energy, weight, (double2*)out);
    AFQMC_LAUNCH_CHECK(c);
    return AFQMC_OK;
}

// ------------------------------------------------------------------------------------------------
// Walker orthogonalisation: thin QR with a real positive diagonal by two passes of Cholesky-QR
//   S = phi^dagger phi (N x N),  S = L L^dagger,  R = L^dagger,  phi <- phi R^{-1}.
// One pass loses cond(phi)^2 * eps of orthogonality, the second pass restores it to eps (the walkers of a
// block stay far below cond 1e7); R = R2 R1 and log det R = log det R1 + log det R2.
// ------------------------------------------------------------------------------------------------
namespace {

constexpr int GR_T = 32;          // Gram tile
constexpr int GR_THREADS = 256;

// S_w[i][j] = sum_p conj(phi_w[p][i]) phi_w[p][j]; CTA = 32 x 32 tile, 2 x 2 outputs per thread
__global__ void __launch_bounds__(GR_THREADS) gram_kernel(int M, int N, const double2* __restrict__ phi,
                                                          double2* __restrict__ S) {
    __shared__ double2 Ai[GR_T][GR_T + 1], Aj[GR_T][GR_T + 1];
    const int i0 = blockIdx.y * GR_T, j0 = blockIdx.x * GR_T, w = blockIdx.z;
    const double2* P = phi + (size_t)w * M * N;
    const int ti = threadIdx.x / 16, tj = threadIdx.x % 16;      // outputs (ti, ti+16) x (tj, tj+16)
    double2 acc[2][2];
    for (int a = 0; a < 2; ++a)
        for (int b = 0; b < 2; ++b) acc[a][b] = make_double2(0.0, 0.0);
    for (int p0 = 0; p0 < M; p0 += GR_T) {
        for (int e = threadIdx.x; e < GR_T * GR_T; e += GR_THREADS) {
            const int p = e / GR_T, c = e % GR_T;
            const bool pok = p0 + p < M;
            Ai[p][c] = (pok && i0 + c < N) ? P[(size_t)(p0 + p) * N + i0 + c] : make_double2(0.0, 0.0);
            Aj[p][c] = (pok && j0 + c < N) ? P[(size_t)(p0 + p) * N + j0 + c] : make_double2(0.0, 0.0);
        }
        __syncthreads();
#pragma unroll 4
        for (int p = 0; p < GR_T; ++p) {
            double2 a[2] = {Ai[p][ti], Ai[p][ti + 16]};
            a[0].y = -a[0].y; a[1].y = -a[1].y;                  // conj
            const double2 b[2] = {Aj[p][tj], Aj[p][tj + 16]};
            for (int x = 0; x < 2; ++x)
                for (int y = 0; y < 2; ++y) acc[x][y] = cfma(a[x], b[y], acc[x][y]);
        }
        __syncthreads();
    }
    for (int x = 0; x < 2; ++x)
        for (int y = 0; y < 2; ++y) {
            const int i = i0 + ti + 16 * x, j = j0 + tj + 16 * y;
            if (i < N && j < N) S[((size_t)w * N + i) * N + j] = acc[x][y];
        }
}

// Cholesky factor (lower, in place in the lower triangle of S) and the inverse of R = L^dagger.
// One CTA per walker; S is staged in shared memory when it fits (use_smem), else worked on in global memory.
// Right-looking, ONE barrier per column: the trailing update of column j and the scaling of column j-1 touch
// disjoint entries.  Then thread c computes column c of L^{-1} by forward substitution (no barriers) and
// stores it, conjugated, as row c of Rinv (upper triangular, zeros below the diagonal).
constexpr int CH_THREADS = 1024;

__global__ void __launch_bounds__(CH_THREADS) cholesky_inverse_kernel(int N, int use_smem, double2* __restrict__ Sg,
                                                                      double2* __restrict__ Rinv, double* __restrict__ logdet_r,
                                                                      int* __restrict__ info) {
    extern __shared__ __align__(16) double2 ch_smem[];
    __shared__ int s_info;
    const int w = blockIdx.x, tid = threadIdx.x;
    double2* G = Sg + (size_t)w * N * N;
    double2* S = use_smem ? ch_smem : G;
    if (use_smem)
        for (int e = tid; e < N * N; e += CH_THREADS) S[e] = G[e];
    if (tid == 0) s_info = 0;
    __syncthreads();
    double ld = 0.0;
    for (int j = 0; j < N; ++j) {
        double dj = S[j * N + j].x;
        if (!(dj > 0.0) || !isfinite(dj)) {
            if (tid == 0 && s_info == 0) s_info = j + 1;
            dj = 1.0;
        }
        if (tid == 0) ld += 0.5 * log(dj);
        const double inv = 1.0 / dj;
        const int nn = N - j - 1;
        for (int e = tid; e < nn * nn; e += CH_THREADS) {
            const int i = j + 1 + e / nn, k = j + 1 + e % nn;
            if (k > i) continue;
            const double2 a = S[i * N + j];
            double2 b = S[k * N + j];
            b.x *= inv; b.y *= -inv;                              // conj(S[k][j]) / d_j
            double2 v = S[i * N + k];
            v.x -= a.x * b.x - a.y * b.y;
            v.y -= a.x * b.y + a.y * b.x;
            S[i * N + k] = v;
        }
        if (j > 0) {                                              // finish column j-1: L[i][j-1] = S[i][j-1]/sqrt(d_{j-1})
            const int c = j - 1;
            double dc = S[c * N + c].x;
            if (!(dc > 0.0) || !isfinite(dc)) dc = 1.0;
            const double r = 1.0 / sqrt(dc);
            for (int i = j + tid; i < N; i += CH_THREADS) {
                double2 v = S[i * N + c];
                v.x *= r; v.y *= r;
                S[i * N + c] = v;
            }
        }
        __syncthreads();
    }
    // diagonal: L[j][j] = sqrt(d_j) (the last column has nothing below it)
    for (int j = tid; j < N; j += CH_THREADS) {
        double dj = S[j * N + j].x;
        if (!(dj > 0.0) || !isfinite(dj)) dj = 1.0;
        S[j * N + j] = make_double2(sqrt(dj), 0.0);
    }
    __syncthreads();
    // X = L^{-1}: X[i][c] = (delta_ic - sum_{k=c}^{i-1} L[i][k] X[k][c]) / L[i][i];  Rinv[c][i] = conj(X[i][c])
    double2* Ri = Rinv + (size_t)w * N * N;
    for (int c = tid; c < N; c += CH_THREADS) {
        double2* row = Ri + (size_t)c * N;
        for (int i = 0; i < c; ++i) row[i] = make_double2(0.0, 0.0);
        for (int i = c; i < N; ++i) {
            double2 s = make_double2(i == c ? 1.0 : 0.0, 0.0);
            for (int k = c; k < i; ++k) {
                const double2 l = S[i * N + k];
                const double2 xk = row[k];                        // conj(X[k][c])
                s.x -= l.x * xk.x + l.y * xk.y;                   // l * conj(xk)
                s.y -= l.y * xk.x - l.x * xk.y;
            }
            const double r = 1.0 / S[i * N + i].x;
            row[i] = make_double2(s.x * r, -s.y * r);
        }
    }
    if (tid == 0) {
        if (logdet_r) logdet_r[w] = ld;
        if (info) info[w] = s_info;
    }
}

// logdet_r[w] = ldr[0][w] + ldr[1][w];  info[w] = first non-zero of (info_in[w], info2[0][w], info2[1][w])
__global__ void ortho_finish_kernel(int nw, const double* __restrict__ ldr, const int* __restrict__ info2,
                                    double* __restrict__ logdet_r, int* __restrict__ info, int keep_info) {
    const int w = blockIdx.x * blockDim.x + threadIdx.x;
    if (w >= nw) return;
    if (logdet_r) logdet_r[w] = ldr[w] + ldr[nw + w];
    if (info) {
        int v = keep_info ? info[w] : 0;
        if (v == 0) v = info2[w];
        if (v == 0) v = info2[nw + w];
        info[w] = v;
    }
}

}  // namespace

static int orthogonalize_i(afqmc_ctx* c, double2* phi, int nw, double* logdet_r, int* info, int keep_info, cudaStream_t st) {
    const Dims& d = c->d;
    const size_t mat = (size_t)d.N * d.N * sizeof(double2);
    const int use_smem = mat + 1024 <= (size_t)c->smem_optin;
    if (use_smem)
        if (int rc = afqmc_smem_optin(c, (const void*)cholesky_inverse_kernel, mat)) return rc;
    const size_t per = (size_t)d.M * d.N;
    for (int pass = 0; pass < 2; ++pass) {
        gram_kernel<<<dim3(ceil_div(d.N, GR_T), ceil_div(d.N, GR_T), nw), GR_THREADS, 0, st>>>(d.M, d.N, phi, c->ws_gram);
        AFQMC_LAUNCH_CHECK(c);
        cholesky_inverse_kernel<<<nw, CH_THREADS, use_smem ? mat : 0, st>>>(d.N, use_smem, c->ws_gram, c->ws_rinv,
                                                                            c->ws_ldr + (size_t)pass * nw, c->ws_info2 + (size_t)pass * nw);
        AFQMC_LAUNCH_CHECK(c);
        zg::Args a = {};
        a.A = phi; a.strideA = (long long)per; a.lda = d.N;
        a.B = c->ws_rinv; a.strideB = (long long)d.N * d.N; a.ldb = d.N;
        a.C = c->ws_T; a.strideC = (long long)per; a.ldc = d.N;
        a.D = nullptr; a.strideD = 0; a.ldd = 0;
        a.M = d.M; a.N = d.N; a.K = d.N; a.alpha = 1.0;
        if (zg::launch<false>(c, a, nw, st) != cudaSuccess) return AFQMC_CUDA_ERROR;
        c->launches++;
        AFQMC_CUDA_TRY(cudaMemcpyAsync(phi, c->ws_T, (size_t)nw * per * sizeof(double2), cudaMemcpyDeviceToDevice, st));
    }
    if (logdet_r || info) {
        ortho_finish_kernel<<<ceil_div(nw, 128), 128, 0, st>>>(nw, c->ws_ldr, c->ws_info2, logdet_r, info, keep_info);
        AFQMC_LAUNCH_CHECK(c);
    }
    return AFQMC_OK;
}

namespace {
__global__ void ortho_merge_kernel(int nw, const double* __restrict__ ldr_dn, const int* __restrict__ info_dn,
                                   double* __restrict__ logdet_r, int* __restrict__ info) {
    const int w = blockIdx.x * blockDim.x + threadIdx.x;
    if (w >= nw) return;
    if (logdet_r) logdet_r[w] += ldr_dn[w];
    if (info && info[w] == 0) info[w] = info_dn[w];
}
}  // namespace

// closed shell: one channel; open shell: each spin channel is orthogonalised on its own (log det R = sum, first non-zero info)
static int orthogonalize_x(afqmc_ctx* c, double2* phi, int nw, double* logdet_r, int* info, int keep_info, cudaStream_t st) {
    int rc = orthogonalize_i(c, phi, nw, logdet_r, info, keep_info, st);
    if (rc != AFQMC_OK || !c->dn) return rc;
    afqmc_ctx* dn = c->dn;
    rc = orthogonalize_i(dn, phi + (size_t)nw * c->d.M * c->d.N, nw, dn->ws_ldr_chan, dn->ws_info_chan, 0, st);
    if (rc != AFQMC_OK) return rc;
    if (logdet_r || info) {
        ortho_merge_kernel<<<ceil_div(nw, 128), 128, 0, st>>>(nw, dn->ws_ldr_chan, dn->ws_info_chan, logdet_r, info);
        AFQMC_LAUNCH_CHECK(c);
    }
    return AFQMC_OK;
}

AFQMC_API int afqmc_orthogonalize(afqmc_ctx* c, void* phi, int nw, double* logdet_r, int* info, void* stream) {
    if (c && c->prec32) return AFQMC_UNSUPPORTED;      // the block calls are FP64-only (boundary32.cu)
    if (!c || !phi || nw < 0 || nw > c->max_walkers) return AFQMC_INVALID_ARGUMENT;
    if (nw == 0) return AFQMC_OK;
    return orthogonalize_x(c, (double2*)phi, nw, logdet_r, info, 0, (cudaStream_t)stream);
}

// ------------------------------------------------------------------------------------------------
// The block: nsteps hybrid steps, energy + mixed estimator, orthogonalisation.
// ------------------------------------------------------------------------------------------------
namespace {
__global__ void info_merge_kernel(int nw, int first, const int* __restrict__ step_info, int* __restrict__ acc) {
    const int w = blockIdx.x * blockDim.x + threadIdx.x;
    if (w >= nw) return;
    const int prev = first ? 0 : acc[w];
    acc[w] = prev != 0 ? prev : step_info[w];
}
}  // namespace

AFQMC_API int afqmc_block(afqmc_ctx* c, void* phi, double* weight, const double* x, double dtau, int order, int nsteps,
                           int nw, void* energy, void* emixed, double* logdet_r, int* info, void* stream) {
    if (c && c->prec32) return AFQMC_UNSUPPORTED;      // the block calls are FP64-only (boundary32.cu)
    if (!c || !phi || !weight || !energy || !emixed || nw < 0 || nw > c->max_walkers || nsteps < 0 || order < 0 ||
        order > 32 || !(dtau >= 0.0) || (nsteps > 0 && !x))
        return AFQMC_INVALID_ARGUMENT;
    if (!c->b1_set) return AFQMC_INVALID_ARGUMENT;
    if (nw == 0) return AFQMC_OK;
    // the block uses the result buffers of pipeline slot 0 (ws_logdet, ws_info): pipelined host steps are completed first
    for (int slot = 0; slot < 2; ++slot)
        if (c->pipe_busy[slot])
            if (int prc = afqmc_step_host_end(c, slot)) return prc;
    const Dims& d = c->d;
    cudaStream_t st = (cudaStream_t)stream;
    double2* ph = (double2*)phi;
    double2* ld[2] = {c->ws_logdet, c->ws_logdet2};
    const size_t xstride = (size_t)nw * d.Nk * d.nchol;
    int rc;
    auto merge = [&](int first) {
        if (!info) return AFQMC_OK;
        info_merge_kernel<<<ceil_div(nw, 128), 128, 0, st>>>(nw, first, c->ws_info, info);
        AFQMC_LAUNCH_CHECK(c);
        return AFQMC_OK;
    };
    AfqmcFuseGuard fuse(c);      // Green's epilogue also writes the force-bias B fragments (zgemm.cuh FragOut)
    if ((rc = afqmc_x_green(c, ph, nw, c->ws_theta, ld[0], c->ws_info, st)) != AFQMC_OK) return rc;
    if ((rc = merge(1)) != AFQMC_OK) return rc;
    for (int s = 0; s < nsteps; ++s) {
        const double* xs = x + (size_t)s * xstride;
        if ((rc = afqmc_x_force_bias(c, c->ws_theta, nw, afqmc_x_vbias_ws(c), st)) != AFQMC_OK) return rc;
        if ((rc = afqmc_i_vhs(c, xs, afqmc_x_vbias_ws(c), dtau, nw, c->ws_vhs, st)) != AFQMC_OK) return rc;
        if ((rc = afqmc_x_apply_onebody(c, ph, nw, st)) != AFQMC_OK) return rc;
        if ((rc = afqmc_x_propagate(c, c->ws_vhs, dtau, order, ph, nw, st)) != AFQMC_OK) return rc;
        if ((rc = afqmc_x_apply_onebody(c, ph, nw, st)) != AFQMC_OK) return rc;
        // overlap of the new walker = Green's function of the next step (or of the energy evaluation)
        if ((rc = afqmc_x_green(c, ph, nw, c->ws_theta, ld[(s + 1) & 1], c->ws_info, st)) != AFQMC_OK) return rc;
        if ((rc = merge(0)) != AFQMC_OK) return rc;
        if ((rc = hybrid_weight_i(c, xs, afqmc_x_vbias_ws(c), dtau, ld[s & 1], ld[(s + 1) & 1], c->ws_info, nw, weight, nullptr, st)) != AFQMC_OK)
            return rc;
    }
    if ((rc = afqmc_i_local_energy(c, c->ws_theta, nw, (double2*)energy, st)) != AFQMC_OK) return rc;
    mixed_estimator_kernel<<<1, 32, 0, st>>>(nw, (const double2*)energy, weight, (double2*)emixed);
    AFQMC_LAUNCH_CHECK(c);
    return orthogonalize_x(c, ph, nw, logdet_r, info, 1, st);
}
