// Batched complex128 GEMM on the FP64 tensor pipe (DMMA m8n8k4), used by a3 (Green) and a6 (Taylor).
//
//   C_b[i][j] = alpha * sum_k A_b[i][k] * B_b[k][j]      (+ optionally  D_b[i][j] += C_b[i][j])
//
// A is row-major with K contiguous (lda).  B is either N-contiguous (B[k*ldb + j], B_KCONTIG=false)
// or K-contiguous (B[j*ldb + k], B_KCONTIG=true).  The complex product is embedded in a real GEMM
// (common.cuh): A rows are used as stored (interleaved re/im = 2K reals); B is expanded to
// [[Br, Bi], [-Bi, Br]] while it is written to shared memory, directly in DMMA fragment order, so the
// inner loop is LDS.64 + DMMA only.  8 real flops per complex multiply-add, no wasted flops.
//
// CTA tile: BM = 16*WGM rows x BN = 4*NT complex columns, WGM warps, each warp 16 rows (2 m-tiles)
// x NT n-tiles (NT complex-column quads).  K chunk BK = 16 complex (8 DMMA k-steps), two shared
// memory stages with register prefetch of the next chunk.
#pragma once
#include "common.cuh"

namespace zg {

constexpr int BK = 16;             // complex K per chunk
constexpr int SA = 2 * BK + 4;     // A row stride in doubles: = 4 (mod 16) -> conflict-free LDS.64 frags

template <int WGM, int NT>
struct Cfg {
    static constexpr int BM = 16 * WGM;
    static constexpr int BN = 4 * NT;
    static constexpr int NTHR = 32 * WGM;
    static constexpr int A_DOUBLES = BM * SA;
    static constexpr int B_DOUBLES = (BK / 2) * NT * 32;
    static constexpr int SMEM_BYTES = 2 * (A_DOUBLES + B_DOUBLES) * 8;
    static constexpr int A_LD = (BM * BK + NTHR - 1) / NTHR;   // double2 loads per thread
    static constexpr int B_LD = (BK * BN + NTHR - 1) / NTHR;
};

// Optional second output of the epilogue (a3 -> a4 fusion): C[i][j] of batch entry w is also stored as an element of the
// force-bias B-fragment operand thetaF (force_bias.cu): row i = (k,a), column j = (k',r), Q = k - k' (table ktab[k*Nk + k']),
// kappa = i*m + r  ->  thetaF[Q][w / (8 NT)][kappa >> 2][(w >> 3) % NT][lane = (w & 7)*4 + (kappa & 3)].
struct FragOut {
    double2* F; const int* ktab;
    int m, n, Nk, NT, nwg, KSf;
};

struct Args {
    FragOut frag;                              // frag.F == nullptr: off
    const double2* A; long long strideA; int lda;
    const double2* B; long long strideB; int ldb;
    double2* C; long long strideC; int ldc;
    double2* D; long long strideD; int ldd;   // nullable accumulate target
    int M, N, K;
    double alpha;
};

template <int WGM, int NT, bool B_KCONTIG>
__global__ void __launch_bounds__(32 * WGM) zgemm_kernel(Args p) {
    using C_ = Cfg<WGM, NT>;
    extern __shared__ __align__(16) double smem[];
    double* As[2] = {smem, smem + C_::A_DOUBLES + C_::B_DOUBLES};
    double* Bs[2] = {smem + C_::A_DOUBLES, smem + 2 * C_::A_DOUBLES + C_::B_DOUBLES};

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int b = blockIdx.z;
    const int i0 = blockIdx.y * C_::BM, j0 = blockIdx.x * C_::BN;
    const double2* A = p.A + (size_t)b * p.strideA;
    const double2* B = p.B + (size_t)b * p.strideB;

    double2 ra[C_::A_LD], rb[C_::B_LD];

    auto load_global = [&](int k0) {
#pragma unroll
        for (int t = 0; t < C_::A_LD; ++t) {
            int e = tid + t * C_::NTHR;
            int k = e % BK, i = e / BK;
            double2 v = make_double2(0.0, 0.0);
            if (e < C_::BM * BK && i0 + i < p.M && k0 + k < p.K) v = A[(size_t)(i0 + i) * p.lda + k0 + k];
            ra[t] = v;
        }
#pragma unroll
        for (int t = 0; t < C_::B_LD; ++t) {
            int e = tid + t * C_::NTHR;
            int k, j;
            if (B_KCONTIG) { k = e % BK; j = e / BK; } else { j = e % C_::BN; k = e / C_::BN; }
            double2 v = make_double2(0.0, 0.0);
            if (e < BK * C_::BN && j0 + j < p.N && k0 + k < p.K)
                v = B_KCONTIG ? B[(size_t)(j0 + j) * p.ldb + k0 + k] : B[(size_t)(k0 + k) * p.ldb + j0 + j];
            rb[t] = v;
        }
    };
    auto store_smem = [&](int buf) {
#pragma unroll
        for (int t = 0; t < C_::A_LD; ++t) {
            int e = tid + t * C_::NTHR;
            int k = e % BK, i = e / BK;
            if (e < C_::BM * BK) *reinterpret_cast<double2*>(&As[buf][i * SA + 2 * k]) = ra[t];
        }
#pragma unroll
        for (int t = 0; t < C_::B_LD; ++t) {
            int e = tid + t * C_::NTHR;
            int k, j;
            if (B_KCONTIG) { k = e % BK; j = e / BK; } else { j = e % C_::BN; k = e / C_::BN; }
            if (e < BK * C_::BN) {
                // fragment (kstep k>>1, ntile j>>2): lane = (2*(j&3)+d)*4 + 2*(k&1)+c
                double* dst = &Bs[buf][((k >> 1) * NT + (j >> 2)) * 32 + (j & 3) * 8 + (k & 1) * 2];
                *reinterpret_cast<double2*>(dst) = make_double2(rb[t].x, -rb[t].y);      // d = 0: (Br, -Bi)
                *reinterpret_cast<double2*>(dst + 4) = make_double2(rb[t].y, rb[t].x);   // d = 1: (Bi,  Br)
            }
        }
    };

    double acc[2][NT][2];
#pragma unroll
    for (int mt = 0; mt < 2; ++mt)
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) acc[mt][nt][0] = acc[mt][nt][1] = 0.0;

    const int nchunks = (p.K + BK - 1) / BK;
    load_global(0);
    store_smem(0);
    __syncthreads();
    const int arow = warp * 16 + (lane >> 2);
    for (int c = 0; c < nchunks; ++c) {
        const int buf = c & 1;
        if (c + 1 < nchunks) load_global((c + 1) * BK);
        const double* as = As[buf] + arow * SA + (lane & 3);
        const double* bs = Bs[buf] + lane;
#pragma unroll
        for (int s = 0; s < BK / 2; ++s) {
            double a0 = as[4 * s], a1 = as[8 * SA + 4 * s];
            double bf[NT];
#pragma unroll
            for (int nt = 0; nt < NT; ++nt) bf[nt] = bs[(s * NT + nt) * 32];
#pragma unroll
            for (int nt = 0; nt < NT; ++nt) {
                dmma884(acc[0][nt][0], acc[0][nt][1], a0, bf[nt]);
                dmma884(acc[1][nt][0], acc[1][nt][1], a1, bf[nt]);
            }
        }
        if (c + 1 < nchunks) store_smem(buf ^ 1);
        __syncthreads();
    }

    // epilogue: lane holds complex element (row = lane>>2, column quad entry lane&3) of each tile
    double2* C = p.C + (size_t)b * p.strideC;
    double2* D = p.D ? p.D + (size_t)b * p.strideD : nullptr;
#pragma unroll
    for (int mt = 0; mt < 2; ++mt) {
        int i = i0 + warp * 16 + mt * 8 + (lane >> 2);
        if (i >= p.M) continue;
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) {
            int j = j0 + nt * 4 + (lane & 3);
            if (j >= p.N) continue;
            double2 v = make_double2(p.alpha * acc[mt][nt][0], p.alpha * acc[mt][nt][1]);
            C[(size_t)i * p.ldc + j] = v;
            if (p.frag.F) {
                const FragOut& f = p.frag;
                const int k2 = j / f.m, r = j - k2 * f.m, kap = i * f.m + r;
                const int Q = f.ktab[(i / f.n) * f.Nk + k2];
                f.F[((((size_t)Q * f.nwg + b / (8 * f.NT)) * f.KSf + (kap >> 2)) * f.NT + ((b >> 3) % f.NT)) * 32 + (b & 7) * 4 + (kap & 3)] = v;
            }
            if (D) {
                double2 o = D[(size_t)i * p.ldd + j];
                o.x += v.x; o.y += v.y;
                D[(size_t)i * p.ldd + j] = o;
            }
        }
    }
}

template <int WGM, int NT, bool B_KCONTIG>
static inline cudaError_t launch_one(afqmc_ctx* c, const Args& a, int batch, cudaStream_t st) {
    using C_ = Cfg<WGM, NT>;
    auto kern = zgemm_kernel<WGM, NT, B_KCONTIG>;
    if (afqmc_smem_optin(c, (const void*)kern, C_::SMEM_BYTES) != AFQMC_OK) return cudaErrorInvalidValue;
    dim3 grid((a.N + C_::BN - 1) / C_::BN, (a.M + C_::BM - 1) / C_::BM, batch);
    kern<<<grid, C_::NTHR, C_::SMEM_BYTES, st>>>(a);
    return cudaGetLastError();
}

// Picks the column-tile width (NT in {7,8,9} quads) that wastes the fewest padded columns.
template <bool B_KCONTIG>
static inline cudaError_t launch(afqmc_ctx* c, const Args& a, int batch, cudaStream_t st) {
    int best = 8;
    long long bestw = -1;
    for (int nt = 7; nt <= 9; ++nt) {
        long long bn = 4 * nt, padded = ((a.N + bn - 1) / bn) * bn;
        if (bestw < 0 || padded < bestw || (padded == bestw && nt > best)) { bestw = padded; best = nt; }
    }
    switch (best) {
        case 7: return launch_one<4, 7, B_KCONTIG>(c, a, batch, st);
        case 9: return launch_one<4, 9, B_KCONTIG>(c, a, batch, st);
        default: return launch_one<4, 8, B_KCONTIG>(c, a, batch, st);
    }
}

}  // namespace zg
