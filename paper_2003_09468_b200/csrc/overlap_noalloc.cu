// afqmc_overlap_noalloc: a1 + a2 (overlap and its log-determinant, PAPER.md:142 Eq. 27-28, :135-146) for callers that
// cannot allocate device memory -- code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.
//
// The other overlap kernels keep the N x N matrices O_w in a context-owned workspace that afqmc_create allocates.  This
// variant needs no context: the caller passes the trial and the walkers, and the matrices live in ONE file-scope
// `static __device__` array of AFQMC_NOALLOC_SCRATCH_BYTES (16 MiB; every GPU that loads the library holds it until the
// process exits).  The entry point calls no cudaMalloc / cudaFree and no allocating library routine.
//
// In HOST code the array's name is a host-side stand-in, not a device address (a kernel given it would fault or, where the
// GPU can reach host memory, silently use the wrong memory), so the address is taken with cudaGetSymbolAddress, once per
// device, with that device current (na_scratch_ptr below), and that pointer is what the kernel receives.
//
// Every call shares the array and finds the previous call's contents in it.  Nothing has to start at zero here: a1 writes
// every element of every O_w that a2 reads (all N x N entries of the nw matrices of the call) before the elimination
// starts, so nothing is cleared.  Two calls that OVERLAP on the GPU (different streams, or graph branches that run side by
// side) race on the array: serialise them.
#include <mutex>
#include <math_constants.h>
#include "common.cuh"

#define AFQMC_NOALLOC_SCRATCH_BYTES (16u << 20)
#define AFQMC_NOALLOC_MAX_N 1024          // row / column buffers of the kernel are static shared memory

static __device__ __align__(256) unsigned char afqmc_noalloc_scratch[AFQMC_NOALLOC_SCRATCH_BYTES];

namespace {

constexpr int NA_MAX_DEVICES = 64;
std::mutex na_mutex;
unsigned char* na_ptr[NA_MAX_DEVICES] = {};      // device address of the array on each device, resolved once

// the device address of afqmc_noalloc_scratch on the CURRENT device (nullptr: *rc holds the error)
unsigned char* na_scratch_ptr(int* rc) {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= NA_MAX_DEVICES) { (void)cudaGetLastError(); *rc = AFQMC_CUDA_ERROR; return nullptr; }
    std::lock_guard<std::mutex> g(na_mutex);
    if (!na_ptr[dev]) {
        unsigned char* p = nullptr;
        if (cudaGetSymbolAddress((void**)&p, afqmc_noalloc_scratch) != cudaSuccess || !p) { (void)cudaGetLastError(); *rc = AFQMC_CUDA_ERROR; return nullptr; }
        na_ptr[dev] = p;
    }
    *rc = AFQMC_OK;
    return na_ptr[dev];
}

inline int na_ld(int N) { return N | 1; }       // odd leading dimension, as the context's workspace uses

constexpr int NA_THREADS = 512;

// One CTA per walker.  O_w at scratch + w*N*LD (global memory, L2-resident); LU with partial pivoting (largest modulus,
// smallest row index on ties: the pivot sequence of the other overlap kernels), det O = (-1)^swaps * prod(pivots).
__global__ void __launch_bounds__(NA_THREADS) overlap_lu_noalloc_kernel(
    int Nk, int m, int n, int N, int M, int LD, const double2* __restrict__ psi_t, const double2* __restrict__ phi,
    double2* scratch, double2* __restrict__ logdet, int* __restrict__ info /*nullable*/) {
    __shared__ double2 rowbuf[AFQMC_NOALLOC_MAX_N];
    __shared__ double2 colbuf[AFQMC_NOALLOC_MAX_N];
    __shared__ double best_val[32];
    __shared__ int best_idx[32];
    __shared__ int piv_row, sh_info, nswaps;
    __shared__ double acc_r, acc_i;
    const int w = blockIdx.x, tid = threadIdx.x, nthr = blockDim.x, lane = tid & 31, warp = tid >> 5;
    double2* a = scratch + (size_t)w * N * LD;
    const double2* ph = phi + (size_t)w * M * N;

    // ---- a1: O[(k,a)][j] = sum_p conj(A_k[p][a]) Phi[(k,p)][j]; every element the elimination reads is written here ----
    for (int e = tid; e < N * N; e += nthr) {
        const int j = e % N, i = e / N, k = i / n, aa = i % n;
        const double2* Ab = psi_t + (size_t)k * m * n + aa;
        const double2* Pb = ph + (size_t)k * m * N + j;
        double2 acc = make_double2(0.0, 0.0);
        for (int p = 0; p < m; ++p) {
            double2 av = Ab[p * n];
            av.y = -av.y;
            acc = cfma(av, Pb[(size_t)p * N], acc);
        }
        a[i * LD + j] = acc;
    }
    if (tid == 0) { sh_info = 0; nswaps = 0; acc_r = 0.0; acc_i = 0.0; }
    __syncthreads();

    // ---- a2: LU with partial pivoting, in place ----
    for (int j = 0; j < N; ++j) {
        double bv = -1.0;
        int bi = 0x7fffffff;
        for (int i = j + tid; i < N; i += nthr) {
            const double2 v = a[i * LD + j];
            const double mag = v.x * v.x + v.y * v.y;
            if (mag > bv) { bv = mag; bi = i; }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const double ov = __shfl_xor_sync(0xffffffffu, bv, o);
            const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
            if (ov > bv || (ov == bv && oi < bi)) { bv = ov; bi = oi; }
        }
        if (lane == 0) { best_val[warp] = bv; best_idx[warp] = bi; }
        __syncthreads();
        if (warp == 0) {
            const int nwarps = nthr >> 5;
            bv = lane < nwarps ? best_val[lane] : -1.0;
            bi = lane < nwarps ? best_idx[lane] : 0x7fffffff;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                const double ov = __shfl_xor_sync(0xffffffffu, bv, o);
                const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
                if (ov > bv || (ov == bv && oi < bi)) { bv = ov; bi = oi; }
            }
            if (lane == 0) {
                if (bi == 0x7fffffff) bi = j;                                   // column of NaNs: stay in range, flagged below
                piv_row = bi;
                if (!(bv > 0.0) && sh_info == 0) sh_info = j + 1;               // exactly-zero (or NaN) pivot
                if (bi != j) nswaps++;
                const double2 pv = a[bi * LD + j];
                acc_r += log(hypot(pv.x, pv.y));
                acc_i += atan2(pv.y, pv.x);
            }
        }
        __syncthreads();
        const int p = piv_row;
        const double2 pv = a[p * LD + j];
        const double den = pv.x * pv.x + pv.y * pv.y;
        const double2 ip = (den > 0.0) ? make_double2(pv.x / den, -pv.y / den) : make_double2(0.0, 0.0);
        __syncthreads();                                  // a[p][j] has been read by everyone before the swap moves it
        // swap rows j <-> p in columns >= j; the pivot row of the trailing block goes to shared memory
        for (int c = j + tid; c < N; c += nthr) {
            const double2 rp = a[p * LD + c];
            if (p != j) { a[p * LD + c] = a[j * LD + c]; a[j * LD + c] = rp; }
            rowbuf[c] = rp;
        }
        __syncthreads();
        for (int i = j + 1 + tid; i < N; i += nthr) colbuf[i] = cmul(a[i * LD + j], ip);     // multipliers
        __syncthreads();
        const int rem = N - 1 - j;
        for (int e = tid; e < rem * rem; e += nthr) {
            const int i = j + 1 + e / rem, c = j + 1 + e % rem;
            double2 f = colbuf[i];
            f.x = -f.x; f.y = -f.y;
            a[i * LD + c] = cfma(f, rowbuf[c], a[i * LD + c]);
        }
        __syncthreads();
    }

    // ---- log det O = sum log(pivot) + i*pi*(#swaps odd), phase wrapped to (-pi, pi] ----
    if (tid == 0) {
        double si = acc_i;
        if (nswaps & 1) si += CUDART_PI;
        si = si - 2.0 * CUDART_PI * ceil((si - CUDART_PI) / (2.0 * CUDART_PI));
        logdet[w] = make_double2(acc_r, si);
        if (info) info[w] = sh_info;
    }
}

}  // namespace

AFQMC_API size_t afqmc_overlap_noalloc_max_bytes(void) { return (size_t)AFQMC_NOALLOC_SCRATCH_BYTES; }

// scratch bytes a call needs (0 for bad dims); pure host arithmetic
AFQMC_API size_t afqmc_overlap_noalloc_bytes(const afqmc_dims* dims, int nw) {
    if (!dims || nw < 0) return 0;
    for (int i = 0; i < 3; ++i) if (dims->g[i] < 1) return 0;
    const long long Nk = (long long)dims->g[0] * dims->g[1] * dims->g[2];
    if (dims->n < 1 || dims->m < dims->n || Nk * dims->n > (1 << 20)) return 0;
    const int N = (int)(Nk * dims->n);
    return (size_t)nw * N * na_ld(N) * sizeof(double2);
}

AFQMC_API int afqmc_overlap_noalloc_setup(void) {
    int rc = AFQMC_OK;
    (void)na_scratch_ptr(&rc);
    return rc;
}

AFQMC_API int afqmc_overlap_noalloc(const afqmc_dims* dims, const void* psi_t, const void* phi, int nw, void* logdet, int* info,
                                    void* stream) {
    if (!dims || !psi_t || !phi || !logdet || nw < 0) return AFQMC_INVALID_ARGUMENT;
    for (int i = 0; i < 3; ++i) if (dims->g[i] < 1) return AFQMC_INVALID_ARGUMENT;
    const long long Nk = (long long)dims->g[0] * dims->g[1] * dims->g[2];
    if (dims->n < 1 || dims->m < dims->n || Nk > AFQMC_MAX_NK) return AFQMC_INVALID_ARGUMENT;
    if (dims->closed_shell != 1 || dims->precision != 0) return AFQMC_UNSUPPORTED;
    if (Nk * dims->n > AFQMC_NOALLOC_MAX_N) return AFQMC_SCRATCH_LIMIT;
    const int N = (int)(Nk * dims->n), M = (int)(Nk * dims->m), LD = na_ld(N);
    if ((size_t)nw * N * LD * sizeof(double2) > (size_t)AFQMC_NOALLOC_SCRATCH_BYTES) return AFQMC_SCRATCH_LIMIT;
    if (nw == 0) return AFQMC_OK;
    int rc = AFQMC_OK;
    unsigned char* scratch = na_scratch_ptr(&rc);
    if (!scratch) return rc;
    const int threads = N * N < 4096 ? 256 : NA_THREADS;
    overlap_lu_noalloc_kernel<<<nw, threads, 0, (cudaStream_t)stream>>>(
        (int)Nk, dims->m, dims->n, N, M, LD, (const double2*)psi_t, (const double2*)phi, reinterpret_cast<double2*>(scratch),
        (double2*)logdet, info);
    if (cudaGetLastError() != cudaSuccess) return AFQMC_CUDA_ERROR;
    return AFQMC_OK;
}
