// Internal declarations shared by the translation units of libafqmc (not part of the ABI).
// Hardware target: sm_100a (B200).  FP64 tensor-core op used throughout: mma.sync m8n8k4 f64
// (SASS DMMA.8x8x4); tcgen05 has no f64 kind, so TMEM/UMMA do not apply to this path.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/afqmc.h"

#define AFQMC_MAX_NK 512
#define AFQMC_FB_MAXKC 16   // max pieces a force-bias tile is cut into (sizes the partial-tile workspace)
#define AFQMC_LX_PAD 1024   // doubles of zero padding after Lx (the exchange kernel prefetches up to 4 k-steps ahead)
// exported C-ABI entry points (everything else in the library has hidden visibility)
#define AFQMC_API extern "C" __attribute__((visibility("default")))

// ----------------------------------------------------------------------------------------
// Dimensions and derived sizes (host + device POD)
// ----------------------------------------------------------------------------------------
struct Dims {
    int g[3];
    int Nk, m, n, nchol;
    int M, N;      // Nk*m, Nk*n
    int KS;        // k-steps (of 4 reals) covering one complex row of length m: ceil(2m/4)
    int NAG;       // groups of 4 occupied orbitals: ceil(n/4)
    int GP;        // pairs of Cholesky vectors: ceil(nchol/2)   (vHS k-steps)
    int GQ;        // quads of Cholesky vectors: ceil(nchol/4)   (exchange tasks: two M-tiles each)
    int PRT;       // octets of (p,r) pairs: ceil(m*m/8)         (vHS M-tiles)
};

// Kernel attributes that were set / queried for this context.  A function attribute belongs to the (function, device)
// pair and a context lives on one device, so the record is per CONTEXT: nothing in the library is process-wide state.
struct FuncAttr { const void* fn; int smem; int occ; int carveout; int occ_smem; };
#define AFQMC_MAX_FATTR 128

// The context.  All pointers are device memory owned by the context.
struct afqmc_ctx {
    alignas(64) unsigned char tmap_lxu[128];   // CUtensorMaps of LxU and ws_thetaU (exchange_tc.cu); valid iff tmap_lxu_ok
    alignas(64) unsigned char tmap_thu[128];      // images of 8 walkers
    alignas(64) unsigned char tmap_thu16[128];    // images of 16 walkers
    int tmap_lxu_ok;
    Dims d;
    int max_walkers;
    // static tables
    int* kminus;   // [Nk(k)][Nk(Q)] -> index of k-Q
    int* kplus;    // [Nk(k)][Nk(Q)] -> index of k+Q
    int* kneg;     // [Nk]           -> index of -Q
    int* units;    // exchange work units, int4-packed (Q,k,k2,mult) [nunits]
    int nunits;
    int ex_parts;     // partial sums per exchange unit written by the last exchange launch (1, or NAG^2 * chunks: exchange3m.cu)
    int ex_parts_max; // ... that ws_expart was sized for
    // static tensors
    double2* psi_t; // [Nk][m][n]
    double2* ht;    // [Nk][n][m]   half-rotated one-body
    double2* Lh;    // half-rotated Cholesky tensor, natural layout [Q][k][a][gamma][r]: computed ONCE in a0; every packed
                    // operand below is a pure re-layout of it
    double* Lxc;    // exchange, generic 3M kernel (exchange3m.cu; default for m > 28): complex fragments [Q][k][ag][gq][ks][lane][4]
    double* Lxr;    // exchange, generic kernel with a REAL operand (real orbitals): real parts only, [Q][k][ag][gq][ks][lane][2]; first use
    double* Lx3t;   // exchange, register-B 3M kernel (default for m <= 28): the three A variants [Q][k][ag][gq][ml][lane][2]
                    // (only the default one of Lxc / Lx3t is packed in a0; the other on first use)
    double* Lx;     // exchange, 4M kernel (energy.cu): [Q][k][ag][gq][s][lane][2]; packed on first use (option exchange_3m = 0)
    float* LxU;     // exchange, tcgen05 TF32 kernel (exchange_tc.cu): shared-memory tile images [Q][k][tile][hi/lo][128 x KP]; first use
    float* LxT;     // exchange, TF32 fragments [Q][k][gq][ks][lane][4] (exchange_tf32.cu; n <= 4 only); packed on first use
    double* Lf;     // force-bias operand Lf3[Q][m-tile][k-step][lane] complex fragments over the flattened K = (k,a,r) (force_bias.cu)
    float* Lff;     // precision = 1: the same in single precision (Lf is then NULL)
    float2* Lv3f;   // precision = 1: the vHS operand in single precision (Lv3 is then NULL): half the bytes of the HBM-bound streams
    double2* Lv3;   // vHS operand [unit][prt][ks][lane] complex fragments (vhs.cu); one block per (Q,-Q) pair if vhs_paired
    int* vunits;    // vHS work units, int4-packed (Q, k, kind, 0) [nvunits]; kind 1 = block + its (-Q,k-Q) partner
    int nvunits;
    int vhs_paired; // 1 = the caller's L satisfies the (Q,-Q) identity (checked in afqmc_create): one block per pair stored
    // workspace (sized by max_walkers)
    double2* ws_O;      // [nw][N][LD]  elimination workspace when the matrix does not fit shared memory
    double2* ws_oinvT;  // [nw][N][N]   transposed inverse overlap
    double2* ws_theta;  // [nw][N][M]
    double2* ws_vbias;  // [nw][Nk][nchol]
    double2* ws_xi;     // [nw][Nk][nchol]
    double2* ws_vhs;    // [nw][M][M]
    double2* ws_T;      // [2][nw][M][N] Taylor ping-pong (legacy GEMM path)
    double* ws_Tx;      // [2][nw][expanded] Taylor ping-pong in the expanded B-fragment layout of tgemm.cuh
    double2* ws_expart; // [nunits][nw]  exchange partial sums
    float* ws_thetaU;   // [Nk][Nk][walker groups of 8][hi/lo][64 x KP] theta blocks as B images of the tcgen05 exchange kernel
    double2* ws_thetaF; // [Nk(Q)][walker groups][k-steps][NT][32] theta as B fragments of the force-bias GEMM (force_bias.cu)
    double2* ws_fbpart; // [AFQMC_FB_MAXKC][nw][Nk][nchol] force-bias partial tiles (stream-K pieces)
    double* ws_x;       // [nw][Nk][nchol] (host-entry staging)
    double2* ws_phi;    // [nw][M][N]     (host-entry staging)
    double2* ws_energy; // [nw][3]
    double2* ws_logdet; // [nw]
    int* ws_info;       // [nw]
    // the block (block.cu)
    double2* b1;        // [Nk][m][m] one-body half-step propagator exp(-dtau/2 h1p); valid iff b1_set
    double2* ws_b1tmp;  // [Nk][3][m][m] scratch of the matrix exponential
    double2* ws_gram;   // [nw][N][N] Gram matrix / Cholesky factor of the orthogonalisation
    double2* ws_rinv;   // [nw][N][N] inverse of the triangular factor
    double2* ws_logdet2;// [nw] overlap of the walker before the propagation
    double* ws_ldr;     // [2][nw] log det R of the two Cholesky-QR passes
    int* ws_info2;      // [2][nw] status of the two Cholesky passes
    int b1_set;
    // open shell (afqmc_dims.closed_shell = 0): this context is the spin-UP channel and owns everything spin independent;
    // `dn` is the spin-DOWN channel (is_child = 1: no vHS operand / workspace, b1 shared).  spin_factor = 2 for a closed
    // shell (one channel stands for both spins: E1, vbias, EX carry it), 1 per channel of an open shell.
    afqmc_ctx* dn;
    int is_child;
    double spin_factor;
    double2* ws_vbtot;  // [nw][Nk][nchol] spin-summed force bias (open shell)
    double2* ws_ld_chan; // [nw] this channel's log det (open shell: combined by openshell.cu)
    int* ws_info_chan;  // [nw] this channel's status
    double* ws_ldr_chan; // [nw] this channel's log det R of the orthogonalisation
    // real orbitals (the dense Gamma-point supercell representation of PAPER.md:260, :276-284): detected in a0 as exactly zero
    // imaginary parts of the half-rotated tensor Lh (force bias, exchange) / of L (vHS); the contractions then need two real
    // products per complex product instead of three.  opt_real = 0 switches the shortcut off (testing aid).
    int real_lh, real_l, opt_real;
    int prec32;         // 1 = complex64 boundary (afqmc_dims.precision = 1, boundary32.cu)
    float* ws_f32;      // precision 1: device staging of afqmc_step_host ([nw][M][N][2] + x + energy + logdet floats)
    int fuse_frag;      // 1 while a composition (afqmc_step, afqmc_block) runs: Green's epilogue also writes ws_thetaF ...
    int frag_nw;        // ... for this many walkers (0: ws_thetaF holds no valid fragments) ...
    const void* frag_src; // ... of the Green's function at this address
    long long launches;
    int opt_exchange_depth; // 0/3 = three k-steps of fragment prefetch, 2 = two
    int opt_exchange_minb;  // tuning aid: 1 = ask for more resident CTAs per SM
    int opt_exchange_tc;    // 1 (default) = the mixed-precision exchange runs on tcgen05.mma / TMEM (exchange_tc.cu), 0 = mma.sync kernel
    int opt_exchange_prec;  // 0 (default) = FP64 exchange kernels; mixed precision on the TF32 tensor cores (n <= 4): 1 = 3xTF32 split, 2 = 1xTF32
    int opt_exchange_3m;    // 1 (default) = 3M exchange kernel when n <= 4, 0 = the 4M kernel of energy.cu
    int opt_exchange_wpc;   // 0 = automatic, else warps per CTA of the exchange kernel (4,5,6,8)
    int opt_exchange_np;    // tuning aid (3M kernel): 0 = automatic, else 1/2/4 walker pairs (n-tiles) per warp
    int opt_exchange_ctas;  // tuning aid: 0 = as many CTAs of the register-B exchange kernel per SM as fit, else at most this many
    int opt_exchange_regb;  // 1 (default) = theta block of a warp in registers when m <= 28 (exchange3m_reg_kernel), 0 = generic kernel
    int opt_timers;     // record stage events in afqmc_step
    int opt_taylor_legacy;  // testing aid: 1 = shared-memory-tiled zgemm for the Taylor chain
    int opt_taylor_wpc;     // tuning aid: 0 = automatic, else 3/4/5 warps per CTA of the Taylor GEMM
    int opt_taylor_groups;  // tuning aid: 0 = automatic, else the number of column groups of the Taylor GEMM
    int opt_taylor_subbatch; // 0 = all walkers per Taylor pass, else walkers per pass (their V stays in L2 across the orders)
    int opt_green_cs;       // tuning aid: 4 = cluster of four CTAs per walker for 64 < N <= 128 (default two)
    int opt_green_legacy;   // testing aid: 1 = shared/global-memory elimination kernel instead of the register-resident one
    cudaStream_t copy_stream;   // afqmc_step_host: downloads the propagated walkers during the energy evaluation
    cudaEvent_t ev_copy[2];
    // afqmc_step_host_begin / _end: two steps in flight.  Slot 0 stages in ws_phi / ws_x / ws_energy / ws_logdet / ws_info,
    // slot 1 in a second set allocated on its first use; uploads run on copyin_stream, the walker download on copy_stream.
    cudaStream_t copyin_stream;
    cudaEvent_t ev_pipe[2][4];   // per slot: inputs on the device | propagated walkers final | step complete | all results downloaded
    double2* pipe_phi; double* pipe_x; double2* pipe_energy; double2* pipe_logdet; int* pipe_info;
    int pipe_busy[2];
    cudaEvent_t ev[AFQMC_NUM_STAGES + 1];
    int ev_valid;
    FuncAttr fattr[AFQMC_MAX_FATTR];   // see afqmc_smem_optin()
    int nfattr;
    int device;         // the CUDA device the context was created on
    int smem_optin;     // max dynamic shared memory per block (bytes)
    int smem_sm;        // shared memory per SM (bytes)
    int num_sms;
};

// ----------------------------------------------------------------------------------------
// Device helpers
// ----------------------------------------------------------------------------------------
#ifdef __CUDACC__

// D(8x8) += A(8x4, row) * B(4x8, col), FP64.  Fragments (lane l):
//   a = A[l>>2][l&3];  b = B[l&3][l>>2];  c0,c1 = C[l>>2][2*(l&3) + {0,1}]
__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(c0), "+d"(c1)
                 : "d"(a), "d"(b));
}

// Real embedding of a complex GEMM  C = A*B  (8 real flops per complex multiply-add, exact):
//   A row -> [Re a_0, Im a_0, Re a_1, Im a_1, ...]            (interleaved storage as is)
//   B     -> for the real-part output column (d=0):  [Re b_k, -Im b_k];  for d=1: [Im b_k, Re b_k]
// A B-fragment lane with K parity c (0: multiplies Re a, 1: multiplies Im a) and output part d
// therefore reads component (c^d) of b and flips its sign iff (c==1 && d==0).
__device__ __forceinline__ double flip_sign(double v, unsigned mask) {
    return __hiloint2double(__double2hiint(v) ^ (int)mask, __double2loint(v));
}

__device__ __forceinline__ double2 cmul(double2 a, double2 b) {
    return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
__device__ __forceinline__ double2 cfma(double2 a, double2 b, double2 c) {  // a*b + c
    c.x = fma(a.x, b.x, c.x); c.x = fma(-a.y, b.y, c.x);
    c.y = fma(a.x, b.y, c.y); c.y = fma(a.y, b.x, c.y);
    return c;
}
// ---- mbarrier / bulk asynchronous copy (TMA engine, SASS UBLKCP) primitives shared by the kernels that stage operands ----
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_fence_init() {
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n.reg .pred p;\nWAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\nbra WAIT_%=;\nDONE_%=:\n}\n" ::"r"(smem_u32(bar)), "r"(parity)
        : "memory");
}
// Orders this thread's earlier generic-proxy accesses to shared memory (LDS) before later async-proxy accesses (the bulk copy
// that refills a ring stage).  Every consumer executes it before it releases a stage: without it the refill of a stage is not
// ordered after the reads of its previous contents (PTX memory model: two proxies), and the vHS kernel's two-product variant
// was seen to read partly refilled stages at 4 resident CTAs per SM (run-to-run differences in whole warp slices).
__device__ __forceinline__ void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory"); }
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
// global -> shared, `bytes` a multiple of 16, both addresses 16-byte aligned; completion is counted on `bar`
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];\n" ::"r"(smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
// the same with an L2 eviction-priority hint (createpolicy below): for a small operand that is re-read all through a kernel
// while a much larger one streams past it
__device__ __forceinline__ void bulk_g2s_hint(void* dst, const void* src, uint32_t bytes, uint64_t* bar, uint64_t policy) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;\n" ::"r"(smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar)), "l"(policy)
                 : "memory");
}
__device__ __forceinline__ uint64_t l2_policy_evict_last() {
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;\n" : "=l"(p));
    return p;
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
#endif  // __CUDACC__

// ----------------------------------------------------------------------------------------
// Host-side helpers
// ----------------------------------------------------------------------------------------
#define AFQMC_CUDA_TRY(expr)                           \
    do {                                               \
        cudaError_t e__ = (expr);                      \
        if (e__ != cudaSuccess) {                      \
            (void)cudaGetLastError();                  \
            return (e__ == cudaErrorMemoryAllocation) ? AFQMC_OUT_OF_MEMORY : AFQMC_CUDA_ERROR; \
        }                                              \
    } while (0)

#define AFQMC_LAUNCH_CHECK(ctx)                        \
    do {                                               \
        (ctx)->launches++;                             \
        cudaError_t e__ = cudaGetLastError();          \
        if (e__ != cudaSuccess) return AFQMC_CUDA_ERROR; \
    } while (0)

static inline int ceil_div(long long a, long long b) { return (int)((a + b - 1) / b); }

// Makes sure kernel `fn` may be launched with `smem` bytes of dynamic shared memory on the context's device.  The limit is
// only ever RAISED (it is shared by every context on the device), and what was done is remembered in the context, not in
// function-local statics: a second context on another device, or a context created after another one was destroyed,
// opts in again.  Returns AFQMC_UNSUPPORTED if the device cannot give that much.
static inline FuncAttr* afqmc_fattr(afqmc_ctx* c, const void* fn) {
    for (int i = 0; i < c->nfattr; ++i)
        if (c->fattr[i].fn == fn) return &c->fattr[i];
    if (c->nfattr == AFQMC_MAX_FATTR) return nullptr;
    FuncAttr* f = &c->fattr[c->nfattr++];
    f->fn = fn; f->smem = 0; f->occ = -1; f->carveout = 0; f->occ_smem = -1;
    return f;
}
// Asks the driver for the largest shared-memory carveout for `fn` (once per context): kernels whose residency is set by
// shared memory (many small CTAs) otherwise get a carveout sized for fewer CTAs than the registers allow.
static inline void afqmc_prefer_smem(afqmc_ctx* c, const void* fn) {
    FuncAttr* f = afqmc_fattr(c, fn);
    if (f && f->carveout) return;
    if (cudaFuncSetAttribute(fn, cudaFuncAttributePreferredSharedMemoryCarveout, (int)cudaSharedmemCarveoutMaxShared) != cudaSuccess)
        (void)cudaGetLastError();
    if (f) { f->carveout = 1; f->occ = -1; }
}
static inline int afqmc_smem_optin(afqmc_ctx* c, const void* fn, size_t smem) {
    if (smem <= 48 * 1024) return AFQMC_OK;
    if (smem > (size_t)c->smem_optin) return AFQMC_UNSUPPORTED;
    FuncAttr* f = afqmc_fattr(c, fn);
    if (f && (size_t)f->smem >= smem) return AFQMC_OK;
    cudaFuncAttributes fa;
    if (cudaFuncGetAttributes(&fa, fn) != cudaSuccess) { (void)cudaGetLastError(); return AFQMC_CUDA_ERROR; }
    if ((size_t)fa.maxDynamicSharedSizeBytes < smem &&
        cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) {
        (void)cudaGetLastError();
        return AFQMC_CUDA_ERROR;
    }
    if (f) { f->smem = (int)smem; f->occ = -1; }
    return AFQMC_OK;
}

// internal entry points used across translation units (all asynchronous on `st`)
int afqmc_i_green(afqmc_ctx* c, const double2* phi, int nw, double2* theta, double2* logdet,
                  int* info, cudaStream_t st);
int afqmc_i_force_bias(afqmc_ctx* c, const double2* theta, int nw, double2* vbias, cudaStream_t st);
int afqmc_i_max_abs_imag(afqmc_ctx* c, const double2* p, size_t n, double* out_host, cudaStream_t st);   // synchronises st
int afqmc_i_pack_force_bias_operand(afqmc_ctx* c, cudaStream_t st);
void afqmc_i_fb_frag_layout(const afqmc_ctx* c, int nw, int* NT, int* nwg, int* KSf);   // layout of ws_thetaF for nw walkers
// switches the Green -> force-bias fragment fusion on / off for a composition (both spin channels)
static inline void afqmc_set_fuse(afqmc_ctx* c, int on) {
    c->fuse_frag = on; c->frag_nw = 0; c->frag_src = nullptr;
    if (c->dn) afqmc_set_fuse(c->dn, on);
}
struct AfqmcFuseGuard {      // on for the lifetime of a composition call, off on every return path
    afqmc_ctx* c;
    explicit AfqmcFuseGuard(afqmc_ctx* ctx) : c(ctx) { afqmc_set_fuse(c, 1); }
    ~AfqmcFuseGuard() { afqmc_set_fuse(c, 0); }
};                     // a0: Lh -> Lf3 (allocates Lf / Lff)
int afqmc_i_vhs(afqmc_ctx* c, const double* x, const double2* vbias, double dtau, int nw,
                double2* vhs, cudaStream_t st);
int afqmc_i_propagate(afqmc_ctx* c, const double2* vhs, double dtau, int order, double2* phi, int nw,
                      cudaStream_t st);
int afqmc_i_local_energy(afqmc_ctx* c, const double2* theta, int nw, double2* energy, cudaStream_t st);
int afqmc_i_exchange3m(afqmc_ctx* c, const double2* theta, int nw, cudaStream_t st);   // AFQMC_UNSUPPORTED only if the staged theta blocks exceed shared memory
int afqmc_i_pack_exchange_operand(afqmc_ctx* c, cudaStream_t st);                       // a0: Lh -> Lx3t (m <= 28) or Lxc
size_t afqmc_i_lxc_doubles(const Dims& d);
int afqmc_i_exchange3m_parts_max(const afqmc_ctx* c);
int afqmc_i_exchange_tc(afqmc_ctx* c, const double2* theta, int nw, cudaStream_t st);    // tcgen05 version; AFQMC_UNSUPPORTED if n > 4 / too large
int afqmc_i_exchange_tf32(afqmc_ctx* c, const double2* theta, int nw, cudaStream_t st);  // AFQMC_UNSUPPORTED if n > 4
int afqmc_i_ensure_lx(afqmc_ctx* c, cudaStream_t st);     // packs the 4M operand Lx from Lh on first use
int afqmc_i_ensure_lxt(afqmc_ctx* c, cudaStream_t st);    // packs the TF32 operand LxT from Lh on first use (n <= 4)
int afqmc_i_pack_lxt(afqmc_ctx* c, cudaStream_t st);
size_t afqmc_i_lxt_floats(const Dims& d);
int afqmc_i_apply_onebody(afqmc_ctx* c, double2* phi, int nw, cudaStream_t st);
int afqmc_i_step(afqmc_ctx* c, double2* phi, const double* x, double dtau, int order, int nw, double2* energy,
                 double2* logdet, int* info, cudaStream_t st, cudaEvent_t phi_final /* nullable: recorded after the propagation */);
// open shell (openshell.cu): `c` is the spin-up context, c->dn the spin-down one; arrays are spin-major (up block, dn block)
int afqmc_os_green(afqmc_ctx* c, const double2* phi, int nw, double2* theta, double2* logdet, int* info, cudaStream_t st);
int afqmc_os_force_bias(afqmc_ctx* c, const double2* theta, int nw, double2* vbias, cudaStream_t st);
int afqmc_os_propagate(afqmc_ctx* c, const double2* vhs, double dtau, int order, double2* phi, int nw, cudaStream_t st);
int afqmc_os_apply_onebody(afqmc_ctx* c, double2* phi, int nw, cudaStream_t st);
// closed / open shell dispatch used by the compositions (step, block): same argument meaning, spin-major arrays when open
static inline int afqmc_x_green(afqmc_ctx* c, const double2* phi, int nw, double2* theta, double2* logdet, int* info, cudaStream_t st) {
    return c->dn ? afqmc_os_green(c, phi, nw, theta, logdet, info, st) : afqmc_i_green(c, phi, nw, theta, logdet, info, st);
}
static inline double2* afqmc_x_vbias_ws(afqmc_ctx* c) { return c->dn ? c->ws_vbtot : c->ws_vbias; }
static inline int afqmc_x_force_bias(afqmc_ctx* c, const double2* theta, int nw, double2* vbias, cudaStream_t st) {
    return c->dn ? afqmc_os_force_bias(c, theta, nw, vbias, st) : afqmc_i_force_bias(c, theta, nw, vbias, st);
}
static inline int afqmc_x_propagate(afqmc_ctx* c, const double2* vhs, double dtau, int order, double2* phi, int nw, cudaStream_t st) {
    return c->dn ? afqmc_os_propagate(c, vhs, dtau, order, phi, nw, st) : afqmc_i_propagate(c, vhs, dtau, order, phi, nw, st);
}
static inline int afqmc_x_apply_onebody(afqmc_ctx* c, double2* phi, int nw, cudaStream_t st) {
    return c->dn ? afqmc_os_apply_onebody(c, phi, nw, st) : afqmc_i_apply_onebody(c, phi, nw, st);
}
// complex numbers of one walker batch entry: all spin channels
static inline size_t afqmc_x_phi_elems(const afqmc_ctx* c) { return (size_t)c->d.M * (c->d.N + (c->dn ? c->dn->d.N : 0)); }
// complex64 boundary (boundary32.cu): same calls on float arrays, staged through the FP64 workspace
int afqmc32_widen_alloc(afqmc_ctx* c, const void* in, size_t ndoubles, double** out, cudaStream_t st);
int afqmc32_green(afqmc_ctx* c, const void* phi, int nw, void* theta, void* logdet, int* info, cudaStream_t st);
int afqmc32_force_bias(afqmc_ctx* c, const void* theta, int nw, void* vbias, cudaStream_t st);
int afqmc32_vhs(afqmc_ctx* c, const void* x, const void* vbias, double dtau, int nw, void* vhs, cudaStream_t st);
int afqmc32_propagate(afqmc_ctx* c, const void* vhs, double dtau, int order, void* phi, int nw, cudaStream_t st);
int afqmc32_local_energy(afqmc_ctx* c, const void* theta, int nw, void* energy, cudaStream_t st);
int afqmc32_step(afqmc_ctx* c, void* phi, const void* x, double dtau, int order, int nw, void* energy, void* logdet,
                 int* info, cudaStream_t st);
int afqmc32_step_host(afqmc_ctx* c, void* phi_host, const void* x_host, double dtau, int order, int nw, void* energy_host,
                      void* logdet_host, int* info_host, cudaStream_t st);
size_t afqmc_i_taylor_ws_doubles(const Dims& d);
size_t afqmc_i_vhs_field_doubles(const Dims& d, int nw);   // doubles of the expanded field operand (workspace ws_xi)   // per-walker doubles of one expanded Taylor buffer
// records stage event i on st when timers are on
static inline void afqmc_mark(afqmc_ctx* c, int i, cudaStream_t st) {
    if (c->opt_timers && c->ev[i]) cudaEventRecord(c->ev[i], st);
}
