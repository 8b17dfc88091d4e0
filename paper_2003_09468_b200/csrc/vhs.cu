// a5 vHS:  field assembly (reading R7) and the contraction of Eq. 48:
//   vhs_w[(k,p),(k-Q,r)] = sum_g L[Q][k][g][p][r] xi_w[Q][g]
//
// Per (Q,k) block this is a complex GEMM on the FP64 tensor pipe: rows = (p,r) pairs, K = gamma, columns = walkers.
//
//  * (Q,-Q) pairing ("only one of the pair needs to be stored").  With the identity
//    L[-Q][k-Q][g][r][p] = conj(L[Q][k][g][p][r]) the partner block of the output is
//        vhs_w[(k-Q,r),(k,p)] = conj( sum_g L[Q][k][g][p][r] conj(xi_w[-Q][g]) ),
//    i.e. the SAME A operand with 32 more columns.  afqmc_create checks the identity on the caller's L (max
//    deviation <= 1e-13 max|L|); if it holds only one block of every pair is stored (half the bytes of L, which
//    is the largest tensor of the problem and the HBM stream that bounds this kernel at small batches) and every
//    stored block is read once per call for both outputs; if not, all blocks are stored and no pairing is used.
//  * 3M complex product (as in exchange3m.cu, Gauss's form): P0 = (Ar+Ai) Br, P1 = Ar (Bi-Br), P2 = Ai (Br+Bi),
//    Re = P0 - P2, Im = P0 + P1: three real GEMMs with K = gamma and one real column per walker, 25 % fewer
//    DMMAs than the real embedding.  A is stored as plain interleaved complex fragments (no expansion: the sum
//    Ar+Ai is one DADD per fragment, amortised over 12 DMMAs); the tiny B operand (the fields) is expanded by the
//    field kernel into the three real variants in fragment order.
//  * Layout  Lv3[unit][prt][ks][lane][2]: rows pr = 8 prt + (lane>>2) (p = pr/m, r = pr%m), gamma = 4 ks + (lane&3),
//    (re, im): one k-step of one m-tile is one coalesced 512-byte LDG.128; an m-tile's k-steps are contiguous.
//  * CTA = (unit, group of row slices, group of <= 32 walkers), 4 warps; a warp owns MT = 2 m-tiles (16 rows).  With
//    pairing warps 0-1 compute the block itself and warps 2-3 the partner block from the same A fragments (same
//    addresses at about the same time: L1 hits, so HBM sees every byte of L once).  The B fragments of the unit
//    (both column sets) stream through a 3-stage shared-memory ring filled by bulk asynchronous copies
//    (cp.async.bulk + mbarrier, SASS UBLKCP) and are shared by the 4 warps.
//  * Single-precision STORAGE of L (precision = 1, the paper's production mode): the same
//    fragments as float2 (Lv3f): half the bytes of the stream that bounds this kernel at small batches (C4, C5); the fragment
//    is widened in registers (one F2F per component) and everything downstream is the FP64 path (FP64 accumulation).
// Every (k,k') block of vhs is written exactly once, so no zero fill is needed.
#include <cstring>
#include <vector>
#include "common.cuh"

namespace {

constexpr int V3_STAGES = 3;
// k-steps per shared-memory stage = the depth D of the A register ring (template parameter of the kernel), so that
// ring entry q always serves k-step q of a stage (static register indexing, no dispatch on a running ring index:
// C3 0.777 -> 0.636 ms)
constexpr int V3_DMAX = 6;
constexpr int V3_WARPS = 4;

// max |L[-Q][k-Q][g][r][p] - conj(L[Q][k][g][p][r])|, max |L| and max |Im L| (as ordered-int atomics on the bit patterns of
// non-negative doubles, which is exact and order independent)
__global__ void pair_symmetry_kernel(Dims d, const int* __restrict__ kminus, const int* __restrict__ kneg,
                                     const double2* __restrict__ L, unsigned long long* __restrict__ out) {
    const size_t total = (size_t)d.Nk * d.Nk * d.nchol * d.m * d.m;
    double dev = 0.0, mx = 0.0, im = 0.0;
    for (size_t idx = blockIdx.x * (size_t)blockDim.x + threadIdx.x; idx < total; idx += (size_t)gridDim.x * blockDim.x) {
        size_t t = idx;
        const int r = (int)(t % d.m); t /= d.m;
        const int p = (int)(t % d.m); t /= d.m;
        const int g = (int)(t % d.nchol); t /= d.nchol;
        const int k = (int)(t % d.Nk);
        const int Q = (int)(t / d.Nk);
        const double2 a = L[idx];
        const int mQ = kneg[Q], kq = kminus[k * d.Nk + Q];
        const double2 b = L[((((size_t)mQ * d.Nk + kq) * d.nchol + g) * d.m + r) * d.m + p];
        dev = fmax(dev, fmax(fabs(a.x - b.x), fabs(a.y + b.y)));
        mx = fmax(mx, fmax(fabs(a.x), fabs(a.y)));
        im = fmax(im, fabs(a.y));
    }
    atomicMax(out, (unsigned long long)__double_as_longlong(dev));
    atomicMax(out + 1, (unsigned long long)__double_as_longlong(mx));
    atomicMax(out + 2, (unsigned long long)__double_as_longlong(im));
}

__device__ __forceinline__ void store_frag(double2* p, double2 z) { *p = z; }
__device__ __forceinline__ void store_frag(float2* p, double2 z) { *p = make_float2((float)z.x, (float)z.y); }
__device__ __forceinline__ double2 load_frag(const double2* p) { return __ldg(p); }
__device__ __forceinline__ double2 load_frag(const float2* p) { const float2 v = __ldg(p); return make_double2((double)v.x, (double)v.y); }

template <typename AT>
__global__ void pack_Lv3_kernel(Dims d, int KS4, int nvu, const int* __restrict__ vunits, const double2* __restrict__ L,
                                AT* __restrict__ Lv3) {
    const size_t total = (size_t)nvu * d.PRT * KS4 * 32;
    for (size_t idx = blockIdx.x * (size_t)blockDim.x + threadIdx.x; idx < total; idx += (size_t)gridDim.x * blockDim.x) {
        size_t t = idx;
        const int lane = (int)(t & 31); t >>= 5;
        const int ks = (int)(t % KS4); t /= KS4;
        const int prt = (int)(t % d.PRT);
        const int u = (int)(t / d.PRT);
        const int Q = vunits[4 * u], k = vunits[4 * u + 1];
        const int pr = 8 * prt + (lane >> 2), gam = 4 * ks + (lane & 3);
        double2 z = make_double2(0.0, 0.0);
        if (pr < d.m * d.m && gam < d.nchol) z = L[(((size_t)Q * d.Nk + k) * d.nchol + gam) * d.m * d.m + pr];
        store_frag(Lv3 + idx, z);
    }
}

}  // namespace

// a0 for the vHS operand: decides the pairing, builds the unit table and packs Lv3.  Synchronises `st` once
// (the decision needs the result of the symmetry check on the host).
int afqmc_i_vhs_setup(afqmc_ctx* c, const double2* L, const std::vector<int>& kminus, const std::vector<int>& kneg,
                      cudaStream_t st) {
    const Dims& d = c->d;
    const int Nk = d.Nk;
    unsigned long long* dchk = nullptr;
    AFQMC_CUDA_TRY(cudaMalloc((void**)&dchk, 3 * sizeof(unsigned long long)));
    cudaMemsetAsync(dchk, 0, 3 * sizeof(unsigned long long), st);
    pair_symmetry_kernel<<<148 * 16, 256, 0, st>>>(d, c->kminus, c->kneg, L, dchk);
    c->launches++;
    unsigned long long h[3] = {0, 0, 0};
    cudaError_t e = cudaMemcpyAsync(h, dchk, sizeof(h), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    cudaFree(dchk);
    if (e != cudaSuccess) { (void)cudaGetLastError(); return AFQMC_CUDA_ERROR; }
    double dev, mx;
    memcpy(&dev, &h[0], 8);
    memcpy(&mx, &h[1], 8);
    c->vhs_paired = (dev <= 1e-13 * mx) ? 1 : 0;
    double im;
    memcpy(&im, &h[2], 8);
    c->real_l = im == 0.0 ? 1 : 0;                 // real orbitals: two real products per complex product in vhs3_kernel

    // units: (Q, k, kind, 0); kind 0 = single block (no pairing, or a self-partner block), 1 = block + partner
    std::vector<int> vu;
    for (int Q = 0; Q < Nk; ++Q)
        for (int k = 0; k < Nk; ++k) {
            int kind = 0;
            if (c->vhs_paired) {
                const int Qp = kneg[Q], kp = kminus[k * Nk + Q];
                const long long me = (long long)Q * Nk + k, pa = (long long)Qp * Nk + kp;
                if (pa < me) continue;
                kind = pa == me ? 0 : 1;
            }
            vu.push_back(Q); vu.push_back(k); vu.push_back(kind); vu.push_back(0);
        }
    c->nvunits = (int)(vu.size() / 4);
    const int KS4 = (d.nchol + 3) / 4;
    AFQMC_CUDA_TRY(cudaMalloc((void**)&c->vunits, vu.size() * sizeof(int)));
    const size_t total = (size_t)c->nvunits * d.PRT * KS4 * 32;
    if (c->prec32) AFQMC_CUDA_TRY(cudaMalloc((void**)&c->Lv3f, total * sizeof(float2)));      // single-precision storage
    else AFQMC_CUDA_TRY(cudaMalloc((void**)&c->Lv3, total * sizeof(double2)));
    AFQMC_CUDA_TRY(cudaMemcpyAsync(c->vunits, vu.data(), vu.size() * sizeof(int), cudaMemcpyHostToDevice, st));
    size_t g = (total + 255) / 256;
    if (g > 148 * 64) g = 148 * 64;
    if (c->prec32) pack_Lv3_kernel<float2><<<(unsigned)g, 256, 0, st>>>(d, KS4, c->nvunits, c->vunits, L, c->Lv3f);
    else pack_Lv3_kernel<double2><<<(unsigned)g, 256, 0, st>>>(d, KS4, c->nvunits, c->vunits, L, c->Lv3);
    AFQMC_LAUNCH_CHECK(c);
    AFQMC_CUDA_TRY(cudaStreamSynchronize(st));      // `vu` must outlive the copy
    return AFQMC_OK;
}

namespace {

// xi_w[Q][gam] = -i (z - zbar)  (R7; zero outside the valid range)
__device__ __forceinline__ double2 xi_value(const Dims& d, int nw, const int* __restrict__ kneg, const double* __restrict__ x,
                                            const double2* __restrict__ vbias, double sqrt_dtau, int Q, int gam, int w) {
    if (gam >= d.nchol || w >= nw) return make_double2(0.0, 0.0);
    const int mq = kneg[Q];
    const double xq = x[((size_t)w * d.Nk + Q) * d.nchol + gam];
    double zr, zi;
    if (mq == Q) { zr = xq; zi = 0.0; }
    else {
        const double xm = x[((size_t)w * d.Nk + mq) * d.nchol + gam];
        const double r2 = 0.70710678118654752440;
        if (Q < mq) { zr = xq * r2; zi = xm * r2; }       // z_Q    = (x_Q + i x_{-Q})/sqrt2
        else        { zr = xm * r2; zi = -xq * r2; }      // z_{-Q} = conj(z_Q)
    }
    if (vbias) {   // zbar = -i sqrt(dtau) vbias[-Q]  (Eq. 17)
        const double2 vb = vbias[((size_t)w * d.Nk + mq) * d.nchol + gam];
        zr -= sqrt_dtau * vb.y;
        zi += sqrt_dtau * vb.x;
    }
    return make_double2(zi, -zr);                          // xi = -i (z - zbar)
}

// The B operand in fragment order:  Bx3[Q][set][wg][ks][prod][nt][lane], lane: gamma = 4ks + (lane&3), walker =
// (wg*NT + nt)*8 + (lane>>2).  set 0: b = xi_w[Q][gamma];  set 1: b = conj(xi_w[-Q][gamma]) (columns of the partner
// block).  prod 0: Re b, 1: Im b - Re b, 2: Re b + Im b  (the B sides of the 3M products).
__global__ void fields3_kernel(Dims d, int nw, int NT, int nwg, int KS4p, const int* __restrict__ kneg,
                               const double* __restrict__ x, const double2* __restrict__ vbias, double sqrt_dtau,
                               double* __restrict__ Bx3) {
    const size_t total = (size_t)d.Nk * 2 * nwg * KS4p * NT * 32;
    for (size_t idx = blockIdx.x * (size_t)blockDim.x + threadIdx.x; idx < total; idx += (size_t)gridDim.x * blockDim.x) {
        size_t t = idx;
        const int lane = (int)(t & 31); t >>= 5;
        const int nt = (int)(t % NT); t /= NT;
        const int ks = (int)(t % KS4p); t /= KS4p;
        const int wg = (int)(t % nwg); t /= nwg;
        const int set = (int)(t & 1);
        const int Q = (int)(t >> 1);
        const int gam = 4 * ks + (lane & 3), w = (wg * NT + nt) * 8 + (lane >> 2);
        double2 b = xi_value(d, nw, kneg, x, vbias, sqrt_dtau, set == 0 ? Q : kneg[Q], gam, w);
        if (set == 1) b.y = -b.y;
        double* dst = Bx3 + ((((((size_t)Q * 2 + set) * nwg + wg) * KS4p + ks) * 3) * NT + nt) * 32 + lane;
        dst[0] = b.x;
        dst[(size_t)NT * 32] = b.y - b.x;
        dst[(size_t)2 * NT * 32] = b.x + b.y;
    }
}

// ---- mbarrier / bulk-copy primitives (PTX) ----

// ---- the contraction kernel: see the header comment ----
// NT = n-tiles (8 walkers each) of one column set.  MERGED (small batches, NT <= 2): one warp computes BOTH column
// sets of its row slice (2 NT n-tiles), so the A stream is read once without relying on L1 and every fragment feeds
// twice as many DMMAs; otherwise warps 0-1 take the block and warps 2-3 its partner.  D = k-steps of A register prefetch
// (deeper for small batches, where the kernel is bound by the HBM stream of L and needs more bytes in flight).
// REAL: L is real (real orbitals, detected in a0): Re = Ar Br, Im = Ar Br + Ar (Bi - Br): the third product and the addition
// Ar + Ai are skipped (the operand keeps its complex fragment layout).
template <int NT, bool MERGED, int D, typename AT, bool REAL>
__global__ void __launch_bounds__(32 * V3_WARPS, 3) vhs3_kernel(
    Dims d, int KS4, int KS4p, int nw, int nwg, int nsg, const int* __restrict__ vunits, const int* __restrict__ kminus,
    const AT* __restrict__ Lv3, const double* __restrict__ Bx3, double2* __restrict__ vhs) {
    extern __shared__ __align__(128) double v3_smem[];
    constexpr int KC = D;                                     // k-steps per stage
    constexpr int SET_DOUBLES = KC * 3 * NT * 32;             // one column set of one stage
    constexpr int STAGE_DOUBLES = 2 * SET_DOUBLES;
    uint64_t* full = reinterpret_cast<uint64_t*>(v3_smem + (size_t)V3_STAGES * STAGE_DOUBLES);
    uint64_t* empty = full + V3_STAGES;

    const int u = blockIdx.x / nsg, sg = blockIdx.x % nsg, wg = blockIdx.y;
    const int Q = vunits[4 * u], k = vunits[4 * u + 1], kind = vunits[4 * u + 2];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nslices = (d.PRT + 1) / 2;
    constexpr int NTT = MERGED ? 2 * NT : NT;                 // n-tiles of one warp
    const int spc = (kind && !MERGED) ? V3_WARPS / 2 : V3_WARPS;   // row slices per CTA
    const int slice0 = sg * spc;
    if (slice0 >= nslices) return;                            // (single-block units need fewer CTAs than paired ones)
    const int set = (kind && !MERGED) ? warp / spc : 0;       // column set of this warp (MERGED: both)
    const int slice = slice0 + warp % spc;
    int nactive = 0;
    for (int wv = 0; wv < V3_WARPS; ++wv) nactive += (slice0 + wv % spc) < nslices ? 1 : 0;
    if (tid == 0) {
        for (int s = 0; s < V3_STAGES; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], nactive); }
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
    }
    __syncthreads();
    if (slice >= nslices) return;

    const int nsets = kind ? 2 : 1;
    const int nchunks = KS4p / KC;
    const double* bsrc0 = Bx3 + ((((size_t)Q * 2 + 0) * nwg + wg) * KS4p) * 3 * NT * 32;
    const double* bsrc1 = Bx3 + ((((size_t)Q * 2 + 1) * nwg + wg) * KS4p) * 3 * NT * 32;
    auto produce = [&](int ch) {       // thread 0 only
        const int s = ch % V3_STAGES;
        mbar_expect_tx(&full[s], (uint32_t)(nsets * SET_DOUBLES * 8));
        double* dst = v3_smem + (size_t)s * STAGE_DOUBLES;
        bulk_g2s(dst, bsrc0 + (size_t)ch * SET_DOUBLES, SET_DOUBLES * 8, &full[s]);
        if (nsets == 2) bulk_g2s(dst + SET_DOUBLES, bsrc1 + (size_t)ch * SET_DOUBLES, SET_DOUBLES * 8, &full[s]);
    };
    if (tid == 0)
        for (int c0 = 0; c0 < V3_STAGES - 1 && c0 < nchunks; ++c0) produce(c0);

    // A stream: two m-tiles, contiguous k-steps; rows beyond the block are clamped (their results are not stored)
    const int prt0 = 2 * slice, prt1 = min(prt0 + 1, d.PRT - 1);
    const AT* pa0 = Lv3 + (((size_t)u * d.PRT + prt0) * KS4) * 32 + lane;
    const AT* pa1 = Lv3 + (((size_t)u * d.PRT + prt1) * KS4) * 32 + lane;
    AT fa0[D], fa1[D];            // kept in the storage type (half the registers for float2); widened at use
#pragma unroll
    for (int q = 0; q < D; ++q) {
        const int ks = min(q, KS4 - 1);
        fa0[q] = __ldg(pa0 + (size_t)ks * 32);
        fa1[q] = __ldg(pa1 + (size_t)ks * 32);
    }
    double acc[3][2][NTT][2];
#pragma unroll
    for (int p = 0; p < 3; ++p)
#pragma unroll
        for (int i = 0; i < 2; ++i)
#pragma unroll
            for (int j = 0; j < NTT; ++j) acc[p][i][j][0] = acc[p][i][j][1] = 0.0;

    int ksg = 0;        // global k-step
    auto kstep = [&](const double* bs, const int qa) {
        const double x0 = (double)fa0[qa].x, y0 = (double)fa0[qa].y, x1 = (double)fa1[qa].x, y1 = (double)fa1[qa].y;
        const double a0[3] = {REAL ? x0 : x0 + y0, x0, y0};
        const double a1[3] = {REAL ? x1 : x1 + y1, x1, y1};
#pragma unroll
        for (int p = 0; p < (REAL ? 2 : 3); ++p) {
            double bf[NTT];
#pragma unroll
            for (int j = 0; j < NTT; ++j) bf[j] = bs[(j / NT) * SET_DOUBLES + (p * NT + j % NT) * 32];
#pragma unroll
            for (int j = 0; j < NTT; ++j) {
                dmma884(acc[p][0][j][0], acc[p][0][j][1], a0[p], bf[j]);
                dmma884(acc[p][1][j][0], acc[p][1][j][1], a1[p], bf[j]);
            }
        }
        const int nk = min(ksg + D, KS4 - 1);          // clamped: the matching B rows are zero
        fa0[qa] = __ldg(pa0 + (size_t)nk * 32);
        fa1[qa] = __ldg(pa1 + (size_t)nk * 32);
        ++ksg;
    };
    for (int ch = 0; ch < nchunks; ++ch) {
        const int s = ch % V3_STAGES;
        mbar_wait(&full[s], (uint32_t)((ch / V3_STAGES) & 1));
        const double* bs = v3_smem + (size_t)s * STAGE_DOUBLES + set * SET_DOUBLES + lane;
#pragma unroll
        for (int q = 0; q < KC; ++q) {
            kstep(bs + q * 3 * NT * 32, q);
            if (q == 0 && tid == 0) {   // producer duty: refill the stage consumed in the previous iteration
                const int nxt = ch + V3_STAGES - 1;
                if (nxt < nchunks) {
                    if (nxt >= V3_STAGES) mbar_wait(&empty[nxt % V3_STAGES], (uint32_t)(((nxt / V3_STAGES) & 1) ^ 1));
                    produce(nxt);
                }
            }
        }
        fence_proxy_async_smem();       // the stage's reads before its refill by the bulk copy (see common.cuh)
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[s]);
    }

    // ---- epilogue: Re = P0 - P2, Im = P0 + P1 (conjugated and transposed for the partner block) ----
    const int kq = kminus[k * d.Nk + Q];
    const int mm = d.m * d.m;
#pragma unroll
    for (int i = 0; i < 2; ++i) {
        const int prt = prt0 + i;
        const int pr = 8 * prt + (lane >> 2);
        if (prt >= d.PRT || pr >= mm) continue;
        const int p = pr / d.m, r = pr % d.m;
        const size_t off_own = ((size_t)k * d.m + p) * d.M + (size_t)kq * d.m + r;
        const size_t off_par = ((size_t)kq * d.m + r) * d.M + (size_t)k * d.m + p;
#pragma unroll
        for (int j = 0; j < NTT; ++j) {
            const int sj = MERGED ? j / NT : set;                 // column set of this n-tile
            if (sj == 1 && !kind) continue;                       // a self-partner block has no second set
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int w = (wg * NT + j % NT) * 8 + 2 * (lane & 3) + e;
                if (w >= nw) continue;
                const double re = acc[0][i][j][e] - acc[2][i][j][e];
                const double im = acc[0][i][j][e] + acc[1][i][j][e];
                vhs[(size_t)w * d.M * d.M + (sj == 0 ? off_own : off_par)] = make_double2(re, sj == 0 ? im : -im);
            }
        }
    }
}

template <int NT, bool MERGED, int D, typename AT, bool REAL>
int launch_vhs3_t(afqmc_ctx* c, const AT* Lv3, int nw, int KS4, int KS4p, double2* vhs, cudaStream_t st) {
    const Dims& d = c->d;
    const int nwg = (nw + 8 * NT - 1) / (8 * NT);
    const int nslices = (d.PRT + 1) / 2;
    const int nsg = (c->vhs_paired && !MERGED) ? (nslices + V3_WARPS / 2 - 1) / (V3_WARPS / 2) : (nslices + V3_WARPS - 1) / V3_WARPS;
    const size_t smem = (size_t)V3_STAGES * 2 * D * 3 * NT * 32 * sizeof(double) + 2 * V3_STAGES * sizeof(uint64_t);
    const long long gx = (long long)c->nvunits * nsg;
    if (gx > 0x7fffffffLL || nwg > 65535) return AFQMC_UNSUPPORTED;
    if (int rc = afqmc_smem_optin(c, (const void*)vhs3_kernel<NT, MERGED, D, AT, REAL>, smem)) return rc;
    vhs3_kernel<NT, MERGED, D, AT, REAL><<<dim3((unsigned)gx, nwg), 32 * V3_WARPS, smem, st>>>(d, KS4, KS4p, nw, nwg, nsg, c->vunits, c->kminus, Lv3,
                                                                            reinterpret_cast<const double*>(c->ws_xi), vhs);
    AFQMC_LAUNCH_CHECK(c);
    return AFQMC_OK;
}

template <int NT, bool MERGED, int D>
int launch_vhs3(afqmc_ctx* c, int nw, int KS4, int KS4p, double2* vhs, cudaStream_t st) {
    if (c->Lv3f) return launch_vhs3_t<NT, MERGED, D, float2, false>(c, c->Lv3f, nw, KS4, KS4p, vhs, st);      // single-precision storage
    if (c->real_l && c->opt_real) return launch_vhs3_t<NT, MERGED, D, double2, true>(c, c->Lv3, nw, KS4, KS4p, vhs, st);   // real orbitals
    return launch_vhs3_t<NT, MERGED, D, double2, false>(c, c->Lv3, nw, KS4, KS4p, vhs, st);
}

}  // namespace

// doubles of the expanded field operand for up to nw walkers (workspace sizing; the largest over the NT choices)
size_t afqmc_i_vhs_field_doubles(const Dims& d, int nw) {
    const int KS4 = (d.nchol + 3) / 4, KS4p = KS4 + V3_DMAX;          // covers the padding to a multiple of any ring depth
    const int ntiles = (nw + 7) / 8;
    return (size_t)d.Nk * 2 * KS4p * 3 * (size_t)((ntiles + 3) / 4 * 4) * 32;
}

int afqmc_i_vhs(afqmc_ctx* c, const double* x, const double2* vbias, double dtau, int nw, double2* vhs,
                cudaStream_t st) {
    const Dims& d = c->d;
    const int NT = nw > 16 ? 4 : (nw > 8 ? 2 : 1);
    const int D = NT == 4 ? 3 : 6;                                       // ring depth = k-steps per stage of the kernel chosen below
    const int KS4 = (d.nchol + 3) / 4, KS4p = (KS4 + D - 1) / D * D;
    const int nwg = (nw + 8 * NT - 1) / (8 * NT);
    {
        const size_t total = (size_t)d.Nk * 2 * nwg * KS4p * NT * 32;
        int T = 256, G = (int)((total + T - 1) / T);
        if (G > 148 * 16) G = 148 * 16;
        fields3_kernel<<<G, T, 0, st>>>(d, nw, NT, nwg, KS4p, c->kneg, x, vbias, sqrt(dtau), reinterpret_cast<double*>(c->ws_xi));
        AFQMC_LAUNCH_CHECK(c);
    }
    if (NT == 4) return launch_vhs3<4, false, 3>(c, nw, KS4, KS4p, vhs, st);
    if (NT == 2) return c->vhs_paired ? launch_vhs3<2, true, 6>(c, nw, KS4, KS4p, vhs, st) : launch_vhs3<2, false, 6>(c, nw, KS4, KS4p, vhs, st);
    return c->vhs_paired ? launch_vhs3<1, true, 6>(c, nw, KS4, KS4p, vhs, st) : launch_vhs3<1, false, 6>(c, nw, KS4, KS4p, vhs, st);
}

AFQMC_API int afqmc_vhs(afqmc_ctx* c, const double* x, const void* vbias, double dtau, int nw, void* vhs,
                         void* stream) {
    if (!c || !x || !vhs || nw < 0 || nw > c->max_walkers || !(dtau >= 0.0)) return AFQMC_INVALID_ARGUMENT;
    if (nw == 0) return AFQMC_OK;
    if (c->prec32) return afqmc32_vhs(c, x, vbias, dtau, nw, vhs, (cudaStream_t)stream);
    return afqmc_i_vhs(c, x, (const double2*)vbias, dtau, nw, (double2*)vhs, (cudaStream_t)stream);
}
