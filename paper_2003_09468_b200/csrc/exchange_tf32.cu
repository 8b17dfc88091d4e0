// a9 exchange energy in MIXED PRECISION (option "exchange_precision" = 1): the same contraction
// as energy.cu / exchange3m.cu (Eq. 49) with the half-rotated Cholesky tensor and the Green's function
// rounded to TF32 and multiplied on the TF32 tensor pipe (mma.sync m16n8k8, FP32 accumulation); the per-task complex
// contraction is FP32, the sums over tasks, warps and work units are FP64.  This is the analogue of the paper's
// production mode ("L stored and contracted in single precision ... energies change by typically < 0.1 mHa",
// PAPER.md:260).  The boundary stays complex128; E1 and EC are still evaluated in FP64.  Tolerance: 1e-4 relative
// on EX (BASELINE.json north_star: "1e-4 for an optional complex64 path"); the FP64 kernels remain the default.
//
// Two modes.  exchange_precision = 1 ("3xTF32"): both operands are split into TF32 high and low parts (x = hi + lo, lo =
// tf32(x - hi)) and every product is three MMAs, Ah Bh + Ah Bl + Al Bh: FP32-equivalent operand accuracy (measured EX error
// ~1e-6 relative).  exchange_precision = 2 ("1xTF32"): operands rounded once to TF32 (10-bit mantissa), one MMA per
// product: the fastest mode, but EX errors of 2e-5 (median) to 2e-3 (worst walker) were measured on the synthetic
// configs, so it does NOT meet the 1e-4 tolerance in general and is offered as a speed/accuracy trade only.
//
// Real embedding (4M): rows = (gamma of a quad, a) = 16 per m-tile, K = (r, re/im) in k-steps of 8 reals, columns =
// (b, re/im) of one walker = one n-tile.  Measured on the B200: mma.sync TF32 278 TFLOP/s against 37 TFLOP/s FP64 DMMA,
// so flops are cheap here and the kernel is bound by fragment traffic; the operand is stored as FP32 fragments
//   LxT[Q][k][gq][ks][lane] = float4 (a0,a1,a2,a3) of the m16n8k8 A fragment (rows g, g+8; columns t, t+4; g = lane>>2,
//   t = lane&3), one coalesced 512-byte LDG.128 per k-step, consecutive k-steps and tasks contiguous.
// The partner tile T2[(gamma,b),(a)] is transposed across lanes by one shuffle per value (same lane map as energy.cu,
// applied to both row halves of the 16 x 8 C fragment).
#include "common.cuh"

namespace {

__device__ __forceinline__ float tf32_of(float f) {
    unsigned u;
    asm("cvt.rna.tf32.f32 %0, %1;\n" : "=r"(u) : "f"(f));
    return __uint_as_float(u);
}

// LxT = [hi plane][pad][lo plane][pad]; plane stride = total_padded floats
__global__ void pack_LxT_kernel(Dims d, int KS8, const double2* __restrict__ Lh, float* __restrict__ LxT, size_t total,
                                size_t total_padded) {
    for (size_t idx = blockIdx.x * (size_t)blockDim.x + threadIdx.x; idx < total; idx += (size_t)gridDim.x * blockDim.x) {
        size_t t_ = idx;
        const int e = (int)(t_ & 3); t_ >>= 2;                // register of the A fragment
        const int lane = (int)(t_ & 31); t_ >>= 5;
        const int ks = (int)(t_ % KS8); t_ /= KS8;
        const int gq = (int)(t_ % d.GQ); t_ /= d.GQ;
        const int k = (int)(t_ % d.Nk);
        const int Q = (int)(t_ / d.Nk);
        const int g = lane >> 2, t = lane & 3;
        const int row = g + 8 * (e & 1), j = 8 * ks + t + 4 * (e >> 1);
        const int gam = 4 * gq + (row >> 2), a = row & 3, r = j >> 1, part = j & 1;
        float v = 0.f, vlo = 0.f;
        if (a < d.n && gam < d.nchol && r < d.m) {
            const double2 z = Lh[((((size_t)Q * d.Nk + k) * d.n + a) * d.nchol + gam) * d.m + r];     // FP64, then rounded
            const float f = (float)(part ? z.y : z.x);
            v = tf32_of(f);
            vlo = tf32_of(f - v);
        }
        LxT[idx] = v;
        LxT[total_padded + idx] = vlo;
    }
    for (size_t idx = total + blockIdx.x * (size_t)blockDim.x + threadIdx.x; idx < total_padded; idx += (size_t)gridDim.x * blockDim.x) {
        LxT[idx] = 0.f;
        LxT[total_padded + idx] = 0.f;
    }
}

__device__ __forceinline__ void mma_tf32(float (&c)[4], const float4& a, const float2& b) {
    asm volatile("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};\n"
                 : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
                 : "r"(__float_as_uint(a.x)), "r"(__float_as_uint(a.y)), "r"(__float_as_uint(a.z)), "r"(__float_as_uint(a.w)),
                   "r"(__float_as_uint(b.x)), "r"(__float_as_uint(b.y)));
}

constexpr int XT_NT = 4;        // walkers per CTA
constexpr int XT_WARPS = 4;
constexpr int XT_PAD = 4096;    // floats of zero padding after LxT (the prefetch runs 2 k-steps past the last task)

template <bool SPLIT>
__global__ void __launch_bounds__(32 * XT_WARPS, 4) exchange_tf32_kernel(
    Dims d, int KS8, size_t lo_offset /* float4 units from the hi plane to the lo plane */, int nw, const int* __restrict__ units, const int* __restrict__ kminus, const int* __restrict__ kplus,
    const int* __restrict__ kneg, const float4* __restrict__ LxT, const double2* __restrict__ theta,
    double2* __restrict__ partial) {
    extern __shared__ __align__(16) float xt_smem[];
    const int nwg = (nw + XT_NT - 1) / XT_NT;
    const int u = blockIdx.x / nwg, w0 = (blockIdx.x % nwg) * XT_NT;
    const int Q = units[4 * u], k = units[4 * u + 1], k2 = units[4 * u + 2];
    const int mQ = kneg[Q];
    const int kq = kminus[k * d.Nk + Q];
    const int k2pq = kplus[k2 * d.Nk + Q];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int GQ = d.GQ;
    // Bs[part: hi, lo][which][ks][walker][lane] float2 (b0, b1)
    const int bs_half = KS8 * XT_NT * 64;
    const int bs_lo = 2 * bs_half;

    const int t_begin = (int)((long long)warp * GQ / XT_WARPS), t_end = (int)((long long)(warp + 1) * GQ / XT_WARPS);
    const int total = (t_end - t_begin) * KS8;
    const float4* la1 = LxT + (((size_t)Q * d.Nk + k) * GQ + t_begin) * KS8 * 32 + lane;
    const float4* la2 = LxT + (((size_t)mQ * d.Nk + k2) * GQ + t_begin) * KS8 * 32 + lane;
    float4 fa1[2], fa2[2], fl1[2], fl2[2];
#pragma unroll
    for (int q = 0; q < 2; ++q) {
        fa1[q] = fa2[q] = fl1[q] = fl2[q] = make_float4(0.f, 0.f, 0.f, 0.f);
        if (total > 0) {
            fa1[q] = __ldg(la1 + q * 32); fa2[q] = __ldg(la2 + q * 32);
            if (SPLIT) { fl1[q] = __ldg(la1 + lo_offset + q * 32); fl2[q] = __ldg(la2 + lo_offset + q * 32); }
        }
    }
    la1 += 64; la2 += 64;

    // ---- stage the B fragments (real embedding of theta, TF32): one thread per complex element (b, walker, r) ----
    //   K row j = 2r + c (c = 0 multiplies Re A, c = 1 multiplies Im A); column 2b + dd:  dd = 0: (Re, -Im), dd = 1: (Im, Re)
    //   fragment: ks = j >> 3, jj = j & 7: register jj >> 2 of lane (col << 2) | (jj & 3)
    {
        const int per_which = 4 * XT_NT * 4 * KS8;                 // (b, walker, r < 4 KS8)
        for (int e = tid; e < 2 * per_which; e += 32 * XT_WARPS) {
            const int which = e / per_which;
            int x = e - which * per_which;
            const int b = x & 3; x >>= 2;
            const int wl = x % XT_NT, r = x / XT_NT;
            const int w = w0 + wl;
            const int rowblk = which == 0 ? k2 : k, colblk = which == 0 ? kq : k2pq;
            double2 v = make_double2(0.0, 0.0);
            if (b < d.n && w < nw && r < d.m)
                v = __ldg(theta + ((size_t)w * d.N + rowblk * d.n + b) * d.M + (size_t)colblk * d.m + r);
            const float fr = (float)v.x, fi = (float)v.y;
            const float re = tf32_of(fr), im = tf32_of(fi);
            const float rel = tf32_of(fr - re), iml = tf32_of(fi - im);
            float* base = xt_smem + which * bs_half + (((2 * r) >> 3) * XT_NT + wl) * 64;
#pragma unroll
            for (int c = 0; c < 2; ++c) {
                const int jj = (2 * r + c) & 7;
#pragma unroll
                for (int dd = 0; dd < 2; ++dd) {
                    const int ln = ((2 * b + dd) << 2) | (jj & 3);
                    base[ln * 2 + (jj >> 2)] = dd == 0 ? (c == 0 ? re : -im) : (c == 0 ? im : re);
                    if (SPLIT) base[bs_lo + ln * 2 + (jj >> 2)] = dd == 0 ? (c == 0 ? rel : -iml) : (c == 0 ? iml : rel);
                }
            }
        }
    }
    __syncthreads();

    double er[XT_NT], ei[XT_NT];
    float acc1[XT_NT][4], acc2[XT_NT][4];
#pragma unroll
    for (int j = 0; j < XT_NT; ++j) {
        er[j] = ei[j] = 0.0;
#pragma unroll
        for (int e = 0; e < 4; ++e) acc1[j][e] = acc2[j][e] = 0.f;
    }
    // lane' holding the (a,b)-transposed element (same map for both row halves of the C fragment)
    const int srcl = (lane & 16) | ((lane & 3) << 2) | ((lane >> 2) & 3);
    const float2* bs1 = reinterpret_cast<const float2*>(xt_smem) + lane;
    const float2* bs2 = reinterpret_cast<const float2*>(xt_smem + bs_half) + lane;
    int ks = 0;
    auto kstep = [&](const int q) {
#pragma unroll
        for (int j = 0; j < XT_NT; ++j) {
            const float2 b1 = bs1[(ks * XT_NT + j) * 32], b2 = bs2[(ks * XT_NT + j) * 32];
            if (SPLIT) {      // small terms first: Al Bh + Ah Bl, then Ah Bh
                const float2 b1l = bs1[bs_lo / 2 + (ks * XT_NT + j) * 32], b2l = bs2[bs_lo / 2 + (ks * XT_NT + j) * 32];
                mma_tf32(acc1[j], fl1[q], b1);
                mma_tf32(acc2[j], fl2[q], b2);
                mma_tf32(acc1[j], fa1[q], b1l);
                mma_tf32(acc2[j], fa2[q], b2l);
            }
            mma_tf32(acc1[j], fa1[q], b1);
            mma_tf32(acc2[j], fa2[q], b2);
        }
        fa1[q] = __ldg(la1); fa2[q] = __ldg(la2);        // 2 k-steps ahead (may run into the next block or the pad)
        if (SPLIT) { fl1[q] = __ldg(la1 + lo_offset); fl2[q] = __ldg(la2 + lo_offset); }
        la1 += 32; la2 += 32;
        if (++ks == KS8) {
            ks = 0;
#pragma unroll
            for (int j = 0; j < XT_NT; ++j)
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const float t1r = acc1[j][2 * h], t1i = acc1[j][2 * h + 1];
                    const float t2r = __shfl_sync(0xffffffffu, acc2[j][2 * h], srcl);
                    const float t2i = __shfl_sync(0xffffffffu, acc2[j][2 * h + 1], srcl);
                    er[j] += (double)(t1r * t2r - t1i * t2i);
                    ei[j] += (double)(t1r * t2i + t1i * t2r);
                    acc1[j][2 * h] = acc1[j][2 * h + 1] = acc2[j][2 * h] = acc2[j][2 * h + 1] = 0.f;
                }
        }
    };
    const int nfull = total - (total & 1);
    for (int g0 = 0; g0 < nfull; g0 += 2) { kstep(0); kstep(1); }
    if (total & 1) kstep(0);

    __syncthreads();
    double* red = reinterpret_cast<double*>(xt_smem);   // reuse: [warp][XT_NT][2]
#pragma unroll
    for (int j = 0; j < XT_NT; ++j) {
        const double r = warp_sum(er[j]), i = warp_sum(ei[j]);
        if (lane == 0) { red[(warp * XT_NT + j) * 2] = r; red[(warp * XT_NT + j) * 2 + 1] = i; }
    }
    __syncthreads();
    if (tid < XT_NT && w0 + tid < nw) {
        double r = 0.0, i = 0.0;
        for (int x = 0; x < XT_WARPS; ++x) { r += red[(x * XT_NT + tid) * 2]; i += red[(x * XT_NT + tid) * 2 + 1]; }
        partial[(size_t)u * nw + w0 + tid] = make_double2(r, i);
    }
}

}  // namespace

size_t afqmc_i_lxt_floats(const Dims& d) {
    const int KS8 = (2 * d.m + 7) / 8;
    return 2 * ((size_t)d.Nk * d.Nk * d.GQ * KS8 * 128 + XT_PAD);      // hi and lo planes
}

int afqmc_i_pack_lxt(afqmc_ctx* c, cudaStream_t st) {
    const Dims& d = c->d;
    const int KS8 = (2 * d.m + 7) / 8;
    const size_t total = (size_t)d.Nk * d.Nk * d.GQ * KS8 * 128;
    size_t g = (total + 255) / 256;
    if (g > 148 * 64) g = 148 * 64;
    pack_LxT_kernel<<<(unsigned)g, 256, 0, st>>>(d, KS8, c->Lh, c->LxT, total, total + XT_PAD);
    AFQMC_LAUNCH_CHECK(c);
    return AFQMC_OK;
}

// Writes the unit partial sums into ws_expart like the FP64 kernels.  AFQMC_UNSUPPORTED for n > 4 (caller falls back).
int afqmc_i_exchange_tf32(afqmc_ctx* c, const double2* theta, int nw, cudaStream_t st) {
    const Dims& d = c->d;
    if (d.NAG != 1 || !c->LxT) return AFQMC_UNSUPPORTED;
    const int KS8 = (2 * d.m + 7) / 8;
    const bool split = c->opt_exchange_prec == 1;
    const size_t plane = (size_t)d.Nk * d.Nk * d.GQ * KS8 * 128 + XT_PAD;
    size_t smem = (size_t)(split ? 4 : 2) * KS8 * XT_NT * 64 * sizeof(float);
    if (smem < (size_t)XT_WARPS * XT_NT * 2 * sizeof(double)) smem = (size_t)XT_WARPS * XT_NT * 2 * sizeof(double);
    if (int rc = afqmc_smem_optin(c, (const void*)exchange_tf32_kernel<true>, smem)) return rc;
    if (int rc = afqmc_smem_optin(c, (const void*)exchange_tf32_kernel<false>, smem)) return rc;
    const long long nblocks = (long long)((nw + XT_NT - 1) / XT_NT) * c->nunits;
    if (nblocks > 0x7fffffffLL) return AFQMC_UNSUPPORTED;
    if (split)
        exchange_tf32_kernel<true><<<(unsigned)nblocks, 32 * XT_WARPS, smem, st>>>(d, KS8, plane / 4, nw, c->units, c->kminus, c->kplus, c->kneg,
                                                                                   reinterpret_cast<const float4*>(c->LxT), theta, c->ws_expart);
    else
        exchange_tf32_kernel<false><<<(unsigned)nblocks, 32 * XT_WARPS, smem, st>>>(d, KS8, plane / 4, nw, c->units, c->kminus, c->kplus, c->kneg,
                                                                                    reinterpret_cast<const float4*>(c->LxT), theta, c->ws_expart);
    AFQMC_LAUNCH_CHECK(c);
    return AFQMC_OK;
}
