// The optional complex64 BOUNDARY (afqmc_dims.precision = 1; BASELINE.json: "an optional complex64 run at 1e-4
// tolerance"; the paper's production runs store and contract in single precision).
//
// Every array of the six step calls, of afqmc_step and of afqmc_step_host is then complex64 / float32.  Inside, the
// arrays are widened into the context's FP64 workspace by conversion kernels, the small algebra (overlap, elimination,
// Green's function, force bias, vHS, Taylor propagation, E1, EC) runs in the FP64 kernels of the default path, and the
// exchange contraction runs on the TF32 tensor cores with the high/low operand split (exchange_tf32.cu, mode
// "3xTF32": FP32-equivalent operand accuracy), unless option "exchange_precision" says otherwise.  Results are
// narrowed back to complex64.  Accuracy against the FP64 oracle is that of FP32 inputs and outputs (relative 1e-6 to
// 1e-5 after the overlap inversion); the tests hold it to 1e-4.  The AFQMC-block calls are FP64-only.
#include "common.cuh"

namespace {

__global__ void f2d_kernel(const float* __restrict__ in, double* __restrict__ out, size_t n) {
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) out[i] = (double)in[i];
}
__global__ void d2f_kernel(const double* __restrict__ in, float* __restrict__ out, size_t n) {
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) out[i] = (float)in[i];
}

int widen(afqmc_ctx* c, const void* in, void* out, size_t n, cudaStream_t st) {
    if (n == 0) return AFQMC_OK;
    size_t g = (n + 255) / 256;
    if (g > 148 * 32) g = 148 * 32;
    f2d_kernel<<<(unsigned)g, 256, 0, st>>>((const float*)in, (double*)out, n);
    AFQMC_LAUNCH_CHECK(c);
    return AFQMC_OK;
}
int narrow(afqmc_ctx* c, const void* in, void* out, size_t n, cudaStream_t st) {
    if (n == 0) return AFQMC_OK;
    size_t g = (n + 255) / 256;
    if (g > 148 * 32) g = 148 * 32;
    d2f_kernel<<<(unsigned)g, 256, 0, st>>>((const double*)in, (float*)out, n);
    AFQMC_LAUNCH_CHECK(c);
    return AFQMC_OK;
}

#define TRY32(expr) do { int rc__ = (expr); if (rc__ != AFQMC_OK) return rc__; } while (0)

}  // namespace

// widening of the static inputs of afqmc_create (device float -> freshly allocated device double; caller frees)
int afqmc32_widen_alloc(afqmc_ctx* c, const void* in, size_t ndoubles, double** out, cudaStream_t st) {
    *out = nullptr;
    AFQMC_CUDA_TRY(cudaMalloc((void**)out, ndoubles * sizeof(double)));
    return widen(c, in, *out, ndoubles, st);
}

int afqmc32_green(afqmc_ctx* c, const void* phi, int nw, void* theta, void* logdet, int* info, cudaStream_t st) {
    const Dims& d = c->d;
    TRY32(widen(c, phi, c->ws_phi, (size_t)nw * d.M * d.N * 2, st));
    TRY32(afqmc_i_green(c, c->ws_phi, nw, theta ? c->ws_theta : nullptr, logdet ? c->ws_logdet : nullptr, info, st));
    if (theta) TRY32(narrow(c, c->ws_theta, theta, (size_t)nw * d.N * d.M * 2, st));
    if (logdet) TRY32(narrow(c, c->ws_logdet, logdet, (size_t)nw * 2, st));
    return AFQMC_OK;
}

int afqmc32_force_bias(afqmc_ctx* c, const void* theta, int nw, void* vbias, cudaStream_t st) {
    const Dims& d = c->d;
    TRY32(widen(c, theta, c->ws_theta, (size_t)nw * d.N * d.M * 2, st));
    TRY32(afqmc_i_force_bias(c, c->ws_theta, nw, c->ws_vbias, st));
    return narrow(c, c->ws_vbias, vbias, (size_t)nw * d.Nk * d.nchol * 2, st);
}

int afqmc32_vhs(afqmc_ctx* c, const void* x, const void* vbias, double dtau, int nw, void* vhs, cudaStream_t st) {
    const Dims& d = c->d;
    TRY32(widen(c, x, c->ws_x, (size_t)nw * d.Nk * d.nchol, st));
    if (vbias) TRY32(widen(c, vbias, c->ws_vbias, (size_t)nw * d.Nk * d.nchol * 2, st));
    TRY32(afqmc_i_vhs(c, c->ws_x, vbias ? c->ws_vbias : nullptr, dtau, nw, c->ws_vhs, st));
    return narrow(c, c->ws_vhs, vhs, (size_t)nw * d.M * d.M * 2, st);
}

int afqmc32_propagate(afqmc_ctx* c, const void* vhs, double dtau, int order, void* phi, int nw, cudaStream_t st) {
    const Dims& d = c->d;
    TRY32(widen(c, vhs, c->ws_vhs, (size_t)nw * d.M * d.M * 2, st));
    TRY32(widen(c, phi, c->ws_phi, (size_t)nw * d.M * d.N * 2, st));
    TRY32(afqmc_i_propagate(c, c->ws_vhs, dtau, order, c->ws_phi, nw, st));
    return narrow(c, c->ws_phi, phi, (size_t)nw * d.M * d.N * 2, st);
}

int afqmc32_local_energy(afqmc_ctx* c, const void* theta, int nw, void* energy, cudaStream_t st) {
    const Dims& d = c->d;
    TRY32(widen(c, theta, c->ws_theta, (size_t)nw * d.N * d.M * 2, st));
    TRY32(afqmc_i_local_energy(c, c->ws_theta, nw, c->ws_energy, st));
    return narrow(c, c->ws_energy, energy, (size_t)nw * 3 * 2, st);
}

int afqmc32_step(afqmc_ctx* c, void* phi, const void* x, double dtau, int order, int nw, void* energy, void* logdet,
                 int* info, cudaStream_t st) {
    const Dims& d = c->d;
    TRY32(widen(c, phi, c->ws_phi, (size_t)nw * d.M * d.N * 2, st));
    TRY32(widen(c, x, c->ws_x, (size_t)nw * d.Nk * d.nchol, st));
    TRY32(afqmc_i_step(c, c->ws_phi, c->ws_x, dtau, order, nw, c->ws_energy, logdet ? c->ws_logdet : nullptr, info, st, nullptr));
    TRY32(narrow(c, c->ws_phi, phi, (size_t)nw * d.M * d.N * 2, st));
    TRY32(narrow(c, c->ws_energy, energy, (size_t)nw * 3 * 2, st));
    if (logdet) TRY32(narrow(c, c->ws_logdet, logdet, (size_t)nw * 2, st));
    return AFQMC_OK;
}

int afqmc32_step_host(afqmc_ctx* c, void* phi_host, const void* x_host, double dtau, int order, int nw, void* energy_host,
                      void* logdet_host, int* info_host, cudaStream_t st) {
    const Dims& d = c->d;
    const size_t nphi = (size_t)nw * d.M * d.N * 2, nx = (size_t)nw * d.Nk * d.nchol;
    float* sphi = c->ws_f32;
    float* sx = sphi + (size_t)c->max_walkers * d.M * d.N * 2;
    float* se = sx + (size_t)c->max_walkers * d.Nk * d.nchol;
    float* sl = se + (size_t)c->max_walkers * 6;
    AFQMC_CUDA_TRY(cudaMemcpyAsync(sphi, phi_host, nphi * sizeof(float), cudaMemcpyHostToDevice, st));
    AFQMC_CUDA_TRY(cudaMemcpyAsync(sx, x_host, nx * sizeof(float), cudaMemcpyHostToDevice, st));
    TRY32(afqmc32_step(c, sphi, sx, dtau, order, nw, se, sl, c->ws_info, st));
    AFQMC_CUDA_TRY(cudaMemcpyAsync(phi_host, sphi, nphi * sizeof(float), cudaMemcpyDeviceToHost, st));
    AFQMC_CUDA_TRY(cudaMemcpyAsync(energy_host, se, (size_t)nw * 6 * sizeof(float), cudaMemcpyDeviceToHost, st));
    if (logdet_host) AFQMC_CUDA_TRY(cudaMemcpyAsync(logdet_host, sl, (size_t)nw * 2 * sizeof(float), cudaMemcpyDeviceToHost, st));
    if (info_host) AFQMC_CUDA_TRY(cudaMemcpyAsync(info_host, c->ws_info, (size_t)nw * sizeof(int), cudaMemcpyDeviceToHost, st));
    AFQMC_CUDA_TRY(cudaStreamSynchronize(st));
    return AFQMC_OK;
}
