// The timed composition: the propagation step of
// PAPER.md:87-107/:142-160 on phi, then the energy evaluation of PAPER.md:306-319 on the new phi.
#include "common.cuh"

static int step_body(afqmc_ctx* c, double2* ph, const double* x, double dtau, int order, int nw, double2* energy,
                     double2* logdet, int* info, cudaStream_t st, cudaEvent_t phi_final) {
    int rc;
    afqmc_mark(c, 0, st);
    if ((rc = afqmc_x_green(c, ph, nw, c->ws_theta, nullptr, nullptr, st)) != AFQMC_OK) return rc;
    afqmc_mark(c, 1, st);
    if ((rc = afqmc_x_force_bias(c, c->ws_theta, nw, afqmc_x_vbias_ws(c), st)) != AFQMC_OK) return rc;
    afqmc_mark(c, 2, st);
    if ((rc = afqmc_i_vhs(c, x, afqmc_x_vbias_ws(c), dtau, nw, c->ws_vhs, st)) != AFQMC_OK) return rc;
    afqmc_mark(c, 3, st);
    if ((rc = afqmc_x_propagate(c, c->ws_vhs, dtau, order, ph, nw, st)) != AFQMC_OK) return rc;
    afqmc_mark(c, 4, st);
    if (phi_final) AFQMC_CUDA_TRY(cudaEventRecord(phi_final, st));      // the propagated walkers are final from here on
    if ((rc = afqmc_x_green(c, ph, nw, c->ws_theta, logdet, info, st)) != AFQMC_OK) return rc;
    afqmc_mark(c, 5, st);
    if ((rc = afqmc_i_local_energy(c, c->ws_theta, nw, energy, st)) != AFQMC_OK) return rc;
    afqmc_mark(c, 8, st);      // marks 6 and 7 are recorded around the exchange kernel inside local_energy
    if (c->opt_timers) c->ev_valid = 1;
    return AFQMC_OK;
}

// Inside the composition both Green's functions live in the library's workspace, so Green's epilogue also writes them as the
// force-bias kernel's B fragments (afqmc_set_fuse; zgemm.cuh FragOut) and the force-bias calls skip their re-layout pass.
int afqmc_i_step(afqmc_ctx* c, double2* ph, const double* x, double dtau, int order, int nw, double2* energy,
                 double2* logdet, int* info, cudaStream_t st, cudaEvent_t phi_final) {
    AfqmcFuseGuard fuse(c);
    return step_body(c, ph, x, dtau, order, nw, energy, logdet, info, st, phi_final);
}

AFQMC_API int afqmc_step(afqmc_ctx* c, void* phi, const double* x, double dtau, int order, int nw,
                          void* energy, void* logdet, int* info, void* stream) {
    if (!c || !phi || !x || !energy || nw < 0 || nw > c->max_walkers || order < 0 || order > 32 || !(dtau >= 0.0))
        return AFQMC_INVALID_ARGUMENT;
    if (nw == 0) return AFQMC_OK;
    if (c->prec32) return afqmc32_step(c, phi, x, dtau, order, nw, energy, logdet, info, (cudaStream_t)stream);
    return afqmc_i_step(c, (double2*)phi, x, dtau, order, nw, (double2*)energy, (double2*)logdet, info, (cudaStream_t)stream, nullptr);
}

AFQMC_API int afqmc_step_host_end(afqmc_ctx* c, int slot);

AFQMC_API int afqmc_step_host(afqmc_ctx* c, void* phi_host, const double* x_host, double dtau, int order,
                               int nw, void* energy_host, void* logdet_host, int* info_host, void* stream) {
    if (!c || !phi_host || !x_host || !energy_host || nw < 0 || nw > c->max_walkers || order < 0 || order > 32 || !(dtau >= 0.0))
        return AFQMC_INVALID_ARGUMENT;
    if (nw == 0) return AFQMC_OK;
    // this call stages in the buffers of pipeline slot 0: steps begun with afqmc_step_host_begin are completed first
    for (int slot = 0; slot < 2; ++slot)
        if (c->pipe_busy[slot])
            if (int rc = afqmc_step_host_end(c, slot)) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    if (c->prec32) return afqmc32_step_host(c, phi_host, x_host, dtau, order, nw, energy_host, logdet_host, info_host, st);
    const Dims& d = c->d;
    const size_t phi_bytes = (size_t)nw * afqmc_x_phi_elems(c) * sizeof(double2);
    const size_t x_bytes = (size_t)nw * d.Nk * d.nchol * sizeof(double);
    // a second stream carries the download of the propagated walkers while the energy of those walkers is evaluated
    if (!c->copy_stream) {
        AFQMC_CUDA_TRY(cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking));
        AFQMC_CUDA_TRY(cudaEventCreateWithFlags(&c->ev_copy[0], cudaEventDisableTiming));
        AFQMC_CUDA_TRY(cudaEventCreateWithFlags(&c->ev_copy[1], cudaEventDisableTiming));
    }
    AFQMC_CUDA_TRY(cudaMemcpyAsync(c->ws_phi, phi_host, phi_bytes, cudaMemcpyHostToDevice, st));
    AFQMC_CUDA_TRY(cudaMemcpyAsync(c->ws_x, x_host, x_bytes, cudaMemcpyHostToDevice, st));
    // the same composition as afqmc_step; ev_copy[0] is recorded when the propagated walkers are final, so that their
    // download (second stream) runs while the energy of those walkers is evaluated
    int rc = afqmc_i_step(c, c->ws_phi, c->ws_x, dtau, order, nw, c->ws_energy, c->ws_logdet, c->ws_info, st, c->ev_copy[0]);
    if (rc != AFQMC_OK) {                          // nothing of this call may still be in flight when it returns
        cudaStreamSynchronize(st);
        (void)cudaGetLastError();
        return rc;
    }
    cudaError_t e = cudaStreamWaitEvent(c->copy_stream, c->ev_copy[0], 0);
    if (e == cudaSuccess) e = cudaMemcpyAsync(phi_host, c->ws_phi, phi_bytes, cudaMemcpyDeviceToHost, c->copy_stream);
    if (e == cudaSuccess) e = cudaEventRecord(c->ev_copy[1], c->copy_stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(energy_host, c->ws_energy, (size_t)nw * 3 * sizeof(double2), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess && logdet_host)
        e = cudaMemcpyAsync(logdet_host, c->ws_logdet, (size_t)nw * sizeof(double2), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess && info_host)
        e = cudaMemcpyAsync(info_host, c->ws_info, (size_t)nw * sizeof(int), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(st, c->ev_copy[1], 0);     // the caller's stream owns the whole result
    // both streams are drained on every path: the caller's host buffers are never written after the call returns
    cudaError_t e1 = cudaStreamSynchronize(c->copy_stream), e2 = cudaStreamSynchronize(st);
    if (e != cudaSuccess || e1 != cudaSuccess || e2 != cudaSuccess) { (void)cudaGetLastError(); return AFQMC_CUDA_ERROR; }
    return AFQMC_OK;
}

// ---------------------------------------------------------------------------------------------------------------------
// Two host-buffer steps in flight (afqmc.h "Pipelined host entry").  The kernels of consecutive steps share the context's
// workspace and therefore run one after the other on the caller's stream; what overlaps is the traffic over the host link:
// the upload of step i+1 (copyin_stream) and the download of the walkers of step i (copy_stream) run while step i computes.
// ---------------------------------------------------------------------------------------------------------------------
static int pipe_setup(afqmc_ctx* c, int slot) {
    if (!c->copy_stream) {
        AFQMC_CUDA_TRY(cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking));
        AFQMC_CUDA_TRY(cudaEventCreateWithFlags(&c->ev_copy[0], cudaEventDisableTiming));
        AFQMC_CUDA_TRY(cudaEventCreateWithFlags(&c->ev_copy[1], cudaEventDisableTiming));
    }
    if (!c->copyin_stream) AFQMC_CUDA_TRY(cudaStreamCreateWithFlags(&c->copyin_stream, cudaStreamNonBlocking));
    for (int e = 0; e < 4; ++e)
        if (!c->ev_pipe[slot][e]) AFQMC_CUDA_TRY(cudaEventCreateWithFlags(&c->ev_pipe[slot][e], cudaEventDisableTiming));
    if (slot == 1 && !c->pipe_phi) {       // the second staging set, sized like the first (max_walkers), on first use
        const Dims& d = c->d;
        const size_t nw = (size_t)c->max_walkers;
        cudaError_t e = cudaMalloc((void**)&c->pipe_phi, nw * afqmc_x_phi_elems(c) * sizeof(double2));
        if (e == cudaSuccess) e = cudaMalloc((void**)&c->pipe_x, nw * d.Nk * d.nchol * sizeof(double));
        if (e == cudaSuccess) e = cudaMalloc((void**)&c->pipe_energy, nw * 3 * sizeof(double2));
        if (e == cudaSuccess) e = cudaMalloc((void**)&c->pipe_logdet, nw * sizeof(double2));
        if (e == cudaSuccess) e = cudaMalloc((void**)&c->pipe_info, nw * sizeof(int));
        if (e != cudaSuccess) {
            (void)cudaGetLastError();
            void* ptrs[] = {c->pipe_phi, c->pipe_x, c->pipe_energy, c->pipe_logdet, c->pipe_info};
            for (void* q : ptrs) if (q) cudaFree(q);
            c->pipe_phi = nullptr; c->pipe_x = nullptr; c->pipe_energy = nullptr; c->pipe_logdet = nullptr; c->pipe_info = nullptr;
            return e == cudaErrorMemoryAllocation ? AFQMC_OUT_OF_MEMORY : AFQMC_CUDA_ERROR;
        }
    }
    return AFQMC_OK;
}

AFQMC_API int afqmc_step_host_end(afqmc_ctx* c, int slot) {
    if (!c || slot < 0 || slot > 1) return AFQMC_INVALID_ARGUMENT;
    if (!c->pipe_busy[slot]) return AFQMC_OK;
    c->pipe_busy[slot] = 0;
    if (cudaEventSynchronize(c->ev_pipe[slot][3]) != cudaSuccess) { (void)cudaGetLastError(); return AFQMC_CUDA_ERROR; }
    return AFQMC_OK;
}

AFQMC_API int afqmc_step_host_begin(afqmc_ctx* c, int slot, const void* phi_host, const double* x_host, double dtau, int order,
                                     int nw, void* phi_out_host, void* energy_host, void* logdet_host, int* info_host,
                                     void* stream) {
    if (!c || slot < 0 || slot > 1 || !phi_host || !x_host || !phi_out_host || !energy_host || nw < 0 || nw > c->max_walkers ||
        order < 0 || order > 32 || !(dtau >= 0.0))
        return AFQMC_INVALID_ARGUMENT;
    if (c->prec32) return AFQMC_UNSUPPORTED;
    int rc = afqmc_step_host_end(c, slot);            // a slot is reused only after its previous step has delivered everything
    if (rc != AFQMC_OK || nw == 0) return rc;
    if ((rc = pipe_setup(c, slot)) != AFQMC_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const Dims& d = c->d;
    const size_t phi_bytes = (size_t)nw * afqmc_x_phi_elems(c) * sizeof(double2);
    const size_t x_bytes = (size_t)nw * d.Nk * d.nchol * sizeof(double);
    double2* phi_d = slot ? c->pipe_phi : c->ws_phi;
    double* x_d = slot ? c->pipe_x : c->ws_x;
    double2* en_d = slot ? c->pipe_energy : c->ws_energy;
    double2* ld_d = slot ? c->pipe_logdet : c->ws_logdet;
    int* info_d = slot ? c->pipe_info : c->ws_info;
    cudaEvent_t* ev = c->ev_pipe[slot];
    // upload on its own stream: it overlaps whatever the caller's stream is still computing (the other slot's step)
    AFQMC_CUDA_TRY(cudaMemcpyAsync(phi_d, phi_host, phi_bytes, cudaMemcpyHostToDevice, c->copyin_stream));
    AFQMC_CUDA_TRY(cudaMemcpyAsync(x_d, x_host, x_bytes, cudaMemcpyHostToDevice, c->copyin_stream));
    AFQMC_CUDA_TRY(cudaEventRecord(ev[0], c->copyin_stream));
    AFQMC_CUDA_TRY(cudaStreamWaitEvent(st, ev[0], 0));
    rc = afqmc_i_step(c, phi_d, x_d, dtau, order, nw, en_d, ld_d, info_d, st, ev[1]);
    if (rc != AFQMC_OK) {                          // nothing of this call may still be in flight when it returns
        cudaStreamSynchronize(c->copyin_stream);
        cudaStreamSynchronize(st);
        (void)cudaGetLastError();
        return rc;
    }
    // every download runs on copy_stream, so that the caller's stream goes straight on to the next step's kernels: the
    // walkers as soon as they are final (during the energy evaluation), the small results once the step is complete (ev[2])
    cudaError_t e = cudaEventRecord(ev[2], st);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(c->copy_stream, ev[1], 0);
    if (e == cudaSuccess) e = cudaMemcpyAsync(phi_out_host, phi_d, phi_bytes, cudaMemcpyDeviceToHost, c->copy_stream);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(c->copy_stream, ev[2], 0);
    if (e == cudaSuccess) e = cudaMemcpyAsync(energy_host, en_d, (size_t)nw * 3 * sizeof(double2), cudaMemcpyDeviceToHost, c->copy_stream);
    if (e == cudaSuccess && logdet_host) e = cudaMemcpyAsync(logdet_host, ld_d, (size_t)nw * sizeof(double2), cudaMemcpyDeviceToHost, c->copy_stream);
    if (e == cudaSuccess && info_host) e = cudaMemcpyAsync(info_host, info_d, (size_t)nw * sizeof(int), cudaMemcpyDeviceToHost, c->copy_stream);
    if (e == cudaSuccess) e = cudaEventRecord(ev[3], c->copy_stream);
    if (e != cudaSuccess) {
        cudaStreamSynchronize(c->copyin_stream); cudaStreamSynchronize(c->copy_stream); cudaStreamSynchronize(st);
        (void)cudaGetLastError();
        return AFQMC_CUDA_ERROR;
    }
    c->pipe_busy[slot] = 1;
    return AFQMC_OK;
}
