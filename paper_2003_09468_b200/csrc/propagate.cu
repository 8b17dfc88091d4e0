// a6 propagation:  phi_w <- sum_{j=0..order} (s V_w)^j / j!  phi_w,  s = -sqrt(dtau)
// (truncated Taylor series of PAPER.md:160), by the recurrence T_0 = phi, T_j = (s/j) V T_{j-1},
// phi += T_j.  Each order is one batched DMMA GEMM (tgemm.cuh) over all walkers: V_w streams from its
// natural layout, T_{j-1} is read in the expanded fragment layout that the previous order's epilogue
// wrote (bulk-copied to shared memory), and the epilogue fuses the scale, the running sum into phi and
// the expanded store of T_j.  T ping-pongs between two workspace buffers.
#include "tgemm.cuh"
#include "zgemm.cuh"

size_t afqmc_i_taylor_ws_doubles(const Dims& d) { return tg::expanded_doubles_max(d.M, d.N); }

int afqmc_i_propagate(afqmc_ctx* c, const double2* vhs, double dtau, int order, double2* phi, int nw,
                      cudaStream_t st) {
    const Dims& d = c->d;
    if (order == 0) return AFQMC_OK;
    const size_t per = (size_t)d.M * d.N;
    const double s = -sqrt(dtau);
    if (c->opt_taylor_legacy) {
        double2* T[2] = {c->ws_T, c->ws_T + (size_t)c->max_walkers * per};
        if (cudaMemcpyAsync(T[0], phi, (size_t)nw * per * sizeof(double2), cudaMemcpyDeviceToDevice, st) != cudaSuccess)
            return AFQMC_CUDA_ERROR;
        for (int j = 1; j <= order; ++j) {
            zg::Args a = {};
            a.A = vhs; a.strideA = (long long)d.M * d.M; a.lda = d.M;
            a.B = T[(j - 1) & 1]; a.strideB = (long long)per; a.ldb = d.N;
            a.C = T[j & 1]; a.strideC = (long long)per; a.ldc = d.N;
            a.D = phi; a.strideD = (long long)per; a.ldd = d.N;
            a.M = d.M; a.N = d.N; a.K = d.M; a.alpha = s / (double)j;
            if (zg::launch<false>(c, a, nw, st) != cudaSuccess) return AFQMC_CUDA_ERROR;
            c->launches++;
        }
        return AFQMC_OK;
    }
    // Walkers per pass: all of them by default.  Option "taylor_subbatch" = b runs the whole series for b walkers at a time, so
    // that their V (b * 16 M^2 bytes) can stay in L2 across the orders instead of being streamed from HBM once per order.
    const int sb = (c->opt_taylor_subbatch > 0 && c->opt_taylor_subbatch < nw) ? c->opt_taylor_subbatch : nw;
    for (int b0 = 0; b0 < nw; b0 += sb) {
        const int nb = nw - b0 < sb ? nw - b0 : sb;
        const int G = c->opt_taylor_groups > 0 ? c->opt_taylor_groups : tg::pick_groups(c, d.M, d.N, nb);
        const size_t perx = tg::expanded_doubles(d.M, d.N, G);
        if (perx > afqmc_i_taylor_ws_doubles(d)) return AFQMC_INVALID_ARGUMENT;   // a forced group count the workspace was not sized for
        double* Tx[2] = {c->ws_Tx, c->ws_Tx + (size_t)c->max_walkers * afqmc_i_taylor_ws_doubles(d)};
        double2* ph = phi + (size_t)b0 * per;
        if (tg::launch_expand<false>(ph, (long long)per, d.N, Tx[0], d.M, d.N, nb, st, G) != cudaSuccess) return AFQMC_CUDA_ERROR;
        c->launches++;
        for (int j = 1; j <= order; ++j) {
            tg::Args a = {};
            a.A = vhs + (size_t)b0 * d.M * d.M; a.strideA = (long long)d.M * d.M; a.lda = d.M;
            a.Bx = Tx[(j - 1) & 1]; a.strideBx = (long long)perx;
            a.Cx = j < order ? Tx[j & 1] : nullptr; a.strideCx = (long long)perx;
            a.D = ph; a.strideD = (long long)per; a.ldd = d.N;
            a.Ct = nullptr; a.strideCt = 0; a.ldct = 0;
            a.M = d.M; a.N = d.N; a.K = d.M; a.alpha = s / (double)j;
            a.wpc = c->opt_taylor_wpc;
            if (tg::launch(c, a, nb, st, G) != cudaSuccess) return AFQMC_CUDA_ERROR;
            c->launches++;
        }
    }
    return AFQMC_OK;
}

AFQMC_API int afqmc_propagate(afqmc_ctx* c, const void* vhs, double dtau, int order, void* phi, int nw,
                               void* stream) {
    if (!c || !vhs || !phi || nw < 0 || nw > c->max_walkers || order < 0 || order > 32 || !(dtau >= 0.0))
        return AFQMC_INVALID_ARGUMENT;
    if (nw == 0) return AFQMC_OK;
    if (c->prec32) return afqmc32_propagate(c, vhs, dtau, order, phi, nw, (cudaStream_t)stream);
    return afqmc_x_propagate(c, (const double2*)vhs, dtau, order, (double2*)phi, nw, (cudaStream_t)stream);
}
