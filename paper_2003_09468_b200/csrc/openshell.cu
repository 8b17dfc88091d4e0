// Open-shell walkers (afqmc_dims.closed_shell = 0): two spin channels with n (up) and n_dn (down)
// occupied orbitals per k-point.  Eq. 36 / Eq. 49 with their explicit sigma sums:
//   overlap     det O = det O_up * det O_dn                      logdet = logdet_up + logdet_dn
//   Green       Theta_up, Theta_dn separately (Eq. 30 per spin)
//   force bias  vbias = vbias_up + vbias_dn   (spin factor 1 per channel)          Eq. 47
//   vHS         spin independent (one matrix per walker)                            Eq. 48
//   propagate   the same Taylor propagator applied to both channels
//   energy      E1 = sum_s;  EC = 1/2 sum (v_up+v_dn)(v_up+v_dn);  EX = -1/2 sum_s sum T^s T^s   (delta_{ss'} on exchange)
// A channel is a complete context of the closed-shell shape with its own n: `c` is the spin-up context and owns what is
// spin independent, `c->dn` the spin-down one.  Arrays at the boundary are SPIN-MAJOR: phi = [nw][M][N_up] followed by
// [nw][M][N_dn]; theta = [nw][N_up][M] followed by [nw][N_dn][M]; psi_t likewise.  Every kernel is the closed-shell one.
#include "common.cuh"

namespace {

__global__ void os_combine_logdet_kernel(int nw, const double2* __restrict__ up, const double2* __restrict__ dn,
                                         const int* __restrict__ info_up, const int* __restrict__ info_dn,
                                         double2* __restrict__ logdet, int* __restrict__ info) {
    const int w = blockIdx.x * blockDim.x + threadIdx.x;
    if (w >= nw) return;
    if (logdet) {
        const double pi = 3.141592653589793238462643, twopi = 6.283185307179586476925287;
        double ph = fmod(up[w].y + dn[w].y + pi, twopi);
        if (ph < 0.0) ph += twopi;
        logdet[w] = make_double2(up[w].x + dn[w].x, ph - pi);
    }
    if (info) info[w] = info_up[w] != 0 ? info_up[w] : info_dn[w];
}

__global__ void os_add_kernel(size_t n, const double2* __restrict__ a, const double2* __restrict__ b, double2* __restrict__ out) {
    for (size_t e = blockIdx.x * (size_t)blockDim.x + threadIdx.x; e < n; e += (size_t)gridDim.x * blockDim.x)
        out[e] = make_double2(a[e].x + b[e].x, a[e].y + b[e].y);
}

}  // namespace

int afqmc_os_green(afqmc_ctx* c, const double2* phi, int nw, double2* theta, double2* logdet, int* info, cudaStream_t st) {
    afqmc_ctx* dn = c->dn;
    const size_t phi_off = (size_t)nw * c->d.M * c->d.N, th_off = (size_t)nw * c->d.N * c->d.M;
    const bool want = logdet || info;
    int rc = afqmc_i_green(c, phi, nw, theta, want ? c->ws_ld_chan : nullptr, want ? c->ws_info_chan : nullptr, st);
    if (rc != AFQMC_OK) return rc;
    rc = afqmc_i_green(dn, phi + phi_off, nw, theta ? theta + th_off : nullptr, want ? dn->ws_ld_chan : nullptr,
                       want ? dn->ws_info_chan : nullptr, st);
    if (rc != AFQMC_OK || !want) return rc;
    os_combine_logdet_kernel<<<ceil_div(nw, 128), 128, 0, st>>>(nw, c->ws_ld_chan, dn->ws_ld_chan, c->ws_info_chan, dn->ws_info_chan, logdet, info);
    AFQMC_LAUNCH_CHECK(c);
    return AFQMC_OK;
}

int afqmc_os_force_bias(afqmc_ctx* c, const double2* theta, int nw, double2* vbias, cudaStream_t st) {
    afqmc_ctx* dn = c->dn;
    int rc = afqmc_i_force_bias(c, theta, nw, c->ws_vbias, st);
    if (rc != AFQMC_OK) return rc;
    if ((rc = afqmc_i_force_bias(dn, theta + (size_t)nw * c->d.N * c->d.M, nw, dn->ws_vbias, st)) != AFQMC_OK) return rc;
    const size_t n = (size_t)nw * c->d.Nk * c->d.nchol;
    int G = (int)((n + 255) / 256);
    if (G > c->num_sms * 8) G = c->num_sms * 8;
    os_add_kernel<<<G, 256, 0, st>>>(n, c->ws_vbias, dn->ws_vbias, vbias);
    AFQMC_LAUNCH_CHECK(c);
    return AFQMC_OK;
}

int afqmc_os_propagate(afqmc_ctx* c, const double2* vhs, double dtau, int order, double2* phi, int nw, cudaStream_t st) {
    int rc = afqmc_i_propagate(c, vhs, dtau, order, phi, nw, st);
    if (rc != AFQMC_OK) return rc;
    return afqmc_i_propagate(c->dn, vhs, dtau, order, phi + (size_t)nw * c->d.M * c->d.N, nw, st);
}

int afqmc_os_apply_onebody(afqmc_ctx* c, double2* phi, int nw, cudaStream_t st) {
    int rc = afqmc_i_apply_onebody(c, phi, nw, st);
    if (rc != AFQMC_OK) return rc;
    c->dn->b1_set = c->b1_set;
    return afqmc_i_apply_onebody(c->dn, phi + (size_t)nw * c->d.M * c->d.N, nw, st);
}
