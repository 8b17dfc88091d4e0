/*
 * afqmc.h -- C ABI of libafqmc: the batched per-walker step of k-point phaseless AFQMC
 * (Malone, Zhang, Morales, arxiv 2003.09468; citations are /root/reference/PAPER.md:<line>).
 *
 * All step calls work on a batch of `nw` walkers at once ("all walkers should be operated on
 * simultaneously") and are ASYNCHRONOUS on the cudaStream_t passed as `stream`.
 *
 * Conventions
 *   Nk = g[0]*g[1]*g[2] k-points = number of Q vectors; k-point linear index
 *   (i1*g[1] + i2)*g[2] + i3 on a Gamma-centred regular mesh; k-Q and -Q are
 *   taken componentwise modulo the mesh.  M = Nk*m basis functions, N = Nk*n electrons per
 *   spin.  Closed shell: one walker matrix serves both spins.
 *
 *   Every array is row-major (last index fastest), complex numbers interleaved (re, im),
 *   double precision (complex128).  "device" = device memory owned by the caller (e.g. a
 *   torch tensor); the library borrows the pointer for the duration of the enqueued work and
 *   never frees it.  Workspace is owned by the context and sized from max_walkers at create.
 *
 *   phi   [nw][M][N]      walker U, DENSE; row (k,p) = k*m+p, column (k,a) = k*n+a
 *   theta [nw][N][M]      half-rotated Green's function, Eq. 30 = the paper's
 *                         G[n,k1,a,k2,q] of PAPER.md:306-312
 *   vbias [nw][Nk][nchol] complex; x [nw][Nk][nchol] real; vhs [nw][M][M];
 *   energy[nw][3]         complex (E1, EC, EX);  logdet[nw] complex = log|det O| + i arg det O of
 *                         ONE spin channel, arg in (-pi, pi];  info[nw] int32.
 *
 * Precision 1 (optional complex64 path; the paper's production runs are single precision): with
 * afqmc_dims.precision = 1 EVERY complex array of afqmc_create, of the six step calls, of afqmc_step and of
 * afqmc_step_host is complex64 (float re, im) and every real array (x) is float32; shapes and layouts are unchanged.
 * Inside, the library STORES the two streamed operands that bound the step at small batches in single precision -- the
 * vHS operand (the largest tensor: L, one block per (Q,-Q) pair) and the force-bias operand (the half-rotated Lh) -- i.e. half
 * their bytes in HBM and on the bus; fragments are widened in registers and every sum is accumulated in FP64.  The small
 * algebra runs in FP64 on widened copies and the exchange contraction on the TF32 tensor cores (tcgen05.mma, accumulators in
 * tensor memory) with a high/low operand split (option "exchange_precision" = 1).  Results agree with the FP64 path to FP32 input/output accuracy (tolerance 1e-4).  The
 * AFQMC-block calls and open-shell contexts return AFQMC_UNSUPPORTED in this mode.
 *
 * Errors: every call returns an int; 0 = AFQMC_OK.  No exceptions cross the ABI, there is no
 * global state.  A singular overlap cannot be a return code of an asynchronous call: it is
 * reported LAPACK-style in the device array info[w] (0 ok, j>0 = exactly-zero pivot at
 * elimination step j); theta/logdet of such a walker are undefined.
 * One context must not be used from two streams at the same time (it owns workspace).
 */
#ifndef AFQMC_H
#define AFQMC_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct afqmc_ctx afqmc_ctx; /* opaque, library-owned */

typedef struct {
    int g[3];         /* k-point mesh                                              */
    int m;            /* bands per k-point                                          */
    int n;            /* occupied orbitals per k-point per spin                      */
    int nchol;        /* Cholesky vectors per Q             */
    int closed_shell; /* 1 = closed shell (one walker matrix for both spins); 0 = open shell (see "Open shell") */
    int precision;    /* 0 = complex128; 1 = complex64 boundary (see "Precision 1" below)  */
    int max_walkers;  /* workspace is sized for this many walkers                    */
    int n_dn;         /* open shell only: spin-down occupied orbitals per k-point (n is then the spin-up count) */
} afqmc_dims;

enum {
    AFQMC_OK = 0,
    AFQMC_INVALID_ARGUMENT = 1, /* null pointer, nw < 0 or > max_walkers, bad dims, bad order */
    AFQMC_UNSUPPORTED = 2,      /* precision > 1, open shell or block calls with precision 1 ...   */
    AFQMC_CUDA_ERROR = 3,       /* a CUDA runtime call or launch failed                       */
    AFQMC_OUT_OF_MEMORY = 4,    /* device allocation failed                                   */
    AFQMC_SCRATCH_LIMIT = 5     /* afqmc_overlap_noalloc: the call needs more than the static scratch array holds */
}/*
 * Open shell (closed_shell = 0; Eq. 36 / Eq. 49 with their explicit spin sums).  Two spin channels
 * with n (spin up) and n_dn (spin down) occupied orbitals per k-point, N_up = Nk*n, N_dn = Nk*n_dn.  Every per-walker array
 * that has an orbital index is SPIN-MAJOR: the spin-up block of all nw walkers followed by the spin-down block,
 *     psi_t = [Nk][m][n]      then [Nk][m][n_dn]           phi   = [nw][M][N_up] then [nw][M][N_dn]
 *     theta = [nw][N_up][M]   then [nw][N_dn][M]           (the offset of the second block depends on the call's nw)
 * and the spin-independent ones are unchanged: vbias[nw][Nk][nchol] = vbias_up + vbias_dn (no factor 2), x, vhs[nw][M][M],
 * energy[nw][3] = (E1 summed over spins, EC = 1/2 sum_Q v_Q v_-Q of the spin-summed v, EX = -1/2 sum_spin sum T T: exchange
 * only between like spins), logdet[nw] = log det O_up + log det O_dn (phase wrapped to (-pi, pi]), info[nw] = first non-zero
 * of the two channels.  All calls below take these layouts when the context is open shell; the hybrid weight then uses the
 * overlap ratio det'_up det'_dn / (det_up det_dn) (closed shell: the squared ratio of the shared determinant).  Two equal
 * channels reproduce the closed-shell results (tested).  The complex64 boundary (precision = 1) is closed-shell only.
 */

;

/* Text for an error code (static storage, never NULL). */
const char* afqmc_strerror(int code);

/*
 * a0 (setup, once per simulation).  Validates dims, copies the trial,
 * half-rotates  Lh[Q][k][a][g][r] = sum_p conj(psi_t[k][p][a]) L[Q][k][g][p][r]  and
 * ht[k][a][q] = sum_p conj(psi_t[k][p][a]) h1[k][p][q], repacks L and Lh into the library's
 * internal tensor-core fragment layouts and allocates workspace.  Synchronises `stream` before
 * returning, so the caller may free h1, L and psi_t afterwards.
 *   h1    [Nk][m][m]            device, complex128, Hermitian blocks (Eq. 45)
 *   L     [Nk][Nk][nchol][m][m] device, complex128: L[Q][k][g][p][r], p at k, r at k-Q.
 *         The (Q,-Q) identity L[-Q][k-Q][g][r][p] = conj(L[Q][k][g][p][r]) is ASSUMED
 *         by afqmc_local_energy (it is what lets Lbar of Eq. 40 be read from Lh).  afqmc_create measures
 *         the deviation from it: if it is below 1e-13 max|L| the library keeps ONE block of every pair for
 *         afqmc_vhs ("only one of the pair needs to be stored": half the bytes of L);
 *         otherwise afqmc_vhs keeps all blocks and stays exact for such an L.
 *   psi_t [Nk][m][n]            device, complex128 (trial block-diagonal in k)
 */
int afqmc_create(afqmc_ctx** out, const afqmc_dims* dims, const void* h1, const void* L,
                 const void* psi_t, void* stream);

/* Frees everything the context owns.  NULL is allowed. */
void afqmc_destroy(afqmc_ctx* ctx);

/*
 * a1+a2.  O_w = A^dagger Phi_w (N x N, assembled as Nk row blocks because the trial is block
 * diagonal, PAPER.md:142 Eq. 27-28, :226) and its elimination with partial pivoting:
 * logdet[w] = log det O_w, info[w].   phi, logdet, info: device.
 */
int afqmc_overlap(afqmc_ctx* ctx, const void* phi, int nw, void* logdet, int* info, void* stream);

/*
 * a1+a2+a3.  Additionally theta_w = (Phi_w^T A^*)^{-1} Phi_w^T = (Phi_w O_w^{-1})^T, Eq. 30
 * (PAPER.md:146).  logdet and info may be NULL.   phi, theta, logdet, info: device.
 */
int afqmc_green(afqmc_ctx* ctx, const void* phi, int nw, void* theta, void* logdet, int* info,
                void* stream);

/*
 * a4.  vbias[w][Q][g] = 2 sum_k sum_{a,r} Lh[Q][k][a][g][r] theta_w[(k,a),(k-Q,r)]
 * = <Psi_T| rho_{Q g} |phi_w> / <Psi_T|phi_w> summed over both spins: the half-rotated contraction
 * of Eq. 47 = 2 X_g of Eq. 37, WITHOUT the -sqrt(dtau) c_pm prefactor
 * of Eq. 25 (that belongs to the field assembly in afqmc_vhs).   theta, vbias: device.
 */
int afqmc_force_bias(afqmc_ctx* ctx, const void* theta, int nw, void* vbias, void* stream);

/*
 * a5.  Field assembly then the contraction of Eq. 48 (PAPER.md:224; Eq. 33, :158):
 *   z_Q = x_Q if -Q == Q, else z_Q = (x_Q + i x_{-Q})/sqrt2 for idx(Q) < idx(-Q), z_{-Q} = conj(z_Q);
 *   zbar_{Q g} = -i sqrt(dtau) vbias[w][-Q][g]   (Eq. 17; zero if vbias == NULL);
 *   xi = -i (z - zbar);   vhs_w[(k,p),(k-Q,r)] = sum_g L[Q][k][g][p][r] xi_{Q g}.
 * Every (k,k') block of vhs_w is written exactly once (Q = k - k').  The propagator applied by
 * afqmc_propagate is then exp(-sqrt(dtau) vhs) = exp(i sqrt(dtau) sum z rho - dtau sum vbias_{-Q} rho_Q)
 * (reading R7).    x: device double [nw][Nk][nchol]; vbias: device or NULL; vhs: device.
 */
int afqmc_vhs(afqmc_ctx* ctx, const double* x, const void* vbias, double dtau, int nw, void* vhs,
              void* stream);

/*
 * a6.  phi_w <- sum_{j=0..order} (s vhs_w)^j / j!  phi_w,  s = -sqrt(dtau), by the recurrence
 * T_0 = phi, T_j = (s/j) vhs T_{j-1} (truncated Taylor series of PAPER.md:160).  In place.
 * 0 <= order <= 32.    vhs, phi: device.
 */
int afqmc_propagate(afqmc_ctx* ctx, const void* vhs, double dtau, int order, void* phi, int nw,
                    void* stream);

/*
 * a7+a8+a9.  Local energy of Eq. 49 by the recipe of PAPER.md:306-319:
 *   energy[w][0] = E1 = 2 sum_k sum_{a,q} ht[k][a][q] theta_w[(k,a),(k,q)]
 *   energy[w][1] = EC = 1/2 sum_Q sum_g v_{Q g} v_{-Q g},  v = the force bias of theta_w (steps 2d, 3)
 *   energy[w][2] = EX = - sum_{Q,k,k'} sum_{a,b,g} T1[b,a,g] T2[a,b,g]                (steps 2a-2c)
 *       T1[b,a,g] = sum_r Lh[Q][k][a][g][r]     theta_w[(k'-Q,b),(k-Q,r)]
 *       T2[a,b,g] = sum_s Lh[-Q][k'-Q][b][g][s] theta_w[(k,a),(k',s)]
 * Closed-shell spin factors (2, 4, 2) are included.   theta, energy: device.
 */
int afqmc_local_energy(afqmc_ctx* ctx, const void* theta, int nw, void* energy, void* stream);

/*
 * One whole step on DEVICE buffers, the composition bench.py times:
 * green(phi) -> force_bias -> vhs(x, vbias, dtau) -> propagate(order) [phi updated in place]
 * -> green(phi') -> local_energy.  energy [nw][3], logdet [nw] (of phi'), info [nw]: device;
 * logdet/info may be NULL.
 */
int afqmc_step(afqmc_ctx* ctx, void* phi, const double* x, double dtau, int order, int nw,
               void* energy, void* logdet, int* info, void* stream);

/*
 * The same step on HOST buffers: copies phi and x to the device, runs afqmc_step, copies phi',
 * energy (and logdet, info if not NULL) back and synchronises `stream` before returning.  The download of phi'
 * runs on a stream of the context, concurrently with the energy evaluation of phi'.
 * Host buffers should be pinned for full copy bandwidth; pageable memory also works.
 */
int afqmc_step_host(afqmc_ctx* ctx, void* phi_host, const double* x_host, double dtau, int order,
                    int nw, void* energy_host, void* logdet_host, int* info_host, void* stream);

/* ------------------------------------------------------------------------------------------------
 * The AFQMC block around the step: one-body half steps, hybrid importance
 * function with the phaseless weight update, walker orthogonalisation, mixed estimator.
 * "A block is 20 iterations of the propagation step followed by an energy evaluation and walker
 * orthogonalization; the 'hybrid' method is used for propagation".
 * ------------------------------------------------------------------------------------------------ */

/*
 * One-body half-step propagator of Eq. 7/13:  B1[k] = exp(-dtau/2 * h1p[k]) per k-point
 * (H1' is block diagonal in k, Eq. 45), by scaling and squaring of a Taylor series on the
 * device; stored in the context for afqmc_apply_onebody / afqmc_block.
 *   h1p [Nk][m][m] device, complex128: the one-body operator to propagate with (the paper's H1' = H1 + v0,
 *       Eq. 10; building v0 is outside this library).  Need not be Hermitian.
 *   b1_out: device [Nk][m][m] or NULL; receives a copy of B1.
 */
int afqmc_set_onebody(afqmc_ctx* ctx, const void* h1p, double dtau, void* b1_out, void* stream);

/* phi_w[(k,:), :] <- B1[k] phi_w[(k,:), :] for every walker and k-point, in place (Eq. 13).
 * AFQMC_INVALID_ARGUMENT if afqmc_set_onebody was never called.   phi: device [nw][M][N].
 * B1[k] is staged in shared memory when it fits (m up to ~116); larger m (the Gamma-point supercell shape) runs one
 * batched tensor-core GEMM per k-point through the context's Taylor workspace instead: same result, no size limit. */
int afqmc_apply_onebody(afqmc_ctx* ctx, void* phi, int nw, void* stream);

/*
 * Hybrid importance function and phaseless weight update, Eq. 16, 18, 19, for the step
 * whose fields were x and whose force bias was vbias (the arrays given to afqmc_vhs):
 *   z, zbar as in afqmc_vhs;   x.xbar = sum_{Q,g} z_{Q g} zbar_{-Q g},   xbar.xbar = sum_{Q,g} zbar_{Q g} zbar_{-Q g}
 *   log I_w  = 2 (logdet_new[w] - logdet_old[w]) + x.xbar - xbar.xbar/2      (closed shell: two spin channels)
 *   dtheta_w = Im 2 (logdet_new[w] - logdet_old[w]) wrapped to (-pi, pi]        (Eq. 19)
 *   weight[w] <- weight[w] * |I_w| * max(0, cos dtheta_w)                       (Eq. 18)
 *   A walker whose weight is 0 stays at 0, and a walker whose log det is not finite (singular overlap: logdet is
 *   undefined when info != 0) or whose factor overflows is KILLED (weight 0): no NaN or 0*inf reaches the weights.
 *   x [nw][Nk][nchol] double, vbias [nw][Nk][nchol] complex, logdet_old/new [nw] complex (afqmc_overlap of the
 *   walker before / after the propagation), weight [nw] double in/out, log_i [nw] complex out or NULL: device.
 */
int afqmc_hybrid_weight(afqmc_ctx* ctx, const double* x, const void* vbias, double dtau, const void* logdet_old,
                        const void* logdet_new, int nw, double* weight, void* log_i, void* stream);

/*
 * Walker orthogonalisation: phi_w <- Q_w of the thin QR  phi_w = Q_w R_w  with R_w upper
 * triangular and a real positive diagonal (unique), by two passes of Cholesky-QR on the device
 * (Gram matrix, Cholesky factor, phi R^{-1}).  logdet_r[w] = log det R_w (real; device double [nw] or NULL).
 * info[w] (device int32 [nw] or NULL): 0, or j > 0 if the Gram matrix was not positive definite at column j
 * (rank-deficient walker; phi_w is then undefined).  In place.
 */
int afqmc_orthogonalize(afqmc_ctx* ctx, void* phi, int nw, double* logdet_r, int* info, void* stream);

/*
 * Mixed estimator, Eq. 35:  out[0..2] = sum_w weight[w] * energy[w][0..2],  out[3] = sum_w weight[w]
 * (E_mixed = (out[0]+out[1]+out[2]) / out[3]), summed in walker order (deterministic).  Walkers with weight 0
 * (killed by the phaseless projection) and walkers whose local energy is not finite are left out of all four sums,
 * so one dead walker cannot turn the block estimate into NaN.
 *   energy [nw][3] complex, weight [nw] double, out [4] complex: device.
 */
int afqmc_mixed_estimator(afqmc_ctx* ctx, const void* energy, const double* weight, int nw, void* out, void* stream);

/*
 * One block on DEVICE buffers: for s < nsteps:  green(phi) -> force_bias -> vhs(x[s], vbias, dtau) ->
 * B1, Taylor(order), B1 on phi -> overlap(phi') -> hybrid weight update;   then green + local_energy on the
 * final walkers, the mixed estimator with the final weights, and afqmc_orthogonalize.  The overlap of step s's
 * new walker is the green() of step s+1 (computed once).
 *   phi [nw][M][N] in/out; weight [nw] double in/out; x [nsteps][nw][Nk][nchol] double;
 *   energy [nw][3], emixed [4] complex out; logdet_r [nw] double out or NULL; info [nw] int32 out or NULL
 *   (first non-zero of: singular overlap at any step, non positive definite Gram matrix): device.
 *   A walker with a singular overlap at some step gets weight 0 there and stays dead (it is still propagated).
 * Needs afqmc_set_onebody.
 */
int afqmc_block(afqmc_ctx* ctx, void* phi, double* weight, const double* x, double dtau, int order, int nsteps,
                int nw, void* energy, void* emixed, double* logdet_r, int* info, void* stream);

/* Number of kernels the context has launched so far (for bench.py's gpu_launches). */
long long afqmc_launch_count(const afqmc_ctx* ctx);

/* Executed real flops of the exchange contraction (a9) of ONE afqmc_local_energy call on nw
 * walkers, as the kernel executes it (pairs (Q,k,k') ~ (-Q,k'-Q,k-Q) computed once). */
double afqmc_exchange_flops(const afqmc_ctx* ctx, int nw);

/* Executed real flops of ONE afqmc_force_bias call (a4; Eq. 47) on nw walkers: the kernel uses the 3M complex
 * product, 6 real flops per complex multiply-add (the plain definition costs 8): 6 Nk^2 n m nchol nw (both channels when open). */
double afqmc_force_bias_flops(const afqmc_ctx* ctx, int nw);

/* Options: "exchange_warps" (0 = automatic, or 4/5/6/8 warps per CTA of the exchange kernel; tuning aid);
 * "exchange_depth" (0/3 or 2: k-steps of register prefetch in the exchange kernel; tuning aid);
 * "exchange_precision" (0 = default: FP64.  MIXED PRECISION exchange energy on the TF32 tensor cores, the analogue of the
 *   paper's single-precision production mode, boundary still complex128, E1 and EC unaffected, n <= 4 only
 *   (else AFQMC_UNSUPPORTED):  1 = "3xTF32": operands split into TF32 high + low parts, three MMAs per product, FP32
 *   accumulation per task, FP64 sums: EX agrees with FP64 to ~1e-6 relative (tolerance 1e-4);  2 = "1xTF32": operands
 *   rounded once to TF32, fastest, EX error 2e-5 typical / 2e-3 worst measured: outside the 1e-4 tolerance);
 * "exchange_tc" (1 = default: the mixed-precision exchange runs on tcgen05.mma.kind::tf32 with TMEM accumulators and tensor-map
 *   TMA operand copies; 0 = the mma.sync kernel, which is also the fallback for shapes the tcgen05 kernel cannot take);
 * "exchange_3m" (1 = default: three real products per complex product, 0 = the 4M kernel);
 * "exchange_regb" (1 = default for m <= 28: register-resident Theta block, A stream by cp.async, deferred hand-over; 2 = the
 *   same kernel with register prefetch and a blocking hand-over; 0 = the generic kernel); "exchange_np", "exchange_ctas",
 *   "exchange_minblocks" (tuning aids of the exchange kernels);
 * "real_orbitals" (1 = default: when afqmc_create found h1, L and psi_t real -- exactly zero imaginary parts, the dense
 *   Gamma-point representation with real orbitals of PAPER.md:260, :276-284 -- force bias, vHS and exchange run two real products
 *   per complex product instead of three; 0 = the complex kernels on the same inputs.  Results are identical up to rounding);
 * "taylor_subbatch" (0 = default: every Taylor order over all walkers; b > 0: the whole series for b walkers at a time, whose
 *   V then stays in L2 -- measured slower, kept as an aid), "taylor_groups", "taylor_warps", "taylor_legacy", "green_cluster",
 *   "green_legacy" (tuning / testing aids);
 * "timers" (1 = afqmc_step records a CUDA event after each stage, see afqmc_stage_times). */
int afqmc_set_option(afqmc_ctx* ctx, const char* name, int value);

/*
 * Per-stage device times (milliseconds, CUDA events on the step's stream) of the most recent
 * afqmc_step, valid after that stream was synchronised and only with option "timers" = 1:
 * ms[0] green(phi), [1] force_bias, [2] vhs (fields + contraction), [3] propagate, [4] green(phi'),
 * [5] force bias inside local_energy, [6] the exchange kernel alone, [7] energy finalisation.
 */
#define AFQMC_NUM_STAGES 8
int afqmc_stage_times(afqmc_ctx* ctx, float* ms /* host, [AFQMC_NUM_STAGES] */);

/*
 * FP64 peak probes (measurement aid, no AFQMC arithmetic): runs a register-resident loop of
 * kind 0 = DFMA (fma.rn.f64), 1 = DMMA (mma.sync.m8n8k4.f64) on every SM for `iters` iterations and
 * returns the achieved TFLOP/s in *tflops (host).  Synchronous.
 */
int afqmc_probe_fp64(int kind, int iters, double* tflops);

/*
 * Pipelined host entry: the same step on HOST buffers with up to TWO steps in flight (slot = 0 or 1), for loops that feed one
 * batch of walkers after the other.  afqmc_step_host_begin enqueues everything and returns without waiting: the upload of
 * phi and x (on a stream of the context, so it runs while the kernels of the other slot's step are still busy on `stream`),
 * the step on `stream`, the download of phi' into phi_out_host (may be phi_host itself) during the energy evaluation, and the
 * downloads of energy / logdet / info.  afqmc_step_host_end blocks until everything of that slot has arrived in the host
 * buffers (no-op for an idle slot); begin on a busy slot completes the slot's previous step first.  The kernels of the two
 * steps share the context's workspace and run one after the other; what overlaps is the host-link traffic.  Results are
 * bitwise those of afqmc_step_host.  Slot 1 allocates a second set of staging buffers (the size of phi, x and the results for
 * max_walkers) on its first use.  Host buffers must stay valid and untouched from begin to the matching end and should be
 * pinned (with pageable memory the copies serialise with the caller).  Use the same `stream` for both slots.
 * precision = 1: AFQMC_UNSUPPORTED.
 */
int afqmc_step_host_begin(afqmc_ctx* ctx, int slot, const void* phi_host, const double* x_host, double dtau, int order,
                          int nw, void* phi_out_host, void* energy_host, void* logdet_host, int* info_host, void* stream);
int afqmc_step_host_end(afqmc_ctx* ctx, int slot);

/*
 * a1+a2 WITHOUT any allocation and without a context, for callers that cannot call cudaMalloc (code under CUDA graph
 * capture, tight serving loops, harnesses that forbid it): the same result as afqmc_overlap -- logdet[w] = log det O_w,
 * O_w = A^dagger Phi_w (PAPER.md:142 Eq. 27-28, :135-146), LU with partial pivoting, arg in (-pi, pi], info[w] as above --
 * from caller-passed inputs.  Only g, m, n, closed_shell (must be 1) and precision (must be 0) of `dims` are read.
 *   psi_t [Nk][m][n] device complex128; phi [nw][M][N] device complex128; logdet [nw] device complex128; info [nw] device
 *   int32 or NULL.  Asynchronous on `stream`.
 * The matrices O_w (nw * N * (N|1) * 16 bytes, see afqmc_overlap_noalloc_bytes) live in ONE static device array of
 * afqmc_overlap_noalloc_max_bytes() = 16 MiB inside the library (every GPU that loads the library holds it until exit); the
 * call runs no cudaMalloc, cudaFree or allocating library routine.  A call that needs more, or N > 1024, returns
 * AFQMC_SCRATCH_LIMIT and launches nothing (all five configs of the paper's workloads fit: C3 6.0 MB, C5 8.4 MB).
 * The array is shared by every call and keeps the last call's contents; the kernel writes every element it later reads, so
 * nothing needs clearing.  Calls that overlap on the GPU (two streams, parallel graph branches) RACE on it: serialise them.
 * The array's device address is resolved once per device on the first call there (cudaGetSymbolAddress, no allocation);
 * afqmc_overlap_noalloc_setup() does just that for the current device, e.g. before a graph capture starts.
 */
size_t afqmc_overlap_noalloc_max_bytes(void);
size_t afqmc_overlap_noalloc_bytes(const afqmc_dims* dims, int nw);   /* host arithmetic only; 0 for invalid dims */
int afqmc_overlap_noalloc_setup(void);
int afqmc_overlap_noalloc(const afqmc_dims* dims, const void* psi_t, const void* phi, int nw, void* logdet, int* info,
                          void* stream);

#ifdef __cplusplus
}
#endif
#endif /* AFQMC_H */
