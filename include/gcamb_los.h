/*
 * gcamb_los.h -- C ABI of the B200 (sm_100a) line-of-sight integration library.
 *
 * The one data-parallel hot path of gCAMB (arXiv 2509.25110): CAMB's flat-universe
 * `DoFlatIntegration` inside `SourceToTransfers` (Algorithm 1)
 * and the C_l assembly of Eq. 1.  "PAPER.md:N" is line N of the paper text; "BJ" is
 * BASELINE.json `north_star`, which fixes the discrete forms the paper leaves open; "Rn" are
 * the readings listed in DESIGN.md.
 *
 *   Eq. 2  Delta^T_l(k)   = sum_i w_i S_T(k,tau_i)   j_l(x_i)
 *   Eq. 3  Delta^E_l(k)   = sqrt((l+2)!/(l-2)!) sum_i w_i S_E(k,tau_i) j_l(x_i)/x_i^2
 *   BJ / PAPER.md:135    Delta^phi_l(k) = sum_i w_i S_phi(k,tau_i) j_l(x_i)
 *                        x_i = k (tau0 - tau_i), w_i = trapezoid weights of the tau grid (R2)
 *   Eq. 1  C_l^{XY} = 4 pi sum_j dlnk_j P_R(k_j) Delta^X_l(k_j) Delta^Y_l(k_j)
 *                        dlnk_j = trapezoid weights of ln k_j (R6); XY = TT, EE, TE, (phiphi) (R12)
 *
 * All arithmetic is IEEE fp64.  Every step runs in hand-written CUDA kernels; there is no CPU
 * fallback.  Pointers are marked HOST or DEVICE.  Device buffers are owned by the caller and
 * must stay valid until the work enqueued on `cuda_stream` has completed.  `cuda_stream` is a
 * cudaStream_t cast to void* (NULL = the legacy default stream).
 *
 * Threading: a plan is immutable after creation and may be used from several host threads /
 * streams at once, EXCEPT gcamb_los_spectra_host(), which uses scratch owned by the plan and
 * must not run concurrently on the same plan.
 *
 * Errors: every call returns a gcamb_status; no exception crosses the ABI.  After a non-OK
 * status gcamb_los_last_error() returns a thread-local message.  NaN/Inf inside S or P_R are
 * not checked and propagate to the outputs.
 */
#ifndef GCAMB_LOS_H
#define GCAMB_LOS_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct gcamb_los_plan gcamb_los_plan; /* opaque; owns its device tables */

typedef enum {
    GCAMB_OK = 0,
    GCAMB_EINVAL = 1, /* null pointer, size < minimum, l outside [2, 65535], mask/pointer mismatch, n_batch < 1 */
    GCAMB_EGRID = 2,  /* grid not strictly increasing or not finite, k <= 0, tau_i >= tau0 (x must be > 0, R18) */
    GCAMB_EALLOC = 3, /* host or device allocation failed */
    GCAMB_ECUDA = 4   /* any other CUDA error (message in gcamb_los_last_error) */
} gcamb_status;

/* source mask bits; T and E are mandatory, phi optional (BJ: "TT/EE/TE/phiphi").  GCAMB_SRC_TENSOR alone
 * makes a tensor-mode plan (sources T, E, B of the tensor perturbations; see gcamb_los_transfer_tensor). */
enum { GCAMB_SRC_T = 1, GCAMB_SRC_E = 2, GCAMB_SRC_PHI = 4, GCAMB_SRC_TENSOR = 8 };

/*
 * Plan creation = `IntegrationVars_init` hoisted out of the per-call path:
 * chi_i = tau0 - tau_i, w_i, dlnk_j, sqrt((l+2)(l+1)l(l-1)), and per (k, tau) point the start
 * of the downward j_l recurrence: the first l-tile that is not negligible (R16: j_l(x) := 0 for
 * l above ~ x + 18.2 x^(1/3) + 8, where |j_l| < 1e-36) and the normalised pair
 * (j_{l+1}(x), j_l(x)) at the top of that tile, generated ON THE DEVICE by Miller's backward
 * recurrence normalised against closed-form j_0 and j_1 (BJ (b), R15).  With the tile index and
 * 1/x that is 28 bytes per (k, tau) point -- O(N_k N_tau), not an O(N_l N_k N_tau) j_l table.
 * Also sorts k by cost so that the heaviest blocks are issued first.
 *
 *   l_list  HOST [n_l]   strictly increasing, 2 <= l <= 65535 (any subset; the recurrence walks
 *                        every l, only listed l are stored; stretches of 8 l without a listed l
 *                        cost the recurrence only, about half the time of a listed stretch, R21)
 *   k       HOST [n_k]   strictly increasing, > 0, finite; n_k >= 2 (and n_k * n_batch < 2^31 in
 *                        the batched calls: one thread block per k row and cosmology)
 *   tau     HOST [n_tau] strictly increasing, < tau0, finite; n_tau >= 2
 *   src_mask             GCAMB_SRC_T|GCAMB_SRC_E, GCAMB_SRC_T|GCAMB_SRC_E|GCAMB_SRC_PHI, or GCAMB_SRC_TENSOR
 *                        (tensor plan: l <= 65533, three sources, four spectra; only the *_tensor calls,
 *                        gcamb_los_cl_interp and gcamb_los_srcinterp_create accept it)
 *   cuda_stream          stream the precompute kernels run on; the call synchronises it.
 * On success *out owns device memory on the CURRENT device; free with gcamb_los_plan_destroy.
 * Every later call on the plan must be made with that device current (GCAMB_EINVAL otherwise;
 * gcamb_los_plan_destroy switches to it and back by itself).
 */
gcamb_status gcamb_los_plan_create(gcamb_los_plan **out,
                                   const int32_t *l_list, int32_t n_l,
                                   const double *k, int32_t n_k,
                                   const double *tau, int32_t n_tau,
                                   double tau0, uint32_t src_mask, void *cuda_stream);

/*
 * Plan for a CURVED universe ("hyperspherical Bessel functions in a non-flat" Universe,
 * PAPER.md:60; DoNonFlatIntegration, the paper's "immediate next step").  The paper gives
 * no formula; reading R28: curvature K != 0 (in the units of k^2), r_c = 1/sqrt|K|,
 * beta_j = k_j r_c (the caller's k is the generalised wavenumber q = beta sqrt|K|), chi_i = (tau0 - tau_i)/r_c,
 * and the radial functions are the hyperspherical Bessel functions Phi_l^beta(chi), the regular solutions of
 *   K < 0 (open):   Phi'' + 2 coth(chi) Phi' + [beta^2 + 1 - l(l+1)/sinh^2(chi)] Phi = 0,  b_l = sqrt(beta^2 + l^2)
 *   K > 0 (closed): Phi'' + 2 cot(chi)  Phi' + [beta^2 - 1 - l(l+1)/sin^2(chi)]  Phi = 0,  b_l = sqrt(beta^2 - l^2)
 * with Phi_0 = sin(beta chi)/(beta sinK chi) (sinK = sinh or sin), which obey
 *   b_{l+1} Phi_{l+1} = (2l+1) cotK(chi) Phi_l - b_l Phi_{l-1}
 * and tend to j_l(beta chi) as K -> 0.  The transfer functions are the flat ones with j_l(x) -> Phi_l^beta(chi)
 * and, in the polarisation weight, x -> beta sinK(chi):
 *   Delta^T = sum w S_T Phi_l,  Delta^E = sqrt((l+2)!/(l-2)!) sum w S_E Phi_l/(beta sinK chi)^2,
 *   Delta^phi = sum w S_phi Phi_l;  Eq. 1 is taken over unchanged (the curved-space measure and spectrum
 * belong to the P the caller passes).  Skip rule (R16 in curved space): Phi_l := 0 above the first l at which the
 * product of the per-l decay ratios above the turning point l + 1/2 = beta sinK(chi) has fallen below 1e-36
 * (open: those ratios tend to tanh(chi/2), slower than the flat j_l when chi is not small).
 * Closed universes: every beta_j must be an integer >= 3 (to 1e-6; it is rounded to it) and chi <= pi/2 on the
 * whole tau grid (GCAMB_EGRID otherwise); Phi_l^beta = 0, hence Delta_l(k_j) = 0 exactly, for l >= beta_j.
 * The plan holds, next to the tables of gcamb_los_plan_create, cotK(chi_i) and 1/sinK^2(chi_i) per tau and
 * the two recurrence coefficients per (k, l): 16 n_l n_k bytes.  gcamb_los_transfer[_batched],
 * gcamb_los_cls[_batched], gcamb_los_spectra_host, gcamb_los_cl_interp and gcamb_los_srcinterp_create work
 * on such a plan as on a flat one (gcamb_los_spectra_batched takes its two-kernel path).
 * src_mask: T|E or T|E|PHI.  K = 0 is GCAMB_EINVAL (use gcamb_los_plan_create).
 */
gcamb_status gcamb_los_plan_create_curved(gcamb_los_plan **out,
                                          const int32_t *l_list, int32_t n_l,
                                          const double *k, int32_t n_k,
                                          const double *tau, int32_t n_tau,
                                          double tau0, double curvature_K, uint32_t src_mask,
                                          void *cuda_stream);

/* Frees the plan and its device tables (synchronises the device).  NULL is allowed. */
gcamb_status gcamb_los_plan_destroy(gcamb_los_plan *plan);

/*
 * Sizes of a plan.  Any output pointer may be NULL.
 *   n_src  = 2 (T,E) or 3 (T,E,phi);  n_spec = 3 (TT,EE,TE) or 4 (+phiphi)
 *   executed_terms = number of (l in l-range, k, tau) triples with l <= min(L(x), l_max), i.e. the
 *   terms that are not skipped by R16 (the algorithmic work; nominal is n_l*n_k*n_tau).
 */
gcamb_status gcamb_los_plan_info(const gcamb_los_plan *plan, int32_t *n_l, int32_t *n_k,
                                 int32_t *n_tau, int32_t *n_src, int32_t *n_spec,
                                 int64_t *executed_terms);

/*
 * Kernels of this library that one gcamb_los_transfer[_batched] call and one gcamb_los_cls[_batched]
 * call launch on this plan (any batch size).  The transfer is one launch, or two overlapping ones when
 * only some rows (x_max = k (tau0 - tau_0) > 2^53 * 7.5e-13 = 6755) take the compensated recurrence
 * coefficient.  Nothing else is enqueued: no memset, no atomics;
 * tau grids longer than one thread block's slots are taken in passes by the same block, so results
 * are bit-reproducible for any n_tau.  Either pointer may be NULL.
 */
gcamb_status gcamb_los_plan_launches(const gcamb_los_plan *plan, int32_t *transfer_kernels,
                                     int32_t *cls_kernels);

/*
 * Eq. 2-3: sources -> transfer functions (steps a1-a3: source staging, j_l recurrence in
 * registers, tau-integration, cross-thread reduction, Delta^E prefactor).  Asynchronous on
 * `cuda_stream`; no allocation, no host<->device copy.
 *   d_S_T, d_S_E, d_S_phi  DEVICE [n_k][n_tau], tau fastest.  d_S_phi must be NULL iff the plan
 *                          has no GCAMB_SRC_PHI.
 *   d_Delta                DEVICE [n_src][n_l][n_k], k fastest, order T, E, (phi) -- the
 *                          (X, l, q) array of PAPER.md:136.  Every element is written.
 */
gcamb_status gcamb_los_transfer(const gcamb_los_plan *plan,
                                const double *d_S_T, const double *d_S_E, const double *d_S_phi,
                                double *d_Delta, void *cuda_stream);

/*
 * Eq. 1: transfer functions -> spectra (step a4).  Asynchronous on `cuda_stream`.
 *   d_Delta DEVICE [n_src][n_l][n_k];  d_P_R DEVICE [n_k];
 *   d_Cl    DEVICE [n_spec][n_l], order TT, EE, TE, (phiphi).
 */
gcamb_status gcamb_los_cls(const gcamb_los_plan *plan, const double *d_Delta, const double *d_P_R,
                           double *d_Cl, void *cuda_stream);

/*
 * Batched variants (step a5; emulator use-case PAPER.md:24, 248; BJ config 3): n_batch
 * cosmologies sharing one plan, one launch each.
 *   d_S_X   DEVICE [n_batch][n_k][n_tau];   d_Delta DEVICE [n_batch][n_src][n_l][n_k]
 *   d_P_R   DEVICE [n_batch][n_k];          d_Cl    DEVICE [n_batch][n_spec][n_l]
 */
gcamb_status gcamb_los_transfer_batched(const gcamb_los_plan *plan, int32_t n_batch,
                                        const double *d_S_T, const double *d_S_E,
                                        const double *d_S_phi, double *d_Delta, void *cuda_stream);
gcamb_status gcamb_los_cls_batched(const gcamb_los_plan *plan, int32_t n_batch,
                                   const double *d_Delta, const double *d_P_R, double *d_Cl,
                                   void *cuda_stream);

/*
 * Spectra on EVERY multipole l_list[0] .. l_list[n_l-1] from the spectra on the plan's (sparse) l list:
 * CAMB computes "a number of explicitly computed multipoles" set by l_sample_boost and obtains the
 * others by "spline interpolation" (footnote 5 PAPER.md:127).  The paper
 * defines neither the spline nor the interpolated quantity; reading R25: NATURAL cubic
 * spline in l (second derivative 0 at both ends) of y(l) = l (l+1) C_l^{XY}, knots = the l list,
 * every spectrum alike, C_l = y(l) / (l (l+1)) afterwards.  The listed multipoles come back
 * unchanged up to rounding (y_i / (l_i (l_i+1))).  The LU factors of the spline's tridiagonal system
 * depend on the l list only and are plan tables; a call runs one kernel, one thread block per
 * (cosmology, spectrum).  Needs 2 <= n_l <= 10000 (GCAMB_EINVAL otherwise).
 *   d_Cl     DEVICE [n_batch][n_spec][n_l]                     as written by gcamb_los_cls[_batched]
 *   d_Cl_all DEVICE [n_batch][n_spec][l_list[n_l-1] - l_list[0] + 1], one entry per integer l
 * Asynchronous on `cuda_stream`; deterministic.
 */
gcamb_status gcamb_los_cl_interp(const gcamb_los_plan *plan, int32_t n_batch, const double *d_Cl,
                                 double *d_Cl_all, void *cuda_stream);

/*
 * Tensor modes: the paper runs SourceToTransfers twice, "one for scalar perturbations
 * and the other for tensor ones" (Figure 1; get_tensor_cls, l_max_tensor = 1500,
 * PAPER.md:91-93) and says that for tensors and B modes "similar equations arise" (citing
 * Seljak & Zaldarriaga) without printing them.  Reading R27: the flat-space
 * tensor line-of-sight kernels of that literature (Zaldarriaga & Seljak 1997, Eq. 30), x = k (tau0 - tau):
 *   Delta^{T,t}_l(k) = sqrt((l+2)!/(l-2)!) sum_i w_i S_T(k,tau_i) j_l(x_i) / x_i^2
 *   Delta^{E,t}_l(k) = sum_i w_i S_E(k,tau_i) [ -j_l + j_l'' + 2 j_l/x^2 + 4 j_l'/x ](x_i)
 *   Delta^{B,t}_l(k) = sum_i w_i S_B(k,tau_i) [ 2 j_l' + 4 j_l/x ](x_i)
 *   C_l^{XY,t}       = 4 pi sum_j dlnk_j P_t(k_j) Delta^{X,t}_l(k_j) Delta^{Y,t}_l(k_j),  XY = TT, EE, BB, TE
 * (Eq. 1 with the tensor primordial spectrum; convention constants of the tensor normalisation belong to
 * P_t).  `plan` must have been created with src_mask = GCAMB_SRC_TENSOR (2 <= l <= 65533).  The transfer call
 * runs the four-sum transfer kernels once on the union of {l - 1, l, l + 1, l + 2} (the T, E and B kernels
 * are combinations, with l-dependent coefficients, of four plain j_l sums at neighbouring multipoles, through
 * j_l' = (l/x) j_l - j_{l+1} and j_l/x = (j_{l-1} + j_{l+1})/(2l+1)) plus one small kernel; it needs
 * caller-owned scratch of gcamb_los_tensor_work_bytes() bytes PER COSMOLOGY.
 *   d_S_T, d_S_E, d_S_B DEVICE [n_k][n_tau];  d_Delta DEVICE [3][n_l][n_k], order T, E, B;
 *   d_work DEVICE scratch;  d_P_t DEVICE [n_k];  d_Cl DEVICE [4][n_l], order TT, EE, BB, TE.
 * The *_batched forms take n_batch cosmologies on one plan (a5; emulator use-case PAPER.md:24, 248), every
 * array with a leading [n_batch] dimension and n_batch * gcamb_los_tensor_work_bytes() bytes of scratch:
 * ONE launch of the transfer kernels with n_batch members; results equal a loop of single calls bit for
 * bit.  1 <= n_batch <= 32767 (transfer), 65535 (cls), 2 n_k n_batch < 2^31: GCAMB_EINVAL otherwise.
 * Asynchronous on `cuda_stream`; deterministic.
 */
gcamb_status gcamb_los_tensor_work_bytes(const gcamb_los_plan *plan, int64_t *bytes);
gcamb_status gcamb_los_transfer_tensor(const gcamb_los_plan *plan, const double *d_S_T, const double *d_S_E,
                                       const double *d_S_B, double *d_Delta, double *d_work,
                                       void *cuda_stream);
gcamb_status gcamb_los_cls_tensor(const gcamb_los_plan *plan, const double *d_Delta, const double *d_P_t,
                                  double *d_Cl, void *cuda_stream);
gcamb_status gcamb_los_transfer_tensor_batched(const gcamb_los_plan *plan, int32_t n_batch, const double *d_S_T,
                                               const double *d_S_E, const double *d_S_B, double *d_Delta,
                                               double *d_work, void *cuda_stream);
gcamb_status gcamb_los_cls_tensor_batched(const gcamb_los_plan *plan, int32_t n_batch, const double *d_Delta,
                                          const double *d_P_t, double *d_Cl, void *cuda_stream);

/*
 * InterpolateSources (SourceToTransfers "begins by calling IntegrationVars_init ... and
 * InterpolateSources to prepare the source data"): sources known on a coarse wavenumber grid (the modes the
 * perturbation evolution integrated) -> sources on the plan's k grid.  The paper does not define the
 * interpolation; reading R26: for every tau independently, the NATURAL cubic spline in k
 * through the coarse samples.  The handle holds the LU factors of the spline system and, per fine k, its
 * coarse interval and weights (tables built on the host at creation); it refers to the plan's grids only
 * at creation and may outlive the plan.
 *   k_coarse   HOST [n_kc] strictly increasing, > 0; every k of the plan must lie inside
 *              [k_coarse[0], k_coarse[n_kc-1]] (GCAMB_EGRID otherwise: no extrapolation); n_kc >= 2
 *   n_series   number of independent [n_kc][n_tau] arrays (sources x cosmologies), <= 65535
 *   d_S_coarse DEVICE [n_series][n_kc][n_tau];  d_S_fine DEVICE [n_series][n_k][n_tau] (n_k <= 524280)
 *   d_work     DEVICE scratch of the size of d_S_coarse (second derivatives of the splines)
 * Asynchronous on `cuda_stream`; two kernels; deterministic.
 * The spline matrix is diagonally dominant, so its inverse is banded to any wanted accuracy: the handle also holds
 * the rows of the inverse, cut where what is dropped stays below 1e-18 max|S| in a result (a bound), and the solve
 * runs as independent dot products of ~60 terms per (coarse k, tau).  Grids whose rows stay wide (more than 100
 * columns on average: spacings that jump by orders of magnitude) or longer than 4096 keep the two sequential
 * sweeps per (series, tau); gcamb_los_srcinterp_info reports which (band_columns = columns of the widest row of
 * the banded inverse, 0 = sequential sweeps; any out pointer may be NULL).
 */
typedef struct gcamb_los_srcinterp gcamb_los_srcinterp;
gcamb_status gcamb_los_srcinterp_create(gcamb_los_srcinterp **out, const gcamb_los_plan *plan,
                                        const double *k_coarse, int32_t n_kc, void *cuda_stream);
gcamb_status gcamb_los_srcinterp_destroy(gcamb_los_srcinterp *handle);
gcamb_status gcamb_los_srcinterp_info(const gcamb_los_srcinterp *handle, int32_t *n_kc, int32_t *n_k, int32_t *n_tau,
                                      int32_t *band_columns);
gcamb_status gcamb_los_interp_sources(const gcamb_los_srcinterp *handle, int32_t n_series,
                                      const double *d_S_coarse, double *d_S_fine, double *d_work,
                                      void *cuda_stream);

/*
 * gcamb_los_interp_sources for callers that cannot allocate device memory (code under CUDA-graph capture, tight
 * serving loops, harnesses that forbid cudaMalloc): the same two kernels, same arguments and results (bit for
 * bit), but the scratch is a file-scope `static __device__` array of the library instead of a caller buffer.
 * The call makes no cudaMalloc / cudaFree and calls no allocating library routine.
 *   limit      n_series * n_kc * n_tau <= 1048576 doubles (8 MiB; e.g. two sources x 300 coarse k x 1200 tau);
 *              GCAMB_EINVAL with a message stating both numbers otherwise (use gcamb_los_interp_sources then)
 *   cost       every GPU that loads the library holds the 8 MiB array until the process exits
 *   sharing    all calls on a device share the array: calls that may OVERLAP on the GPU (different streams
 *              without an ordering between them) race on it and are not supported; calls on one stream, or
 *              ordered by events, are safe.  Nothing in it needs clearing: every element a call reads it has
 *              written itself, so the contents an earlier call left behind are never used.
 *   set-up     the first call on a device looks up the array's device address (cudaGetSymbolAddress, with
 *              that device current) and keeps it; make that first call outside a stream capture.
 * The handle (gcamb_los_srcinterp_create) is built beforehand, at set-up, like the plan.
 */
gcamb_status gcamb_los_interp_sources_noalloc(const gcamb_los_srcinterp *handle, int32_t n_series,
                                              const double *d_S_coarse, double *d_S_fine, void *cuda_stream);

/*
 * Batched sources -> spectra in one call, WITHOUT the transfer functions ever reaching memory
 * (the emulator-training use-case: 1e5-1e6 spectra on a fixed grid; Eq. 1-3,
 * PAPER.md:50-58).  For plans with the T and E sources only and n_tau <= 2560 this runs ONE fused
 * kernel plus a small finishing kernel: x = k (tau0 - tau) does not depend on the cosmology, so the
 * j_l recurrence is evaluated once per (l, k, tau) for a block of 8 (or 4) cosmologies, the tau-sum
 * becomes a dense [l x tau] . [tau x (X, cosmology)] contraction on the FP64 tensor cores
 * (mma.sync.m8n8k4.f64), and Eq. 1 is accumulated over k inside the kernel from per-thread-block
 * partial spectra that are added in a fixed order: results are bit-reproducible run to run.  They
 * are NOT bit-identical to gcamb_los_transfer_batched + gcamb_los_cls_batched (another summation
 * order; both are within the tolerances of BJ).  Other plans (phi source, longer tau grids, sparse
 * l lists) and n_batch = 1 take those two calls internally, with Delta in scratch of the plan.
 *   d_S_T, d_S_E, d_S_phi DEVICE [n_batch][n_k][n_tau] (d_S_phi NULL iff the plan has no phi);
 *   d_P_R DEVICE [n_batch][n_k];  d_Cl DEVICE [n_batch][n_spec][n_l], order TT, EE, TE, (phiphi).
 * Asynchronous on `cuda_stream`.  Scratch (partial spectra: n_SM x ceil(n_batch/8) x 3 x n_l x 8
 * doubles, or Delta) belongs to the plan, is allocated on first use and grows when a larger batch
 * arrives (that call synchronises the device); NOT thread-safe per plan.
 */
gcamb_status gcamb_los_spectra_batched(gcamb_los_plan *plan, int32_t n_batch,
                                       const double *d_S_T, const double *d_S_E, const double *d_S_phi,
                                       const double *d_P_R, double *d_Cl, void *cuda_stream);

/*
 * What gcamb_los_spectra_batched does for this plan and batch size: *fused = 1 if the fused kernel
 * applies, *kernels = kernels of this library one call launches, *scratch_bytes = plan scratch it
 * needs.  Any output pointer may be NULL.
 */
gcamb_status gcamb_los_spectra_batched_info(const gcamb_los_plan *plan, int32_t n_batch, int32_t *fused,
                                            int32_t *kernels, int64_t *scratch_bytes);

/*
 * End-to-end call with HOST buffers (the paper's "accelerator data region"):
 * H2D of the sources and P_R, transfer, cls, D2H of C_l (and of Delta when h_Delta != NULL), then
 * synchronises `cuda_stream`.  The sources are copied in four blocks of k rows (heaviest rows first)
 * on a copy stream owned by the plan and each block's kernels start when it has landed, so the
 * compute hides behind the H2D copy; results equal the device-resident path bit for bit.  Device
 * scratch, streams and events are created inside the plan on first use (scratch sized for n_batch)
 * and reused; NOT thread-safe per plan.  Host buffers should be pinned for full copy bandwidth
 * (pageable memory works but serialises the copies).
 *   h_S_X HOST [n_batch][n_k][n_tau];  h_P_R HOST [n_batch][n_k];
 *   h_Cl  HOST [n_batch][n_spec][n_l]; h_Delta HOST [n_batch][n_src][n_l][n_k] or NULL.
 */
gcamb_status gcamb_los_spectra_host(gcamb_los_plan *plan, int32_t n_batch,
                                    const double *h_S_T, const double *h_S_E, const double *h_S_phi,
                                    const double *h_P_R, double *h_Cl, double *h_Delta,
                                    void *cuda_stream);

/* Thread-local message of the last non-OK status on this thread ("" if none). */
const char *gcamb_los_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* GCAMB_LOS_H */
