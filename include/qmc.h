/*
 * qmc.h -- C ABI of the B200-native batched Slater-Jastrow electron-move engine.
 *
 * The library implements, in hand-written CUDA for sm_100a, the hot path behind the double-precision
 * DMC runs of arXiv 2504.07948: the walker-batched particle-by-particle electron move for a
 * Slater-Jastrow trial function in a contracted-Gaussian (LCAO) basis.
 *
 *   Psi_T = exp[J] D_up D_dn,  phi_j = sum_l C_lj Phi_l            PAPER.md L125-127 (eq. 2), M = 1
 *   A_pj = phi_j(r_p) and its inverse
 *   d ln D / d lambda = tr(A^-1 dA/d lambda)                       PAPER.md L173 (eq. 3)
 *   walker-level batching of all of the above
 *   fixed-node rejection
 * Everything the paper leaves open (basis functional form, Pade Jastrow, drift-diffusion proposal,
 * Philox stream, delayed rank-k update, local energy) follows BASELINE.json `north_star`/`configs`
 * with the readings listed in DESIGN.md ("Readings").
 *
 * Conventions
 *   - Units: bohr and hartree.  All floating point is IEEE FP64.
 *   - Electrons 0..n_up-1 are spin-up, n_up..n_up+n_dn-1 spin-down.  One "step" of qmc_sweep is one
 *     sweep: one proposed move for every electron, ups first, index ascending, all walkers in lockstep.
 *   - Every function returns QMC_OK (0) or a negative error code; nothing throws, aborts or prints.
 *     qmc_last_error() gives a thread-local message for the last failing call.
 *   - Pointer arguments marked "host or device" may be either (unified virtual addressing decides);
 *     inputs are copied before the call returns, so the caller may free them afterwards.
 *   - Output buffers are caller-owned (normally torch tensors).  Device buffers are written
 *     asynchronously on the walker set's stream -- a caller that reads them on ANOTHER stream must order that
 *     stream after the walker set's (an event, or qmc_synchronize); host buffers are written synchronously.
 *   - The library owns its internal state (cudaMalloc at create time, freed at destroy).  Scratch of the
 *     row-f2 / f3 getters and the staging buffer of host-pointer getters are allocated by the first call that
 *     needs them and kept (qmc_release_scratch frees them); no other call allocates.
 *   - A system lives on the CUDA device that was current at qmc_init; every call on it or on its walker sets
 *     runs there whatever the calling thread's current device is (restored on return).
 *   - Relative to the signatures sketched in SURVEY.md 8(b): qmc_walkers_create takes a `flags` word (logging,
 *     path selection, screening) and qmc_basis carries `n_prim_total` (the length of alpha / coef, needed to copy
 *     them); rows f1-f4 and the stage-level / timing entry points are additions, each marked below.
 *   - There is NO CPU fallback: every entry point fails with QMC_ERR_CUDA when no sm_100 device works.
 */
#ifndef QMC_B200_H
#define QMC_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define QMC_OK 0
#define QMC_ERR_ARG (-1)      /* null pointer, inconsistent sizes, l > 2, delay_k < 1, tau <= 0, ... */
#define QMC_ERR_CUDA (-2)     /* a CUDA call failed (message in qmc_last_error) */
#define QMC_ERR_SINGULAR (-3) /* zero pivot while inverting a Slater matrix at walker creation */
#define QMC_ERR_NOMEM (-4)
#define QMC_ERR_STATE (-5)    /* call not valid in the current state (e.g. log requested but not enabled) */

/* flags of qmc_walkers_create */
#define QMC_LOG_RATIOS 1u /* also record rho_D*exp(dJ) and p_acc of every proposed move */
#define QMC_SCREEN_MO 4u  /* optional screening of the MO contraction (off by default; SURVEY 8(d).1 allows it where the
                             parity tolerances still hold): a 128-row x 32-function stage of the basis matrix Phi whose
                             largest |entry| (value, gradient, Laplacian) is below QMC_SCREEN_THETA is not contracted.  With
                             orthonormal MO columns the orbital rows change by at most sqrt(N_b) * theta ~ 1e-22 absolute,
                             far below the rounding of the sums.  The work saved depends on how localised the crowd's
                             electron is; qmc_get_mo_work reports it. */
#define QMC_SCREEN_THETA 1e-24
#define QMC_LARGE_PATH 2u /* never use the one-launch small-system path (row f4): systems with <= 32 electrons per spin
                             whose per-walker state fits in shared memory otherwise run a whole qmc_sweep / qmc_dmc_step
                             call in one kernel, one warp per walker, with rank-1 updates (delay_k then only changes
                             rounding, reading A13) */

#define QMC_ONE_LANE 8u   /* never split the crowd into two lanes.  By default a large crowd (rows of the inverse longer than
                             256, per-electron kernels, a walker count that splits without padding the contraction) moves
                             through the electron steps as two half crowds on two streams, so that the HBM-bound kernels of
                             one run in the shadow of the other's contraction; results differ from the one-lane run only by
                             the rounding of the stream-K partition (it depends on the row count). */

#define QMC_PER_ELECTRON 16u /* never use the window kernel of the mid-size path: systems with 33..256 electrons per spin whose
                               basis fits (5 x 4 rows of N_b functions in shared memory) otherwise run all electron steps of a
                               delay window in ONE launch -- four walkers per CTA, basis functions and MO rows never leaving
                               the SM -- followed by the flush.  Same arithmetic; the contraction sums in another order
                               (rounding). */

#define QMC_STEP_ONEPASS 32u /* use the one-pass step kernel (the delay window read once, as an FP64 DMMA pass against eight
                               vectors; csrc/step_onepass.cuh) whatever the size.  It is the default of the per-electron
                               kernels for rows of the inverse longer than 256; the flag forces it for shorter rows (tests). */

typedef struct qmc_system qmc_system;   /* immutable after qmc_init: atoms, basis, MO coefficients, Jastrow (device) */
typedef struct qmc_walkers qmc_walkers; /* mutable crowd state */

typedef struct {
    int n_atoms;
    const double* xyz; /* [n_atoms][3], host or device */
    const double* Z;   /* [n_atoms] charge used by the e-n Jastrow and the bare Coulomb potential */
} qmc_atoms;

/* Contracted Gaussian shells, Phi = S_lm(x) * sum_p coef_p exp(-alpha_p |x|^2), x = r - R_atom.
 * l = 0: {1};  l = 1: {x, y, z};
 * l = 2: {sqrt3 xy, sqrt3 yz, z^2 - (x^2+y^2)/2, sqrt3 xz, (sqrt3/2)(x^2-y^2)}  (5 components, reading A1).
 * Basis-function order: shells in input order, functions of a shell in the order above.
 * coef already contains all normalisation (the library never normalises); alpha = 0 is legal. */
typedef struct {
    int n_shells;
    const int* atom;        /* [n_shells] index into qmc_atoms */
    const int* l;           /* [n_shells] 0, 1 or 2 */
    const int* n_prim;      /* [n_shells] >= 1 */
    const int* prim_offset; /* [n_shells] offset into alpha / coef */
    int n_prim_total;
    const double* alpha; /* [n_prim_total] */
    const double* coef;  /* [n_prim_total] */
} qmc_basis;

typedef struct {
    int n_basis; /* must equal sum over shells of 2l+1 */
    int n_up, n_dn;
    const double* C_up; /* [n_basis][n_up] row-major: C_up[l][j] = coefficient of Phi_l in orbital j */
    const double* C_dn; /* [n_basis][n_dn]; may be NULL when n_dn == 0 */
} qmc_mo;

/* u_ee(r) = a r / (1 + b_ee r), a = a_anti (opposite spins) or a_para (same spin);
 * u_en(r) = -Z_I r / (1 + b_en r);  Psi ~ exp(+J). */
typedef struct {
    double a_anti, a_para, b_ee, b_en;
} qmc_jastrow;

/* Build the immutable system on the current CUDA device.  `cuda_stream` is a cudaStream_t (may be 0). */
int qmc_init(qmc_system** out, const qmc_atoms* atoms, const qmc_basis* basis, const qmc_mo* mo,
             const qmc_jastrow* jastrow, void* cuda_stream);
void qmc_finalize(qmc_system* sys);

/* Create a crowd of n_walkers walkers at `positions` ([n_walkers][n_elec][3], ups first, host or device).
 * Evaluates all orbital rows, inverts the Slater matrices on the device (Gauss-Jordan with partial pivoting; from 256
 * electrons per spin a blocked form with implicit row pivoting whose rank-16 updates are FP64 DMMA GEMMs; one
 * Newton-Schulz refinement step either way), and sets log|Psi|, sign, E_L and unit weights.  RNG streams are keyed (seed; first_walker_id + w, step,
 * electron) with the step counter starting at first_step, so any crowd is a slice of one infinite
 * crowd (reading A20) and sweeps can be resumed bit for bit.  Returns QMC_ERR_SINGULAR if any Slater
 * matrix has a zero pivot.  All later work is enqueued on `cuda_stream`. */
int qmc_walkers_create(const qmc_system* sys, qmc_walkers** out, int n_walkers, const double* positions,
                       uint64_t seed, uint32_t first_walker_id, uint32_t first_step, uint32_t flags,
                       void* cuda_stream);
void qmc_walkers_destroy(qmc_walkers* w);

/* Run nsteps sweeps with time step tau (> 0) and delay rank delay_k (1 <= delay_k <= 128).
 * Per electron i, for all walkers (BASELINE.json north_star items 1-6):
 *   drift G = grad_i ln|Psi|; r' = r + tau G + sqrt(tau) chi (Philox4x32-10 -> Box-Muller);
 *   basis functions and orbital rows at r' (FP64 contraction C^T Phi); rho_D from the effective
 *   inverse column; Pade Jastrow ratio; accept iff u < rho_D^2 exp(2 dJ + Delta) and rho_D > 0;
 *   accepted rows enter a delay window that is flushed into A^-1 every delay_k proposals and at the
 *   end of each spin block as FP64 GEMMs.  E_L = K + V is evaluated at the end of every sweep.
 * delay_k changes performance only; results differ from delay_k = 1 by rounding.
 * Asynchronous on the walker set's stream.  The accept log of this call replaces the previous one. */
int qmc_sweep(qmc_walkers* w, int nsteps, double tau, int delay_k);

/* Getters.  `out` may be host or device memory. */
int qmc_get_positions(const qmc_walkers* w, double* out /* [W][n_elec][3] */);
/* out[w][p][j] = (A^-1)[j][p] of spin (0 up, 1 down): row p is the vector dotted with a new orbital row (A18) */
int qmc_get_Ainv(const qmc_walkers* w, int spin, double* out /* [W][n_s][n_s] */);
int qmc_get_logpsi(const qmc_walkers* w, double* logabs /* [W] */, int8_t* sign /* [W], may be NULL */);
int qmc_get_eloc(const qmc_walkers* w, double* eloc /* [W], K+V */, double* ekin /* [W], may be NULL */);
/* log of the most recent qmc_sweep call: bits[t][i][w], bit0 = accepted, bit1 = tie-flagged
 * (|u - p_acc| < 1e-12 or |rho_D| < 1e-12), bit2 = non-finite value seen (move rejected). */
int qmc_get_accept_log(const qmc_walkers* w, uint8_t* bits /* [T][n_elec][W] */);
/* needs QMC_LOG_RATIOS: ratio = rho_D * exp(dJ), pacc = p_acc (0 when rejected at the node) */
int qmc_get_ratio_log(const qmc_walkers* w, double* ratio /* [T][n_elec][W] */, double* pacc /* may be NULL */);
/* totals since creation */
int qmc_get_stats(const qmc_walkers* w, uint64_t* n_proposed, uint64_t* n_accepted, uint64_t* n_ties,
                  uint64_t* n_nonfinite);
int qmc_synchronize(const qmc_walkers* w);

/* ---- Row f1 of the scope table: the DMC generation (fixed-node DMC, eq. 1; the paper prints no
 * weight or branching rule, so these follow Umrigar-Nightingale-Runge 1993 -- readings A28-A30 of DESIGN.md).
 *
 * qmc_dmc_step: n_generations times { one sweep exactly as qmc_sweep, except that the drift of every proposal (forward
 * and reverse) is limited, vbar = v (-1 + sqrt(1 + 2 a v^2 tau)) / (a v^2 tau) with a = limiter_a (0: no limiter);
 * E_L; tau_eff = tau * (sum over accepted moves of |sqrt(tau) chi|^2) / (sum over all proposals of it);
 * weight *= exp(-tau_eff ((E_old + E_new) / 2 - e_trial)) }.  Weights start at 1 at creation and persist across calls;
 * E_old of the first generation of a call is the current E_L.  Asynchronous on the stream; the accept log covers the
 * call like qmc_sweep's.  Errors: QMC_ERR_ARG as qmc_sweep, or limiter_a < 0 / non-finite e_trial. */
int qmc_dmc_step(qmc_walkers* w, int n_generations, double tau, int delay_k, double e_trial, double limiter_a);
/* weights[W] (and tau_eff[W] of the last generation; may be NULL); host or device buffers. */
int qmc_get_weights(const qmc_walkers* w, double* weights, double* tau_eff);
/* Fixed-population "comb" reconfiguration: with c_i the cumulative weights (summed in index order) and one uniform xi
 * (Philox counter (0xFFFFFFFF, step, 0xFFFFFFFF, 3), first word pair), walker i gets as many copies as teeth
 * (j + xi) W_tot / W, j = 0..W-1, fall in [c_{i-1}, c_i).  Walkers with >= 1 copy keep their slot; the k-th slot with
 * none (ascending) receives the k-th extra copy, donors in ascending order; every weight becomes W_tot / W.
 * source[W] (int32, host or device, may be NULL): slot j now holds a copy of old walker source[j].  e_mixed (may be
 * NULL): sum w E_L / sum w before the reconfiguration.  Must be called between sweeps (the delay window is empty then);
 * synchronises the stream. */
int qmc_branch(qmc_walkers* w, int32_t* source, double* e_mixed);
/* A DMC run with population control, the whole loop on the device (no host round trip between generations; DESIGN.md
 * reading A32; "walkers ... branching", L279-302 the production runs):
 *   E_T = e_trial0
 *   for g = 0 .. n_generations-1:  one qmc_dmc_step generation with E_T
 *       if branch_every > 0 and (g + 1) % branch_every == 0:
 *           qmc_branch;  E_T <- e_mixed - feedback * ln(W_tot / W)      (W_tot / W: the weight every walker leaves with)
 * e_trial_out (may be NULL): E_T after the run.  branch_log (may be NULL): [n_generations / branch_every][3] =
 * {e_mixed, E_T after, W_tot / W} of every reconfiguration.  sources (int32, may be NULL): [n_generations /
 * branch_every][W] slot maps as qmc_branch's.  All three host or device.  The accept / ratio logs cover all
 * n_generations.  Synchronises the stream once, at the end.  Errors: as qmc_dmc_step; QMC_ERR_ARG if branch_every < 0
 * or feedback / e_trial0 is not finite. */
int qmc_dmc_run(qmc_walkers* w, int n_generations, double tau, int delay_k, double e_trial0, double limiter_a, int branch_every,
                double feedback, double* e_trial_out, double* branch_log, int32_t* sources);

/* ---- Row f2, first half: out[W][n_atoms][3] = d ln|Psi| / d R_a at the current configuration -- the paper's eq. (3)
 * (d ln D / d lambda = tr(A^-1 dA/d lambda)) with the nuclear coordinates as parameters, basis functions
 * moving with their nucleus, plus the electron-nucleus Jastrow term.  This is the wave-function ("Pulay") term of a QMC
 * force estimator; qmc_get_deloc_dR below is the other term (eq. 4).  out: host or device.  Call between sweeps; uses a
 * [W][N_s][N_b] scratch (12.9 GB at config 2; allocated by the first call, kept) and synchronises the stream.
 * QMC_ERR_NOMEM if that does not fit. */
int qmc_get_dlogpsi_dR(qmc_walkers* w, double* out);
/* ---- Row f2, second half: deloc[W][n_atoms][3] = d E_L / d R_a at the current configuration by the paper's eq. (4)
 * (PAPER.md L177-181): tr(A^-1 dB/dR_a - X dA/dR_a), X = A^-1 B A^-1, summed over both spins, plus the derivative of the
 * Jastrow and potential terms of E_L that are not inside the trace (reading A33).  Electrons fixed; basis
 * functions and electron-nucleus Jastrow terms move with their nucleus; MO coefficients and Jastrow parameters constant
 * (no orbital relaxation, no space warp).  dlogpsi (may be NULL): the same call also returns qmc_get_dlogpsi_dR's
 * result from the shared C A^-1 product -- the two pieces of the force estimator
 * F_a = -< dE_L/dR_a + 2 (E_L - <E_L>) d ln|Psi|/dR_a >.  deloc, dlogpsi: host or device.  Call between sweeps;
 * uses 2 [W][N_s][N_b] + 4 [W][N_s^2] doubles of scratch (allocated by the first call, kept) and synchronises the
 * stream.  QMC_ERR_NOMEM if that does not fit. */
int qmc_get_deloc_dR(qmc_walkers* w, double* deloc, double* dlogpsi);
/* Frees the scratch kept by qmc_get_dlogpsi_dR / qmc_get_deloc_dR / qmc_get_vnl and the staging buffer of the
 * host-pointer getters (they come back on the next call that needs them).  Synchronises the stream. */
int qmc_release_scratch(qmc_walkers* w);

/* ---- Row f3: non-local pseudopotential energy by spherical quadrature ("ccECP pseudopotentials", L180;
 * DESIGN.md reading A34).  qmc_set_ecp attaches the non-local channels to a system: channel c sits on atom ch_atom[c],
 * projects on angular momentum ch_l[c] (0..2), has the radial function ch_beta[c] exp(-ch_alpha[c] r^2); atom I acts on
 * electrons closer than rcut[I] (n_atoms entries; 0 = none).  Arrays host or device, copied.  May be called again
 * (replaces the table).  QMC_ERR_ARG on out-of-range entries. */
int qmc_set_ecp(qmc_system* s, int n_channels, const int32_t* ch_atom, const int32_t* ch_l, const double* ch_beta,
                const double* ch_alpha, const double* rcut);
/* vnl[W] (host or device) = sum over electrons i and atoms I with |r_i - R_I| < rcut_I of
 *     sum_q (1/12) [ sum_l (2l+1) v_l(r) P_l(cos th_q) ] Psi(.., r_q, ..) / Psi(.., r_i, ..),   r_q = R_I + r O_q,
 * O_q the 12 icosahedron vertices under a uniform random rotation drawn per (walker, sweep counter, electron) from Philox
 * blocks 4 and 5 (three uniforms -> unit quaternion), cos th_q = O_q . (r_i - R_I)/r; the ratio is the determinant ratio
 * (orbital values at r_q against the electron's row of A^-T) times exp(J(r_q) - J(r_i)).  Not part of qmc_get_eloc's E_L:
 * the caller adds it.  n_pairs (may be NULL): (electron, atom) pairs inside the cut-offs, all walkers.  Call between
 * sweeps; synchronises the stream (the number of pairs is read back once per spin).  QMC_ERR_ARG without qmc_set_ecp. */
int qmc_get_vnl(qmc_walkers* w, double* vnl, uint64_t* n_pairs);

/* Several crowds per GPU: walker sets created on different streams run concurrently, and the HBM-bound stages of one
 * (k_basis, k_step) can overlap the tensor-bound contraction of another only if that persistent kernel leaves some SMs
 * free.  n_ctas (1..number of SMs; 0 = all, the default) is the grid of this set's contraction from now on (the
 * stream-K workspace is sized for all SMs, so any value fits).  Results change only through the stream-K partition
 * (rounding). */
int qmc_set_mo_ctas(qmc_walkers* w, int n_ctas);
/* qmc_sweep of n_sets walker sets ("crowds") of ONE system together: the host enqueues electron p of every set, each
 * on its own stream, before electron p + 1 of any.  Every set does exactly what qmc_sweep(set, nsteps, tau, delay_k)
 * would do -- its results do not depend on the other sets -- but sets created on DIFFERENT streams overlap on the GPU
 * (with qmc_set_mo_ctas leaving SMs free, the basis / step kernels of one crowd run beside the contraction of another:
 * +5 % at config 2 with two crowds of 128 and 124 CTAs).  Asynchronous like qmc_sweep.  Errors: as qmc_sweep;
 * QMC_ERR_ARG if the sets belong to different systems or one appears twice. */
int qmc_sweep_crowds(qmc_walkers* const* sets, int n_sets, int nsteps, double tau, int delay_k);
/* (tile, k-block) iterations of the MO contraction since creation: executed, and what the dense contraction would
 * have done; equal unless QMC_SCREEN_MO is set (counted only for screened walker sets, else both 0). */
int qmc_get_mo_work(const qmc_walkers* w, uint64_t* executed, uint64_t* dense);

/* Stage-level entry points (used by the per-stage parity tests and the per-stage roofline bench).
 * Basis functions at n_points positions: out[n][5][n_basis] = value, d/dx, d/dy, d/dz, laplacian. */
int qmc_eval_basis(const qmc_system* sys, int n_points, const double* xyz /* [n][3] */, double* out, void* cuda_stream);
/* Orbital rows at n_points positions: out[n][5][n_s] (basis kernel + FP64 contraction kernel). */
int qmc_eval_mo(const qmc_system* sys, int spin, int n_points, const double* xyz, double* out, void* cuda_stream);
/* qmc_eval_basis for callers that may not allocate device memory (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): the same basis kernel (the AO values, gradients
 * and Laplacians of one electron position) and the same export kernel, with the pre-tiled A operand -- the kernel's
 * scratch -- in a fixed array inside the library instead of a per-call allocation.
 *   xyz  DEVICE pointer, [n_points][3] doubles (the caller's; read only)
 *   out  DEVICE pointer, [n_points][5][n_basis] doubles (the caller's; value, d/dx, d/dy, d/dz, laplacian)
 * Both must be device (or managed) memory of the system's device: a host pointer is rejected with QMC_ERR_ARG.
 * Limit: ceil(5 n_points / 128) * ceil(n_basis / 32) * 36864 bytes <= QMC_NOALLOC_SCRATCH_BYTES (the used part of the
 * array is cleared on the stream first); beyond it the call returns QMC_ERR_ARG and qmc_last_error() names the largest
 * n_points this system allows.  The call makes no cudaMalloc / cudaFree and calls no allocating routine; it only
 * enqueues (memset, two kernels) on `cuda_stream` and does NOT synchronise: `out` is complete when that work is.
 * Every GPU that loads the library holds the array (8 MiB) until the process exits.  All calls on a device share it and
 * it keeps the last call's contents: two calls whose work overlaps on the GPU (different streams, no ordering between
 * them) race; calls on one stream are safe. */
#define QMC_NOALLOC_SCRATCH_BYTES (8u << 20)
int qmc_eval_basis_noalloc(const qmc_system* sys, int n_points, const double* xyz, double* out, void* cuda_stream);
/* Time `reps` launches of one stage of the move on the walker set's current state with CUDA events on its
 * stream (no state is committed).  stage: 0 = step kernel, proposal half only (effective column + drift + RNG +
 * Jastrow), 1 = basis, 2 = MO contraction, 3 = step kernel with both halves (ratio/accept with the decision
 * suppressed + proposal), 4 = delayed-update flush at full window (A^-1 unchanged: zero correction),
 * 5 = local energy.  Returns mean milliseconds per launch. */
int qmc_time_stage(qmc_walkers* w, int stage, int spin, int delay_k, int reps, double* ms_per_launch);
/* In-situ stage timing: with stride > 0, qmc_sweep brackets the three per-electron launches (fused step
 * kernel = stage 3, basis, MO contraction) of every stride-th electron, and every half-step launch (stage 0:
 * the first proposal and the last accept of a delay window), flush and local-energy evaluation, with CUDA
 * events on the walker set's stream.  qmc_get_stage_times synchronises and returns accumulated milliseconds
 * and launch counts per stage id (a "launch" of stage 4 is the whole flush = 4 kernels, of stage 5 two
 * kernels; stage 6 = one window kernel of the mid-size path, QMC_PER_ELECTRON).  stride = 0 turns it off and clears
 * the totals. */
int qmc_set_profiling(qmc_walkers* w, int stride);
int qmc_get_stage_times(qmc_walkers* w, double* ms /* [7] */, uint64_t* counts /* [7] */);
/* Lanes of a walker set (see QMC_ONE_LANE): *n_lanes = 1 or 2; walkers_per_lane[2] (may be NULL) = their sizes. */
int qmc_get_lanes(const qmc_walkers* w, int* n_lanes, int* walkers_per_lane);
/* Time on the GPU of the contraction launches that the in-situ profiling sampled (qmc_set_profiling stride > 0): every CTA
 * of such a launch stamps %globaltimer when it starts and when it ends.  The SPAN of a launch is last end - first start
 * (mean_us, min_us over the launches); the RESIDENCY of a launch is the mean over its CTAs of end - start (mean_cta_us,
 * averaged over the launches).  The kernel is persistent with equal shares per CTA, so the residency is what the launch
 * costs on the SMs it holds; with two lanes the span (and the stream events of qmc_get_stage_times) also counts the time
 * most CTAs of a launch wait for the SMs the other lane's contraction still holds.  Any of the three may be NULL;
 * *n_launches launches (at most 8192 are recorded).  Synchronises the stream(s). */
int qmc_get_mo_spans(qmc_walkers* w, double* mean_us, double* min_us, double* mean_cta_us, uint64_t* n_launches);
/* Register-resident DMMA issue-rate loop for `ms_target` milliseconds: the FP64 ceiling of this GPU as
 * it runs now (used as the roofline denominator of the contraction stages). */
int qmc_measure_fp64_peak(double ms_target, double* tflops, void* cuda_stream);
/* The random generator of the move kernels on caller-chosen inputs (reading A11: Philox4x32-10): ctr_key [n][6] =
 * counter words 0..3 and key words 0..1, out [n][4] = the four output words.  Host or device buffers; synchronous.
 * Exists so that the GPU's raw words can be compared with an independent implementation. */
int qmc_philox_words(int n, const uint32_t* ctr_key, uint32_t* out, void* cuda_stream);
/* number of kernels this library launched on this thread's calls since load (for bench.py gpu_launches) */
uint64_t qmc_launch_count(void);

const char* qmc_last_error(void);
/* Diagnostic: the last non-sticky CUDA error that an entry point found PENDING on the calling thread when it was entered
 * -- left there by an earlier runtime call of another library that shares the thread -- and dropped, with the entry point's
 * name; "" if there never was one.  (Without this, the cudaGetLastError() after our next kernel launch would report it as
 * that launch's failure.) */
const char* qmc_stale_error(void);
const char* qmc_version(void);

#ifdef __cplusplus
}
#endif
#endif /* QMC_B200_H */
