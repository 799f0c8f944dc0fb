/*
 * lm.h -- C ABI of the B200-native open-boundary RPY mobility solver ("liblm").
 *
 * The calls follow the solver interface of libMobility (arXiv 2510.02135; citations are
 * PAPER.md:LINE of the paper text this repo was built from):
 *
 *   paper                                            here
 *   -----------------------------------------------  ---------------------------------
 *   NBody("open","open","open") + initialize(         lm_create
 *     viscosity, hydrodynamicRadius, includeAngular)
 *   NBody("open","open","single_wall") +              lm_create + lm_set_wall
 *     setParameters(wallHeight)
 *   setPositions                                      lm_set_positions
 *   Mdot(forces, torques) -> (linear, angular)        lm_mdot, lm_mdot_batch
 *   sqrtMdotW()           -> (linear, angular)        lm_sqrt_mdot_w
 *   mf + dwf + drift (the sum the example forms)      lm_hydrodynamic_velocities PAPER.md:78 (eq. 9), 137-138
 *   eq. (13) steric force, eq. (14) AB time step       lm_steric_forces, lm_bd_step
 *   divM()                                            lm_thermal_drift (zero for open boundaries,
 *                                                     PAPER.md:87, 151), lm_thermal_drift_rfd (eq. 11)
 *
 * What is computed.  U = M.[F;T] with M the 6N x 6N grand mobility of eq. (7)
 * whose blocks are the free-space Rotne-Prager-Yamakawa pair tensors, summed over
 * all ordered pairs (i,j) INCLUDING j = i (self term = r -> 0 limit), with the overlap (r < 2a)
 * regularisation; and y = M^{1/2} W by the Lanczos iteration.  The closed
 * forms and every reading of the paper are listed in DESIGN.md.
 *
 * Conventions for every call
 *   - Precision is fixed per handle (LM_F32 / LM_F64); all `void*` arrays hold that type.
 *   - Arrays are interleaved xyz, length 3N: element 3*i+k is component k of particle i (the
 *     (N,3) row-major arrays of PAPER.md:128-138).  Batches are [nrhs][3N], contiguous.
 *   - Plain entry points take DEVICE pointers; the `_host` variants take HOST pointers and do
 *     the host<->device copies themselves on the given stream ("the library will
 *     automatically copy the data to the GPU").  Pinned host memory makes those copies async.
 *   - The caller owns every buffer it passes; the library never frees or retains them beyond
 *     the call (`_host` variants and Lanczos calls return only after the stream has drained).
 *     The handle owns its packed position copy, staging and Lanczos workspace (freed by
 *     lm_destroy).  Inputs and outputs must not alias.
 *   - `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).  lm_set_positions,
 *     lm_mdot and lm_mdot_batch are asynchronous on it.  lm_sqrt_mdot_w and
 *     lm_hydrodynamic_velocities (with noise) synchronise the stream internally: the Lanczos
 *     stopping test reads two scalars per iteration on the host.
 *   - Return value: LM_OK (0) or a negative LM_E_* code; lm_last_error(h) gives the message of
 *     the last failing call on that handle.  No exceptions, no global state, no CPU fallback:
 *     without a CUDA device every compute call returns LM_E_CUDA.
 *   - A handle must not be used from two threads at once.
 */
#ifndef LM_H
#define LM_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct lm_solver lm_solver; /* opaque */

enum { LM_F32 = 0, LM_F64 = 1 };

enum {
    LM_OK = 0,
    LM_E_INVALID = -1, /* bad argument: N <= 0, eta <= 0, a <= 0, unknown precision, nrhs < 1, tol <= 0; non-finite values in the
                          noise or the positions given to a Lanczos call (seen as a non-finite |z|, alpha_k or beta_k) */
    LM_E_NOPOS = -2,   /* compute call before lm_set_positions */
    LM_E_ANGULAR = -3, /* torques / angular output given but include_angular == 0, or angular output missing */
    LM_E_NULL = -4,    /* a required pointer is NULL */
    LM_E_CUDA = -5,    /* CUDA runtime error (message in lm_last_error) */
    LM_E_NOCONV = -6   /* Lanczos reached max_iter before meeting tol; the last iterate IS written */
};

/* Create a solver for N equal spheres of hydrodynamic radius a in an unbounded fluid of viscosity
 * eta.  include_angular != 0: torques are accepted and angular velocities returned (dof = 6N),
 * else forces -> linear velocities only (dof = 3N; "more efficient").  Uses the
 * current CUDA device; all later calls on the handle must run with that device current.
 * Any consistent unit system works, SI included (a = 1e-6, eta = 1e-3 ...): internally lengths are stored
 * multiplied by the power of two nearest 1/a (exact), so the kernels always see a radius of order one.
 * One caveat is the method's, not the kernels': with include_angular the 6N x 6N matrix mixes blocks
 * ~ 1/(eta a) and ~ 1/(eta a^3), so its square root (lm_sqrt_mdot_w) is well scaled only in units with a of
 * order one; in fp32 use such units for the angular noise. */
int lm_create(lm_solver** out, int precision, int64_t N, double eta, double a, int include_angular);
int lm_destroy(lm_solver* h);

/* Geometry ("open","open","single_wall") of the paper's NBody solver: a no-slip wall in
 * the plane z = wall_height, fluid above it (setParameters(wallHeight)).  enabled = 0 returns to
 * open boundaries.  Every entry point then works with the single-wall mobility
 *     M~ = B M(x~) B,
 * M = free-space RPY blocks + the wall correction of the "Swan-Brady kernel" (ref. [37]): the Faxen operators
 * applied to the image part of the half-space Green's function, which is eq. (8) exactly for spheres that do not
 * cut the wall (closed forms: DESIGN.md appendix A); x~ = the positions with every height above the wall raised to at
 * least a, B = diag(b_i) on all six components of particle i, b_i = min(1, max(h_i, 0)/a) -- the "damping matrix
 * approach" that keeps M~ symmetric positive (semi-)definite and takes a particle's mobility to zero continuously
 * as it reaches the wall (readings S18-S20).  lm_thermal_drift_rfd then estimates a
 * non-zero drift, lm_steric_forces / lm_bd_step add the particle-wall repulsion of eq. (13) with
 * r = height of the centre and d = a.  Call before lm_set_positions (it invalidates the positions). */
int lm_set_wall(lm_solver* h, int enabled, double wall_height);

/* Store the particle positions (3N).  The library keeps its own packed copy; `pos` may be reused
 * by the caller as soon as the stream has passed this call. */
int lm_set_positions(lm_solver* h, const void* pos, void* stream);

/* U = M.[F;T]  (eq. (7)).  forces / torques: 3N each or NULL; NULL means zeros
 * ("one or both of forces and torques"), but not both NULL.  lin_out: 3N, required.  ang_out: 3N,
 * required iff include_angular.  torques != NULL or ang_out != NULL without include_angular
 * -> LM_E_ANGULAR. */
int lm_mdot(lm_solver* h, const void* forces, const void* torques, void* lin_out, void* ang_out, void* stream);

/* nrhs independent right-hand sides sharing one position set: the pair geometry is evaluated
 * once per pair and applied to every force vector.  forces/torques [nrhs][3N] -> lin_out/ang_out
 * [nrhs][3N].  Same NULL rules as lm_mdot. */
int lm_mdot_batch(lm_solver* h, int nrhs, const void* forces, const void* torques, void* lin_out,
                  void* ang_out, void* stream);

/* y = M^{1/2} W by Lanczos.  noise: dof values, [3N linear | 3N angular]
 * (the caller draws W ~ N(0,1); the paper's sqrtMdotW() draws it internally).
 * tol: relative error requested of the iterate, as estimated by the stopping rule (LM_OPT_LANCZOS_RULE below;
 * DESIGN.md reading S3: the default rule's estimate is within x0.5 ... x2 of the true error).
 * lin_out 3N, ang_out 3N (iff include_angular).  iters_out: HOST int*, may be NULL.
 * LM_E_NOCONV if max_iter is reached (result still written).  The iteration also ends, with an exact result, on
 * breakdown beta_k <= eps |alpha_k| (invariant subspace): eps = 1e-6 on fp32 handles (beta_k carries fp32 rounding of
 * relative size ~1e-7), 1e-14 on fp64 handles.  A non-finite value in the noise or the positions -> LM_E_INVALID. */
int lm_sqrt_mdot_w(lm_solver* h, const void* noise, double tol, void* lin_out, void* ang_out,
                   int* iters_out, void* stream);

/* nvec independent noise vectors sharing one position set: y_q = M^{1/2} W_q, q < nvec.  The Lanczos
 * recurrences run in lockstep in groups of 4 / 2 / 1 vectors (angular or single wall: 2 / 1) so that ONE multi-right-
 * hand-side pair-kernel launch per iteration serves a whole group (the pair geometry is evaluated once
 * per pair, as in lm_mdot_batch); each vector has its own alpha, beta, Gram matrix and stopping test
 * and stops contributing to the result at its own step.  noise: [nvec][dof]; lin_out / ang_out:
 * [nvec][3N]; iters_out: HOST int[nvec] or NULL.  Each y_q equals what lm_sqrt_mdot_w returns for W_q up
 * to the summation order of the pair kernel.  LM_E_NOCONV if any vector reached max_iter. */
int lm_sqrt_mdot_w_batch(lm_solver* h, int nvec, const void* noise, double tol, void* lin_out, void* ang_out,
                         int* iters_out, void* stream);

/* out = M.[F;T] + noise_prefactor * M^{1/2} W  (+ 0 thermal drift): the right-hand
 * side of eq. (9) for dt = 1 with noise_prefactor = sqrt(2 k_B T / dt) supplied by the caller
 * (PAPER.md:116-118).  noise == NULL: deterministic part only (tol ignored). */
int lm_hydrodynamic_velocities(lm_solver* h, const void* forces, const void* torques, const void* noise,
                               double noise_prefactor, double tol, void* lin_out, void* ang_out, void* stream);

/* Host-pointer variants: identical semantics, all array pointers are HOST memory in the handle's
 * precision.  Each copies its inputs to the device, runs the device path above and copies the
 * results back, all on `stream`, and returns after the results have landed. */
int lm_set_positions_host(lm_solver* h, const void* pos, void* stream);
int lm_mdot_host(lm_solver* h, const void* forces, const void* torques, void* lin_out, void* ang_out, void* stream);
int lm_mdot_batch_host(lm_solver* h, int nrhs, const void* forces, const void* torques, void* lin_out,
                       void* ang_out, void* stream);
int lm_sqrt_mdot_w_host(lm_solver* h, const void* noise, double tol, void* lin_out, void* ang_out,
                        int* iters_out, void* stream);
int lm_hydrodynamic_velocities_host(lm_solver* h, const void* forces, const void* torques, const void* noise,
                                    double noise_prefactor, double tol, void* lin_out, void* ang_out, void* stream);

/* ---- Free-space Brownian-dynamics step built on the calls above (sec. 5.1) ----
 *
 * lm_steric_forces: forces_out = ext_forces + the soft pairwise repulsion of eq. (13)
 *   U(r) = U0 (1 + (d - r)/b) for r < d,  U0 exp((d - r)/b) for r >= d,  d = 2a (particle-particle),
 * summed over all ordered pairs j != i at the positions of the last lm_set_positions:
 *   F_i = ext_i + sum_j m(r_ij) (x_i - x_j)/r_ij,  m = -U' = U0/b (r < d), (U0/b) exp((d - r)/b) (r >= d).
 * Pairs beyond r_c = d + 20 b (fp32) / d + 40 b (fp64) are dropped (exp below the type's epsilon);
 * exactly coincident particles exert nothing on each other.  ext_forces: 3N or NULL.  forces_out: 3N.
 * Asynchronous on `stream`.  b <= 0 -> LM_E_INVALID.
 *
 * lm_bd_step: one step of the stochastic Adams-Bashforth scheme, eq. (14), in place:
 *   X^{n+1} = X^n + dt (3/2 M^n F^n - 1/2 M^{n-1} F^{n-1}) + sqrt(2 kT dt) (M^n)^{1/2} W^n
 * with F^n = lm_steric_forces(X^n; U0, b) + ext_forces (U0 == 0: no steric term), external torques
 * ext_torques (include_angular only; the spheres' orientations are not tracked), and the thermal-drift
 * terms of eq. (14) identically zero for open boundaries.  The first step after
 * lm_create / lm_bd_reset has no history and is forward Euler.  pos: 3N, read and overwritten.
 * noise: W^n, dof values as for lm_sqrt_mdot_w, or NULL (or kT == 0) for a deterministic step; tol:
 * Lanczos tolerance.  The handle keeps M^n F^n for the next step.  Synchronises the stream when noise
 * is given.  After the call the handle's positions are the new X^{n+1} (as if lm_set_positions(pos) had
 * been called).  Returns LM_E_NOCONV if Lanczos hit max_iter (the step is still taken). */
int lm_steric_forces(lm_solver* h, double U0, double b, const void* ext_forces, void* forces_out, void* stream);
int lm_bd_step(lm_solver* h, void* pos, const void* ext_forces, const void* ext_torques, const void* noise,
               double dt, double kT, double U0, double b, double tol, void* stream);
int lm_bd_step_host(lm_solver* h, void* pos, const void* ext_forces, const void* ext_torques, const void* noise,
                    double dt, double kT, double U0, double b, double tol, void* stream);
int lm_bd_reset(lm_solver* h);                        /* forget the Adams-Bashforth history */
/* lm_bd_step with the thermal-drift terms of eq. (14) ("we also include the thermal drift term in the
 * deterministic part of the time stepping scheme as it has non-zero mean"): the deterministic velocity becomes
 *   v^n = M^n F^n + kT * (1/rfd_delta) [ M(X^n + rfd_delta W~/2) - M(X^n - rfd_delta W~/2) ] W~,
 * ONE random-finite-difference sample of kT d/dX . M^n (eq. (11)) with W~ = rfd_noise (3N values ~ N(0,1),
 * independent of `noise`), and enters the Adams-Bashforth combination 3/2 v^n - 1/2 v^{n-1} as a whole.  Two more M.F
 * applies per step.  rfd_noise == NULL (or kT == 0): exactly lm_bd_step.  Meant for lm_set_wall geometries; for open
 * boundaries the term has zero mean. */
int lm_bd_step_rfd(lm_solver* h, void* pos, const void* ext_forces, const void* ext_torques, const void* noise,
                   const void* rfd_noise, double rfd_delta, double dt, double kT, double U0, double b, double tol, void* stream);
int lm_bd_step_rfd_host(lm_solver* h, void* pos, const void* ext_forces, const void* ext_torques, const void* noise,
                        const void* rfd_noise, double rfd_delta, double dt, double kT, double U0, double b, double tol, void* stream);

/* ---- Thermal drift  d/dX . M  (the paper's divM) ----
 * lm_thermal_drift: the library default for open boundaries -- the divergence of the free-space mobility
 * is identically zero ("the default implementation simply sets the thermal drift to
 * zero"): writes zeros to lin_out (3N) and ang_out (3N, iff include_angular).  After lm_set_wall(h, 1, ...) the
 * divergence is not zero and the call returns LM_E_INVALID, writing nothing: use lm_thermal_drift_rfd
 * (or lm_bd_step_rfd) there.
 * lm_thermal_drift_rfd: ONE realisation of the random finite difference of eq. (11),
 *   (1/delta) [ M(X + delta W/2) W - M(X - delta W/2) W ],
 * at the positions X of the last lm_set_positions (which stay set), W = noise: 3N values ~ N(0,1)
 * acting as forces (the mobility depends on positions only); rows: linear (lin_out) and,
 * with include_angular, angular (ang_out) velocities.  Its average over realisations estimates d/dX . M,
 * zero here; it is exported because eq. (11) is part of the paper's generic machinery and because it
 * costs exactly two M.F applies.  delta <= 0 -> LM_E_INVALID.  Asynchronous on `stream`. */
int lm_thermal_drift(lm_solver* h, void* lin_out, void* ang_out, void* stream);
int lm_thermal_drift_rfd(lm_solver* h, const void* noise, double delta, void* lin_out, void* ang_out, void* stream);

/* ---- Row-sharded applies across GPUs (one process per GPU) ----
 * The target rows of M.[F;T] are independent, so G ranks can each compute a block of rows against ALL
 * sources.  SPMD with replicated inputs and outputs: every rank creates a handle for the same N, calls
 * the same functions in the same order with the same positions / forces / noise, computes only its row
 * block  [r B, min((r+1) B, N)),  B = ceil(N / G)  (lm_dist_row_block), and one grouped ncclAllGather
 * per pair-kernel launch (over NVLink / NVSwitch) completes every output on every rank.  All entry points
 * (lm_mdot*, lm_sqrt_mdot_w*, lm_hydrodynamic_velocities, lm_thermal_drift_rfd, lm_steric_forces,
 * lm_bd_step) then work unchanged; only the O(N) vector kernels are replicated.  Ranks must run the
 * same GPU model.  The Lanczos stopping verdict acted upon is rank 0's, broadcast after every iteration, so ranks
 * cannot part ways even if their scalars ever differed in the last bit.
 *   lm_dist_unique_id : 128-byte NCCL unique id (host buffer); call on ONE rank and broadcast it to the
 *                       others by any means (torch.distributed, MPI, a file).
 *   lm_dist_init      : collective; creates this handle's communicator (current CUDA device) and fixes
 *                       its row block.  nranks = 1 is allowed.  NCCL is loaded at run time (the libnccl
 *                       already in the process, else the system one); LM_E_CUDA if it cannot be.
 *   lm_dist_row_block : host-only helper, the row block of `rank` (needs no GPU).
 *   lm_mdot_rows      : WITHOUT a communicator: compute only rows [row_begin, row_begin + row_count) of
 *                       lm_mdot and write them at their places in the full-length outputs (the other
 *                       entries are left untouched) -- the building block for a caller's own sharding. */
int lm_dist_row_block(int64_t N, int nranks, int rank, int64_t* row_begin, int64_t* row_end);
int lm_dist_unique_id(void* out128);
int lm_dist_init(lm_solver* h, int nranks, int rank, const void* unique_id128);
int lm_mdot_rows(lm_solver* h, int64_t row_begin, int64_t row_count, const void* forces, const void* torques,
                 void* lin_out, void* ang_out, void* stream);

/* Lanczos controls and introspection.
 * lm_set_option: per-handle switches (no environment variables, no global state):
 *   LM_OPT_LANCZOS_RULE       LM_RULE_ESTIMATE (default) | LM_RULE_STEP -- what `tol` bounds (reading S3; the
 *                             paper states no rule).  With s_k = |y_k - y_{k-1}| / |y_{k-1}|:
 *                             STEP: stop at the first k >= 2 with s_k <= tol (the rule of ref. [35]; it under-states the
 *                             true error by the factor rho/(1 - rho) when the steps shrink slowly: measured 15-20 x tol
 *                             at N = 131072, phi = 5 %);  ESTIMATE: stop at the first k >= 3 with
 *                             e_k = max(s_k, s_{k-1}) max(1, rho/(1 - rho)) <= tol, rho = the step ratio per iteration
 *                             over the trailing min(10, (k-1)/2) steps, capped at 0.98 -- measured within x0.5 ... x2
 *                             of the true relative error from N = 12 to N = 131072.
 *   LM_OPT_GRAPH_REPLAY       1 (default) | 0: replay short applies / Lanczos iterations as CUDA graphs, or launch
 *                             every kernel directly.
 *   LM_OPT_SHARE_FIRST_APPLY  1 (default) | 0: in lm_hydrodynamic_velocities / lm_bd_step, M.[F;T] rides along with the
 *                             first Lanczos apply in one 2-right-hand-side launch, or is a launch of its own.
 *   LM_OPT_SMALL_KERNEL       1 (default): small applies (N up to a few thousand) run as ONE launch of the cluster kernel
 *                             of csrc/rpy_small.cuh (reads the caller's arrays, sums the source splits through
 *                             distributed shared memory) where the launch chooser prefers it | 0: never (always pack,
 *                             pair kernel, reduce) | (cluster << 8 | warps), cluster and warps in {1, 2, 4, 8}: always,
 *                             with that shape (plan sweeps; a shape whose shared memory does not fit falls back to the
 *                             general path and a cluster size above what the device can co-schedule is clamped:
 *                             lm_pair_kernel_name / lm_pair_launch_config report what the next apply will really run --
 *                             check them after forcing a shape).  Same results up to summation order (PAPER.md:435-437:
 *                             the small-N regime where launch overhead, not arithmetic, sets the time).  An apply on
 *                             this path takes no host decision and synchronises nothing, so a caller may capture
 *                             batches of lm_mdot / lm_mdot_batch calls into a CUDA graph of their own and replay them.
 *   LM_OPT_J_SPLITS           0 (default): the launch chooser sizes the grid | s > 0: the general path deals the sources to
 *                             exactly s j-splits (clamped to what the problem allows) -- for plan sweeps; results are
 *                             the same up to summation order.
 *   LM_OPT_GATHER_IN_PLACE    1 (default): a row-sharded apply (lm_dist_init) whose row blocks tile [0, N) exactly (the
 *                             number of ranks divides N) all-gathers straight into the caller's output arrays | 0: always
 *                             through the handle's own all-gather buffers and a device-to-device copy (the path taken
 *                             anyway when the last block is short).
 *   LM_OPT_ACCUMULATE_F64     0 (default) | 1, fp32 handles only: mixed precision -- fp32 pair arithmetic, but the packed fp32
 *                             accumulators are flushed every 32 sources into fp64 totals, the j-split partial sums are
 *                             kept and added in fp64, and each result is rounded to fp32 once.  The error of an fp32
 *                             apply is dominated by the length of its fp32 summation runs: measured on config 3
 *                             (N = 131072) rel-L2 5.5e-7 -> 1.6e-7, the floor set by the fp32 pair arithmetic being 0.8e-7,
 *                             for 2.7 % more time.  Always the general path (no one-launch kernel).
 * lm_lanczos_history: what the last Lanczos call measured for noise vector `vec` of its (last) group: for iteration
 *   i + 1 (i < cap): alpha[i], beta[i], step[i] = s_{i+1} (NaN for i = 0), estimate[i] = e_{i+1} (NaN for i < 2; NaN
 *   throughout under LM_RULE_STEP).  Any output may be NULL.  Returns the number of iterations recorded. */
enum { LM_RULE_ESTIMATE = 0, LM_RULE_STEP = 1 };
enum { LM_OPT_LANCZOS_RULE = 0, LM_OPT_GRAPH_REPLAY = 1, LM_OPT_SHARE_FIRST_APPLY = 2, LM_OPT_SMALL_KERNEL = 3, LM_OPT_J_SPLITS = 4, LM_OPT_GATHER_IN_PLACE = 5, LM_OPT_ACCUMULATE_F64 = 6 };
int lm_set_option(lm_solver* h, int option, int value);
int lm_set_max_iter(lm_solver* h, int max_iter);     /* default 100; 1 <= max_iter <= 1000 */
int lm_last_iterations(const lm_solver* h);           /* iterations of the last Lanczos call (or < 0) */
int lm_lanczos_history(const lm_solver* h, int vec, int cap, double* alpha, double* beta, double* step, double* estimate);
const char* lm_last_error(const lm_solver* h);        /* never NULL; "" if the last call succeeded */

/* Launch accounting for benchmarks.  Counters accumulate from lm_create or the last reset.
 * With profiling on (lm_set_profiling(h, 1)) every pair-kernel launch is bracketed by CUDA events
 * on its stream; lm_get_stats then waits for those events and reports their summed time.
 * pair_kernel_launches: O(N^2) kernel launches; aux_launches: O(N) pack / reduce / vector kernels;
 * pair_kernel_ms: summed device time of the pair kernel (0 unless profiling);
 * pairs: ordered (i,j) pair evaluations performed (N^2 per launch, all right-hand sides share it). */
int lm_set_profiling(lm_solver* h, int on);
int lm_reset_stats(lm_solver* h);
int lm_get_stats(lm_solver* h, int64_t* pair_kernel_launches, int64_t* aux_launches, double* pair_kernel_ms,
                 double* pairs);

/* The launch configuration the next lm_mdot_batch(nrhs) would use: grid = i_tiles x j_splits CTAs
 * of `block` threads, `targets_per_thread` targets each, `smem_bytes` dynamic shared memory.  For the one-launch
 * small-N kernel j_splits is the cluster size (the CTA's block / 32 warps split the sources further). */
int lm_pair_launch_config(lm_solver* h, int nrhs, int* i_tiles, int* j_splits, int* block,
                          int* targets_per_thread, int* smem_bytes);

/* Name of the O(N^2) kernel that launch would run (static storage): "rpy_small_kernel" (one launch per apply, small N,
 * LM_OPT_SMALL_KERNEL) or "rpy_pair_kernel" (pack, pair kernel, split-j reduce); "" for an unsupported nrhs. */
const char* lm_pair_kernel_name(lm_solver* h, int nrhs);

/* ---- M.F without any allocation (csrc/lm_static.cu) ----
 * For callers that cannot let a library allocate device memory: an engine or framework allocator that claimed the whole
 * card for its own arena (a later cudaMalloc fails or eats its headroom), a latency-tuned stepping loop (cudaMalloc and
 * cudaFree synchronise the whole device at a moment the caller does not choose), a process held to a fixed device-memory
 * budget.  A handle (lm_create) owns cudaMalloc'ed buffers and may grow them on a later call; this call owns none:
 *   lm_mdot_static : lin_out = M_uF . forces for N equal spheres in free space (the translational block of lm_mdot:
 *       PAPER.md:173, eq. (8)), precision LM_F32 or LM_F64, on the CURRENT device.  positions, forces,
 *       lin_out: DEVICE pointers, 3N reals of that precision, interleaved xyz, owned by the caller; inputs are not
 *       modified; lin_out is overwritten.  Asynchronous on `stream`.  Results equal lm_mdot's up to summation order.
 *       It calls no cudaMalloc / cudaFree / allocating library routine, on the first call or later.  Its scratch (packed
 *       positions and forces, j-split partial sums) is a static device array of LM_STATIC_SCRATCH_BYTES inside the
 *       library image: every GPU the process touches with liblm loaded holds those bytes until exit.
 *       Limit: 1 <= N <= LM_STATIC_MAX_N, otherwise LM_E_INVALID and nothing is launched.  Other errors: LM_E_INVALID
 *       (precision, eta, a), LM_E_NULL (a NULL pointer), LM_E_CUDA.  lm_mdot_static_error() gives the message of the
 *       calling thread's last lm_mdot_static call ("" after success; static thread-local storage).
 *       Sharing: ONE array per GPU serves every call.  Calls whose kernels may overlap on the GPU (two streams, two
 *       unordered host threads) race on it; order them on one stream or with events.  The array keeps the previous call's
 *       contents; a call reads only what it has itself written, so nothing needs clearing between calls.
 *       First call on each device: one-time set-up with that device current (resolves the array's device address with
 *       cudaGetSymbolAddress, sets kernel attributes, queries occupancy).  Make that first call before any stream
 *       capture begins; later calls only launch three kernels (pack, pair kernel, split reduce).
 *   lm_mdot_static_max_n : LM_STATIC_MAX_N, for callers that bind at run time. */
#define LM_STATIC_MAX_N 65536
#define LM_STATIC_SCRATCH_BYTES (16u << 20)
int lm_mdot_static(int precision, int64_t N, double eta, double a, const void* positions, const void* forces,
                   void* lin_out, void* stream);
int64_t lm_mdot_static_max_n(void);
const char* lm_mdot_static_error(void);

/* Library version string (static storage). */
const char* lm_version(void);

#ifdef __cplusplus
}
#endif
#endif /* LM_H */
