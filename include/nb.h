/*
 * nb.h -- C-ABI of libnb: the hot path of the HiGPUs method (arXiv 1207.2367) on one B200.
 *
 * What the library computes (citations are PAPER.md line + section/equation; "Gn" are the
 * readings of DESIGN.md section 3 where the paper is silent or garbled):
 *
 *   6th-order Hermite integration with hierarchical block time steps of the softened
 *   Newtonian N-body problem (Eq. 2; section 3), G = 1.
 *   Per block step:  next block (Table 1 row 1)  ->  predictor for all N
 *   (Eq. 3-7)  ->  evaluation of acceleration, jerk and snap of the m active
 *   particles against all N predicted particles (Eq. 8-10; split over j when
 *   m is small)  ->  corrector (Eq. 11-14)  ->  new
 *   power-of-two time steps (Eq. 15-16).  Diagnostics: Eq. 20.
 *
 * Conventions
 *   - All arithmetic is IEEE binary64 (unless nb_set_precision selects the paper's mixed
 *     evaluation).  Every step runs in CUDA kernels on the device the
 *     context was created on; there is no CPU fallback.  A call made without a usable
 *     CUDA device fails with NB_ECUDA.
 *   - Pointers marked [dev|host] may be device pointers or host pointers (pinned host memory
 *     makes the copy asynchronous); the library moves the data with cudaMemcpyAsync(...,
 *     cudaMemcpyDefault) on the context stream and never keeps the pointer.  Pointers
 *     marked [host] are plain host memory written before the call returns.
 *   - Layouts are row-major: pos/vel/acc/jerk/snap are [n][3] doubles, mass/t/dt are [n].
 *   - Ownership: the library copies its inputs and owns every internal buffer; the caller
 *     owns every argument buffer.  Nothing returned points into library memory except the
 *     string of nb_last_error (valid until the next call on that context).
 *   - Errors: every call returns NB_OK (0) or a negative code; nothing throws, aborts or
 *     prints.  nb_last_error(ctx) describes the last failure on that context.
 *   - Ordering: calls enqueue work on the context stream.  [dev] outputs are valid after
 *     that stream is synchronised; calls that return [host] scalars (nb_next_block,
 *     nb_energy, nb_get_stats, nb_run_until) synchronise it themselves.  A context is not
 *     thread-safe.
 */
#ifndef NB_H
#define NB_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct nb_ctx nb_ctx; /* opaque; owns all device state */

enum {
    NB_OK = 0,
    NB_EINVAL = -1, /* bad argument: N < 1, null pointer, eps < 0, eta <= 0, n_active out of [0, N],
                       t earlier than the current time, limits not powers of two ...              */
    NB_ESTATE = -2, /* wrong call order, e.g. nb_correct_and_step before nb_force                 */
    NB_ECUDA = -3,  /* a CUDA runtime call or kernel launch failed (message in nb_last_error)     */
    NB_ENOMEM = -4  /* device or host allocation failed                                           */
};

/* Create a context for N particles at t = 0 (state of a particle: PAPER.md:54-56).
 *   pos, vel [dev|host] [N][3];  mass [dev|host] [N];  eps >= 0 softening (Eq. 2);
 *   eta > 0 accuracy parameter of Eq. 15;  cuda_stream: a cudaStream_t (NULL =
 *   the legacy default stream) on which every later call of this context enqueues.
 * After nb_init: t_i = 0, all derivatives 0, the predicted arrays hold (pos, vel, a_pred = 0)
 * so nb_force may be called at once (force-only use); time-step limits are the paper's
 * 2^-25 and 2^-3, eta_init = 0.01 (G8).  *ctx is NULL on failure.
 * nb_init does NOT run the start-up S0 (SURVEY.md section 8(b) sketched it inside nb_init): S0 is
 * nb_startup, because it costs two full-N evaluations (2 N^2 pairs: 6 s at N = 2^20, 6 min at 2^23)
 * that force-only use (configs 3, 4) and a context that loads a checkpoint (nb_set_full_state) must
 * not pay, and because nb_set_limits / nb_set_precision must be able to act before it.
 * nb_run_until / nb_run_steps run it implicitly when it has not run.                        */
int nb_init(nb_ctx **ctx, int64_t N, const double *pos, const double *vel, const double *mass,
            double eps, double eta, void *cuda_stream);

/* Time-step limits (powers of two, dt_min <= dt_max) and the start-up
 * parameter eta_init (G8).  Only before nb_startup.                                         */
int nb_set_limits(nb_ctx *ctx, double dt_min, double dt_max, double eta_init);

/* Start-up S0 (paper silent; G8): pass 1 evaluates a, jerk with a_pred = 0, pass 2 evaluates
 * a, jerk, snap with a_pred = a; crackle = 0; dt_i = pow2floor(eta_init * min(|a|/|jerk|,
 * sqrt(|a|/|snap|))) clamped to the limits.  Two full-N evaluations (2 N^2 pairs).
 * NB_ESTATE when a proper j-slice is set (nb_set_j_range): a sliced start-up needs the exchange
 * between its passes and is driven call by call with nb_startup_commit.                      */
int nb_startup(nb_ctx *ctx);

/* The two commits of nb_startup as separate calls, for callers that must exchange the evaluated
 * values between the passes (j-sharding, nb_set_j_range):  nb_predict(ctx, 0) ->
 * nb_force(NULL, N) -> [exchange] -> nb_startup_commit(ctx, 1)  (a_pred <- a)  ->
 * nb_force(NULL, N) -> [exchange] -> nb_startup_commit(ctx, 2)  (commit a, jerk, snap; crackle = 0;
 * initial dt; the context is started).                                                       */
int nb_startup_commit(nb_ctx *ctx, int pass);

/* Table 1 row 1: t_next = min_i(t_i + dt_i) and the ascending list of the
 * particles with t_i + dt_i == t_next, built on the device.  Returns both [host].           */
int nb_next_block(nb_ctx *ctx, double *t_next, int64_t *n_active);

/* Copy the scheduler's current active list (ascending, int32) to idx [dev|host] [n_active]. */
int nb_get_active(nb_ctx *ctx, int32_t *idx);

/* Predictor, Eq. 3-7 for ALL N particles to time t, interval t - t_i (G2).
 * t must be >= every t_i (i.e. >= the time of the last committed block).                    */
int nb_predict(nb_ctx *ctx, double t);

/* Evaluation, Eq. 8-10 with the Eq. 2 softening in every r_ij^2 (G3), of
 * the particles active_idx[0..n_active) against all N predicted particles (j = i excluded).
 *   active_idx [dev|host] int32 [n_active], values in [0, N), or NULL:
 *       NULL with n_active == N  -> all particles in index order;
 *       NULL otherwise           -> the scheduler's set (n_active must equal its size).
 *   acc, jerk, snap [dev|host] [n_active][3], each may be NULL (not returned).
 * The evaluated values are also kept inside the context for nb_correct_and_step.
 * Needs valid predicted data: after nb_init, nb_set_pred, nb_predict or nb_startup.
 * The indices are NOT range-checked on the hot path (an index outside [0, N) reads outside the
 * predicted stream); nb_set_debug(ctx, 1) adds a device-side check that makes the call return
 * NB_EINVAL, naming the first offending slot, before anything is evaluated.
 * With a proper j-slice set (nb_set_j_range) the values are slice partials: nb_correct_and_step
 * refuses them until nb_set_forces has stored the reduced buffer.                            */
int nb_force(nb_ctx *ctx, const int32_t *active_idx, int64_t n_active, double *acc,
             double *jerk, double *snap);

/* Corrector Eq. 11-14 for the set just evaluated (must be the scheduler's
 * set, predicted to its t_next), end-point a^(3..5) of the quintic Hermite interpolant (G6),
 * commit (a, jerk, snap <- evaluated, crackle <- a^(3)(t1), t_i <- t_next; G7, G16), then
 * the new step of Eq. 15-16 with p = 6 quantised to a power of two
 * (G9).                                                                       */
int nb_correct_and_step(nb_ctx *ctx);

/* Block steps (next block, predict, force, correct) repeated while the next block time is
 * <= t_end; bit-identical results to the call sequence.  n_steps [host] (may be NULL) receives
 * the number of block steps taken.  Runs nb_startup first if it has not run.  By default the
 * loop is driven from the device (nb_set_loop_mode): batches of block steps replayed as one
 * CUDA graph whose kernels read (t_next, n_active) from device memory; the host synchronises
 * once per batch instead of once per step (Table 1 rows 1, 2, 6, 9 disappear). */
int nb_run_until(nb_ctx *ctx, double t_end, int64_t *n_steps);

/* Exactly `n` block steps (config 5: "advance 8 block steps").  Optional per-step log
 * [host]: log_t[k] = block time, log_m[k] = active count, log_ms[k] = device time of the
 * step in milliseconds (CUDA events); each may be NULL.                                     */
int nb_run_steps(nb_ctx *ctx, int64_t n, double *log_t, int64_t *log_m, float *log_ms);

/* Diagnostics at the current time (Eq. 2; Eq. 20):
 * out [host] = {E, K, W, Px, Py, Pz, Lx, Ly, Lz}; W = -sum_{i<j} m_i m_j/sqrt(r_ij^2+eps^2).
 * Particles not at the current time are predicted to it first (Eq. 3-7), into a scratch buffer:
 * the predicted arrays that nb_force reads (nb_predict, nb_set_pred, nb_set_pred_acc) are left
 * untouched.  With eps = 0 two DISTINCT particles at the same position are outside the domain
 * (G12); such a pair contributes nothing instead of an infinite W.                           */
int nb_energy(nb_ctx *ctx, double out[9]);

/* Copy out the committed state; any pointer may be NULL.  pos, vel [dev|host] [N][3];
 * t, dt [dev|host] [N].                                                                     */
int nb_get_state(nb_ctx *ctx, double *pos, double *vel, double *t, double *dt);

/* Committed derivatives: acc, jerk, snap, crackle [dev|host] [N][3]; any may be NULL.       */
int nb_get_derivs(nb_ctx *ctx, double *acc, double *jerk, double *snap, double *crackle);

/* Predicted arrays of the last nb_predict: pos, vel, acc [dev|host] [N][3]; any may be NULL.*/
int nb_get_pred(nb_ctx *ctx, double *pos, double *vel, double *acc);

/* Force-only use (configs 3, 4; G8): overwrite the predicted accelerations a_j that the
 * snap term of Eq. 10 needs.  acc_pred [dev|host] [N][3].                                   */
int nb_set_pred_acc(nb_ctx *ctx, const double *acc_pred);

/* Force-only use: overwrite all predicted data (pos, vel, acc [dev|host] [N][3]; acc may be
 * NULL = zeros) without touching the committed state.                                       */
int nb_set_pred(nb_ctx *ctx, const double *pos, const double *vel, const double *acc);

/* Checkpoint in/out of the complete integrator state, 21 doubles per particle:
 * state [dev|host] [N][21] = {m, t, dt, r[3], v[3], a[3], jerk[3], snap[3], crackle[3]}.
 * nb_set_full_state marks the context as started at t_now = max_i t_i.                      */
int nb_get_full_state(nb_ctx *ctx, double *state);
int nb_set_full_state(nb_ctx *ctx, const double *state);

/* Counters since nb_init: out [host] = {block steps, pair interactions evaluated (as a
 * double), kernels launched, current time}; hist [host] (may be NULL) [64]: number of block
 * steps with floor(log2(n_active)) == b (Fig. 7 analogue).               */
int nb_get_stats(nb_ctx *ctx, double out[4], int64_t hist[64]);

/* Tuning knobs of the evaluation kernel, for the split-j on/off experiment (PAPER.md:256,
 * Fig. 8): split = 0 chooses the number of j-splits automatically (default), split >= 1
 * forces it.  jlanes = 0 automatic, else lanes of a warp that share one i (1, 2, 4 .. 32).
 * The resident loops (nb_set_loop_mode 3, 4) split the j-range by construction (one piece per CTA) and honour
 * jlanes only.                                                                               */
int nb_set_tuning(nb_ctx *ctx, int split, int jlanes);

/* j-sharding across GPUs (the paper's decomposition; Table 1 row 7): every
 * process holds the whole (replicated) state, evaluates the active particles against its own
 * slice [j_begin, j_end) of the predicted particles only, and the partial (acc, jerk, snap) of
 * all processes are summed before the corrector:
 *     nb_next_block -> nb_predict -> nb_force(NULL, m, ...) -> nb_get_forces(buf)
 *     -> all-reduce(sum) of buf over the processes -> nb_set_forces(buf) -> nb_correct_and_step.
 * j_begin and j_end must be multiples of 128 (j_end may also be N).  Default [0, N).  With a
 * proper slice set, nb_run_until / nb_run_steps refuse (NB_ESTATE): the exchange is the caller's. */
int nb_set_j_range(nb_ctx *ctx, int64_t j_begin, int64_t j_end);

/* The (acc, jerk, snap) of the set just evaluated, as one contiguous buffer the caller can
 * all-reduce: buf [dev|host] [9][n_eval] = {ax, ay, az, jx, jy, jz, sx, sy, sz} x n_eval.
 * nb_set_forces stores a buffer of that layout back as the evaluated values that
 * nb_correct_and_step will use.                                                             */
int nb_get_forces(nb_ctx *ctx, double *buf);
int nb_set_forces(nb_ctx *ctx, const double *buf);

/* Arithmetic of the evaluation step.  0 (default): IEEE binary64 throughout.  1: the paper's own
 * mixed scheme (section 5.7): predicted data stay double, the nine differences
 * r_ij, v_ij, a_ij are formed in double and rounded to float, the pair arithmetic of Eq. 8-10 is
 * float, pair terms are summed in float within a j-tile (at most 128 j) and the tile sums in double
 * (reading G27).  2: the same, but the acceleration and jerk terms of every pair are added in
 * double -- 9 + 6 = the 15 double-precision operations per pair that PAPER.md:301 counts (reading G27b).
 * Relative error of a force ~1e-7 of sum_j |pair term| instead of ~1e-16; everything else (predictor,
 * corrector, time steps, energy) stays binary64.                                            */
int nb_set_precision(nb_ctx *ctx, int mode);

/* Debug switch (Errors): 1 = nb_force range-checks a caller-supplied
 * active_idx on the device (one extra small kernel and a stream synchronisation per call) and
 * returns NB_EINVAL instead of reading out of bounds; 0 (default) = no check, no cost.       */
int nb_set_debug(nb_ctx *ctx, int on);

/* Driver of nb_run_until / nb_run_steps:
 *   0  the host issues nb_next_block / nb_predict / nb_force / nb_correct_and_step per step;
 *   1  device-driven CUDA-graph batches (kernels read (t_next, n_active) from device memory);
 *   2  the same graph with its kernels chained by programmatic dependent launch (measured slower than
 *      plain graph edges on B200, kept for comparison);
 *   3  ONE kernel resident on one thread-block cluster (up to 16 SMs) keeps the whole system in shared
 *      memory and runs every step, its phases separated by the hardware cluster barrier: no launch, no host
 *      round trip and no trip to L2 per step (the small blocks).  Serves N <= 2048 (NB_EINVAL
 *      above).
 *   4  ONE cooperative kernel on ALL SMs, one CTA per SM, each keeping its share of the particles (state and
 *      predicted records) in shared memory; a block step costs two grid barriers and a few reads of small
 *      L2-resident buffers instead of three kernels.  Serves N up to 704 particles per SM (104 192 on a B200;
 *      NB_EINVAL above).  Block steps with 2048 or more active particles are handed, one at a time, to the
 *      call sequence of mode 0 (the streaming evaluation kernel at full occupancy) and the kernel is launched again.
 * Modes 0, 1, 2 give bit-identical states.  Modes 3 and 4 add the pair terms of a particle in their own fixed order
 * (per owner CTA, then over the CTAs), so their results agree with modes 0-2 to rounding, not bit for bit (any order
 * is correct, G18), and are bit-reproducible from run to run.
 * Default: 3 for N <= 1024, 4 while the system fits the shared memory of the device, else 1.  nb_run_steps with a
 * per-step log always uses 0.                                                                 */
int nb_set_loop_mode(nb_ctx *ctx, int device_driven);

/* The driver nb_run_until / nb_run_steps will use on this context (0..4, as above) -> *mode [host].          */
int nb_get_loop_mode(nb_ctx *ctx, int *mode);

/* What the last nb_force launched: out [host] = {threads per CTA, j-lanes per i, j-splits,
 * CTAs, j-tile length}.                                                                     */
int nb_get_launch(nb_ctx *ctx, int64_t out[5]);

/* DFMA-only micro-benchmark on the context's device: `iters` dependent-free FMA rounds on
 * every SM; returns achieved FP64 flop/s in *flops [host] and the kernel time in *ms [host].
 * It is the measured denominator quoted beside the nominal FP64 peak. */
int nb_probe_fp64_peak(nb_ctx *ctx, int64_t iters, double *flops, float *ms);

/* The evaluation of nb_force (Eq. 8-10, Eq. 2 softening; j-splits as in PAPER.md:108-114) for
 * callers that cannot allocate -- code under CUDA-graph capture, serving loops, harnesses that forbid cudaMalloc.
 * No context: the call packs the caller's arrays into the record layout, evaluates and sums the j-splits in a
 * fixed 16 MiB `static __device__` array inside the library (every GPU that loads libnb.so holds it until the process
 * exits), and calls no cudaMalloc, cudaFree or allocating routine.  Binary64 only.
 *   N in [1, NB_STATIC_MAX_N]; larger N is refused with NB_EINVAL (use nb_init + nb_force).
 *   pos, vel [dev] [N][3], mass [dev] [N]; acc_pred [dev] [N][3] or NULL (= zeros): the predicted a_j of Eq. 10.
 *   eps >= 0.  active_idx [dev] int32 [n_active], values in [0, N), not range-checked; NULL = all N in index order
 *   (n_active must be N).  acc, jerk, snap [dev] [n_active][3], each may be NULL.  ALL pointers are DEVICE pointers.
 *   cuda_stream: a cudaStream_t on the CURRENT device (NULL = legacy default stream); the kernels are enqueued on
 *   it and the call returns without synchronising.  err [host] (may be NULL): receives the message of a failure,
 *   at most err_len bytes.
 * The first call on a device also does the one-time set-up for that device (symbol address, SM count, occupancy
 * query; nothing allocates): make it before a capture starts -- n_active = 0 does the set-up and nothing else.
 * The array is shared by all calls of the process on that device and keeps the last call's contents; the call
 * rewrites whatever it reads (padding records are zeroed every time).  Calls that OVERLAP on the GPU (two
 * streams, two graphs replayed at once) race on it: serialise them.  Results: the split rule sees this array's
 * partial-sum budget instead of a context's, so the number of j-splits, hence the summation order, may differ from
 * nb_force's: equal to rounding (G18), bit-reproducible from call to call.           */
#define NB_STATIC_MAX_N 65536
int nb_force_static(int64_t N, const double *pos, const double *vel, const double *acc_pred, const double *mass,
                    double eps, const int32_t *active_idx, int64_t n_active, double *acc, double *jerk, double *snap,
                    void *cuda_stream, char *err, int64_t err_len);

const char *nb_last_error(const nb_ctx *ctx);
void nb_free(nb_ctx *ctx);

/* Library version string, e.g. "nb-b200 0.3 (sm_100a)".                                     */
const char *nb_version(void);

#ifdef __cplusplus
}
#endif
#endif /* NB_H */
