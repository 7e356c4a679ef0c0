// nb_internal.cuh -- context layout and kernel-launcher declarations shared by the .cu files
// of libnb.  Nothing here is visible through the C-ABI (include/nb.h).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <limits.h>

#include "../../include/nb.h"

namespace nb {

// ---------------------------------------------------------------------------------------
// Data layout in HBM.
//   committed state : SoA, one array of Npad doubles per scalar; 3-vectors are three
//                     consecutive planes x|y|z of Npad doubles each.
//   predicted stream: one packed record of REC = 10 doubles per particle
//                     {x, y, z, vx, vy, vz, ax, ay, az, m}; a j-tile of TJ particles is one
//                     contiguous 80*TJ-byte block that a single bulk copy (TMA, UBLKCP)
//                     moves into shared memory.  Records N..Npad-1 are all-zero (m = 0), so
//                     they contribute exactly nothing to any sum.
//   evaluated forces: f1[c][k], c = 0..8 (ax ay az jx jy jz sx sy sz), k = slot in the
//                     active list, plane stride Npad.
// ---------------------------------------------------------------------------------------
constexpr int REC = 10;        // doubles per predicted record
constexpr int TILE_ALIGN = 128; // Npad is a multiple of this; every j-tile length divides it

struct Sched {                 // device-written, host-read (pinned, mapped)
    double t_next;
    long long n_active;
};

// Launch geometry of one evaluation: which kernel variant, how many
// lanes share one i (JL), how many j-splits (S) of how many tiles each (tps), how many i-blocks.
struct ForceGeom {
    int JL;       // lanes of a warp that share one i (1: one i per thread; 2..32 when the set is small)
    int S, tps;   // j-splits, tiles per split
    int n_ib;     // i-blocks of NT_E / JL particles
    int mpad;     // set size rounded up to 32 (row length of the split-major partial buffer)
    int pad_;
};

// Control block of the device-resident block-step loop (nb_graph.cu): lives in device memory,
// written by the kernels of a step, copied to a pinned mirror once per graph launch.
struct StepCtl {
    // Double-buffered by the parity p of the step inside a batch (a kernel argument fixed at capture):
    // tmin[p] = bits of min_i(t_i + dt_i) of THIS step, complete when the step starts; tmin[1 - p]
    // collects the minimum for the next step.  cnt[p] = append counter of this step's active list.
    unsigned long long tmin[2];
    int cnt[2];
    unsigned int work;             // next work item of the persistent evaluation kernel (dynamic distribution)
    int done;                      // set when the next block lies beyond t_end / no steps left
    unsigned int ticket;           // blocks of the gather kernel that have finished (the last one chooses the geometry)
    double t_next, t_end, t_now;
    long long n_active, steps_left, n_steps;
    double n_pairs;
    ForceGeom g;
    long long hist[64];
};

#ifdef __CUDACC__
// Programmatic dependent launch (sm_90+, PTX griddepcontrol), loop mode 2: the kernels of the
// device-driven loop are launched with cudaLaunchAttributeProgrammaticStreamSerialization, let their
// successor start launching at once (pdl_trigger) and wait for the COMPLETION of their predecessor
// (pdl_wait: all its blocks done, its writes visible) before they read anything it wrote.  Every
// kernel of the chain waits, so completion is transitive; without the launch attribute (mode 1, the
// default: plain graph edges measured faster) both are no-ops.
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

template <typename... KArgs, typename... Args>
inline cudaError_t launch_chain(void (*kern)(KArgs...), dim3 grid, dim3 block, cudaStream_t stream, bool pdl,
                                size_t smem, Args... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, KArgs(args)...);
}
#endif

constexpr int NT_E = 128, TJ_E = 128, MINB_E = 4;   // evaluation CTA: 128 threads, j-tiles of 128 records, 4 CTAs per SM
constexpr int JL_MAX = 32;                           // at most one warp shares one i
constexpr int64_t L2_CHUNK_BYTES = 24 << 20;         // j-stream piece kept L2-resident across i-block waves
constexpr int GEOM_CACHE_M = 4096;                   // the device loop remembers the geometry of set sizes up to this
constexpr int MAX_WAVES = 255;                      // the split search considers 1..MAX_WAVES work items per SM
constexpr int64_t RES_MAX_N = 2048;                  // the cluster-resident loop (nb_resident.cu) keeps N up to this on chip
constexpr int64_t RES_AUTO_N = 1024;                 // ... and is the default driver up to this (measured: 7.7 against 10.5 us per
                                                     // step at N = 512, 10.4 / 11.1 at 1024, 16.6 / 11.9 at 2048 for modes 3 / 4)
constexpr int GR_M_BIG_DEFAULT = 2048;               // grid-resident loop (nb_gridres.cu): steps with this many active particles
                                                     // or more go to the streaming kernels

// Number of j-splits.  The evaluation is bound by the FP64 pipe of the SM, which the CTAs resident on an SM
// share: what a launch costs is the work of the most loaded SM, (work items on it) x (tiles per item + a
// fixed 0.15 tile per item), in integer thousandths so that host and device take the identical decision.
// Items are handed out one by one (block scheduler / the work counter of the persistent kernel), so the most
// loaded SM holds ceil(items / SMs) of them.  (Round 1 counted waves of SMs x resident CTAs: 683 CTAs on
// 148 SMs x 5 are "one wave", but 91 SMs hold five items and 57 four -- 8 % lost; measured at N = 2^20,
// m = 128: 497 us with 683 splits of 12 tiles, 453 us with 2048 splits of 4.)  Half an item is added for the
// ramp-up and the tail of a launch, which shorter items shrink.  An SM needs about four
// resident CTAs (4 warps per sub-partition) to cover the DFMA latency: fewer items per SM are charged
// in proportion.  0.002 S accounts for the partial sums (0.004, 0.008 S when 16, 32 lanes share an i: a tile is
// then 8, 4 pairs per thread, and m <= 4 is bound by HBM, not by the pipe: measured best 586 splits at m = 1, 1171 at m >= 8).  For w items per SM the best S is the largest that
// still fits, so only the candidates w = 0..MAX_WAVES are scored (w = 0 stands for S = 1); the first candidate
// with the least cost wins.
struct SplitProblem {
    int64_t n_ib, tiles, slots, s_cap, n_sm, jl;
};
// candidate w -> its S; returns the cost, or INT64_MAX when the candidate does not exist
__host__ __device__ inline int64_t split_candidate(const SplitProblem &p, int64_t w, int *S_out)
{
    int64_t s_cap = p.s_cap;
    if (s_cap > p.tiles) s_cap = p.tiles;
    if (s_cap > 65535) s_cap = 65535;
    if (s_cap < 1) s_cap = 1;
    int64_t S = (w == 0) ? 1 : (w * p.n_sm) / p.n_ib;
    if (S < 1) { *S_out = 1; return INT64_MAX; }
    if (S > s_cap) S = s_cap;
    const int64_t tps = (p.tiles + S - 1) / S;
    S = (p.tiles + tps - 1) / tps;  // splits that actually get tiles
    const int64_t per_sm = (p.n_ib * S + p.n_sm - 1) / p.n_sm;   // items on the most loaded SM
    int64_t cost = per_sm * (tps * 1000 + 150) + 500 * tps;      // + half an item of ramp-up / tail
    const int64_t want = p.slots / p.n_sm < 4 ? p.slots / p.n_sm : 4;
    if (per_sm < want) cost = cost * want / per_sm;              // too few warps to keep the FP64 pipe busy
    *S_out = (int)S;
    return cost + S * (p.jl > 8 ? p.jl / 4 : 2);                 // the partial sums; dearer against the short tiles of many lanes per i
}
__host__ __device__ inline int choose_split(const SplitProblem &p)
{
    int64_t best = INT64_MAX;
    int best_s = 1;
    for (int64_t w = 0; w <= MAX_WAVES; ++w) {
        int S;
        const int64_t cost = split_candidate(p, w, &S);
        if (cost < best) { best = cost; best_s = S; }
    }
    return best_s;
}

// Geometry of the evaluation of m particles against Npad records, in two halves so that the
// device can score the split candidates with one thread each (geom_finish takes the winner).
// Lanes per i: as many (a power of two, at most one warp) as keep m * JL within one CTA, so that a small
// set still fills the lanes of its CTA; the j-splits then fill the machine.
__host__ __device__ inline SplitProblem geom_begin(ForceGeom &g, int64_t m, int64_t Npad, int n_sm, int occ,
                                                   int64_t partials_cap, int force_jlanes)
{
    int JL = 1;
    if (force_jlanes >= 1) JL = force_jlanes < JL_MAX ? force_jlanes : JL_MAX;
    else { while (JL < JL_MAX && m * (JL * 2) <= NT_E) JL *= 2; }
    const int64_t slots_per_cta = NT_E / JL;
    SplitProblem p;
    p.n_ib = (m + slots_per_cta - 1) / slots_per_cta;
    p.tiles = Npad / TJ_E;
    p.slots = (int64_t)n_sm * occ;
    p.n_sm = n_sm;
    p.jl = JL;
    const int64_t mpad = (m + 31) & ~(int64_t)31;
    p.s_cap = partials_cap / (9 * mpad);
    g.JL = JL; g.n_ib = (int)p.n_ib; g.mpad = (int)mpad; g.pad_ = 0;
    return p;
}
__host__ __device__ inline void geom_finish(ForceGeom &g, const SplitProblem &p, int S_auto, int force_split)
{
    int S = force_split >= 1 ? (int)(force_split < p.tiles ? force_split : p.tiles) : S_auto;
    if (force_split < 1 && p.n_ib > p.slots) {
        // More than one wave of i-blocks re-reads the whole j-stream once per wave.  Keep the piece
        // that the concurrently running CTAs stream below L2_CHUNK_BYTES (a cyclic sweep over more
        // than the L2 of one die misses on every pass), when the partial sums fit.
        const int64_t tps_max = L2_CHUNK_BYTES / ((int64_t)TJ_E * REC * 8);
        const int64_t s_min = (p.tiles + tps_max - 1) / tps_max;
        if (s_min > S && s_min <= p.s_cap) S = (int)s_min;
    }
    if (S > p.s_cap) S = (int)(p.s_cap < 1 ? 1 : p.s_cap);
    const int64_t tps = (p.tiles + S - 1) / S;
    S = (int)((p.tiles + tps - 1) / tps);
    g.S = S; g.tps = (int)tps;
}
__host__ __device__ inline ForceGeom choose_geom(int64_t m, int64_t Npad, int n_sm, int occ,
                                                 int64_t partials_cap, int force_split, int force_jlanes)
{
    ForceGeom g;
    const SplitProblem p = geom_begin(g, m, Npad, n_sm, occ, partials_cap, force_jlanes);
    geom_finish(g, p, force_split >= 1 ? 1 : choose_split(p), force_split);
    return g;
}

}  // namespace nb

struct nb_ctx {
    int64_t N, Npad;
    double eps, eps2, eta, eta_init, dt_min, dt_max;
    cudaStream_t stream;
    int device, n_sm;

    // state flags
    bool started;      // nb_startup has run (or a full state was loaded)
    bool pred_valid;   // predicted stream holds data
    double t_pred;     // time of the predicted stream
    bool have_block;   // nb_next_block selected a set that is not yet committed
    bool evaluated;    // nb_force evaluated the scheduler's set at t_next (complete sums: corrector may run)
    bool eval_partial; // the same, but over a proper j-slice: becomes `evaluated` when nb_set_forces stores the reduced sums
    int debug;         // nb_set_debug: range-check caller-supplied index lists
    double t_now, t_next;
    int64_t n_active;       // scheduler's set
    int64_t n_eval;         // size of the last evaluated set

    // device buffers
    double *mass, *t, *dt;          // [Npad]
    double *r, *v, *a, *j, *s, *c;  // [3][Npad]
    double *jp;                     // [Npad][REC]
    int32_t *active;                // [Npad] scheduler's list
    int32_t *user_idx;              // [Npad] copy of a caller-supplied list
    double *f1;                     // [9][Npad]
    double *stage;                  // staging for [n][3] / [n][21] in/out copies and the scratch prediction of
                                    // nb_energy; stage_cap doubles, grown on demand (reserve_stage)
    size_t stage_cap;
    double *partials;               // [S][9][mpad]
    size_t partials_cap;            // in doubles (grown on demand up to partials_limit)
    size_t partials_limit;          // most the split search can ask for: bounds S in choose_geom
    unsigned long long *d_tmin;     // scheduler scalar: bits of min(t+dt)
    int32_t *blk_count;             // per-block match counts / offsets
    int64_t n_sched_blocks;
    double *red;                    // reduction scratch (energy)
    int32_t *h_dbg, *d_dbg;         // pinned, mapped {number of bad indices, first bad slot} of the debug check
    nb::Sched *h_sched;             // pinned host mirror
    nb::Sched *d_sched;             // device alias of h_sched
    nb::StepCtl *ctl;               // device control block of the graph-driven block-step loop
    nb::StepCtl *h_ctl;             // pinned host copy, refreshed after every graph launch
    nb::ForceGeom *geom_cache;      // [GEOM_CACHE_M + 1], S == 0: not computed yet (device loop only)
    cudaGraphExec_t step_graph;     // `graph_batch` block steps captured once per context
    int graph_batch;
    int graph_split, graph_jlanes, graph_precision;  // knobs the captured graph was built with
    int64_t launches_per_batch;     // kernels in one replay of step_graph
    int use_graph;                  // loop mode: 0 host-issued calls; 1, 2 graph batches (2: with PDL); 3 cluster-resident loop
    int res_cluster;                // CTAs of the resident loop's cluster (16, or 8 where 16 cannot be scheduled)
    bool loop_auto;                 // the loop mode is the default for this N (not set by nb_set_loop_mode)
    int graph_pdl;                  // the captured graph uses programmatic dependent launch
    void *gr_hdr;                   // grid-resident loop (nb_gridres.cu): per-CTA headers, candidates' records, partial sums,
    double *gr_cand, *gr_part;      // barrier counter; allocated at the first run in loop mode 4
    unsigned long long *gr_bar;
    int gr_m_big, gr_m_big_alloc;

    // tuning
    int force_split, force_jlanes;
    int64_t j_begin, j_end;         // j-shard evaluated by nb_force (nb_set_j_range); default [0, N)
    int precision;                  // 0: FP64 throughout (default); 1: the paper's mixed SP/DP pair arithmetic
    int64_t last_launch[5];
    int occ[8];                     // resident CTAs per SM: [0] k_force (the geometry rule uses it), [1] k_force_persistent

    // statistics
    int64_t n_steps;
    double n_pairs;
    int64_t n_launch;
    int64_t hist[64];

    char err[512];
};

namespace nb {

// ----- nb_force.cu
// Evaluate (acc, jerk, snap) of `m` particles (active == nullptr: particles 0..m-1) against the
// Npad predicted records; result in ctx->f1[c][k].  no_snap = true (start-up pass 1, G8) launches the
// SNAP = false instantiation of the pair body: acceleration and jerk only, 31 instead of 53 FP64
// instructions per pair; the snap planes of f1 are then written as zeros.
int launch_force(nb_ctx *ctx, const int32_t *active, int64_t m, bool no_snap = false);
int launch_check_indices(nb_ctx *ctx, const int32_t *idx, int64_t m);   // debug: fills ctx->h_dbg (after a sync)
int query_force_occupancy(nb_ctx *ctx);
int enqueue_force_persistent(nb_ctx *ctx);   // evaluation of the graph-driven loop; set size and geometry come from ctx->ctl
// f1[c][k] -> out[q][k][3] (q = 0 acc, 1 jerk, 2 snap) contiguous in ctx->stage
int launch_unpack_f1(nb_ctx *ctx, int64_t m);
int launch_f1_contig(nb_ctx *ctx, int64_t m, double *buf, bool to_f1);
int reserve_partials(nb_ctx *ctx, size_t doubles);

// ----- nb_step.cu
int launch_load_state(nb_ctx *ctx, const double *pos_dev, const double *vel_dev, const double *mass_dev);
int launch_predict(nb_ctx *ctx, double t, double *records = nullptr);   // records: destination (default ctx->jp)
int launch_set_pred(nb_ctx *ctx, const double *pos, const double *vel, const double *acc, bool pos_vel, bool acc_valid);
int launch_get_pred(nb_ctx *ctx, double *pos, double *vel, double *acc);
int launch_pack3(nb_ctx *ctx, const double *soa, double *aos);      // [3][Npad] -> [N][3]
int launch_next_block(nb_ctx *ctx);                                  // fills active, d_sched
int launch_correct(nb_ctx *ctx, const int32_t *active, int64_t m, double t_next);
int launch_startup_commit(nb_ctx *ctx, int pass);                    // pass 1: a,j <- f1 ; pass 2: a,j,s <- f1 + dt
int launch_full_state(nb_ctx *ctx, double *state, bool to_ctx);
int launch_tmax(nb_ctx *ctx);                                        // d_sched->t_next = max t_i

int enqueue_graph_gather_predict(nb_ctx *ctx, int parity);           // active list + predictor of one step
int enqueue_graph_correct(nb_ctx *ctx, int parity);           // split sums + corrector + bookkeeping
int launch_graph_begin(nb_ctx *ctx, double t_end, int64_t steps);    // seeds ctl (t_end, steps_left, tmin)

// ----- nb_graph.cu
int graph_run(nb_ctx *ctx, double t_end, int64_t max_steps, int64_t *n_steps);
void graph_release(nb_ctx *ctx);

// ----- nb_resident.cu
int resident_run(nb_ctx *ctx, double t_end, int64_t max_steps, int64_t *n_steps);

// ----- nb_gridres.cu
int gridres_run(nb_ctx *ctx, double t_end, int64_t max_steps, int64_t *n_steps);
bool gridres_fits(const nb_ctx *ctx);
void gridres_release(nb_ctx *ctx);

// ----- nb_energy.cu
int launch_energy(nb_ctx *ctx, const double *records, double out_host[9]);

// ----- nb_probe.cu
int launch_probe(nb_ctx *ctx, int64_t iters, double *flops, float *ms);

// ----- nb_api.cu
int reserve_stage(nb_ctx *ctx, size_t doubles);
// one block step through the call sequence (next block [sync], predict, evaluate, correct) unless the next block lies beyond t_end
int host_block_step(nb_ctx *ctx, double t_end, bool *stepped);

int set_err(nb_ctx *ctx, int code, const char *fmt, ...);

#define NB_CUDA(ctx, call)                                                                   \
    do {                                                                                     \
        cudaError_t e_ = (call);                                                             \
        if (e_ != cudaSuccess)                                                               \
            return nb::set_err((ctx), e_ == cudaErrorMemoryAllocation ? NB_ENOMEM : NB_ECUDA, \
                               "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_),       \
                               __FILE__, __LINE__);                                          \
    } while (0)

#define NB_LAUNCH_CHECK(ctx, name)                                                           \
    do {                                                                                     \
        cudaError_t e_ = cudaGetLastError();                                                 \
        if (e_ != cudaSuccess)                                                               \
            return nb::set_err((ctx), NB_ECUDA, "launch of %s failed: %s", name,             \
                               cudaGetErrorString(e_));                                      \
        (ctx)->n_launch += 1;                                                                \
    } while (0)

}  // namespace nb
