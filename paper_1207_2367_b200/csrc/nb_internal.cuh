// nb_internal.cuh -- context layout and kernel-launcher declarations shared by the .cu files
// of libnb.  Nothing here is visible through the C-ABI (include/nb.h).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

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
    bool evaluated;    // nb_force evaluated the scheduler's set at t_next
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
    double *stage;                  // [9*Npad] staging for [n][3] in/out copies
    double *partials;               // [S][9][mpad]
    size_t partials_cap;            // in doubles
    unsigned long long *d_tmin;     // scheduler scalar: bits of min(t+dt)
    int32_t *blk_count;             // per-block match counts / offsets
    int64_t n_sched_blocks;
    double *red;                    // reduction scratch (energy)
    nb::Sched *h_sched;             // pinned host mirror
    nb::Sched *d_sched;             // device alias of h_sched

    // tuning
    int force_split, force_jlanes;
    int64_t last_launch[5];
    int occ[8];                     // resident CTAs per SM of each evaluation-kernel variant

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
// Npad predicted records; result in ctx->f1[c][k].  with_snap = false skips nothing in the
// arithmetic (the body is the same); it only exists for symmetry of the start-up passes.
int launch_force(nb_ctx *ctx, const int32_t *active, int64_t m);
int query_force_occupancy(nb_ctx *ctx);
// f1[c][k] -> out[q][k][3] (q = 0 acc, 1 jerk, 2 snap) contiguous in ctx->stage
int launch_unpack_f1(nb_ctx *ctx, int64_t m);

// ----- nb_step.cu
int launch_load_state(nb_ctx *ctx, const double *pos_dev, const double *vel_dev, const double *mass_dev);
int launch_predict(nb_ctx *ctx, double t);
int launch_set_pred(nb_ctx *ctx, const double *pos, const double *vel, const double *acc, bool pos_vel, bool acc_valid);
int launch_get_pred(nb_ctx *ctx, double *pos, double *vel, double *acc);
int launch_pack3(nb_ctx *ctx, const double *soa, double *aos);      // [3][Npad] -> [N][3]
int launch_next_block(nb_ctx *ctx);                                  // fills active, d_sched
int launch_correct(nb_ctx *ctx, const int32_t *active, int64_t m, double t_next);
int launch_startup_commit(nb_ctx *ctx, int pass);                    // pass 1: a,j <- f1 ; pass 2: a,j,s <- f1 + dt
int launch_full_state(nb_ctx *ctx, double *state, bool to_ctx);
int launch_tmax(nb_ctx *ctx);                                        // d_sched->t_next = max t_i

// ----- nb_energy.cu
int launch_energy(nb_ctx *ctx, double out_host[9]);

// ----- nb_probe.cu
int launch_probe(nb_ctx *ctx, int64_t iters, double *flops, float *ms);
int launch_probe_operands(nb_ctx *ctx, int mode, int64_t iters, double sm_mhz, double *cycles_per_inst);

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
