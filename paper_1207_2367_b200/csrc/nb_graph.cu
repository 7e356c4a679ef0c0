// nb_graph.cu -- the block-step loop driven from the device.
//
// The paper's loop returns to the host every block step: the CPU finds the active set, copies
// indices in and forces out (Table 1 rows 1, 2, 6, 9), and for the smallest
// blocks that overhead is most of the step.  Here the kernels of a step read
// (t_next, m) and the evaluation geometry from a control block in device memory, so their launch
// configurations are fixed and `graph_batch` consecutive block steps (three kernels each:
// gather+predict, evaluation, split sums+corrector) are captured ONCE per context as a CUDA graph.  The host replays the graph and looks at the control block only
// once per batch; steps past t_end (or past the requested count) find `done` set and return
// without touching the state, so overshooting inside a batch is harmless.
//
// The arithmetic of a step is that of the call sequence nb_next_block -> nb_predict -> nb_force
// -> nb_correct_and_step (same kernels' device functions, same geometry rule, same summation
// order), so both drivers produce bit-identical states; tests/test_gpu_graph.py checks it.
#include "nb_internal.cuh"

namespace nb {

static int steps_per_batch(const nb_ctx *ctx)
{
    // an idle (done) step still scans t and dt once: keep the overshoot cheap when N is large
    return ctx->N <= ((int64_t)1 << 18) ? 64 : (ctx->N <= ((int64_t)1 << 21) ? 16 : 4);
}

static int build_graph(nb_ctx *ctx)
{
    cudaStream_t cap = nullptr;
    NB_CUDA(ctx, cudaStreamCreateWithFlags(&cap, cudaStreamNonBlocking));
    cudaStream_t user = ctx->stream;
    const int64_t launches = ctx->n_launch;
    ctx->stream = cap;  // the enqueue helpers launch on ctx->stream; capture cannot use the legacy stream
    cudaGraph_t graph = nullptr;
    int rc = NB_OK;
    cudaError_t e = cudaStreamBeginCapture(cap, cudaStreamCaptureModeThreadLocal);
    if (e != cudaSuccess) rc = set_err(ctx, NB_ECUDA, "cudaStreamBeginCapture failed: %s", cudaGetErrorString(e));
    const int B = steps_per_batch(ctx);
    for (int b = 0; b < B && rc == NB_OK; ++b) {
        if ((rc = enqueue_graph_gather_predict(ctx, b & 1)) != NB_OK) break;
        if ((rc = enqueue_force_persistent(ctx)) != NB_OK) break;
        rc = enqueue_graph_correct(ctx, b & 1);
    }
    if (e == cudaSuccess) {
        const cudaError_t e2 = cudaStreamEndCapture(cap, &graph);
        if (e2 != cudaSuccess && rc == NB_OK)
            rc = set_err(ctx, NB_ECUDA, "cudaStreamEndCapture failed: %s", cudaGetErrorString(e2));
    }
    ctx->stream = user;
    ctx->launches_per_batch = ctx->n_launch - launches;
    ctx->n_launch = launches;  // captured, not launched
    cudaStreamDestroy(cap);
    if (rc != NB_OK) { if (graph) cudaGraphDestroy(graph); return rc; }
    // the remembered geometries belong to the knobs this graph is captured with
    NB_CUDA(ctx, cudaMemsetAsync(ctx->geom_cache, 0, ((size_t)GEOM_CACHE_M + 1) * sizeof(ForceGeom), ctx->stream));
    const cudaError_t e3 = cudaGraphInstantiate(&ctx->step_graph, graph, 0);
    cudaGraphDestroy(graph);
    if (e3 != cudaSuccess) return set_err(ctx, NB_ECUDA, "cudaGraphInstantiate failed: %s", cudaGetErrorString(e3));
    ctx->graph_batch = B;
    ctx->graph_split = ctx->force_split; ctx->graph_jlanes = ctx->force_jlanes;
    ctx->graph_precision = ctx->precision;
    ctx->graph_pdl = ctx->use_graph == 2;
    return NB_OK;
}

void graph_release(nb_ctx *ctx)
{
    if (ctx->step_graph) cudaGraphExecDestroy(ctx->step_graph);
    ctx->step_graph = nullptr;
}

// Advance while the next block time is <= t_end and fewer than max_steps steps were taken.
int graph_run(nb_ctx *ctx, double t_end, int64_t max_steps, int64_t *n_steps)
{
    // tuning knobs are kernel arguments of the captured nodes: re-capture when they changed
    if (ctx->step_graph && (ctx->graph_split != ctx->force_split || ctx->graph_jlanes != ctx->force_jlanes ||
                            ctx->graph_precision != ctx->precision || ctx->graph_pdl != (ctx->use_graph == 2)))
        graph_release(ctx);
    {
        const int rc = reserve_partials(ctx, ctx->partials_limit);  // no allocation inside a replay
        if (rc != NB_OK) return rc;
    }
    if (!ctx->step_graph) {
        const int rc = build_graph(ctx);
        if (rc != NB_OK) return rc;
    }
    {
        const int rc = launch_graph_begin(ctx, t_end, max_steps);
        if (rc != NB_OK) return rc;
    }
    for (;;) {
        NB_CUDA(ctx, cudaGraphLaunch(ctx->step_graph, ctx->stream));
        ctx->n_launch += ctx->launches_per_batch;
        NB_CUDA(ctx, cudaMemcpyAsync(ctx->h_ctl, ctx->ctl, sizeof(StepCtl), cudaMemcpyDeviceToHost, ctx->stream));
        NB_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
        if (ctx->h_ctl->done) break;
    }
    const StepCtl *h = ctx->h_ctl;
    if (h->n_steps > 0) {
        ctx->t_now = h->t_now;
        ctx->pred_valid = true; ctx->t_pred = h->t_now;
    }
    ctx->n_steps += h->n_steps;
    ctx->n_pairs += h->n_pairs;
    for (int b = 0; b < 64; ++b) ctx->hist[b] += h->hist[b];
    ctx->have_block = false; ctx->evaluated = false; ctx->eval_partial = false;
    if (n_steps) *n_steps = h->n_steps;
    return NB_OK;
}

}  // namespace nb
