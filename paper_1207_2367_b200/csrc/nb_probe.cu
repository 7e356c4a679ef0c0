// nb_probe.cu -- DFMA-only micro-benchmark: the measured FP64 ALU rate that bench.py prints beside
// the derived peak.  Not on the hot path.
#include "nb_internal.cuh"

namespace nb {

// ---------------------------------------------------------------------------------------
// DFMA-only probe: 16 independent FMA chains per thread, 8 warps per SM sub-partition.
__global__ void __launch_bounds__(256, 4) k_probe_dfma(const long long iters, const double x0, double *__restrict__ sink)
{
    double a[16];
#pragma unroll
    for (int q = 0; q < 16; ++q) a[q] = x0 + q + threadIdx.x;
    const double m = 0.999999, c = 1e-9;
    for (long long it = 0; it < iters; ++it) {
#pragma unroll
        for (int q = 0; q < 16; ++q) a[q] = fma(a[q], m, c);
    }
    double t = 0.0;
#pragma unroll
    for (int q = 0; q < 16; ++q) t += a[q];
    if (t == 123.456) sink[0] = t;  // never true: keeps the chains alive
}

int launch_probe(nb_ctx *ctx, int64_t iters, double *flops, float *ms)
{
    cudaEvent_t e0, e1;
    NB_CUDA(ctx, cudaEventCreate(&e0));
    NB_CUDA(ctx, cudaEventCreate(&e1));
    const int grid = ctx->n_sm * 4;
    k_probe_dfma<<<grid, 256, 0, ctx->stream>>>(iters / 16 + 1, 1.0, ctx->red);  // warm-up
    NB_CUDA(ctx, cudaEventRecord(e0, ctx->stream));
    k_probe_dfma<<<grid, 256, 0, ctx->stream>>>(iters, 1.0, ctx->red);
    NB_CUDA(ctx, cudaEventRecord(e1, ctx->stream));
    NB_LAUNCH_CHECK(ctx, "k_probe_dfma");
    ctx->n_launch += 1;
    NB_CUDA(ctx, cudaEventSynchronize(e1));
    float t = 0.f;
    NB_CUDA(ctx, cudaEventElapsedTime(&t, e0, e1));
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (ms) *ms = t;
    if (flops) *flops = 2.0 * 16.0 * (double)iters * 256.0 * (double)grid / ((double)t * 1e-3);
    return NB_OK;
}

}  // namespace nb
