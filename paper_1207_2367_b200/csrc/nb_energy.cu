// nb_energy.cu -- diagnostics: E = K + W with the softened pair potential of Eq. 2
// (PAPER.md:40), total momentum and angular momentum (Eq. 20), computed from the
// predicted stream (positions and velocities at the current time).
//   W = -sum_i m_i sum_{j > i} m_j / sqrt(|r_ij|^2 + eps^2)   (every pair once, as Eq. 2 is
//   written; the j = i term is excluded by index: with eps > 0 it is NOT zero).  Thread i sums
//   over j > i only, so the blocks have triangular work (the block scheduler balances them).
// Reductions are fixed-order trees, so the result is bit-reproducible.
#include "nb_internal.cuh"

namespace nb {

constexpr int EN_THREADS = 128;
constexpr int EN_TJ = 128;
static_assert(EN_THREADS == EN_TJ, "the triangular loop starts at the block's own tile");

__device__ __forceinline__ double rsqrt_full(double s)
{
    // hardware seed on the upper word + one third-order step (as in the evaluation kernel)
    double y0;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y0) : "d"(s));
    const double e = fma(-s, y0 * y0, 1.0);
    return fma(y0 * e, fma(0.375, e, 0.5), y0);
}

__device__ __forceinline__ double block_sum(double v, double *sm)
{
    // fixed-order tree: butterfly inside each warp, then over the warps
    for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
    __syncthreads();
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = v;
    __syncthreads();
    double tot = 0.0;
    for (int w = 0; w < (int)(blockDim.x >> 5); ++w) tot += sm[w];
    return tot;
}

// per-block partials: part[b][0..8] = {unused, K, W, Px, Py, Pz, Lx, Ly, Lz}
__global__ void __launch_bounds__(EN_THREADS)
    k_energy(const int64_t N, const int64_t Npad, const double eps2, const double *__restrict__ jp,
             double *__restrict__ part)
{
    __shared__ __align__(16) double tile[EN_TJ * 4];
    __shared__ double red[EN_THREADS / 32];
    const int64_t i = (int64_t)blockIdx.x * EN_THREADS + threadIdx.x;
    const bool live = i < N;
    const double *pi = jp + (live ? i : 0) * REC;
    const double xi = pi[0], yi = pi[1], zi = pi[2], vx = pi[3], vy = pi[4], vz = pi[5];
    const double mi = live ? pi[9] : 0.0;
    double pot = 0.0;
    // first tile that holds a j > i for some i of this block (blocks and tiles are both 128 long)
    for (int64_t j0 = (int64_t)blockIdx.x * EN_THREADS; j0 < Npad; j0 += EN_TJ) {
        __syncthreads();
        {
            const double *pj = jp + (j0 + threadIdx.x) * REC;
            tile[4 * threadIdx.x + 0] = pj[0];
            tile[4 * threadIdx.x + 1] = pj[1];
            tile[4 * threadIdx.x + 2] = pj[2];
            tile[4 * threadIdx.x + 3] = pj[9];
        }
        __syncthreads();
        double p = 0.0;
#pragma unroll 12
        for (int jj = 0; jj < EN_TJ; ++jj) {
            const double2 a = *reinterpret_cast<const double2 *>(tile + 4 * jj);
            const double2 b = *reinterpret_cast<const double2 *>(tile + 4 * jj + 2);
            const double dx = a.x - xi, dy = a.y - yi, dz = b.x - zi;
            const double s = fma(dx, dx, fma(dy, dy, fma(dz, dz, eps2)));
            double y = rsqrt_full(s);
            // pairs with j <= i belong to the other particle's sum; padded / massless records add
            // nothing (integer test on the bits: +0.0 only, no FP64 pipe slot)
            if (j0 + jj <= i || __double_as_longlong(b.y) == 0) y = 0.0;
            p = fma(b.y, y, p);
        }
        pot += p;
    }
    double vals[8];
    vals[0] = 0.5 * mi * (vx * vx + vy * vy + vz * vz);
    vals[1] = -mi * pot;
    vals[2] = mi * vx; vals[3] = mi * vy; vals[4] = mi * vz;
    vals[5] = mi * (yi * vz - zi * vy);
    vals[6] = mi * (zi * vx - xi * vz);
    vals[7] = mi * (xi * vy - yi * vx);
    if (!live) {  // lanes beyond N: their pot may be NaN (eps = 0 against record 0); they own nothing
#pragma unroll
        for (int q = 0; q < 8; ++q) vals[q] = 0.0;
    }
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        const double tot = block_sum(vals[q], red);
        if (threadIdx.x == 0) part[(int64_t)blockIdx.x * 9 + 1 + q] = tot;
    }
}

// one block: pairwise (tree) sum of the per-block partials, fixed order
__global__ void k_energy_final(const int nb, const double *__restrict__ part, double *__restrict__ out)
{
    __shared__ double sm[256];
    for (int q = 1; q < 9; ++q) {
        double v = 0.0;
        for (int b = threadIdx.x; b < nb; b += 256) v += part[(int64_t)b * 9 + q];
        sm[threadIdx.x] = v;
        __syncthreads();
        for (int off = 128; off > 0; off >>= 1) {
            if ((int)threadIdx.x < off) sm[threadIdx.x] += sm[threadIdx.x + off];
            __syncthreads();
        }
        if (threadIdx.x == 0) out[q] = sm[0];
        __syncthreads();
    }
    if (threadIdx.x == 0) out[0] = out[1] + out[2];
}

int launch_energy(nb_ctx *ctx, double out_host[9])
{
    const int64_t N = ctx->N;
    const int nb = (int)((N + EN_THREADS - 1) / EN_THREADS);
    double *part = ctx->red;  // [nb][9] + 9
    k_energy<<<nb, EN_THREADS, 0, ctx->stream>>>(N, ctx->Npad, ctx->eps2, ctx->jp, part + 9);
    NB_LAUNCH_CHECK(ctx, "k_energy");
    k_energy_final<<<1, 256, 0, ctx->stream>>>(nb, part + 9, part);
    NB_LAUNCH_CHECK(ctx, "k_energy_final");
    NB_CUDA(ctx, cudaMemcpyAsync(out_host, part, 9 * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    NB_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return NB_OK;
}

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

// Operand-fetch probe: 12 independent DFMA chains per thread, 24 DFMAs per loop trip, operands
// pinned by inline PTX so that ptxas cannot fold them.
template <int MODE>
__global__ void __launch_bounds__(512) k_probe_operands(const long long iters, const double seed, double *__restrict__ sink)
{
    double x[12], a[12], b[12];
    const double tf = (double)threadIdx.x;
#pragma unroll
    for (int k = 0; k < 12; ++k) {
        x[k] = seed + k + tf;
        // loaded, not computed: ptxas would otherwise re-materialise them inside the timed loop
        a[k] = sink[1 + k] + tf * 1e-15;
        b[k] = sink[13 + k] + tf * 1e-16;
    }
    for (long long it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 2; ++r) {
#pragma unroll
            for (int k = 0; k < 12; ++k) {
                if (MODE == 0) asm volatile("fma.rn.f64 %0, %0, 0d3FEFFFFDE7210BE9, 0d3E112E0BE826D695;" : "+d"(x[k]));
                if (MODE == 1) asm volatile("fma.rn.f64 %0, %1, %2, %0;" : "+d"(x[k]) : "d"(a[k]), "d"(b[k]));
                if (MODE == 2) asm volatile("fma.rn.f64 %0, %1, %2, %0;" : "+d"(x[k]) : "d"(a[k / 3]), "d"(b[k]));
                if (MODE == 3) asm volatile("fma.rn.f64 %0, %1, %1, %0;" : "+d"(x[k]) : "d"(a[k]));
                if (MODE == 4) asm volatile("fma.rn.f64 %0, %1, %2, %0;" : "+d"(x[k]) : "d"(a[0]), "d"(b[k]));
                if (MODE == 5) {  // 3-register DFMA, then a DADD that shares one operand with it (1 fresh read)
                    if (k % 2 == 0) asm volatile("fma.rn.f64 %0, %1, %2, %0;" : "+d"(x[k]) : "d"(a[k]), "d"(b[k]));
                    else asm volatile("add.f64 %0, %1, %0;" : "+d"(x[k]) : "d"(a[k - 1]));
                }
            }
        }
    }
    double t = 0.0;
#pragma unroll
    for (int k = 0; k < 12; ++k) t += x[k];
    if (t == 123.456) sink[0] = t;
}

int launch_probe_operands(nb_ctx *ctx, int mode, int64_t iters, double sm_mhz, double *cycles_per_inst)
{
    cudaEvent_t e0, e1;
    NB_CUDA(ctx, cudaEventCreate(&e0));
    NB_CUDA(ctx, cudaEventCreate(&e1));
    const int grid = ctx->n_sm, threads = 512;  // 4 warps per SM sub-partition, as in the evaluation kernel
    for (int pass = 0; pass < 2; ++pass) {
        const long long n = pass ? iters : iters / 8 + 1;
        if (pass) NB_CUDA(ctx, cudaEventRecord(e0, ctx->stream));
        switch (mode) {
            case 0: k_probe_operands<0><<<grid, threads, 0, ctx->stream>>>(n, 1.0, ctx->red); break;
            case 1: k_probe_operands<1><<<grid, threads, 0, ctx->stream>>>(n, 1.0, ctx->red); break;
            case 2: k_probe_operands<2><<<grid, threads, 0, ctx->stream>>>(n, 1.0, ctx->red); break;
            case 3: k_probe_operands<3><<<grid, threads, 0, ctx->stream>>>(n, 1.0, ctx->red); break;
            case 4: k_probe_operands<4><<<grid, threads, 0, ctx->stream>>>(n, 1.0, ctx->red); break;
            default: k_probe_operands<5><<<grid, threads, 0, ctx->stream>>>(n, 1.0, ctx->red); break;
        }
        NB_LAUNCH_CHECK(ctx, "k_probe_operands");
    }
    NB_CUDA(ctx, cudaEventRecord(e1, ctx->stream));
    NB_CUDA(ctx, cudaEventSynchronize(e1));
    float t = 0.f;
    NB_CUDA(ctx, cudaEventElapsedTime(&t, e0, e1));
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    const double warp_inst_per_smsp = (double)iters * 24.0 * (threads / 32) / 4.0;
    if (cycles_per_inst) *cycles_per_inst = (double)t * 1e-3 * sm_mhz * 1e6 / warp_inst_per_smsp;
    return NB_OK;
}

}  // namespace nb
