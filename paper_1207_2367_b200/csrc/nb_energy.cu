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
            // nothing, nor does a coincident pair at eps = 0 (s = +0: outside the domain, G12) -- integer
            // tests on the bits, no FP64 pipe slot
            if (j0 + jj <= i || __double_as_longlong(b.y) == 0 || __double_as_longlong(s) == 0) y = 0.0;
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

int launch_energy(nb_ctx *ctx, const double *records, double out_host[9])
{
    const int64_t N = ctx->N;
    const int nb = (int)((N + EN_THREADS - 1) / EN_THREADS);
    double *part = ctx->red;  // [nb][9] + 9
    k_energy<<<nb, EN_THREADS, 0, ctx->stream>>>(N, ctx->Npad, ctx->eps2, records, part + 9);
    NB_LAUNCH_CHECK(ctx, "k_energy");
    k_energy_final<<<1, 256, 0, ctx->stream>>>(nb, part + 9, part);
    NB_LAUNCH_CHECK(ctx, "k_energy_final");
    NB_CUDA(ctx, cudaMemcpyAsync(out_host, part, 9 * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    NB_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return NB_OK;
}

}  // namespace nb
