// nb_static.cu -- nb_force_static: the evaluation step (Eq. 8-10, Eq. 2 softening, split over j as in
// PAPER.md:108-114) for callers that cannot allocate: code under CUDA-graph capture, serving loops, harnesses that
// forbid cudaMalloc.  It is a variant of k_force (nb_force.cu) with the same device functions (force_item, the
// fixed-order split sums); what nb_force keeps in buffers of a context -- the packed predicted records and the
// j-split partial sums -- lives here in ONE file-scope device array of fixed size.  No context, no cudaMalloc /
// cudaFree / allocating library call anywhere on this path; existing entry points are untouched.
//
// The array is shared by every call in the process (per device) and keeps the last call's contents.  Nothing in
// it has to start at zero except the padding records N..Npad-1, which k_static_pack writes as zeros on every
// call; every partial sum that is read was written by the same call.  Two calls that overlap on the GPU (different
// streams, or graphs replayed concurrently) race on it.
#include <math.h>
#include <mutex>
#include <stdarg.h>
#include <stdio.h>

#include "nb_internal.cuh"
#include "nb_force_dev.cuh"

// 16 MiB per GPU that loads the library, held until the process exits.
#define NB_STATIC_MAX_N_ 65536
constexpr size_t STATIC_REC_DOUBLES = (size_t)nb::REC * NB_STATIC_MAX_N_;     // packed records: 5 MiB
constexpr size_t STATIC_DOUBLES = (size_t)2 << 20;                            // the whole array: 16 MiB
constexpr size_t STATIC_PART_DOUBLES = STATIC_DOUBLES - STATIC_REC_DOUBLES;   // split partials / single-split sums: 11 MiB
static_assert(NB_STATIC_MAX_N_ == NB_STATIC_MAX_N, "nb.h states the limit");
static_assert(9 * (size_t)NB_STATIC_MAX_N_ <= STATIC_PART_DOUBLES, "one split of the largest set must fit");

// In host code this name is a host-side stand-in for the symbol, NOT a device address: the host obtains the
// address once per device with cudaGetSymbolAddress (static_setup) and passes that pointer to the kernels.
static __device__ __align__(256) double nb_static_scratch[STATIC_DOUBLES];

namespace nb {

// pos, vel, acc_pred [N][3], mass [N]  ->  records [Npad][REC]; records N..Npad-1 are written as zeros (m = 0)
__global__ void k_static_pack(const double *__restrict__ pos, const double *__restrict__ vel, const double *__restrict__ acc,
                              const double *__restrict__ mass, const int N, const int Npad, double *__restrict__ rec)
{
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= Npad) return;
    double *q = rec + (size_t)p * REC;
    if (p < N) {
        q[0] = pos[3 * (size_t)p]; q[1] = pos[3 * (size_t)p + 1]; q[2] = pos[3 * (size_t)p + 2];
        q[3] = vel[3 * (size_t)p]; q[4] = vel[3 * (size_t)p + 1]; q[5] = vel[3 * (size_t)p + 2];
        q[6] = acc ? acc[3 * (size_t)p] : 0.0; q[7] = acc ? acc[3 * (size_t)p + 1] : 0.0; q[8] = acc ? acc[3 * (size_t)p + 2] : 0.0;
        q[9] = mass[p];
    } else {
#pragma unroll
        for (int c = 0; c < REC; ++c) q[c] = 0.0;
    }
}

// k_force with its records and its output in the static array (pointers passed by the host)
template <int JL, bool GUARD0>
__global__ void __launch_bounds__(NT_E, MINB_E)
    k_force_static(const double *__restrict__ rec, const int32_t *__restrict__ active, const int m, const int tiles_total,
                   const int tiles_per_split, const double eps2, double *__restrict__ out, const size_t cstride,
                   const size_t kstride, const size_t sstride)
{
    __shared__ __align__(128) double tile[2][TJ_E * REC];
    __shared__ __align__(8) uint64_t full[2];
    if (threadIdx.x == 0) {
        mbar_init(&full[0], 1);
        mbar_init(&full[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    unsigned tc = 0;
    force_item<NT_E, TJ_E, JL, GUARD0, 0, 12>(rec, rec, active, m, blockIdx.x, blockIdx.y, tiles_total, tiles_per_split, eps2, out,
                                              cstride, kstride, sstride, tile, full, tc);
}

// one warp per slot k: fixed-order sum over the S splits (sum_splits_thread / sum_splits_warp, the additions of
// every other driver), written straight into the caller's [m][3] arrays
__global__ void k_static_finish(const double *__restrict__ part, const int S, const int m, const size_t cstride,
                                const size_t kstride, const size_t sstride, double *__restrict__ acc,
                                double *__restrict__ jerk, double *__restrict__ snap)
{
    const int k = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (k >= m) return;
    double v = 0.0;
    if (S < 32) {
        if (lane < 9) v = sum_splits_thread(part + lane * cstride + (size_t)k * kstride, S, sstride);
    } else {
        for (int c = 0; c < 9; ++c) {
            const double a = sum_splits_warp(part + c * cstride + (size_t)k * kstride, S, lane);
            if (lane == c) v = a;
        }
    }
    if (lane < 9) {
        double *dst = lane < 3 ? acc : (lane < 6 ? jerk : snap);
        if (dst) dst[3 * (size_t)k + lane % 3] = v;
    }
}

}  // namespace nb

using namespace nb;

namespace {

struct StaticDev {
    bool ready;
    double *scratch;   // device address of nb_static_scratch on this device
    int n_sm, occ;
};
constexpr int MAX_DEVICES = 64;
StaticDev g_dev[MAX_DEVICES];
std::mutex g_dev_lock;

int fail(char *err, int64_t err_len, int code, const char *fmt, ...)
{
    if (err && err_len > 0) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(err, (size_t)err_len, fmt, ap);
        va_end(ap);
    }
    return code;
}

#define NBS_CUDA(call)                                                                                        \
    do {                                                                                                      \
        const cudaError_t e_ = (call);                                                                        \
        if (e_ != cudaSuccess)                                                                                \
            return fail(err, err_len, NB_ECUDA, "nb_force_static: %s failed: %s", #call, cudaGetErrorString(e_)); \
    } while (0)

// once per device, with that device current: the array's device address and the launch constants.  None of
// these calls allocates.
int static_setup(StaticDev **out, char *err, int64_t err_len)
{
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) {
        cudaGetLastError();
        return fail(err, err_len, NB_ECUDA, "nb_force_static: no usable CUDA device (there is no CPU path)");
    }
    if (dev < 0 || dev >= MAX_DEVICES) return fail(err, err_len, NB_ECUDA, "nb_force_static: device ordinal %d not supported", dev);
    std::lock_guard<std::mutex> hold(g_dev_lock);
    StaticDev &d = g_dev[dev];
    if (!d.ready) {
        int major = 0, n_sm = 0, occ = 0;
        NBS_CUDA(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
        if (major < 10) return fail(err, err_len, NB_ECUDA, "nb_force_static: built for sm_100a, device %d is sm_%d*", dev, major);
        NBS_CUDA(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
        NBS_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_force_static<1, false>, NT_E, 0));
        double *ptr = nullptr;
        NBS_CUDA(cudaGetSymbolAddress((void **)&ptr, nb_static_scratch));
        if (!ptr) return fail(err, err_len, NB_ECUDA, "nb_force_static: cudaGetSymbolAddress returned a null address");
        d.scratch = ptr; d.n_sm = n_sm; d.occ = occ > 0 ? occ : 1;
        d.ready = true;
    }
    *out = &d;
    return NB_OK;
}

template <int JL>
void launch_static_lanes(dim3 grid, cudaStream_t st, bool g0, const double *rec, const int32_t *active, int m, int tiles, int tps,
                         double eps2, double *out, const PartLayout &L)
{
    if (g0) k_force_static<JL, true><<<grid, NT_E, 0, st>>>(rec, active, m, tiles, tps, eps2, out, L.cstride, L.kstride, L.sstride);
    else k_force_static<JL, false><<<grid, NT_E, 0, st>>>(rec, active, m, tiles, tps, eps2, out, L.cstride, L.kstride, L.sstride);
}

}  // namespace

extern "C" int nb_force_static(int64_t N, const double *pos, const double *vel, const double *acc_pred, const double *mass,
                               double eps, const int32_t *active_idx, int64_t n_active, double *acc, double *jerk, double *snap,
                               void *cuda_stream, char *err, int64_t err_len)
{
    if (err && err_len > 0) err[0] = 0;
    if (N < 1 || !pos || !vel || !mass) return fail(err, err_len, NB_EINVAL, "nb_force_static: need N >= 1 and pos, vel, mass");
    if (N > NB_STATIC_MAX_N)
        return fail(err, err_len, NB_EINVAL, "nb_force_static: N = %lld exceeds NB_STATIC_MAX_N = %d (the fixed %zu MiB device "
                    "array holds the packed records of at most that many particles); use nb_init + nb_force",
                    (long long)N, NB_STATIC_MAX_N, STATIC_DOUBLES * sizeof(double) >> 20);
    if (!(eps >= 0.0) || !isfinite(eps) || (eps > 0.0 && !(eps * eps >= 2.2250738585072014e-308)))
        return fail(err, err_len, NB_EINVAL, "nb_force_static: eps must be 0 or have a normal square");
    if (n_active < 0 || n_active > N) return fail(err, err_len, NB_EINVAL, "nb_force_static: n_active = %lld outside [0, N]", (long long)n_active);
    if (!active_idx && n_active != 0 && n_active != N)
        return fail(err, err_len, NB_EINVAL, "nb_force_static: active_idx is NULL but n_active = %lld is not N = %lld", (long long)n_active, (long long)N);
    StaticDev *d = nullptr;
    const int rc = static_setup(&d, err, err_len);
    if (rc != NB_OK) return rc;
    if (n_active == 0) return NB_OK;   // set-up only (e.g. before a capture starts)

    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int64_t Npad = (N + TILE_ALIGN - 1) / TILE_ALIGN * TILE_ALIGN;
    const int64_t m = n_active;
    double *rec = d->scratch;
    double *part = d->scratch + STATIC_REC_DOUBLES;
    // the split rule of every other driver, its partial-sum budget being what the array holds
    const ForceGeom g = choose_geom(m, Npad, d->n_sm, d->occ, (int64_t)STATIC_PART_DOUBLES, 0, 0);
    if ((size_t)g.S * 9 * (size_t)g.mpad > STATIC_PART_DOUBLES)   // cannot happen (geom_finish caps S); never write past the array
        return fail(err, err_len, NB_EINVAL, "nb_force_static: %d splits of %d slots exceed the static array", g.S, g.mpad);
    PartLayout L = part_layout(g.S, g.mpad, Npad);
    if (g.S <= 1) { L.cstride = (size_t)g.mpad; L.kstride = 1; L.sstride = 0; }   // one split: [9][mpad] in the array

    k_static_pack<<<(unsigned)((Npad + 255) / 256), 256, 0, st>>>(pos, vel, acc_pred, mass, (int)N, (int)Npad, rec);
    NBS_CUDA(cudaGetLastError());
    const dim3 grid((unsigned)g.n_ib, (unsigned)g.S, 1);
    const int tiles = (int)(Npad / TJ_E);
    const bool g0 = eps == 0.0;
    const double eps2 = eps * eps;
    switch (g.JL) {
        case 1: launch_static_lanes<1>(grid, st, g0, rec, active_idx, (int)m, tiles, g.tps, eps2, part, L); break;
        case 2: launch_static_lanes<2>(grid, st, g0, rec, active_idx, (int)m, tiles, g.tps, eps2, part, L); break;
        case 4: launch_static_lanes<4>(grid, st, g0, rec, active_idx, (int)m, tiles, g.tps, eps2, part, L); break;
        case 8: launch_static_lanes<8>(grid, st, g0, rec, active_idx, (int)m, tiles, g.tps, eps2, part, L); break;
        case 16: launch_static_lanes<16>(grid, st, g0, rec, active_idx, (int)m, tiles, g.tps, eps2, part, L); break;
        default: launch_static_lanes<32>(grid, st, g0, rec, active_idx, (int)m, tiles, g.tps, eps2, part, L); break;
    }
    NBS_CUDA(cudaGetLastError());
    if (acc || jerk || snap) {
        k_static_finish<<<(unsigned)((m * 32 + 255) / 256), 256, 0, st>>>(part, g.S, (int)m, L.cstride, L.kstride, L.sstride, acc, jerk, snap);
        NBS_CUDA(cudaGetLastError());
    }
    return NB_OK;
}
