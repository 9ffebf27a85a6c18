// Per-DM mean and standard deviation of the plane (the step that
// feeds mu, sigma of eq. (4)/(5) into the hot path).
//
// PAPER.md:720-726 (sec. 4.6.2): "a streaming algorithm by Chan et al. [1983]" for the mean and
// the standard deviation, and "point-wise outlier rejection. Each point is compared with the
// current estimate of the mean and standard deviation and rejected if it is significantly
// different (the threshold is user defined). This is repeated until convergence."
//
// Reading (A14): pass 0 takes every sample; each further pass takes the samples with
// |x - mu| <= clip * sigma of the previous pass (comparison in float32 on the float32 mu, sigma
// the caller receives - the oracle decides in double and counts the border-line samples); sigma is
// the population standard deviation (ddof 0, as reading A6).  The caller fixes the number of
// rejection passes (spd_row_stats), or gives a limit and a tolerance (spd_row_stats_converge):
// "until convergence" is then tested on the device, per row, on the double-precision estimates of
// consecutive passes, and the blocks of a converged row return at once in the passes that follow.
//
// Partial statistics (n, mean, M2) are combined with the pairwise update of Chan, Golub &
// LeVeque: delta = mean_b - mean_a, mean = mean_a + delta n_b / n,
// M2 = M2_a + M2_b + delta^2 n_a n_b / n.  A thread accumulates its samples as shifted sums
// (shift = first sample of its block's part; four samples at a time in float32, then double), threads and parts are then merged
// pairwise in a fixed order, so the result does not depend on scheduling.
// One pass reads the plane once: 4 B per sample, HBM-bound.
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#include <algorithm>
#include <mutex>

#include "spd_internal.h"

namespace spd {
namespace {

constexpr int kStatThreads = 256;

struct Moments {
    double n, mean, m2;
};

// Per-row state of the iteration (plan workspace): estimates of the last pass in double.
struct RowState {
    int32_t converged, passes;
    double mu, sg;
};

__device__ __forceinline__ Moments merge(const Moments a, const Moments b) {
    if (b.n == 0.0) return a;
    if (a.n == 0.0) return b;
    Moments r;
    r.n = a.n + b.n;
    const double delta = b.mean - a.mean;
    const double f = b.n / r.n;
    r.mean = a.mean + delta * f;
    r.m2 = a.m2 + b.m2 + delta * delta * a.n * f;
    return r;
}

__device__ __forceinline__ Moments shfl_down(const Moments v, int o) {
    Moments r;
    r.n = __shfl_down_sync(0xffffffffu, v.n, o);
    r.mean = __shfl_down_sync(0xffffffffu, v.mean, o);
    r.m2 = __shfl_down_sync(0xffffffffu, v.m2, o);
    return r;
}

// Block b of row d reduces samples [b * part, min((b+1) * part, n_t)) to one Moments.
// clip_on: keep only |x - mu[d]| <= clip * sigma[d] (float32 comparison).
template <bool VEC>
__global__ void __launch_bounds__(kStatThreads) row_moments_kernel(const float* __restrict__ plane, long long n_t,
                                                                   long long part, int parts, int clip_on,
                                                                   float clip, const float* __restrict__ mean,
                                                                   const float* __restrict__ sigma,
                                                                   const RowState* __restrict__ state,
                                                                   Moments* __restrict__ out) {
    __shared__ Moments warp_m[kStatThreads / 32];
    const long long d = blockIdx.x / parts;
    if (clip_on && state[d].converged) return;  // this row's iteration has stopped
    const int b = blockIdx.x - static_cast<int>(d) * parts;
    const float* __restrict__ row = plane + d * n_t;
    const long long lo = static_cast<long long>(b) * part;
    const long long hi = min(lo + part, n_t);
    float mu = 0.f, lim = 0.f;
    if (clip_on) {
        mu = mean[d];
        lim = clip * sigma[d];
    }
    const float shift = lo < hi ? __ldg(row + lo) : 0.f;
    // Shifted sums: x - shift and the sums over one float4 in float32 (a sum of 4 terms each
    // rounded to 2^-24 relative), everything longer in double.
    double s1 = 0.0, s2 = 0.0;
    unsigned int cnt = 0;
    auto keep = [&](float x) { return !clip_on || fabsf(x - mu) <= lim; };
    if constexpr (VEC) {  // n_t % 4 == 0, part % 4 == 0 and an aligned plane: float4 loads
#pragma unroll 4
        for (long long n = lo + 4ll * threadIdx.x; n < hi; n += 4ll * kStatThreads) {
            const float4 v = __ldg(reinterpret_cast<const float4*>(row + n));
            const bool k0 = keep(v.x), k1 = keep(v.y), k2 = keep(v.z), k3 = keep(v.w);
            const float a0 = k0 ? v.x - shift : 0.f, a1 = k1 ? v.y - shift : 0.f;
            const float a2 = k2 ? v.z - shift : 0.f, a3 = k3 ? v.w - shift : 0.f;
            s1 += static_cast<double>((a0 + a1) + (a2 + a3));
            s2 += static_cast<double>((a0 * a0 + a1 * a1) + (a2 * a2 + a3 * a3));
            cnt += static_cast<unsigned>(k0) + k1 + k2 + k3;
        }
    } else {
        for (long long n = lo + threadIdx.x; n < hi; n += kStatThreads) {
            const float x = __ldg(row + n);
            if (keep(x)) {
                const float a = x - shift;
                s1 += static_cast<double>(a);
                s2 += static_cast<double>(a * a);
                ++cnt;
            }
        }
    }
    Moments m;
    m.n = static_cast<double>(cnt);
    m.mean = cnt ? static_cast<double>(shift) + s1 / m.n : 0.0;
    m.m2 = cnt ? fmax(s2 - s1 * s1 / m.n, 0.0) : 0.0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const Moments other = shfl_down(m, o);
        m = merge(m, other);
    }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (lane == 0) warp_m[warp] = m;
    __syncthreads();
    if (threadIdx.x == 0) {
        Moments t = warp_m[0];
#pragma unroll
        for (int w = 1; w < kStatThreads / 32; ++w) t = merge(t, warp_m[w]);
        out[blockIdx.x] = t;
    }
}

// One thread per row: merge its parts in order, write float32 mean and population sigma, and decide
// whether the row's iteration stops ("repeated until convergence").
__global__ void row_moments_finish_kernel(const Moments* __restrict__ parts_m, int parts, long long n_dm, int pass,
                                          float rel_tol, RowState* __restrict__ state, float* __restrict__ mean,
                                          float* __restrict__ sigma, int32_t* __restrict__ n_passes) {
    const long long d = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (d >= n_dm) return;
    RowState st = state[d];
    if (pass == 0) {
        st.converged = 0;
        st.passes = 0;
    } else if (st.converged) {
        return;
    }
    Moments t = parts_m[d * parts];
    for (int b = 1; b < parts; ++b) t = merge(t, parts_m[d * parts + b]);
    if (t.n == 0.0) {
        // no sample survived the rejection: keep the previous estimate and stop
        st.converged = 1;
    } else {
        const double mu = t.mean, sg = sqrt(t.m2 / t.n);
        if (pass > 0) {
            st.passes = pass;
            if (rel_tol >= 0.0f && fabs(mu - st.mu) <= static_cast<double>(rel_tol) * st.sg &&
                fabs(sg - st.sg) <= static_cast<double>(rel_tol) * st.sg)
                st.converged = 1;
        }
        st.mu = mu;
        st.sg = sg;
        mean[d] = static_cast<float>(mu);
        sigma[d] = static_cast<float>(sg);
    }
    state[d] = st;
    if (n_passes) n_passes[d] = st.passes;
}

}  // namespace

int stats_configure(spd_plan* plan) {
    // enough blocks to fill the machine, parts a multiple of 1024 samples
    const long long want = 16ll * plan->sm_count;
    long long parts = std::max<long long>(1, std::min<long long>(256, (want + plan->n_dm - 1) / plan->n_dm));
    long long part = (plan->n_t + parts - 1) / parts;
    part = (part + 1023) / 1024 * 1024;
    parts = (plan->n_t + part - 1) / part;
    plan->stats_parts = static_cast<int>(parts);
    plan->stats_part = part;
    if (plan->n_dm * parts > 0x7fffffffll) {
        set_error("plane too large for the statistics grid");
        return SPD_ERR_INVALID_ARG;
    }
    const size_t bytes = sizeof(Moments) * static_cast<size_t>(plan->n_dm) * static_cast<size_t>(parts);
    const cudaError_t e = cudaMalloc(&plan->d_stats, bytes);
    if (e != cudaSuccess) {
        set_error("device allocation of the statistics workspace (%zu bytes) failed: %s", bytes,
                  cudaGetErrorString(e));
        cudaGetLastError();
        return SPD_ERR_ALLOC;
    }
    plan->workspace_bytes += static_cast<int64_t>(bytes);
    const size_t sbytes = sizeof(RowState) * static_cast<size_t>(plan->n_dm);
    void* st = nullptr;
    const cudaError_t e2 = cudaMalloc(&st, sbytes);
    if (e2 != cudaSuccess) {
        set_error("device allocation of the statistics state (%zu bytes) failed: %s", sbytes, cudaGetErrorString(e2));
        cudaGetLastError();
        return SPD_ERR_ALLOC;
    }
    plan->d_stats_state = static_cast<int32_t*>(st);
    plan->workspace_bytes += static_cast<int64_t>(sbytes);
    return SPD_OK;
}

void stats_release(spd_plan* plan) {
    cudaFree(plan->d_stats);
    cudaFree(plan->d_stats_state);
    plan->d_stats = nullptr;
    plan->d_stats_state = nullptr;
}

int stats_run(const spd_plan* plan, const float* plane, float clip, int n_iter, float rel_tol, float* mean,
              float* sigma, int32_t* n_passes, cudaStream_t stream) {
    Moments* ws = static_cast<Moments*>(plan->d_stats);
    RowState* state = reinterpret_cast<RowState*>(plan->d_stats_state);
    const int parts = plan->stats_parts;
    const unsigned grid = static_cast<unsigned>(plan->n_dm * parts);
    const bool vec = plan->n_t % 4 == 0 && (reinterpret_cast<uintptr_t>(plane) & 15u) == 0;
    const unsigned fin_grid = static_cast<unsigned>((plan->n_dm + 127) / 128);
    for (int pass = 0; pass <= n_iter; ++pass) {
        const int clip_on = pass > 0;
        if (vec)
            row_moments_kernel<true><<<grid, kStatThreads, 0, stream>>>(plane, plan->n_t, plan->stats_part, parts,
                                                                        clip_on, clip, mean, sigma, state, ws);
        else
            row_moments_kernel<false><<<grid, kStatThreads, 0, stream>>>(plane, plan->n_t, plan->stats_part, parts,
                                                                         clip_on, clip, mean, sigma, state, ws);
        row_moments_finish_kernel<<<fin_grid, 128, 0, stream>>>(ws, parts, plan->n_dm, pass, rel_tol, state, mean,
                                                                sigma, n_passes);
    }
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "launching the statistics kernels");
    return SPD_OK;
}

// ------------------------------------------------------------------------------------------------------------
// spd_row_stats_static: the same two kernels with their scratch (partial moments per (row, part), per-row state)
// in a file-scope device array instead of a plan workspace, for callers that may not allocate (CUDA graph
// capture, serving loops).  No plan, no cudaMalloc / cudaFree, nothing but kernel launches and one memset on
// the caller's stream.
// ------------------------------------------------------------------------------------------------------------
namespace {

constexpr long long kStaticMaxRows = SPD_STATIC_MAX_ROWS;          // RowState entries
constexpr long long kStaticMaxPartials = SPD_STATIC_MAX_PARTIALS;  // Moments entries (rows x parts)
constexpr size_t kStaticStateOff = sizeof(Moments) * static_cast<size_t>(kStaticMaxPartials);
constexpr size_t kStaticBytes = kStaticStateOff + sizeof(RowState) * static_cast<size_t>(kStaticMaxRows);
static_assert(kStaticBytes == SPD_STATIC_SCRATCH_BYTES, "spd.h states the size of the scratch");
static_assert(kStaticStateOff % 256 == 0, "the per-row state starts on a 256-byte boundary");
static_assert(kStaticBytes <= (2u << 20), "the static scratch is meant to stay modest (2 MiB)");

// Held by every device that loads the library, until exit.  In host code this NAME is a host-side stand-in,
// not a device address: host code takes the address with cudaGetSymbolAddress (static_scratch below).
static __device__ __align__(256) unsigned char g_stats_scratch[kStaticBytes];

constexpr int kMaxDevices = 64;
struct StaticSlot {
    bool ready = false;
    unsigned char* base = nullptr;  // device address of g_stats_scratch on this device
    int sm_count = 0;
};
StaticSlot g_static_slot[kMaxDevices];
std::mutex g_static_mutex;

// Set-up, once per device, with that device current: device check (sm_100 only, as every other entry point),
// SM count, device address of the scratch array.
int static_scratch(StaticSlot* out) {
    int device = -1;
    cudaError_t e = cudaGetDevice(&device);
    if (e != cudaSuccess) {
        set_error("no usable CUDA device: %s (this library has no CPU fallback)", cudaGetErrorString(e));
        cudaGetLastError();
        return SPD_ERR_UNSUPPORTED_DEVICE;
    }
    if (device < 0 || device >= kMaxDevices) {
        set_error("spd_row_stats_static: device ordinal %d outside 0 .. %d", device, kMaxDevices - 1);
        return SPD_ERR_UNSUPPORTED_DEVICE;
    }
    std::lock_guard<std::mutex> lock(g_static_mutex);
    StaticSlot& slot = g_static_slot[device];
    if (!slot.ready) {
        int major = 0, sms = 0;
        if ((e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, device)) != cudaSuccess ||
            (e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device)) != cudaSuccess) {
            set_error("cannot query the CUDA device: %s", cudaGetErrorString(e));
            cudaGetLastError();
            return SPD_ERR_UNSUPPORTED_DEVICE;
        }
        if (major != 10) {
            set_error("device compute capability %d.x is not supported: this library is built for sm_100a only", major);
            return SPD_ERR_UNSUPPORTED_DEVICE;
        }
        void* ptr = nullptr;
        e = cudaGetSymbolAddress(&ptr, g_stats_scratch);
        if (e != cudaSuccess || !ptr) {
            set_error("spd_row_stats_static: cudaGetSymbolAddress of the scratch array failed: %s",
                      cudaGetErrorString(e));
            cudaGetLastError();
            return SPD_ERR_CUDA;
        }
        slot.base = static_cast<unsigned char*>(ptr);
        slot.sm_count = sms;
        slot.ready = true;
    }
    *out = slot;
    return SPD_OK;
}

}  // namespace
}  // namespace spd

extern "C" int spd_row_stats_static(const float* plane, int64_t n_dm, int64_t n_t, float clip_sigma,
                                    int32_t n_reject_passes, float* mean, float* sigma, void* cuda_stream) {
    using namespace spd;
    if (!plane || !mean || !sigma) {
        set_error("spd_row_stats_static: NULL argument");
        return SPD_ERR_INVALID_ARG;
    }
    if (n_dm < 1 || n_t < 1) {
        set_error("spd_row_stats_static: need n_dm >= 1 and n_t >= 1 (got %lld, %lld)", static_cast<long long>(n_dm),
                  static_cast<long long>(n_t));
        return SPD_ERR_INVALID_ARG;
    }
    if (n_reject_passes < 0 || n_reject_passes > 64 || (n_reject_passes > 0 && !(clip_sigma > 0.0f))) {
        set_error("spd_row_stats_static: need 0 <= n_reject_passes <= 64 and clip_sigma > 0 when rejecting (got %d, %g)",
                  n_reject_passes, static_cast<double>(clip_sigma));
        return SPD_ERR_INVALID_ARG;
    }
    if (n_dm > kStaticMaxRows) {
        set_error("spd_row_stats_static: n_dm = %lld exceeds the static scratch (SPD_STATIC_MAX_ROWS = %lld rows); "
                  "use spd_row_stats with a plan",
                  static_cast<long long>(n_dm), kStaticMaxRows);
        return SPD_ERR_INVALID_ARG;
    }
    StaticSlot slot;
    const int rc = static_scratch(&slot);
    if (rc != SPD_OK) return rc;

    // the work split of stats_configure (enough blocks to fill the machine, parts a multiple of 1024 samples),
    // with the parts per row also bounded by the scratch
    const long long want = 16ll * slot.sm_count;
    long long parts = std::max<long long>(1, std::min<long long>(256, (want + n_dm - 1) / n_dm));
    parts = std::max<long long>(1, std::min<long long>(parts, kStaticMaxPartials / n_dm));
    long long part = (n_t + parts - 1) / parts;
    part = (part + 1023) / 1024 * 1024;
    parts = (n_t + part - 1) / part;

    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    Moments* const ws = reinterpret_cast<Moments*>(slot.base);
    RowState* const state = reinterpret_cast<RowState*>(slot.base + kStaticStateOff);
    // the array keeps the last call's contents: the per-row state starts at zero (not converged, no pass done);
    // the partial moments are all written by pass 0 before they are read
    cudaError_t e = cudaMemsetAsync(state, 0, sizeof(RowState) * static_cast<size_t>(n_dm), stream);
    if (e != cudaSuccess) return cuda_fail(e, "clearing the static statistics state");
    const unsigned grid = static_cast<unsigned>(n_dm * parts);  // <= kStaticMaxPartials
    const bool vec = n_t % 4 == 0 && (reinterpret_cast<uintptr_t>(plane) & 15u) == 0;
    const unsigned fin_grid = static_cast<unsigned>((n_dm + 127) / 128);
    for (int pass = 0; pass <= n_reject_passes; ++pass) {
        const int clip_on = pass > 0;
        if (vec)
            row_moments_kernel<true><<<grid, kStatThreads, 0, stream>>>(plane, n_t, part, static_cast<int>(parts), clip_on,
                                                                        clip_sigma, mean, sigma, state, ws);
        else
            row_moments_kernel<false><<<grid, kStatThreads, 0, stream>>>(plane, n_t, part, static_cast<int>(parts),
                                                                         clip_on, clip_sigma, mean, sigma, state, ws);
        row_moments_finish_kernel<<<fin_grid, 128, 0, stream>>>(ws, static_cast<int>(parts), n_dm, pass, -1.0f, state,
                                                                mean, sigma, nullptr);
    }
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "launching the statistics kernels (static scratch)");
    return SPD_OK;
}
