// Threshold + 1-D peak candidate stage.
//
// The paper only names this stage ("candidates are selected using a peak-finding
// algorithm"; "basic candidate selection (peak-finding)").
// Reading A9: (d, n) is a candidate iff Y[d,n] >= thr, Y[d,n] > Y[d,n-1]
// and Y[d,n] >= Y[d,n+1], row ends comparing against -inf, i.e. the first sample of
// a local-maximum plateau.  Candidates are appended to a bounded list with one
// atomic per warp; the count keeps running past the capacity (overflow report).
#include <cuda_runtime.h>
#include <stdint.h>

#include "spd_internal.h"

namespace spd {
namespace {

constexpr int kCandThreads = 256;
constexpr int kCandPerThread = 4;
constexpr int kCandTile = kCandThreads * kCandPerThread;

__global__ void __launch_bounds__(kCandThreads) find_candidates_kernel(
    const float* __restrict__ snr, const int32_t* __restrict__ width, long long n_t, long long tiles_per_row,
    float thr, spd_candidate* __restrict__ list, unsigned long long capacity, unsigned long long* __restrict__ n_found) {
    const long long d = blockIdx.x / tiles_per_row;
    const long long tile = blockIdx.x - d * tiles_per_row;
    const float* y = snr + d * n_t;
    const long long n0 = tile * kCandTile + static_cast<long long>(threadIdx.x) * kCandPerThread;
    const float ninf = __int_as_float(0xff800000);
    const unsigned lane = threadIdx.x & 31u;

    // y[n0-1 .. n0+4]; n_t % 4 == 0 is not assumed, so loads are scalar and guarded.
    float v[kCandPerThread + 2];
#pragma unroll
    for (int i = 0; i < kCandPerThread + 2; ++i) {
        const long long n = n0 - 1 + i;
        v[i] = (n >= 0 && n < n_t) ? __ldg(y + n) : ninf;
    }
#pragma unroll
    for (int i = 0; i < kCandPerThread; ++i) {
        const long long n = n0 + i;
        const float c = v[i + 1];
        const bool hit = n < n_t && c >= thr && c > v[i] && c >= v[i + 2];
        const unsigned mask = __ballot_sync(0xffffffffu, hit);
        if (mask == 0u) continue;
        unsigned long long base = 0;
        const int leader = __ffs(mask) - 1;
        if (static_cast<int>(lane) == leader) base = atomicAdd(n_found, static_cast<unsigned long long>(__popc(mask)));
        base = __shfl_sync(0xffffffffu, base, leader);
        if (hit) {
            const unsigned long long slot = base + __popc(mask & ((1u << lane) - 1u));
            if (slot < capacity) {
                spd_candidate cnd;
                cnd.dm = static_cast<int32_t>(d);
                cnd.t = static_cast<int32_t>(n);
                cnd.snr = c;
                cnd.width_idx = __ldg(width + d * n_t + n);
                list[slot] = cnd;
            }
        }
    }
}

}  // namespace

int candidates_run(const spd_plan* plan, const float* out_snr, const int32_t* out_width, float threshold,
                   spd_candidate* list, int64_t capacity, int64_t* n_found, cudaStream_t stream) {
    cudaError_t e = cudaMemsetAsync(n_found, 0, sizeof(int64_t), stream);
    if (e != cudaSuccess) return cuda_fail(e, "clearing the candidate counter");
    const long long tiles = (plan->n_t + kCandTile - 1) / kCandTile;
    if (plan->n_dm * tiles > 0x7fffffffll) {
        set_error("plane too large for the candidate grid");
        return SPD_ERR_INVALID_ARG;
    }
    find_candidates_kernel<<<static_cast<unsigned>(plan->n_dm * tiles), kCandThreads, 0, stream>>>(
        out_snr, out_width, plan->n_t, tiles, threshold, list, static_cast<unsigned long long>(capacity),
        reinterpret_cast<unsigned long long*>(n_found));
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "launching the candidate kernel");
    return SPD_OK;
}

}  // namespace spd
