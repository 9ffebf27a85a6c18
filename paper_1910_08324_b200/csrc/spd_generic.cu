// Any-width-set path (SURVEY.md sec. 8(a) rows a2-a7 for width sets the dyadic tree does
// not cover: the "ideal" set 1..L_max of PAPER.md:193, BoxDIT eq. (14), IGRID eq. (18), ...).
//
// Partial sums are reused through one running sum per DM row, kept in double precision in a
// plan-owned workspace:  C_d[n] = sum_{j<n} (x[d,j] - mu_d),  X_L[n] - L mu_d = C_d[n+L] - C_d[n]
// (eq. 2 with eq. 5).  Three small kernels build C (block sums, scan of the
// block sums, in-block scan); the fourth evaluates eq. (4) and the max / arg-max of eq. (12)
// for every sample, visiting the widths in ascending order with a strict '>'.
// This path favours generality over speed; the dyadic tree (spd_tree.cu) is the fast path.
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#include "spd_internal.h"

namespace spd {
namespace {

constexpr int kScanThreads = 256;
constexpr int kScanItems = 8;
constexpr int kScanBlock = kScanThreads * kScanItems;  // samples per scan block

// Block-wide inclusive scan of one double per thread; returns the exclusive prefix of the
// calling thread and the block total in *total.
__device__ __forceinline__ double block_exclusive_scan(double v, double* smem, double* total) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    double incl = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const double u = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += u;
    }
    if (lane == 31) smem[warp] = incl;
    __syncthreads();
    if (warp == 0) {
        double w = lane < (kScanThreads / 32) ? smem[lane] : 0.0;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const double u = __shfl_up_sync(0xffffffffu, w, o);
            if (lane >= o) w += u;
        }
        if (lane < (kScanThreads / 32)) smem[32 + lane] = w;  // inclusive over warps
    }
    __syncthreads();
    const double warp_off = warp > 0 ? smem[32 + warp - 1] : 0.0;
    *total = smem[32 + kScanThreads / 32 - 1];
    return warp_off + incl - v;
}

__global__ void __launch_bounds__(kScanThreads) generic_block_sums(const float* __restrict__ plane,
                                                                     const float* __restrict__ mean, long long n_t,
                                                                     long long blocks_per_row,
                                                                     double* __restrict__ blocksum) {
    __shared__ double smem[64];
    const long long d = blockIdx.x / blocks_per_row;
    const long long b = blockIdx.x - d * blocks_per_row;
    const float* row = plane + d * n_t;
    const double mu = static_cast<double>(mean[d]);
    const long long base = b * kScanBlock;
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < kScanItems; ++i) {
        const long long n = base + threadIdx.x + static_cast<long long>(i) * kScanThreads;
        if (n < n_t) s += static_cast<double>(row[n]) - mu;
    }
    double total;
    block_exclusive_scan(s, smem, &total);
    if (threadIdx.x == 0) blocksum[blockIdx.x] = total;
}

// One block per row: exclusive scan of that row's block sums, in place.
__global__ void __launch_bounds__(kScanThreads) generic_scan_block_sums(double* __restrict__ blocksum,
                                                                          long long blocks_per_row) {
    __shared__ double smem[64];
    double* row = blocksum + static_cast<long long>(blockIdx.x) * blocks_per_row;
    const long long per = (blocks_per_row + kScanThreads - 1) / kScanThreads;
    const long long lo = min(static_cast<long long>(threadIdx.x) * per, blocks_per_row);
    const long long hi = min(lo + per, blocks_per_row);
    double s = 0.0;
    for (long long i = lo; i < hi; ++i) s += row[i];
    double total;
    double run = block_exclusive_scan(s, smem, &total);
    for (long long i = lo; i < hi; ++i) {
        const double v = row[i];
        row[i] = run;
        run += v;
    }
}

// C_d[n + 1] for the samples of one scan block; C_d[0] = 0.
__global__ void __launch_bounds__(kScanThreads) generic_write_prefix(const float* __restrict__ plane,
                                                                       const float* __restrict__ mean, long long n_t,
                                                                       long long blocks_per_row,
                                                                       const double* __restrict__ blocksum,
                                                                       double* __restrict__ prefix) {
    __shared__ double smem[64];
    const long long d = blockIdx.x / blocks_per_row;
    const long long b = blockIdx.x - d * blocks_per_row;
    const float* row = plane + d * n_t;
    double* crow = prefix + d * (n_t + 1);
    const double mu = static_cast<double>(mean[d]);
    const long long first = b * kScanBlock + static_cast<long long>(threadIdx.x) * kScanItems;
    double v[kScanItems];
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < kScanItems; ++i) {
        const long long n = first + i;
        v[i] = n < n_t ? static_cast<double>(row[n]) - mu : 0.0;
        s += v[i];
    }
    double total;
    double run = blocksum[blockIdx.x] + block_exclusive_scan(s, smem, &total);
    if (b == 0 && threadIdx.x == 0) crow[0] = 0.0;
#pragma unroll
    for (int i = 0; i < kScanItems; ++i) {
        const long long n = first + i;
        run += v[i];
        if (n < n_t) crow[n + 1] = run;
    }
}

__global__ void __launch_bounds__(256) generic_eval(const double* __restrict__ prefix,
                                                    const float* __restrict__ sigma,
                                                    const int32_t* __restrict__ widths,
                                                    const float* __restrict__ wscale, int n_w, long long n_t,
                                                    long long tiles_per_row, float* __restrict__ out_snr,
                                                    int32_t* __restrict__ out_width) {
    const long long d = blockIdx.x / tiles_per_row;
    const long long tile = blockIdx.x - d * tiles_per_row;
    const long long n = tile * 256 + threadIdx.x;
    if (n >= n_t) return;
    const double* crow = prefix + d * (n_t + 1);
    const float inv = 1.0f / sigma[d];
    const double c0 = crow[n];
    const long long room = n_t - n;
    float best = __int_as_float(0xff800000);
    int idx = -1;
    for (int k = 0; k < n_w; ++k) {
        const int L = __ldg(widths + k);
        if (L > room) break;  // valid windows only (reading A3); widths ascend
        const float x = static_cast<float>(crow[n + L] - c0);
        const float snr = x * (__ldg(wscale + k) * inv);  // eq. (4) with eq. (5)
        if (snr > best) {                                 // strict '>'
            best = snr;
            idx = k;
        }
    }
    out_snr[d * n_t + n] = best;
    out_width[d * n_t + n] = idx;
}

}  // namespace

int generic_configure(spd_plan* plan) {
    const int n_w = static_cast<int>(plan->widths.size());
    std::vector<float> scale(n_w);
    for (int k = 0; k < n_w; ++k) scale[k] = static_cast<float>(1.0 / sqrt(static_cast<double>(plan->widths[k])));
    plan->generic_blocks_per_row = (plan->n_t + kScanBlock - 1) / kScanBlock;
    const size_t prefix_bytes = sizeof(double) * static_cast<size_t>(plan->n_dm) * static_cast<size_t>(plan->n_t + 1);
    const size_t bs_bytes = sizeof(double) * static_cast<size_t>(plan->n_dm) * plan->generic_blocks_per_row;
    if (plan->n_dm * plan->generic_blocks_per_row > 0x7fffffffll ||
        plan->n_dm * ((plan->n_t + 255) / 256) > 0x7fffffffll) {
        set_error("plane too large for the generic path's 1-D grids");
        return SPD_ERR_INVALID_ARG;
    }
    cudaError_t e;
    if ((e = cudaMalloc(&plan->d_widths, sizeof(int32_t) * n_w)) != cudaSuccess ||
        (e = cudaMalloc(&plan->d_wscale, sizeof(float) * n_w)) != cudaSuccess ||
        (e = cudaMalloc(&plan->d_prefix, prefix_bytes)) != cudaSuccess ||
        (e = cudaMalloc(&plan->d_blocksum, bs_bytes)) != cudaSuccess) {
        set_error("device allocation of the generic workspace (%zu bytes) failed: %s", prefix_bytes + bs_bytes,
                  cudaGetErrorString(e));
        cudaGetLastError();
        generic_release(plan);
        return SPD_ERR_ALLOC;
    }
    plan->workspace_bytes = static_cast<int64_t>(prefix_bytes + bs_bytes);
    if ((e = cudaMemcpy(plan->d_widths, plan->widths.data(), sizeof(int32_t) * n_w, cudaMemcpyHostToDevice)) !=
            cudaSuccess ||
        (e = cudaMemcpy(plan->d_wscale, scale.data(), sizeof(float) * n_w, cudaMemcpyHostToDevice)) != cudaSuccess) {
        generic_release(plan);
        return cuda_fail(e, "uploading the width table");
    }
    return SPD_OK;
}

void generic_release(spd_plan* plan) {
    cudaFree(plan->d_widths);
    cudaFree(plan->d_wscale);
    cudaFree(plan->d_prefix);
    cudaFree(plan->d_blocksum);
    plan->d_widths = nullptr;
    plan->d_wscale = nullptr;
    plan->d_prefix = nullptr;
    plan->d_blocksum = nullptr;
}

int generic_run(const spd_plan* plan, int64_t n_dm, const float* plane, const float* mean, const float* sigma,
                float* out_snr, int32_t* out_width, cudaStream_t stream) {
    const long long n_t = plan->n_t;
    const long long bpr = plan->generic_blocks_per_row;
    const unsigned scan_grid = static_cast<unsigned>(n_dm * bpr);
    generic_block_sums<<<scan_grid, kScanThreads, 0, stream>>>(plane, mean, n_t, bpr, plan->d_blocksum);
    generic_scan_block_sums<<<static_cast<unsigned>(n_dm), kScanThreads, 0, stream>>>(plan->d_blocksum, bpr);
    generic_write_prefix<<<scan_grid, kScanThreads, 0, stream>>>(plane, mean, n_t, bpr, plan->d_blocksum,
                                                                 plan->d_prefix);
    const long long tiles = (n_t + 255) / 256;
    generic_eval<<<static_cast<unsigned>(n_dm * tiles), 256, 0, stream>>>(
        plan->d_prefix, sigma, plan->d_widths, plan->d_wscale, static_cast<int>(plan->widths.size()), n_t, tiles,
        out_snr, out_width);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "launching the generic kernels");
    return SPD_OK;
}

}  // namespace spd
