// Standard deviation per boxcar width, measured on the data (second half).
//
// PAPER.md:728 (sec. 4.6.2): "we calculate values of the standard deviation only for time-series
// which are decimations of the input time-series in time, i.e. we calculate the standard deviation
// only for boxcar filters of width that are equal to a powers of two.  We then interpolate values of
// standard deviation for all intermediate boxcar widths."  It replaces eq. (5)'s white-noise
// sigma(X_L) = sqrt(L) sigma on real data (Fig. 24).
//
// Reading (A17): level j is the series of sums of 2^j consecutive samples,
// x^j[m] = sum_{i < 2^j} x[2^j m + i], m < floor(n_t / 2^j) (eq. 13 with D = 2, without its shift);
// sigma_j is its population standard deviation; for 2^j <= L < 2^(j+1) sigma_L is linear in L
// between sigma_j and sigma_(j+1); above the last level with two elements, sqrt(L) from that level.
//
// width_moments_kernel: a block walks "super-blocks" of 8192 samples of one row; the decimations
// are formed by repeated pairwise sums in float32 - levels 0..5 in a thread's registers (32
// consecutive samples each), 5..8 in the registers of one warp, 8..13 across its lanes by shuffles -
// and every level adds its elements to shifted sums S1 = sum(v - 2^j mu), S2 = sum(v - 2^j mu)^2 kept
// in double.  Block-reduced in a fixed order -> one partial per (row, part, level); the super-block
// totals are kept for the levels above 8192.  width_sigma_finish_kernel (one block per row) merges the
// partials in order, builds the levels above 8192 from the totals, and interpolates the plan's
// widths.  Reads the plane once: 4 B per sample, HBM-bound; results do not depend on scheduling.
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#include <algorithm>

#include "spd_internal.h"
#include "spd_tree_common.cuh"  // mbarrier + 1-D bulk copy helpers

namespace spd {
namespace {

constexpr int kWsgThreads = 256;
constexpr int kWsgLog = 13;
constexpr int kWsgBlock = 1 << kWsgLog;  // samples per super-block
constexpr int kWsgLevels = kWsgLog + 1;  // levels 0 .. 13 inside a super-block
constexpr int kWsgMaxLevels = 32;

struct LevelSums {
    double s1, s2;
};

__device__ __forceinline__ double block_sum(double v, double* scratch) {
    // fixed order: lanes by shuffle, then warps serially
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    __syncthreads();
    if (lane == 0) scratch[warp] = v;
    __syncthreads();
    double t = 0.0;
    if (threadIdx.x == 0)
        for (int w = 0; w < kWsgThreads / 32; ++w) t += scratch[w];
    return t;  // valid in thread 0
}

// Adds the n values v[0..n) of level j (sums of 2^j samples, first sample at `first` of the
// super-block) to the level's shifted sums; only groups that end inside the row count.
template <int N>
__device__ __forceinline__ void level_add(const float (&v)[N], int j, long long first, long long avail, float shift,
                                          double& s1, double& s2) {
    float a = 0.f, b = 0.f;
#pragma unroll
    for (int i = 0; i < N; ++i) {
        if (first + (static_cast<long long>(i + 1) << j) <= avail) {
            const float u = v[i] - shift;
            a += u;
            b = fmaf(u, u, b);
        }
    }
    s1 += static_cast<double>(a);
    s2 += static_cast<double>(b);
}

// TMA variant (rows 16-byte aligned): the full super-blocks of a block's part arrive by 1-D bulk copies through
// a ring of kWsgStages stages of 32 KB, so that two to three super-blocks per block are in flight whatever the
// threads are doing (with plain loads a thread's 128 B were requested, awaited and consumed in turn: 3.2 TB/s).
// A thread reads its 8 float4 in the order q ^ (t & 7): consecutive threads are 128 B apart, the rotation spreads
// a quarter-warp over all banks; XOR by a constant maps aligned blocks of 2^k float4 onto aligned blocks, so every
// level still sums the same groups - only the order of a thread's additions changes.
constexpr int kWsgStages = 3;
constexpr size_t kWsgRingBytes = static_cast<size_t>(kWsgStages) * kWsgBlock * sizeof(float);

// One block walks super-blocks of 8192 samples.  Thread t owns the 32 consecutive samples
// 32 t .. 32 t + 31: levels 0..5 in its registers; the 256 level-5 sums go through shared memory to
// warp 0, whose lane l owns 8 of them: levels 5..8 in registers, levels 8..13 across lanes by
// shuffles.  One block barrier per super-block (two buffers).  Sums of a few values are formed in
// float32 (they ARE the decimated series), the running S1 / S2 of each level in double.
template <bool TMA>
__global__ void __launch_bounds__(kWsgThreads) width_moments_kernel(const float* __restrict__ plane,
                                                                      const float* __restrict__ mean, long long n_t,
                                                                      int sb_per_row, int sb_per_part, int parts,
                                                                      LevelSums* __restrict__ partial,
                                                                      double* __restrict__ totals) {
    __shared__ float v5[2][kWsgThreads];
    __shared__ double scratch[kWsgThreads / 32];
    __shared__ __align__(8) uint64_t full[kWsgStages];
    extern __shared__ __align__(128) float ring[];  // TMA: kWsgStages stages of kWsgBlock floats
    const int d = blockIdx.x / parts;
    const int part = blockIdx.x - d * parts;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const float* __restrict__ row = plane + static_cast<long long>(d) * n_t;
    const float mu = mean[d];
    double s1[kWsgLevels], s2[kWsgLevels];
#pragma unroll
    for (int j = 0; j < kWsgLevels; ++j) s1[j] = s2[j] = 0.0;
    const int sb_lo = part * sb_per_part;
    const int sb_hi = min(sb_lo + sb_per_part, sb_per_row);
    // super-blocks [sb_lo, sb_full) are complete (only a row's last one can be ragged): they go through the ring
    const int sb_full = TMA ? min(sb_hi, static_cast<int>(n_t / kWsgBlock)) : sb_lo;
    if constexpr (TMA) {
        if (tid == 0) {
#pragma unroll
            for (int i = 0; i < kWsgStages; ++i) mbar_init(&full[i], 1);
            fence_mbar_init();
            fence_proxy_async();
#pragma unroll
            for (int i = 0; i < kWsgStages; ++i) {
                if (sb_lo + i < sb_full) {
                    mbar_arrive_expect_tx(&full[i], kWsgBlock * 4);
                    bulk_g2s(ring + i * kWsgBlock, row + static_cast<long long>(sb_lo + i) * kWsgBlock, kWsgBlock * 4,
                             &full[i]);
                }
            }
        }
        __syncthreads();
    }
    int buf = 0;
    for (int sb = sb_lo; sb < sb_hi; ++sb, buf ^= 1) {
        const long long base = static_cast<long long>(sb) * kWsgBlock;
        const long long avail = n_t - base;  // samples of the row from here on (> 0)
        const long long mine = 32ll * tid;
        const int k = sb - sb_lo, stage = k % kWsgStages;
        float x[32];
        if (TMA && sb < sb_full) {
            mbar_wait(&full[stage], (k / kWsgStages) & 1);
            const float4* s4 = reinterpret_cast<const float4*>(ring + stage * kWsgBlock) + 8 * tid;
#pragma unroll
            for (int q = 0; q < 8; ++q) {
                const float4 f = s4[q ^ (tid & 7)];
                x[4 * q] = f.x;
                x[4 * q + 1] = f.y;
                x[4 * q + 2] = f.z;
                x[4 * q + 3] = f.w;
            }
        } else if (mine + 32 <= avail && ((reinterpret_cast<uintptr_t>(row + base) & 15u) == 0)) {
            const float4* p4 = reinterpret_cast<const float4*>(row + base + mine);
#pragma unroll
            for (int q = 0; q < 8; ++q) {
                const float4 f = __ldg(p4 + q);
                x[4 * q] = f.x;
                x[4 * q + 1] = f.y;
                x[4 * q + 2] = f.z;
                x[4 * q + 3] = f.w;
            }
        } else {
#pragma unroll
            for (int i = 0; i < 32; ++i) x[i] = mine + i < avail ? __ldg(row + base + mine + i) : 0.f;
        }
        // levels 0..5 in registers (level j + 1 = sums of pairs of level j)
        level_add(x, 0, mine, avail, mu, s1[0], s2[0]);
        float y16[16], y8[8], y4[4], y2[2], y1[1];
#pragma unroll
        for (int i = 0; i < 16; ++i) y16[i] = x[2 * i] + x[2 * i + 1];
        level_add(y16, 1, mine, avail, 2.f * mu, s1[1], s2[1]);
#pragma unroll
        for (int i = 0; i < 8; ++i) y8[i] = y16[2 * i] + y16[2 * i + 1];
        level_add(y8, 2, mine, avail, 4.f * mu, s1[2], s2[2]);
#pragma unroll
        for (int i = 0; i < 4; ++i) y4[i] = y8[2 * i] + y8[2 * i + 1];
        level_add(y4, 3, mine, avail, 8.f * mu, s1[3], s2[3]);
#pragma unroll
        for (int i = 0; i < 2; ++i) y2[i] = y4[2 * i] + y4[2 * i + 1];
        level_add(y2, 4, mine, avail, 16.f * mu, s1[4], s2[4]);
        y1[0] = y2[0] + y2[1];
        v5[buf][tid] = y1[0];
        __syncthreads();  // the other buffer is free again: its readers passed this barrier one trip ago
        if constexpr (TMA) {
            // every thread has read this stage: refill it with the super-block kWsgStages ahead
            if (tid == 0 && sb < sb_full && sb + kWsgStages < sb_full) {
                mbar_arrive_expect_tx(&full[stage], kWsgBlock * 4);
                bulk_g2s(ring + stage * kWsgBlock, row + static_cast<long long>(sb + kWsgStages) * kWsgBlock,
                         kWsgBlock * 4, &full[stage]);
            }
        }
        // the upper levels of a super-block are one warp's work: the warps take turns (every thread's sums are
        // block-reduced at the end, so it does not matter whose registers hold them)
        if (warp == (TMA ? (k & (kWsgThreads / 32 - 1)) : 0)) {
            // lane l: level-5 sums 8 l .. 8 l + 7 of the super-block (first sample 256 l)
            const long long first = 256ll * lane;
            float z8[8], z4[4], z2[2], z1[1];
#pragma unroll
            for (int i = 0; i < 8; ++i) z8[i] = v5[buf][8 * lane + i];
            level_add(z8, 5, first, avail, 32.f * mu, s1[5], s2[5]);
#pragma unroll
            for (int i = 0; i < 4; ++i) z4[i] = z8[2 * i] + z8[2 * i + 1];
            level_add(z4, 6, first, avail, 64.f * mu, s1[6], s2[6]);
#pragma unroll
            for (int i = 0; i < 2; ++i) z2[i] = z4[2 * i] + z4[2 * i + 1];
            level_add(z2, 7, first, avail, 128.f * mu, s1[7], s2[7]);
            z1[0] = z2[0] + z2[1];
            // levels 8..13 across lanes: after step q the lanes that are multiples of 2^q hold level 8 + q
            float v = z1[0];
#pragma unroll
            for (int q = 0; q <= 5; ++q) {
                if ((lane & ((1 << q) - 1)) == 0) {
                    const float one[1] = {v};
                    level_add(one, 8 + q, first, avail, static_cast<float>(256 << q) * mu, s1[8 + q], s2[8 + q]);
                }
                if (q < 5) v += __shfl_down_sync(0xffffffffu, v, 1 << q);
            }
            if (lane == 0) totals[static_cast<long long>(d) * sb_per_row + sb] = static_cast<double>(v);
        }
    }
    LevelSums* out = partial + (static_cast<long long>(d) * parts + part) * kWsgLevels;
#pragma unroll
    for (int j = 0; j < kWsgLevels; ++j) {
        const double a = block_sum(s1[j], scratch);
        const double b = block_sum(s2[j], scratch);
        if (tid == 0) {
            out[j].s1 = a;
            out[j].s2 = b;
        }
    }
}

__global__ void __launch_bounds__(64) width_sigma_finish_kernel(const LevelSums* __restrict__ partial,
                                                                const double* __restrict__ totals,
                                                                const float* __restrict__ mean, long long n_t,
                                                                int sb_per_row, int parts, int n_levels,
                                                                const int32_t* __restrict__ widths, int n_w,
                                                                float* __restrict__ sigma_w) {
    __shared__ double sig[kWsgMaxLevels];
    __shared__ int n_valid;
    const int d = blockIdx.x;
    const int j = threadIdx.x;
    if (j < n_levels) {
        double sd = -1.0;  // < 0: level has fewer than two elements
        if (j < kWsgLevels) {
            double a = 0.0, b = 0.0;
            const LevelSums* p = partial + static_cast<long long>(d) * parts * kWsgLevels + j;
            for (int q = 0; q < parts; ++q) {
                a += p[q * kWsgLevels].s1;
                b += p[q * kWsgLevels].s2;
            }
            const double n = static_cast<double>(n_t >> j);  // every full group of the row was counted once
            if (n >= 2.0) sd = sqrt(fmax(0.0, (b - a * a / n) / n));
        } else {
            // groups of 2^(j - 13) complete super-blocks
            const long long g = 1ll << (j - kWsgLog);
            const long long n_groups = (n_t >> j);
            const double shift = static_cast<double>(mean[d]) * static_cast<double>(1ll << j);
            const double* t = totals + static_cast<long long>(d) * sb_per_row;
            double a = 0.0, b = 0.0;
            for (long long m = 0; m < n_groups; ++m) {
                double v = 0.0;
                for (long long i = 0; i < g; ++i) v += t[m * g + i];
                v -= shift;
                a += v;
                b += v * v;
            }
            const double n = static_cast<double>(n_groups);
            if (n_groups >= 2) sd = sqrt(fmax(0.0, (b - a * a / n) / n));
        }
        sig[j] = sd;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        int nv = 0;
        while (nv < n_levels && sig[nv] >= 0.0) ++nv;
        n_valid = nv;  // >= 1 whenever n_t >= 2
    }
    __syncthreads();
    const int nv = n_valid;
    for (int k = threadIdx.x; k < n_w; k += blockDim.x) {
        const long long L = widths[k];
        int jj = 0;
        while ((2ll << jj) <= L) ++jj;  // 2^jj <= L < 2^(jj+1)
        double sd;
        if (nv == 0) {
            sd = 0.0;
        } else if (jj + 1 < nv) {
            const double lo = static_cast<double>(1ll << jj);
            sd = sig[jj] + (sig[jj + 1] - sig[jj]) * (static_cast<double>(L) - lo) / lo;
        } else {
            const int top = nv - 1;
            sd = sig[top] * sqrt(static_cast<double>(L) / static_cast<double>(1ll << top));
        }
        sigma_w[static_cast<long long>(d) * n_w + k] = static_cast<float>(sd);
    }
}

}  // namespace

int wsig_configure(spd_plan* plan) {
    const int64_t sb_per_row = (plan->n_t + kWsgBlock - 1) / kWsgBlock;
    // parts: enough blocks to fill the machine
    const int64_t want = std::max<int64_t>(1, (16 * int64_t(plan->sm_count) + plan->n_dm - 1) / plan->n_dm);
    const int64_t parts = std::max<int64_t>(1, std::min<int64_t>(sb_per_row, want));
    plan->wsig_sb_per_part = static_cast<int>((sb_per_row + parts - 1) / parts);
    plan->wsig_parts = static_cast<int>((sb_per_row + plan->wsig_sb_per_part - 1) / plan->wsig_sb_per_part);
    plan->wsig_sb_per_row = static_cast<int>(sb_per_row);
    int levels = 0;
    while ((int64_t(1) << levels) <= plan->max_width) ++levels;  // floor(log2(max_width)) + 1
    plan->wsig_levels = std::min(levels + 1, kWsgMaxLevels);       // one above, for the interpolation
    if (plan->n_dm * int64_t(plan->wsig_parts) > 0x7fffffffll) {
        set_error("plane too large for the width-sigma grid");
        return SPD_ERR_INVALID_ARG;
    }
    const size_t pb = sizeof(LevelSums) * static_cast<size_t>(plan->n_dm) * plan->wsig_parts * kWsgLevels;
    const size_t tb = sizeof(double) * static_cast<size_t>(plan->n_dm) * sb_per_row;
    const size_t wb = sizeof(int32_t) * plan->widths.size();
    cudaError_t e;
    if ((e = cudaMalloc(&plan->d_wsig_partial, pb)) != cudaSuccess ||
        (e = cudaMalloc(&plan->d_wsig_totals, tb)) != cudaSuccess ||
        (e = cudaMalloc(&plan->d_wsig_widths, wb)) != cudaSuccess ||
        (e = cudaMemcpy(plan->d_wsig_widths, plan->widths.data(), wb, cudaMemcpyHostToDevice)) != cudaSuccess) {
        set_error("device allocation of the width-sigma workspace failed: %s", cudaGetErrorString(e));
        cudaGetLastError();
        wsig_release(plan);
        return SPD_ERR_ALLOC;
    }
    plan->workspace_bytes += static_cast<int64_t>(pb + tb + wb);
    return SPD_OK;
}

void wsig_release(spd_plan* plan) {
    cudaFree(plan->d_wsig_partial);
    cudaFree(plan->d_wsig_totals);
    cudaFree(plan->d_wsig_widths);
    plan->d_wsig_partial = nullptr;
    plan->d_wsig_totals = nullptr;
    plan->d_wsig_widths = nullptr;
}

int wsig_run(const spd_plan* plan, const float* plane, const float* mean, float* sigma_w, cudaStream_t stream) {
    LevelSums* partial = static_cast<LevelSums*>(plan->d_wsig_partial);
    double* totals = static_cast<double*>(plan->d_wsig_totals);
    const unsigned grid = static_cast<unsigned>(plan->n_dm * plan->wsig_parts);
    if (plan->n_t % 4 == 0 && (reinterpret_cast<uintptr_t>(plane) & 15u) == 0) {  // rows 16-byte aligned: bulk copies
        static bool configured = false;  // per process; the attribute is sticky
        if (!configured) {
            const cudaError_t ea = cudaFuncSetAttribute(width_moments_kernel<true>,
                                                        cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                        static_cast<int>(kWsgRingBytes));
            if (ea != cudaSuccess) return cuda_fail(ea, "configuring the width-sigma kernel");
            configured = true;
        }
        width_moments_kernel<true><<<grid, kWsgThreads, kWsgRingBytes, stream>>>(
            plane, mean, plan->n_t, plan->wsig_sb_per_row, plan->wsig_sb_per_part, plan->wsig_parts, partial, totals);
    } else {
        width_moments_kernel<false><<<grid, kWsgThreads, 0, stream>>>(
            plane, mean, plan->n_t, plan->wsig_sb_per_row, plan->wsig_sb_per_part, plan->wsig_parts, partial, totals);
    }
    width_sigma_finish_kernel<<<static_cast<unsigned>(plan->n_dm), 64, 0, stream>>>(
        partial, totals, mean, plan->n_t, plan->wsig_sb_per_row, plan->wsig_parts, plan->wsig_levels,
        static_cast<const int32_t*>(plan->d_wsig_widths), static_cast<int>(plan->widths.size()), sigma_w);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "launching the width-sigma kernels");
    return SPD_OK;
}

}  // namespace spd
