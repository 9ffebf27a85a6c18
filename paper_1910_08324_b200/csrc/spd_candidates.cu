// Threshold + 1-D peak candidate stage and the 2-D (DM x time) peak stage over
// its list (sec. 8(f) row f4, cluster_candidates_kernel below).
//
// The paper only names this stage ("candidates are selected using a peak-finding
// algorithm"; "basic candidate selection (peak-finding)").
// Reading A9: (d, n) is a candidate iff Y[d,n] >= thr, Y[d,n] > Y[d,n-1]
// and Y[d,n] >= Y[d,n+1], row ends comparing against -inf, i.e. the first sample of
// a local-maximum plateau.  Candidates are appended to a bounded list with one
// atomic per warp; the count keeps running past the capacity (overflow report).
//
// Two kernels apply the same rule:
//   * find_candidates_kernel visits every sample (any plane, any alignment);
//   * find_candidates_flagged_kernel visits only the blocks of samples whose byte in the
//     activity map is set.  The map is written by the kernel that produced Y (the
//     threshold test is fused into spd_tree.cu), so on planes where detections are rare
//     this stage reads a few per cent of Y instead of all of it.  A persistent grid of
//     warps scans the map (32 blocks per warp step) and each warp walks its flagged blocks
//     with 128-bit loads, neighbours coming from the adjacent lanes.
#include <cuda_runtime.h>
#include <stdint.h>

#include <algorithm>

#include "spd_internal.h"

namespace spd {
namespace {

constexpr int kCandThreads = 256;
constexpr int kCandPerThread = 4;
constexpr int kCandTile = kCandThreads * kCandPerThread;

// W[d, n] of a plane stored as int32, or as uint8 with 255 for -1 (SPD_FLAG_WIDTH_U8).
__device__ __forceinline__ int32_t load_width(const void* __restrict__ width, long long i, int wbytes) {
    if (wbytes == 4) return __ldg(static_cast<const int32_t*>(width) + i);
    const unsigned v = __ldg(static_cast<const uint8_t*>(width) + i);
    return v == 255u ? -1 : static_cast<int32_t>(v);
}

// Warp-aggregated append of the lanes with `hit` set.
__device__ __forceinline__ void append_hits(bool hit, long long d, long long n, float c,
                                            const void* __restrict__ width, int wbytes, long long dm_offset,
                                            long long n_t,
                                            spd_candidate* __restrict__ list, unsigned long long capacity,
                                            unsigned long long* __restrict__ n_found, unsigned lane) {
    const unsigned mask = __ballot_sync(0xffffffffu, hit);
    if (mask == 0u) return;
    unsigned long long base = 0;
    const int leader = __ffs(mask) - 1;
    if (static_cast<int>(lane) == leader) base = atomicAdd(n_found, static_cast<unsigned long long>(__popc(mask)));
    base = __shfl_sync(0xffffffffu, base, leader);
    if (hit) {
        const unsigned long long slot = base + __popc(mask & ((1u << lane) - 1u));
        if (slot < capacity) {
            spd_candidate cnd;
            cnd.dm = static_cast<int32_t>(dm_offset + d);
            cnd.t = static_cast<int32_t>(n);
            cnd.snr = c;
            cnd.width_idx = load_width(width, d * n_t + n, wbytes);
            list[slot] = cnd;
        }
    }
}

__global__ void __launch_bounds__(kCandThreads) find_candidates_kernel(
    const float* __restrict__ snr, const void* __restrict__ width, int wbytes, long long dm_offset, long long n_t,
    long long tiles_per_row, float thr, spd_candidate* __restrict__ list, unsigned long long capacity,
    unsigned long long* __restrict__ n_found) {
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
        append_hits(hit, d, n, c, width, wbytes, dm_offset, n_t, list, capacity, n_found, lane);
    }
}

// Peak test of the 4 samples a lane holds -> 4-bit mask (bit i: sample n + i is a candidate).
__device__ __forceinline__ unsigned peak_bits(float4 v, float prev, float next, float thr) {
    unsigned m = 0;
    if (v.x >= thr && v.x > prev && v.x >= v.y) m |= 1u;
    if (v.y >= thr && v.y > v.x && v.y >= v.z) m |= 2u;
    if (v.z >= thr && v.z > v.y && v.z >= v.w) m |= 4u;
    if (v.w >= thr && v.w > v.z && v.w >= next) m |= 8u;
    return m;
}

// One warp per flagged block of `block` samples (block % 128 == 0, n_t % 4 == 0), walked in
// pieces of kPiece samples: the piece's peaks are first collected as bits (4 per lane and
// 128-sample step), counted across the warp, reserved with ONE atomic per piece, and then
// written.  On planes that flood the threshold (config 5: baseline drift) this keeps the
// single counter off the critical path.
constexpr int kPiece = 2048;             // samples per reservation
constexpr int kPieceSteps = kPiece / 128;  // 16 steps x 4 bits = 64 bits per lane

__global__ void __launch_bounds__(kCandThreads) find_candidates_flagged_kernel(
    const float* __restrict__ snr, const void* __restrict__ width, int wbytes, long long dm_offset,
    const uint8_t* __restrict__ activity, long long n_flags, long long flags_per_row, long long block, long long n_t,
    float thr,
    spd_candidate* __restrict__ list, unsigned long long capacity, unsigned long long* __restrict__ n_found) {
    const unsigned lane = threadIdx.x & 31u;
    const long long warp = (static_cast<long long>(blockIdx.x) * kCandThreads + threadIdx.x) >> 5;
    const long long n_warps = (static_cast<long long>(gridDim.x) * kCandThreads) >> 5;
    const float ninf = __int_as_float(0xff800000);
    // 32 flags per warp step (one per lane): marked blocks spread over as many warps as possible
    const long long n_steps = (n_flags + 31) / 32;
    for (long long step = warp; step < n_steps; step += n_warps) {
        const long long mine = step * 32 + lane;
        const unsigned flag = mine < n_flags ? __ldg(activity + mine) : 0u;
        unsigned pending = __ballot_sync(0xffffffffu, flag != 0u);
        while (pending) {
            const int src = __ffs(pending) - 1;
            pending &= pending - 1;
            {
                const long long fi = step * 32 + src;
                const long long d = fi / flags_per_row;
                const long long b = fi - d * flags_per_row;
                const float* __restrict__ y = snr + d * n_t;
                const long long lo = b * block;
                const long long hi = min(lo + block, n_t);  // multiples of 4
                for (long long p0 = lo; p0 < hi; p0 += kPiece) {
                    const long long p1 = min(p0 + kPiece, hi);
                    // value before the first sample of the piece
                    float carry = p0 > 0 ? __ldg(y + p0 - 1) : ninf;
                    unsigned long long bits = 0ull;
                    // all loads of the piece first: one memory latency per piece, not per step
                    float4 pv[kPieceSteps];
#pragma unroll
                    for (int it = 0; it < kPieceSteps; ++it) {
                        const long long n = p0 + 128ll * it + 4 * lane;
                        pv[it] = n < p1 ? __ldg(reinterpret_cast<const float4*>(y + n))
                                        : make_float4(ninf, ninf, ninf, ninf);
                    }
#pragma unroll
                    for (int it = 0; it < kPieceSteps; ++it) {
                        const long long n = p0 + 128ll * it + 4 * lane;
                        const bool in = n < p1;
                        const float4 v = pv[it];
                        float prev = __shfl_up_sync(0xffffffffu, v.w, 1);
                        if (lane == 0) prev = carry;
                        float next = __shfl_down_sync(0xffffffffu, v.x, 1);
                        if (lane == 31) next = (in && n + 4 < n_t) ? __ldg(y + n + 4) : ninf;
                        carry = __shfl_sync(0xffffffffu, v.w, 31);
                        if (in) bits |= static_cast<unsigned long long>(peak_bits(v, prev, next, thr)) << (4 * it);
                    }
                    const unsigned mine = __popcll(bits);
                    if (!__any_sync(0xffffffffu, mine != 0u)) continue;
                    // exclusive scan of the per-lane counts, one reservation for the piece
                    unsigned incl = mine;
#pragma unroll
                    for (int o = 1; o < 32; o <<= 1) {
                        const unsigned u = __shfl_up_sync(0xffffffffu, incl, o);
                        if (lane >= static_cast<unsigned>(o)) incl += u;
                    }
                    const unsigned total = __shfl_sync(0xffffffffu, incl, 31);
                    unsigned long long base = 0;
                    if (lane == 0) base = atomicAdd(n_found, static_cast<unsigned long long>(total));
                    base = __shfl_sync(0xffffffffu, base, 0);
                    unsigned long long slot = base + (incl - mine);
                    while (bits && slot < capacity) {
                        const int bpos = __ffsll(static_cast<long long>(bits)) - 1;
                        bits &= bits - 1;
                        const long long n = p0 + 128ll * (bpos >> 2) + 4 * lane + (bpos & 3);
                        spd_candidate cnd;
                        cnd.dm = static_cast<int32_t>(dm_offset + d);
                        cnd.t = static_cast<int32_t>(n);
                        cnd.snr = __ldg(y + n);
                        cnd.width_idx = load_width(width, d * n_t + n, wbytes);
                        list[slot++] = cnd;
                    }
                }
            }
        }
    }
}

// 2-D (DM x time) peak stage over the 1-D candidates (reading A18 - the paper
// only names "peak-finding"): candidate (d, n) with best width L is kept iff no sample of
// the window |d' - d| <= R, |n' - n| <= L has a larger Y and none earlier in (d, n) order an equal one.
// One warp per candidate; the window is scanned from the candidate's own time outwards, 32 samples on
// either side per step and row, and the warp leaves at the first step that finds a dominating sample -
// the ripples around a pulse die within a step or two, only the few survivors pay for the whole window.
__global__ void __launch_bounds__(kCandThreads) cluster_candidates_kernel(
    const float* __restrict__ snr, long long n_dm, long long n_t, const int32_t* __restrict__ widths, int n_w,
    const spd_candidate* __restrict__ in, const unsigned long long* __restrict__ n_in, unsigned long long cap_in, int R,
    spd_candidate* __restrict__ out, unsigned long long cap_out, unsigned long long* __restrict__ n_out) {
    const unsigned lane = threadIdx.x & 31u;
    const long long warp = (static_cast<long long>(blockIdx.x) * kCandThreads + threadIdx.x) >> 5;
    const long long n_warps = (static_cast<long long>(gridDim.x) * kCandThreads) >> 5;
    const unsigned long long total = min(*n_in, cap_in);
    for (unsigned long long i = warp; i < total; i += n_warps) {
        const spd_candidate c = in[i];
        const long long d = c.dm, n = c.t;
        const long long L = (c.width_idx >= 0 && c.width_idx < n_w) ? __ldg(widths + c.width_idx) : 1;
        const float v = __ldg(snr + d * n_t + n);
        const long long d_lo = max(0ll, d - R), d_hi = min(n_dm - 1, d + R);
        const long long n_lo = max(0ll, n - L), n_hi = min(n_t - 1, n + L);
        bool dominated = false;
        // offsets 0 .. L on the right (own sample included: other rows need it), 1 .. L on the left
        for (long long o = 0; o <= L && !dominated; o += 32) {
            const long long nr = n + o + lane, nl = n - 1 - o - lane;
            bool bad = false;
            for (long long dd = d_lo; dd <= d_hi; ++dd) {
                const float* __restrict__ y = snr + dd * n_t;
                if (nr <= n_hi) {
                    const float u = __ldg(y + nr);
                    bad |= u > v || (u == v && (dd < d || (dd == d && nr < n)));
                }
                if (nl >= n_lo) {
                    const float u = __ldg(y + nl);
                    bad |= u > v || (u == v && (dd < d || dd == d));  // nl < n always
                }
            }
            dominated = __any_sync(0xffffffffu, bad);
        }
        if (!dominated && lane == 0) {
            const unsigned long long slot = atomicAdd(n_out, 1ull);
            if (slot < cap_out) out[slot] = c;
        }
    }
}

}  // namespace

int64_t activity_block(const spd_plan* plan) {
    if (!runs_tree_kernel(plan)) return 4096;
    return plan->tree.act_block > 0 ? plan->tree.act_block : plan->tree.chunk;
}
int64_t activity_per_row(const spd_plan* plan) {
    const int64_t b = activity_block(plan);
    return (plan->n_t + b - 1) / b;
}

int candidates_run(const spd_plan* plan, int64_t n_rows, int64_t dm_offset, const float* out_snr,
                   const void* out_width, const uint8_t* activity, float threshold, spd_candidate* list,
                   int64_t capacity, int64_t* n_found, bool clear, cudaStream_t stream) {
    cudaError_t e = cudaSuccess;
    if (clear && (e = cudaMemsetAsync(n_found, 0, sizeof(int64_t), stream)) != cudaSuccess)
        return cuda_fail(e, "clearing the candidate counter");
    // the any-width-set path marks everything: visiting every sample with the dense kernel is
    // the same work with more parallelism (BoxDIT plans: the streaming kernel fills the map, 4096 samples per flag)
    if (activity && (runs_tree_kernel(plan) || plan->boxdit.B > 0)) {
        const long long per_row = activity_per_row(plan);
        const long long n_flags = n_rows * per_row;
        const long long steps = (n_flags + 31) / 32;
        const long long warps_per_block = kCandThreads / 32;
        long long blocks = (steps + warps_per_block - 1) / warps_per_block;
        blocks = std::max<long long>(1, std::min<long long>(blocks, static_cast<long long>(plan->sm_count) * 16));
        find_candidates_flagged_kernel<<<static_cast<unsigned>(blocks), kCandThreads, 0, stream>>>(
            out_snr, out_width, plan->width_bytes, dm_offset, activity, n_flags, per_row, activity_block(plan),
            plan->n_t, threshold, list, static_cast<unsigned long long>(capacity),
            reinterpret_cast<unsigned long long*>(n_found));
    } else {
        const long long tiles = (plan->n_t + kCandTile - 1) / kCandTile;
        if (n_rows * tiles > 0x7fffffffll) {
            set_error("plane too large for the candidate grid");
            return SPD_ERR_INVALID_ARG;
        }
        find_candidates_kernel<<<static_cast<unsigned>(n_rows * tiles), kCandThreads, 0, stream>>>(
            out_snr, out_width, plan->width_bytes, dm_offset, plan->n_t, tiles, threshold, list,
            static_cast<unsigned long long>(capacity), reinterpret_cast<unsigned long long*>(n_found));
    }
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "launching the candidate kernel");
    return SPD_OK;
}

int cluster_run(const spd_plan* plan, const float* out_snr, const spd_candidate* list_in, const int64_t* n_in,
                int64_t capacity_in, int dm_radius, spd_candidate* list_out, int64_t capacity_out, int64_t* n_out,
                cudaStream_t stream) {
    cudaError_t e = cudaMemsetAsync(n_out, 0, sizeof(int64_t), stream);
    if (e != cudaSuccess) return cuda_fail(e, "clearing the cluster counter");
    // a persistent grid of warps strides over the list (its length is known on the device only)
    const unsigned blocks = static_cast<unsigned>(plan->sm_count) * 8u;
    cluster_candidates_kernel<<<blocks, kCandThreads, 0, stream>>>(
        out_snr, plan->n_dm, plan->n_t, static_cast<const int32_t*>(plan->d_wsig_widths),
        static_cast<int>(plan->widths.size()), list_in, reinterpret_cast<const unsigned long long*>(n_in),
        static_cast<unsigned long long>(capacity_in), dm_radius, list_out,
        static_cast<unsigned long long>(capacity_out), reinterpret_cast<unsigned long long*>(n_out));
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "launching the 2-D peak kernel");
    return SPD_OK;
}

}  // namespace spd
