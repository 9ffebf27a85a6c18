// Any-width-set path (SURVEY.md sec. 8(a) rows a2-a7 for width sets the dyadic tree does
// not cover: the "ideal" set 1..L_max of PAPER.md:193, BoxDIT eq. (14), IGRID eq. (18), ...).
//
// Partial sums are reused through one running sum per DM row,
//   C_d[n] = sum_{j<n} (x[d,j] - mu_d),  X_L[n] - L mu_d = C_d[n+L] - C_d[n]
// (eq. 2 with eq. 5); eq. (4) and the max / arg-max of eq. (12) then visit
// the widths in ascending order with a strict '>'.
//
// Tile kernel (max_width up to ~40 K): a block stages one time tile of a row plus its
// max_width - 1 look-ahead in shared memory as a two-level running sum - a float32
// exclusive sum inside 64-sample sub-blocks (magnitude of a few sigma, so differences keep
// ~1e-6 sigma) and a double running sum of the sub-block totals - and evaluates every width
// of every sample of the tile from it.  Nothing but x is read and Y, W written; the work is
// O(|B|) shared-memory loads per sample, so this path is bound by the L1/issue pipes, not by
// HBM, and is not the tuned path (the dyadic tree, spd_tree.cu, is).
//
// Workspace kernels (fallback for larger max_width): the same running sum kept in double in
// a plan-owned device workspace, built by three scan kernels and read by an evaluation kernel.
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#include <algorithm>
#include <cstdlib>

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

// ---- tile kernel --------------------------------------------------------------------
constexpr int kTileThreads = 1024;
constexpr int kSub = 64;                 // samples per float32 sub-block
constexpr int kTileSpanMax = 48 * 1024;  // floats of shared memory for tile + look-ahead
constexpr int kTileWidthsMax = 1024;     // width table kept in shared memory up to this many widths

// Phases 1 and 2 of a tile: the two-level running sum of (x - mu) over `span` samples from t0:
// c[i] = float32 exclusive sum inside the 64-sample sub-block of i, B[j] = double running sum
// of the sub-block totals, so that C[i] = B[i / kSub] + c[i].  Ends with a block barrier.
__device__ __forceinline__ void build_running_sum(const float* __restrict__ row, long long t0, long long avail,
                                                  float mu, int n_sub, int span, double* __restrict__ B,
                                                  float* __restrict__ c) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    // phase 1: sub-block sums; samples beyond the row count as x = mu (never used by a valid window).
    // A warp takes every 32nd sub-block; the loads of kAhead of them are issued before the first
    // is scanned, so that a tile pays a few memory latencies instead of one per sub-block.
    constexpr int kAhead = 4;
    constexpr int kWarps = kTileThreads / 32;
    for (int sb0 = warp; sb0 < n_sub; sb0 += kAhead * kWarps) {
        float2 raw[kAhead];
#pragma unroll
        for (int u = 0; u < kAhead; ++u) {
            const int i = (sb0 + u * kWarps) * kSub + 2 * lane;
            raw[u].x = (sb0 + u * kWarps < n_sub && i < avail) ? __ldg(row + t0 + i) : mu;
            raw[u].y = (sb0 + u * kWarps < n_sub && i + 1 < avail) ? __ldg(row + t0 + i + 1) : mu;
        }
#pragma unroll
        for (int u = 0; u < kAhead; ++u) {
            const int sb = sb0 + u * kWarps;
            if (sb >= n_sub) break;
            const int i = sb * kSub + 2 * lane;
            const float x0 = raw[u].x - mu;
            const float x1 = raw[u].y - mu;
            const float s = x0 + x1;
            float incl = s;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const float v = __shfl_up_sync(0xffffffffu, incl, o);
                if (lane >= o) incl += v;
            }
            c[i] = incl - s;
            c[i + 1] = incl - s + x0;
            // sub-block total in double (pairwise over the lanes)
            double tot = static_cast<double>(x0) + static_cast<double>(x1);
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) tot += __shfl_xor_sync(0xffffffffu, tot, o);
            if (lane == 0) B[sb + 1] = tot;
        }
    }
    __syncthreads();
    // phase 2: running sum of the totals (one warp, consecutive runs per lane)
    if (warp == 0) {
        const int per = (n_sub + 31) / 32;
        const int lo = min(lane * per, n_sub), hi = min(lo + per, n_sub);
        double run = 0.0;
        for (int j = lo; j < hi; ++j) run += B[j + 1];
        double incl = run;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const double u = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += u;
        }
        double acc = incl - run;
        for (int j = lo; j < hi; ++j) {
            const double t = B[j + 1];
            B[j + 1] = acc + t;
            acc += t;
        }
        if (lane == 0) {
            B[0] = 0.0;
            c[span] = 0.f;  // C at the end of the last sub-block = B[n_sub] + 0
        }
    }
    __syncthreads();
}

__global__ void __launch_bounds__(kTileThreads) generic_tile_kernel(
    const float* __restrict__ plane, const float* __restrict__ mean, const float* __restrict__ sigma,
    const int32_t* __restrict__ widths, const float* __restrict__ wscale, int n_w, long long n_t, int tile,
    int span, long long tiles_per_row, float* __restrict__ out_snr, int32_t* __restrict__ out_width,
    const float* __restrict__ sigma_w) {
    extern __shared__ __align__(16) unsigned char gsm[];
    const int n_sub = span / kSub;  // span is a multiple of kSub
    double* const B = reinterpret_cast<double*>(gsm);                        // [n_sub + 1] running sum of sub-block totals
    float* const c = reinterpret_cast<float*>(gsm + (n_sub + 2) / 2 * 16);  // [span + 1] exclusive sum inside a sub-block
    int32_t* const sw = reinterpret_cast<int32_t*>(c + (span + 4) / 4 * 4);   // [kTileWidthsMax] widths
    float* const ss = reinterpret_cast<float*>(sw + kTileWidthsMax);          // [kTileWidthsMax] 1 / (sqrt(L) sigma)
    const long long d = blockIdx.x / tiles_per_row;
    const long long t0 = (blockIdx.x - d * tiles_per_row) * tile;
    const float* __restrict__ row = plane + d * n_t;
    const float mu = mean[d];
    // sigma_w: measured standard deviation per (row, width) instead of eq. (5)'s sqrt(L) sigma
    // (PAPER.md:728); only with the width table in shared memory (checked by the caller)
    const float inv = sigma_w ? 1.0f : 1.0f / sigma[d];
    const long long avail = n_t - t0;  // samples of the row from t0 on
    const bool table_in_smem = n_w <= kTileWidthsMax;
    if (table_in_smem) {
        for (int k = threadIdx.x; k < n_w; k += kTileThreads) {
            sw[k] = __ldg(widths + k);
            ss[k] = sigma_w ? 1.0f / __ldg(sigma_w + d * n_w + k) : __ldg(wscale + k) * inv;
        }
    }
    const int32_t* __restrict__ wp = table_in_smem ? sw : widths;
    const float* __restrict__ sp = table_in_smem ? ss : wscale;
    const float post = table_in_smem ? 1.0f : inv;  // 1/sigma already folded into ss

    build_running_sum(row, t0, avail, mu, n_sub, span, B, c);
    // phase 3: every width of every sample of the tile.  C[i] = B[i / kSub] + c[i].
    const int n_out = static_cast<int>(min(static_cast<long long>(tile), avail));
    const int max_w = __ldg(widths + n_w - 1);
    for (int i = threadIdx.x; i < n_out; i += kTileThreads) {
        const long long room = avail - i;
        const float c0 = c[i];
        const double b0 = B[i / kSub];
        float best = __int_as_float(0xff800000);
        int idx = -1;
        auto visit = [&](int k, int L) {
            const int e = i + L;
            const float x = static_cast<float>(B[e / kSub] - b0) + (c[e] - c0);
            const float snr = x * sp[k] * post;  // eq. (4) with eq. (5)
            if (snr > best) {                    // strict '>'
                best = snr;
                idx = k;
            }
        };
        if (room >= max_w) {  // every width fits: no test inside the loop, loads of 4 widths in flight
            int k = 0;
            for (; k + 4 <= n_w; k += 4) {
                const int L0 = wp[k], L1 = wp[k + 1], L2 = wp[k + 2], L3 = wp[k + 3];
                visit(k, L0);
                visit(k + 1, L1);
                visit(k + 2, L2);
                visit(k + 3, L3);
            }
            for (; k < n_w; ++k) visit(k, wp[k]);
        } else {
            for (int k = 0; k < n_w; ++k) {
                const int L = wp[k];
                if (L > room) break;  // valid windows only (reading A3); widths ascend
                visit(k, L);
            }
        }
        out_snr[d * n_t + t0 + i] = best;
        out_width[d * n_t + t0 + i] = idx;
    }
}

// ---- per-width boxcar separation (the paper's decimated grids) ----
// Width k is evaluated only at samples that are multiples of its separation L_s[k] = 2^shift
// (BoxDIT iteration i: every D^(i)-th point, Alg. 1; DIT: width 2^i every 2^i,
// Alg. 3; IGRID with P layers: 2^i / P); one merged plane
// Y[n] = max over the widths whose grid contains n (reading A16).  Widths ascend and their
// separations do not decrease, so the widths form groups of equal separation (the paper's
// iterations).  The tile's running sum is built as in generic_tile_kernel; then the groups are
// visited in turn, one thread per grid point of the group (equal work per thread: a group's
// widths), the running best of every sample of the tile living in shared memory between groups.
__global__ void __launch_bounds__(kTileThreads) grid_tile_kernel(
    const float* __restrict__ plane, const float* __restrict__ mean, const float* __restrict__ sigma,
    const int32_t* __restrict__ widths, const float* __restrict__ wscale, int n_w, const GridGroups groups,
    long long n_t, int tile, int span, long long tiles_per_row, float* __restrict__ out_snr,
    int32_t* __restrict__ out_width, const float* __restrict__ sigma_w) {
    extern __shared__ __align__(16) unsigned char gsm[];
    const int n_sub = span / kSub;
    double* const B = reinterpret_cast<double*>(gsm);
    float* const c = reinterpret_cast<float*>(gsm + (n_sub + 2) / 2 * 16);
    int32_t* const sw = reinterpret_cast<int32_t*>(c + (span + 4) / 4 * 4);
    float* const ss = reinterpret_cast<float*>(sw + kTileWidthsMax);
    const long long d = blockIdx.x / tiles_per_row;
    const long long t0 = (blockIdx.x - d * tiles_per_row) * tile;
    const float* __restrict__ row = plane + d * n_t;
    const float mu = mean[d];
    const float inv = sigma_w ? 1.0f : 1.0f / sigma[d];
    const long long avail = n_t - t0;
    for (int k = threadIdx.x; k < n_w; k += kTileThreads) {  // n_w <= kTileWidthsMax (checked at plan creation)
        sw[k] = __ldg(widths + k);
        ss[k] = sigma_w ? 1.0f / __ldg(sigma_w + d * n_w + k) : __ldg(wscale + k) * inv;
    }
    build_running_sum(row, t0, avail, mu, n_sub, span, B, c);

    const int n_out = static_cast<int>(min(static_cast<long long>(tile), avail));
    // running best of every sample of the tile, in shared memory between the groups
    float* const sbest = ss + kTileWidthsMax;                     // [tile]
    int32_t* const sidx = reinterpret_cast<int32_t*>(sbest + tile);  // [tile]
    for (int i = threadIdx.x; i < n_out; i += kTileThreads) {
        sbest[i] = __int_as_float(0xff800000);  // samples on no grid at all keep -inf / -1
        sidx[i] = -1;
    }
    __syncthreads();
    for (int g = 0; g < groups.n; ++g) {
        const int sh = groups.shift[g];
        const int kb = groups.kb[g], ke = groups.ke[g];
        const long long step = 1ll << sh;
        const int i0 = static_cast<int>((step - (t0 & (step - 1))) & (step - 1));  // first grid point of the tile
        const int count = i0 < n_out ? static_cast<int>((n_out - i0 + step - 1) >> sh) : 0;
        for (int item = threadIdx.x; item < count; item += kTileThreads) {
            const int i = i0 + (item << sh);
            const long long room = avail - i;
            const float c0 = c[i];
            const double b0 = B[i / kSub];
            float best = sbest[i];
            int idx = sidx[i];
            for (int k = kb; k < ke; ++k) {
                const int L = sw[k];
                if (L > room) break;  // valid windows only (reading A3); widths ascend
                const int e = i + L;
                const float x = static_cast<float>(B[e / kSub] - b0) + (c[e] - c0);
                const float snr = x * ss[k];  // eq. (4) with eq. (5)
                if (snr > best) {             // strict '>' in ascending width order
                    best = snr;
                    idx = k;
                }
            }
            sbest[i] = best;
            sidx[i] = idx;
        }
        __syncthreads();
    }
    float* const ysnr = out_snr + d * n_t + t0;
    int32_t* const yidx = out_width + d * n_t + t0;
    for (int i = threadIdx.x; i < n_out; i += kTileThreads) {
        ysnr[i] = sbest[i];
        yidx[i] = sidx[i];
    }
}

// ---- output separated by iteration (eq. 12) ----------------------------------------------
// The same tile and running sum as grid_tile_kernel, but the groups of equal separation (the paper's iterations)
// are not merged: group g writes its own decimated plane Y^g[d][m], W^g[d][m], point m = sample m * 2^shift,
// at out + off[g] + d * npts[g] + m.  One thread per grid point and group; a point where no width of the group
// fits the row gets -inf / -1 (reading A3).
struct GridIterLayout {
    long long off[kGridGroupsMax];   // element offset of group g's plane in the concatenated outputs
    long long npts[kGridGroupsMax];  // points per row: ceil(n_t / 2^shift)
};

__global__ void __launch_bounds__(kTileThreads) grid_iter_kernel(
    const float* __restrict__ plane, const float* __restrict__ mean, const float* __restrict__ sigma,
    const int32_t* __restrict__ widths, const float* __restrict__ wscale, int n_w, const GridGroups groups,
    const GridIterLayout lay, long long n_t, int tile, int span, long long tiles_per_row,
    float* __restrict__ out_snr, int32_t* __restrict__ out_width) {
    extern __shared__ __align__(16) unsigned char gsm[];
    const int n_sub = span / kSub;
    double* const B = reinterpret_cast<double*>(gsm);
    float* const c = reinterpret_cast<float*>(gsm + (n_sub + 2) / 2 * 16);
    int32_t* const sw = reinterpret_cast<int32_t*>(c + (span + 4) / 4 * 4);
    float* const ss = reinterpret_cast<float*>(sw + kTileWidthsMax);
    const long long d = blockIdx.x / tiles_per_row;
    const long long t0 = (blockIdx.x - d * tiles_per_row) * tile;
    const float* __restrict__ row = plane + d * n_t;
    const float mu = mean[d];
    const float inv = 1.0f / sigma[d];
    const long long avail = n_t - t0;
    for (int k = threadIdx.x; k < n_w; k += kTileThreads) {  // n_w <= kTileWidthsMax (checked at plan creation)
        sw[k] = __ldg(widths + k);
        ss[k] = __ldg(wscale + k) * inv;
    }
    build_running_sum(row, t0, avail, mu, n_sub, span, B, c);
    const int n_out = static_cast<int>(min(static_cast<long long>(tile), avail));
    for (int g = 0; g < groups.n; ++g) {
        const int sh = groups.shift[g];
        const int kb = groups.kb[g], ke = groups.ke[g];
        const long long step = 1ll << sh;
        const int i0 = static_cast<int>((step - (t0 & (step - 1))) & (step - 1));  // first grid point of the tile
        const int count = i0 < n_out ? static_cast<int>((n_out - i0 + step - 1) >> sh) : 0;
        float* const ys = out_snr + lay.off[g] + d * lay.npts[g];
        int32_t* const yw = out_width + lay.off[g] + d * lay.npts[g];
        for (int item = threadIdx.x; item < count; item += kTileThreads) {
            const int i = i0 + (item << sh);
            const long long room = avail - i;
            const float c0 = c[i];
            const double b0 = B[i / kSub];
            float best = __int_as_float(0xff800000);
            int idx = -1;
            for (int k = kb; k < ke; ++k) {
                const int L = sw[k];
                if (L > room) break;  // valid windows only (reading A3); widths ascend
                const int e = i + L;
                const float x = static_cast<float>(B[e / kSub] - b0) + (c[e] - c0);
                const float snr = x * ss[k];  // eq. (4) with eq. (5)
                if (snr > best) {             // strict '>' in ascending width order
                    best = snr;
                    idx = k;
                }
            }
            const long long m = (t0 + i) >> sh;
            ys[m] = best;
            yw[m] = idx;
        }
    }
}

}  // namespace

// Iterations of a grid plan = its groups of equal separation; points per row of group g.
int64_t grid_iter_points(const spd_plan* plan, int g) {
    const int64_t step = int64_t(1) << plan->grid.shift[g];
    return (plan->n_t + step - 1) / step;
}

int generic_run_iterations(const spd_plan* plan, const float* plane, const float* mean, const float* sigma,
                           float* out_snr, int32_t* out_width, cudaStream_t stream) {
    if (plan->boxdit.B > 0)  // Alg. 1's widths on Alg. 1's grids: the BoxDIT streaming kernel keeps its levels apart
        return boxdit_run_iterations(plan, plane, mean, sigma, out_snr, out_width, stream);
    static bool configured = false;  // per process; the attribute is sticky
    if (!configured) {
        const cudaError_t e = cudaFuncSetAttribute(grid_iter_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                   227 * 1024);  // the most a block can have
        if (e != cudaSuccess) return cuda_fail(e, "configuring the per-iteration kernel");
        configured = true;
    }
    GridIterLayout lay = {};
    long long off = 0;
    for (int g = 0; g < plan->grid.n; ++g) {
        lay.off[g] = off;
        lay.npts[g] = grid_iter_points(plan, g);
        off += plan->n_dm * lay.npts[g];
    }
    grid_iter_kernel<<<static_cast<unsigned>(plan->n_dm * plan->generic_tiles_per_row), kTileThreads, plan->generic_smem,
                       stream>>>(plane, mean, sigma, plan->d_widths, plan->d_wscale,
                                 static_cast<int>(plan->widths.size()), plan->grid, lay, plan->n_t, plan->generic_tile,
                                 plan->generic_span, plan->generic_tiles_per_row, out_snr, out_width);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "launching the per-iteration kernel");
    return SPD_OK;
}

int generic_configure(spd_plan* plan) {
    const int n_w = static_cast<int>(plan->widths.size());
    std::vector<float> scale(n_w);
    for (int k = 0; k < n_w; ++k) scale[k] = static_cast<float>(1.0 / sqrt(static_cast<double>(plan->widths[k])));
    cudaError_t e;
    if ((e = cudaMalloc(&plan->d_widths, sizeof(int32_t) * n_w)) != cudaSuccess ||
        (e = cudaMalloc(&plan->d_wscale, sizeof(float) * n_w)) != cudaSuccess) {
        set_error("device allocation of the width table failed: %s", cudaGetErrorString(e));
        cudaGetLastError();
        generic_release(plan);
        return SPD_ERR_ALLOC;
    }
    if ((e = cudaMemcpy(plan->d_widths, plan->widths.data(), sizeof(int32_t) * n_w, cudaMemcpyHostToDevice)) !=
            cudaSuccess ||
        (e = cudaMemcpy(plan->d_wscale, scale.data(), sizeof(float) * n_w, cudaMemcpyHostToDevice)) != cudaSuccess) {
        generic_release(plan);
        return cuda_fail(e, "uploading the width table");
    }

    // ---- tile kernel: no workspace -------------------------------------------------------
    const int64_t M = plan->max_width;
    plan->generic_tile = 0;
    const bool is_grid = !plan->separations.empty();
    if (is_grid && (M - 1 + 4096 > kTileSpanMax || n_w > kTileWidthsMax)) {
        set_error("a plan with boxcar separations needs max_width <= %d and at most %d widths",
                  kTileSpanMax - 4095, kTileWidthsMax);
        generic_release(plan);
        return SPD_ERR_INVALID_ARG;
    }
    if (M - 1 + 4096 <= kTileSpanMax && (is_grid || !(plan->flags & SPD_FLAG_GENERIC_WORKSPACE))) {
        // a grid plan also keeps 8 bytes of running best per sample of the tile in shared memory
        const int64_t tile_max = is_grid ? std::max<int64_t>(1024, ((200 << 10) - 4 * M) / 12 / 1024 * 1024)
                                         : (kTileSpanMax - (M - 1)) / kSub * kSub;
        // enough tiles to fill the machine, but none so short that its look-ahead dominates
        const int64_t tiles_wanted = std::max<int64_t>(1, (2 * plan->sm_count + plan->n_dm - 1) / plan->n_dm);
        int64_t tile = ((plan->n_t + tiles_wanted - 1) / tiles_wanted + 1023) / 1024 * 1024;
        tile = std::max<int64_t>(tile, std::min<int64_t>(tile_max, (M + 1023) / 1024 * 1024));
        tile = std::min<int64_t>(tile, tile_max);
        const int64_t span = (tile + M - 1 + kSub - 1) / kSub * kSub;
        const int64_t n_sub = span / kSub;
        plan->generic_tile = static_cast<int>(tile);
        plan->generic_span = static_cast<int>(span);
        plan->generic_smem = static_cast<size_t>((n_sub + 2) / 2 * 16 + (span + 4) / 4 * 16 + kTileWidthsMax * 8) +
                             (is_grid ? static_cast<size_t>(tile) * 8 : 0);
        plan->generic_tiles_per_row = (plan->n_t + tile - 1) / tile;
        if (plan->n_dm * plan->generic_tiles_per_row > 0x7fffffffll) {
            set_error("plane too large for the generic path's 1-D grid");
            generic_release(plan);
            return SPD_ERR_INVALID_ARG;
        }
        e = is_grid ? cudaFuncSetAttribute(grid_tile_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                           static_cast<int>(plan->generic_smem))
                    : cudaFuncSetAttribute(generic_tile_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                           static_cast<int>(plan->generic_smem));
        if (e != cudaSuccess) {
            generic_release(plan);
            return cuda_fail(e, "configuring the any-width-set tile kernel");
        }
        return SPD_OK;
    }

    // ---- workspace kernels (max_width too large for a shared-memory tile) -----------------
    plan->generic_blocks_per_row = (plan->n_t + kScanBlock - 1) / kScanBlock;
    const size_t prefix_bytes = sizeof(double) * static_cast<size_t>(plan->n_dm) * static_cast<size_t>(plan->n_t + 1);
    const size_t bs_bytes = sizeof(double) * static_cast<size_t>(plan->n_dm) * plan->generic_blocks_per_row;
    if (plan->n_dm * plan->generic_blocks_per_row > 0x7fffffffll ||
        plan->n_dm * ((plan->n_t + 255) / 256) > 0x7fffffffll) {
        set_error("plane too large for the generic path's 1-D grids");
        generic_release(plan);
        return SPD_ERR_INVALID_ARG;
    }
    if ((e = cudaMalloc(&plan->d_prefix, prefix_bytes)) != cudaSuccess ||
        (e = cudaMalloc(&plan->d_blocksum, bs_bytes)) != cudaSuccess) {
        set_error("device allocation of the generic workspace (%zu bytes) failed: %s", prefix_bytes + bs_bytes,
                  cudaGetErrorString(e));
        cudaGetLastError();
        generic_release(plan);
        return SPD_ERR_ALLOC;
    }
    plan->workspace_bytes = static_cast<int64_t>(prefix_bytes + bs_bytes);
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
                float* out_snr, int32_t* out_width, cudaStream_t stream, const float* sigma_w) {
    const long long n_t = plan->n_t;
    if (dense_applicable(plan))  // max_width <= 64: running sums in registers (spd_dense.cu)
        return dense_run(plan, n_dm, plane, mean, sigma, out_snr, out_width, stream, sigma_w);
    if (sigma_w && (plan->generic_tile <= 0 || static_cast<int>(plan->widths.size()) > kTileWidthsMax)) {
        set_error("a standard deviation per width needs the shared-memory tile kernel (max_width <= %d, at most %d "
                  "widths)", kTileSpanMax - 4095, kTileWidthsMax);
        return SPD_ERR_INVALID_ARG;
    }
    if (plan->boxdit.B > 0)  // Alg. 1's widths on Alg. 1's grids (spd_boxdit.cu)
        return boxdit_run(plan, n_dm, plane, mean, sigma, out_snr, out_width, stream, sigma_w);
    if (!plan->separations.empty()) {
        grid_tile_kernel<<<static_cast<unsigned>(n_dm * plan->generic_tiles_per_row), kTileThreads, plan->generic_smem,
                           stream>>>(plane, mean, sigma, plan->d_widths, plan->d_wscale,
                                     static_cast<int>(plan->widths.size()), plan->grid, n_t, plan->generic_tile,
                                     plan->generic_span, plan->generic_tiles_per_row, out_snr, out_width, sigma_w);
        const cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return cuda_fail(e, "launching the boxcar-separation tile kernel");
        return SPD_OK;
    }
    if (plan->generic_tile > 0) {
        generic_tile_kernel<<<static_cast<unsigned>(n_dm * plan->generic_tiles_per_row), kTileThreads,
                              plan->generic_smem, stream>>>(
            plane, mean, sigma, plan->d_widths, plan->d_wscale, static_cast<int>(plan->widths.size()), n_t,
            plan->generic_tile, plan->generic_span, plan->generic_tiles_per_row, out_snr, out_width, sigma_w);
        const cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return cuda_fail(e, "launching the any-width-set tile kernel");
        return SPD_OK;
    }
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
