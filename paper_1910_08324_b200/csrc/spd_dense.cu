// Any width set with max_width <= 64 ("dense" plans: BASELINE config 1's ideal algorithm, all widths 1 .. 64,
// PAPER.md:193; and any subset of them) - rows a1-a7 in one kernel, partial sums reused by the running sum
// X_L[n] = X_{L-1}[n] + x[n + L - 1] (eq. 2 with the reuse of eq. 16/17: "the longest sum is
// reused", here within a thread's registers).
//
//   * a block stages a tile of 1024 samples plus 64 of look-ahead with one 1-D cp.async.bulk (TMA) and an
//     mbarrier; thread t owns the float4 4t .. 4t+3 and walks the widths 1 .. max_width with four running sums in
//     registers; the samples entering the windows arrive as one aligned 128-bit shared-memory load per four
//     widths (conflict-free; a 32-bit load per width would hit every fourth bank);
//   * every width of the plan (a 64-bit presence mask, a warp-uniform test) contributes a key: the sum times
//     1 / (sqrt(L) sigma_d) - or 1 / sigma_{d,L} measured - with the inverted width index in the six
//     low mantissa bits (<= 63 ulp), folded with a max; ascending widths and the inverted tag give
//     the smallest width on exact ties;
//   * windows that cross the end of the row are skipped (reading A3).
// Per sample and width: one add, one multiply, one tag, one max - the same ALU-pipe work per key as the tree
// kernels, 64 keys per sample for config 1.
#include <cuda_runtime.h>
#include <stdint.h>

#include <algorithm>

#include "spd_tree_common.cuh"

namespace spd {
namespace {

constexpr int kDenseThreads = 256;
constexpr int kDenseTile = 4 * kDenseThreads;  // samples per block
constexpr int kDenseMaxW = 64;
constexpr int kDenseSpan = kDenseTile + kDenseMaxW;  // floats staged
constexpr uint32_t kDenseTagMask = ~63u;

struct DenseParams {
    const float* plane;
    const float* mean;
    const float* sigma;    // or nullptr with sigma_w
    const float* sigma_w;  // [n_dm][n_w] or nullptr
    float* out_snr;
    int32_t* out_width;
    long long n_t;
    int tiles_per_row;
    int n_w, max_w;
    unsigned long long present;  // bit L-1: width L is in the plan
    uint32_t full_groups;        // bit g: the widths 4g+1 .. 4g+4 are all in the plan
    uint8_t index_of[kDenseMaxW + 1];  // width -> index in the ascending table
};

__global__ void __launch_bounds__(kDenseThreads, 7) spd_dense_kernel(const DenseParams p) {
    __shared__ __align__(128) float xs[kDenseSpan];
    __shared__ __align__(16) float scale[kDenseMaxW];     // [L - 1]: 1 / (sqrt(L) sigma_d) or 1 / sigma_{d,L}; 0 = not in the plan
    __shared__ __align__(16) uint32_t codes[kDenseMaxW];  // [L - 1]: 63 - index, the smaller width carries the larger tag
    __shared__ __align__(8) uint64_t bar;
    const int tid = threadIdx.x;
    const long long d = blockIdx.x / p.tiles_per_row;
    const long long t0 = static_cast<long long>(blockIdx.x - d * p.tiles_per_row) * kDenseTile;
    const float* __restrict__ row = p.plane + d * p.n_t;
    const long long left = p.n_t - t0;                                    // samples of the row from the tile's start
    const int staged = static_cast<int>(left < kDenseSpan ? left : kDenseSpan);  // multiple of 4 (n_t % 4 == 0)
    if (tid == 0) {
        mbar_init(&bar, 1);
        fence_mbar_init();
        mbar_arrive_expect_tx(&bar, static_cast<uint32_t>(staged) * 4u);
        bulk_g2s(xs, row + t0, static_cast<uint32_t>(staged) * 4u, &bar);
    }
    if (tid >= 32 && tid < 32 + kDenseMaxW) {
        const int L = tid - 31;
        float s = 0.f;
        uint32_t c = 0;
        if ((p.present >> (L - 1)) & 1ull) {
            const int k = p.index_of[L];
            c = 63u - k;
            s = p.sigma_w ? 1.0f / __ldg(p.sigma_w + d * p.n_w + k) : rsqrtf(static_cast<float>(L)) / __ldg(p.sigma + d);
        }
        scale[L - 1] = s;
        codes[L - 1] = c;
    }
    __syncthreads();
    mbar_wait(&bar, 0);
    const long long n = t0 + 4ll * tid;
    if (n >= p.n_t) return;
    const float mu = __ldg(p.mean + d);
    const int lim = static_cast<int>(min(p.n_t - n, 1ll << 20));  // samples from n to the end of the row
    const float ninf = __int_as_float(0xff800000);
    const float4* const x4 = reinterpret_cast<const float4*>(xs) + tid;
    const float4* const scale4 = reinterpret_cast<const float4*>(scale);
    const uint4* const codes4 = reinterpret_cast<const uint4*>(codes);
    float4 cur = norm4(x4[0], mu);
    float S[4] = {0.f, 0.f, 0.f, 0.f};
    float best[4] = {ninf, ninf, ninf, ninf};
    // groups of four consecutive widths that are all in the plan take the short way when every window of this
    // thread fits the row (all threads but the last 17 of a row)
    const uint32_t fast = lim >= p.max_w + 3 ? p.full_groups : 0u;
    const int n_groups = (p.max_w + 3) >> 2;
    for (int g = 0; g < n_groups; ++g) {
        // the four samples that enter the windows during these four widths (past the staged span - beyond the end
        // of the row - only windows that are skipped use them)
        const float4 nxt = norm4(x4[1 + g], mu);
        const float win[8] = {cur.x, cur.y, cur.z, cur.w, nxt.x, nxt.y, nxt.z, nxt.w};
        const float4 sc4 = scale4[g];
        const uint4 cd4 = codes4[g];
        const float sc[4] = {sc4.x, sc4.y, sc4.z, sc4.w};
        const uint32_t cd[4] = {cd4.x, cd4.y, cd4.z, cd4.w};
        if ((fast >> g) & 1u) {
            float key[4][4];
#pragma unroll
            for (int u = 0; u < 4; ++u)
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    S[i] += win[i + u];  // X_L[n+i] = X_{L-1}[n+i] + x[n+i+L-1]
                    key[u][i] = __uint_as_float((__float_as_uint(S[i] * sc[u]) & kDenseTagMask) | cd[u]);
                }
#pragma unroll
            for (int i = 0; i < 4; ++i)
                best[i] = fmax3(fmax3(best[i], key[0][i], key[1][i]), key[2][i], key[3][i]);
        } else {
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int L = 4 * g + u + 1;
#pragma unroll
                for (int i = 0; i < 4; ++i) S[i] += win[i + u];
                if (sc[u] != 0.f) {  // the width is in the plan
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        float key = __uint_as_float((__float_as_uint(S[i] * sc[u]) & kDenseTagMask) | cd[u]);
                        if (L > lim - i) key = ninf;  // the window crosses the end of the row (reading A3)
                        best[i] = fmaxf(best[i], key);
                    }
                }
            }
        }
        cur = nxt;
    }
    float4 y;
    int4 w;
    float* yy = &y.x;
    int* ww = &w.x;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const uint32_t b = __float_as_uint(best[i]);
        const bool none = best[i] == ninf;
        yy[i] = none ? ninf : __uint_as_float(b & kDenseTagMask);
        ww[i] = none ? -1 : static_cast<int>(63u - (b & 63u));
    }
    *reinterpret_cast<float4*>(p.out_snr + d * p.n_t + n) = y;
    *reinterpret_cast<int4*>(p.out_width + d * p.n_t + n) = w;
}

}  // namespace

bool dense_applicable(const spd_plan* plan) {
    return plan->separations.empty() && plan->max_width <= kDenseMaxW && plan->n_t % 4 == 0 &&
           !(plan->flags & SPD_FLAG_GENERIC_WORKSPACE) && plan->widths.size() <= 64;
}

int dense_blocks(const spd_plan* plan) { return static_cast<int>(plan->n_dm * ((plan->n_t + kDenseTile - 1) / kDenseTile)); }

int dense_run(const spd_plan* plan, int64_t n_dm, const float* plane, const float* mean, const float* sigma,
              float* out_snr, int32_t* out_width, cudaStream_t stream, const float* sigma_w) {
    DenseParams prm = {};
    prm.plane = plane;
    prm.mean = mean;
    prm.sigma = sigma;
    prm.sigma_w = sigma_w;
    prm.out_snr = out_snr;
    prm.out_width = out_width;
    prm.n_t = plan->n_t;
    const int64_t tiles = (plan->n_t + kDenseTile - 1) / kDenseTile;
    if (n_dm * tiles > 0x7fffffffll) {
        set_error("plane too large for the dense kernel's grid");
        return SPD_ERR_INVALID_ARG;
    }
    prm.tiles_per_row = static_cast<int>(tiles);
    prm.n_w = static_cast<int>(plan->widths.size());
    prm.max_w = plan->widths.back();
    for (int k = 0; k < prm.n_w; ++k) {
        const int L = plan->widths[k];
        prm.present |= 1ull << (L - 1);
        prm.index_of[L] = static_cast<uint8_t>(k);
    }
    for (int g = 0; g < kDenseMaxW / 4; ++g)
        if (((prm.present >> (4 * g)) & 15ull) == 15ull) prm.full_groups |= 1u << g;
    spd_dense_kernel<<<static_cast<unsigned>(n_dm * tiles), kDenseThreads, 0, stream>>>(prm);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "launching the dense kernel");
    return SPD_OK;
}

}  // namespace spd
