// The BoxDIT algorithm (Alg. 1, eq. 13-15) as one streaming kernel - row f2 for the paper's
// BD-4/8/16/32 grids with D = 2: iteration i evaluates the widths (2^i - 1) B + 2^i m, m = 1 .. B (eq. 14,
// B = L_max per iteration) at every 2^i-th sample of the row, from the decimated series x^i and the longest
// boxcar X^{i-1} of the iteration before (eq. 15).
//
// What is kept of the paper's design: the iteration structure, the shifted decimation of eq. (13) - with it the
// window of iteration i starts exactly where the windows of iterations < i end, so X_L[n] = X^{i-1}[n] + the first
// m elements of x^i from n's own grid point on - and the fusion of boxcars and decimation in one pass
// (PAPER.md:229).  What differs: the paper launches one kernel per iteration and passes x^i and X^i through
// device memory ("doubles the size of the input"); here all iterations of a chunk of the row run
// inside one block with x^i, X^i and the running best key in shared memory, so the plane is read once
// (4 B per sample) and Y, W written once (8 B), and the rows are walked backwards in time (like the
// streaming trees): the elements of x^i past the chunk's end are the first B of the chunk
// processed just before, a carry of B floats per iteration instead of a look-ahead of L_MAX samples.
//
//   chunk of T samples, NT threads, iterations ("levels") i = 0 .. I-1 one after the other, a block barrier
//   between them; level i has T / 2^i grid points, a task is four consecutive points:
//     window   x^i[4a .. 4a+B+3]                         (B/4 + 1 aligned 128-bit shared-memory loads)
//     sums     t_j <- X^{i-1}[point j];  t_j += x^i[4a+j+m-1], m = 1 .. B          (eq. 15; B adds per point)
//     keys     t_j * 1/(sqrt(L) sigma_d) (or 1/sigma_{d,L}) tagged with the inverted width index
//              in the low 7 (<= 128 widths) or 8 mantissa bits, folded with 3-input maxima
//     out      x^{i+1}[2a], [2a+1] = pairs of the window's last four (eq. 13);  X^i at points 0 and 2;
//              the four best keys, stored where X^{i-1} came from
//   then the thread that owns samples n .. n+3 at level 0 gathers the keys of the levels whose grid holds them
//   (sample n: levels 0, 1, 2 and on while 2^i | n; n+2: levels 0, 1), splits key and tag, and stores Y, W.
// Per sample: 2 B keys (B = 8: 16, PAPER.md:702 footnote 9), each one add, one multiply (FMA pipe), one LOP3 and
// half an FMNMX3 (ALU pipe) - DESIGN.md sec. 7b.
#include <cuda_runtime.h>
#include <stdint.h>

#include <algorithm>

#include "spd_tree_common.cuh"

namespace spd {
namespace {

constexpr int kBdThreads = 256;
constexpr int kBdChunk = 4096;      // samples per chunk: level i has kBdChunk >> i points, at least one task
constexpr int kBdMaxLevels = 11;    // kBdChunk >> 10 = 4 points

struct BdParams {
    const float* plane;
    const float* mean;
    const float* sigma;    // or nullptr with sigma_w
    const float* sigma_w;  // [n_dm][n_w] or nullptr
    float* out_snr;
    int32_t* out_width;
    long long n_t;
    int chunks_per_row;
    int segs_per_row;
    int seg_chunks;
    int warm_chunks;   // chunks run ahead of a segment to fill the carries (ceil(L_MAX / T))
    int n_levels;      // I
    int n_w;           // widths in the plan
    int last_count;    // widths of the last level (1 .. B; a width set cut by max_width)
    int l_max_total;   // the largest width
    uint32_t tag_mask;  // ~127 or ~255
    // output separated by iteration (eq. 12; spd_run_iterations): level i's plane Y^i, W^i [n_dm][it_npts[i]] at
    // element offset it_off[i] of it_snr / it_width; out_snr / out_width are not written then
    // threshold test of row a8 fused (spd_run_flagged): a chunk with a key >= thr_key sets activity[d][c]
    uint8_t* activity;  // [n_dm][chunks_per_row] or nullptr (cleared by the host)
    float thr_key;      // threshold in SNR units, lowered by the tag's perturbation so that rounding only adds chunks
    float* it_snr;
    int32_t* it_width;
    long long it_off[kBdMaxLevels];
    long long it_npts[kBdMaxLevels];
};

template <int B>
__host__ __device__ constexpr int bd_smem_floats() {
    // x^0 twice (TMA double buffer), x^i for i >= 1, X / best for i >= 1, scale table
    return 2 * (kBdChunk + B) + (kBdChunk + kBdMaxLevels * B) + kBdChunk + kBdMaxLevels * B;
}

// offset of level i >= 1 inside the x^i region (T/2 + T/4 + .. + B each) and inside the X / best region
template <int B>
__device__ __forceinline__ int bd_off_x(int i) { return kBdChunk - 2 * (kBdChunk >> i) + (i - 1) * B; }
__device__ __forceinline__ int bd_off_b(int i) { return kBdChunk - 2 * (kBdChunk >> i); }

// One task of level `level`: points 4a .. 4a+3 of the chunk's level-`level` grid.
//   A        x^level of this chunk (B more elements behind the chunk's own: the carry)
//   xin      X^{level-1} at the four points (level 0: zero)
//   sc       this level's B scales (shared memory), code0 the tag of its first width (the tags count down)
//   mlim[j]  MASKED: how many of the level's widths fit the row (or the plan) at point j
template <int B, bool FIRST, bool MASKED>
__device__ __forceinline__ void bd_task(const float* __restrict__ A, const float4 xin, const int a, const float mu,
                                        const float* __restrict__ sc, const uint32_t code0, const uint32_t tag_mask,
                                        const bool last, float* __restrict__ A_next, float* __restrict__ X_next,
                                        const int (&mlim)[4], float (&best)[4]) {
    float w[B + 4];
    const float4* const A4 = reinterpret_cast<const float4*>(A) + a;
#pragma unroll
    for (int v = 0; v < B / 4 + 1; ++v) {
        float4 q = A4[v];
        if (FIRST) q = norm4(q, mu);  // x^0 arrives raw: remove the row's mean before any sum
        w[4 * v] = q.x;
        w[4 * v + 1] = q.y;
        w[4 * v + 2] = q.z;
        w[4 * v + 3] = q.w;
    }
    // the four running sums as two packed pairs (FADD2 / FMUL2: one issue slot for two points)
    float2 t01 = make_float2(xin.x, xin.y), t23 = make_float2(xin.z, xin.w);
    const float ninf = __int_as_float(0xff800000);
    float pend[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) best[j] = ninf;
#pragma unroll
    for (int m = 0; m < B; ++m) {
        const float s = sc[m];
        const float2 ss = make_float2(s, s);
        const uint32_t code = code0 - m;
        // eq. (15): the boxcar of m + 1 elements of x^level on top of X^{level-1}
        t01 = __fadd2_rn(t01, make_float2(w[m], w[m + 1]));
        t23 = __fadd2_rn(t23, make_float2(w[m + 2], w[m + 3]));
        const float2 k01 = __fmul2_rn(t01, ss), k23 = __fmul2_rn(t23, ss);
        float key[4] = {k01.x, k01.y, k23.x, k23.y};
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            key[j] = __uint_as_float((__float_as_uint(key[j]) & tag_mask) | code);
            if (MASKED && m >= mlim[j]) key[j] = ninf;  // does not fit the row (reading A3) or is not in the plan
            if (m & 1)
                best[j] = fmax3(best[j], pend[j], key[j]);
            else
                pend[j] = key[j];
        }
    }
    const float t[4] = {t01.x, t01.y, t23.x, t23.y};
    if (!last) {
        // eq. (13): x^{level+1}[q'] = x^level[2q' + B] + x^level[2q' + B + 1]; and X^level at the even points
        *reinterpret_cast<float2*>(A_next + 2 * a) = make_float2(w[B] + w[B + 1], w[B + 2] + w[B + 3]);
        *reinterpret_cast<float2*>(X_next + 2 * a) = make_float2(t[0], t[2]);
    }
}

// ITER: the best key of the four points of a task goes to its iteration's own plane (tag split off), scalar stores
// (a decimated row starts at any alignment); point q of level `level` is sample q << level of the row.
__device__ __forceinline__ void bd_store_iteration(const BdParams& p, const long long d, const int level,
                                                   const long long q0, const float (&key)[4]) {
    const uint32_t code_top = ~p.tag_mask;
    const long long npts = p.it_npts[level];
    const long long base = p.it_off[level] + d * npts;
    float* const ys = p.it_snr + base;
    int32_t* const yw = p.it_width + base;
    float y[4];
    int w[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const uint32_t b = __float_as_uint(key[j]);
        const bool none = key[j] == __int_as_float(0xff800000);
        y[j] = none ? key[j] : __uint_as_float(b & p.tag_mask);
        w[j] = none ? -1 : static_cast<int>(code_top - (b & code_top));
    }
    if (((base + q0) & 3) == 0 && q0 + 3 < npts) {  // the usual case (row lengths that are multiples of 2^(level+2))
        *reinterpret_cast<float4*>(ys + q0) = make_float4(y[0], y[1], y[2], y[3]);
        *reinterpret_cast<int4*>(yw + q0) = make_int4(w[0], w[1], w[2], w[3]);
        return;
    }
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        if (q0 + j < npts) {
            ys[q0 + j] = y[j];
            yw[q0 + j] = w[j];
        }
    }
}

template <int B, bool ITER>
__global__ void __launch_bounds__(kBdThreads) spd_boxdit_kernel(const BdParams p) {
    constexpr int T = kBdChunk, NT = kBdThreads, TASKS0 = T / 4 / NT;
    extern __shared__ __align__(128) float sm[];
    float* const x0 = sm;                                   // [2][T + B]
    float* const xl = x0 + 2 * (T + B);                     // x^i, i >= 1
    float* const xb = xl + T + kBdMaxLevels * B;            // X^{i-1} in, best keys out, i >= 1
    float* const scale = xb + T;                            // [I][B]
    __shared__ __align__(8) uint64_t full[2];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int I = p.n_levels;
    const long long d = blockIdx.x / p.segs_per_row;
    const int seg = static_cast<int>(blockIdx.x - d * p.segs_per_row);
    const int c_lo = seg * p.seg_chunks;                                      // chunks [c_lo, c_hi) are this block's
    const int c_hi = min(c_lo + p.seg_chunks, p.chunks_per_row);
    const int c_start = min(c_hi + p.warm_chunks, p.chunks_per_row) - 1;      // first chunk walked (latest in time)
    const float* __restrict__ row = p.plane + d * p.n_t;
    const int n_t = static_cast<int>(p.n_t);

    // carries start as zeros: past the end of the row nothing is added (and those windows are skipped); a
    // segment that starts inside the row warms up over warm_chunks >= L_MAX samples first
    for (int u = tid; u < bd_smem_floats<B>(); u += NT) sm[u] = 0.f;
    __syncthreads();
    {
        const float inv = p.sigma_w ? 1.f : 1.0f / __ldg(p.sigma + d);
        for (int k = tid; k < p.n_w; k += NT) {  // width index k = level * B + m
            const int i = k / B, m = k - i * B;
            const float L = static_cast<float>((((1 << i) - 1) * B) + ((m + 1) << i));  // eq. (14)
            scale[i * B + m] = p.sigma_w ? 1.0f / __ldg(p.sigma_w + d * p.n_w + k) : rsqrtf(L) * inv;
        }
    }
    const float mu = __ldg(p.mean + d);
    auto chunk_floats = [&](int c) { return min(T, n_t - c * T); };
    if (tid == 0) {
        mbar_init(&full[0], 1);
        mbar_init(&full[1], 1);
        fence_mbar_init();
        fence_proxy_async();
        for (int s = 0; s < 2; ++s) {
            const int c = c_start - s;
            if (c >= c_lo) {
                const uint32_t bytes = static_cast<uint32_t>(chunk_floats(c)) * 4u;
                mbar_arrive_expect_tx(&full[s], bytes);
                bulk_g2s(x0 + s * (T + B), row + static_cast<long long>(c) * T, bytes, &full[s]);
            }
        }
    }
    __syncthreads();

    const uint32_t code_top = ~p.tag_mask;  // tag of width index 0: all tag bits set
    int step = 0;
    for (int c = c_start; c >= c_lo; --c, ++step) {
        const int buf = step & 1;
        float* const A0 = x0 + buf * (T + B);
        mbar_wait(&full[buf], (step >> 1) & 1);
        const int t0 = c * T;
        const bool store = c < c_hi;  // chunks walked ahead of the segment only fill the carries
        // a window of this chunk may cross the end of the row: per-key test of fit
        const bool masked = static_cast<long long>(t0) + T + p.l_max_total > p.n_t;
        // ---- level 0 --------------------------------------------------------------------
        if (warp == 0 && lane < B) x0[(buf ^ 1) * (T + B) + T + lane] = A0[lane];  // the carry of x^0
        float best0[TASKS0][4];
        {
            const bool last = I == 1;
            float* const A1 = xl + bd_off_x<B>(1);
            float* const X1 = xb + bd_off_b(1);
#pragma unroll
            for (int k = 0; k < TASKS0; ++k) {
                const int a = tid + k * NT;
                int mlim[4] = {B, B, B, B};
                if (masked || (last && p.last_count < B)) {
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        const int fit = n_t - (t0 + 4 * a + j);  // samples from the point to the row's end
                        mlim[j] = min(fit, last ? p.last_count : B);
                    }
                    bd_task<B, true, true>(A0, make_float4(0.f, 0.f, 0.f, 0.f), a, mu, scale, code_top, p.tag_mask,
                                           last, A1, X1, mlim, best0[k]);
                } else {
                    bd_task<B, true, false>(A0, make_float4(0.f, 0.f, 0.f, 0.f), a, mu, scale, code_top, p.tag_mask,
                                            last, A1, X1, mlim, best0[k]);
                }
                if constexpr (ITER) {
                    if (store) bd_store_iteration(p, d, 0, static_cast<long long>(t0) + 4 * a, best0[k]);
                }
            }
        }
        __syncthreads();
        if (tid == 0 && c - 2 >= c_lo) {  // x^0 of this chunk is consumed: fetch the chunk two ahead into it
            const uint32_t bytes = static_cast<uint32_t>(chunk_floats(c - 2)) * 4u;
            fence_proxy_async();
            mbar_arrive_expect_tx(&full[buf], bytes);
            bulk_g2s(A0, row + static_cast<long long>(c - 2) * T, bytes, &full[buf]);
        }
        // ---- levels 1 .. I-1 ----------------------------------------------------------------
        for (int i = 1; i < I; ++i) {
            const bool last = i == I - 1;
            const float* const A = xl + bd_off_x<B>(i);
            float* const XB = xb + bd_off_b(i);
            float* const An = xl + bd_off_x<B>(i + 1);
            float* const Xn = xb + bd_off_b(i + 1);
            const int n_tasks = (T >> i) >> 2;
            const uint32_t code0 = code_top - static_cast<uint32_t>(i * B);
            const int base = ((1 << i) - 1) * B;  // L_MAX of the levels before (eq. 14)
            const bool slow = masked || (last && p.last_count < B);
            for (int a = tid; a < n_tasks; a += NT) {
                const float4 xin = *reinterpret_cast<const float4*>(XB + 4 * a);
                int mlim[4] = {B, B, B, B};
                float best[4];
                if (slow) {
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        const int fit = n_t - (t0 + ((4 * a + j) << i)) - base;  // room for the level's own part
                        mlim[j] = min(fit >> i, last ? p.last_count : B);       // (negative: nothing fits)
                    }
                    bd_task<B, false, true>(A, xin, a, mu, scale + i * B, code0, p.tag_mask, last, An, Xn, mlim, best);
                } else {
                    bd_task<B, false, false>(A, xin, a, mu, scale + i * B, code0, p.tag_mask, last, An, Xn, mlim, best);
                }
                if constexpr (ITER) {
                    if (store) bd_store_iteration(p, d, i, (static_cast<long long>(t0) >> i) + 4 * a, best);
                } else if (i <= 2) {
                    *reinterpret_cast<float4*>(XB + 4 * a) = make_float4(best[0], best[1], best[2], best[3]);
                } else {
                    // point q of level i is sample q * 2^i = entry q * 2^(i-2) of level 2's array: the best keys of the
                    // levels above 2 are folded into it here, so that the gather below reads three values per task
                    // instead of walking the levels (levels run one after the other: no two writers per entry)
                    float* const fin = xb + bd_off_b(2) + ((4 * a) << (i - 2));
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        float* const q = fin + (j << (i - 2));
                        *q = fmaxf(*q, best[j]);
                    }
                }
            }
            __syncthreads();
        }
        // ---- gather the levels per sample, store; carry x^i, i >= 1 -------------------------------
#pragma unroll
        for (int k = 0; k < (ITER ? 0 : TASKS0); ++k) {
            const int a = tid + k * NT;
            float* const key = best0[k];
            if (I > 1) {
                const float2 b1 = *reinterpret_cast<const float2*>(xb + bd_off_b(1) + 2 * a);
                key[0] = fmaxf(key[0], b1.x);
                key[2] = fmaxf(key[2], b1.y);
            }
            if (I > 2) key[0] = fmaxf(key[0], xb[bd_off_b(2) + a]);  // level 2 and, folded into it, the levels above
            if (p.activity && store && fmax3(fmaxf(key[0], key[1]), key[2], key[3]) >= p.thr_key)
                p.activity[d * p.chunks_per_row + c] = 1;  // any thread of the block may set it
            const int n = t0 + 4 * a;
            if (store && n < n_t) {
                float4 y;
                int4 wi;
                float* const yy = &y.x;
                int* const ww = &wi.x;
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const uint32_t b = __float_as_uint(key[j]);
                    const bool none = key[j] == __int_as_float(0xff800000);
                    yy[j] = none ? key[j] : __uint_as_float(b & p.tag_mask);
                    ww[j] = none ? -1 : static_cast<int>(code_top - (b & code_top));
                }
                *reinterpret_cast<float4*>(p.out_snr + d * p.n_t + n) = y;
                *reinterpret_cast<int4*>(p.out_width + d * p.n_t + n) = wi;
            }
        }
        for (int i = 1 + warp; i < I; i += NT / 32) {  // x^i[T_i + j] of the next chunk = x^i[j] of this one
            float* const A = xl + bd_off_x<B>(i);
            const float v = lane < B ? A[lane] : 0.f;
            __syncwarp();
            if (lane < B) A[(T >> i) + lane] = v;
        }
        __syncthreads();
    }
}

template <int B>
int bd_launch(const BdParams& prm, unsigned blocks, cudaStream_t stream) {
    static bool configured = false;  // per process and instantiation; the attribute is sticky
    const size_t smem = static_cast<size_t>(bd_smem_floats<B>()) * sizeof(float);
    if (!configured) {
        cudaError_t e =
            cudaFuncSetAttribute(spd_boxdit_kernel<B, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem));
        if (e == cudaSuccess)
            e = cudaFuncSetAttribute(spd_boxdit_kernel<B, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem));
        if (e != cudaSuccess) return cuda_fail(e, "configuring the BoxDIT kernel");
        configured = true;
    }
    if (prm.it_snr)
        spd_boxdit_kernel<B, true><<<blocks, kBdThreads, smem, stream>>>(prm);
    else
        spd_boxdit_kernel<B, false><<<blocks, kBdThreads, smem, stream>>>(prm);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "launching the BoxDIT kernel");
    return SPD_OK;
}

}  // namespace

// The plan's widths are exactly Alg. 1's (eq. 14, D = 2, B = 4, 8, 16 or 32 per iteration, possibly cut by
// max_width inside the last iteration) and every iteration sits on its own grid 2^i: fills plan->boxdit.
bool boxdit_configure(spd_plan* plan) {
    plan->boxdit = BoxditConfig();
    const std::vector<int32_t>& w = plan->widths;
    const std::vector<int32_t>& s = plan->separations;
    if (s.size() != w.size() || plan->n_t % 4 != 0 || plan->n_t > 0x7fffffffll - 2 * kBdChunk || w.size() > 256) return false;
    int B = 0;
    while (B < static_cast<int>(s.size()) && s[B] == 1) ++B;
    if (B != 4 && B != 8 && B != 16 && B != 32) return false;
    int levels = 0;
    for (size_t k = 0; k < w.size(); ++k) {
        const int i = static_cast<int>(k) / B, m = static_cast<int>(k) % B;
        if (i >= kBdMaxLevels) return false;
        if (w[k] != ((1 << i) - 1) * B + ((m + 1) << i) || s[k] != (1 << i)) return false;
        levels = i + 1;
    }
    if (levels > 1 && static_cast<int>(w.size()) <= B) return false;
    BoxditConfig& c = plan->boxdit;
    c.B = B;
    c.levels = levels;
    c.last_count = static_cast<int>(w.size()) - (levels - 1) * B;
    c.chunks_per_row = static_cast<int>((plan->n_t + kBdChunk - 1) / kBdChunk);
    c.warm_chunks = (w.back() + kBdChunk - 1) / kBdChunk;
    // segments: 32 warm-up lengths each (the replay then costs 3 %), shorter only to reach ~16 blocks per SM
    int seg_chunks;
    if (plan->segs_option > 0) {
        seg_chunks = (c.chunks_per_row + plan->segs_option - 1) / plan->segs_option;
    } else {
        seg_chunks = std::min(c.chunks_per_row, 32 * c.warm_chunks);
        const int64_t want_blocks = static_cast<int64_t>(plan->sm_count) * 16;
        while (seg_chunks > 4 * c.warm_chunks &&
               plan->n_dm * ((c.chunks_per_row + seg_chunks - 1) / seg_chunks) < want_blocks)
            seg_chunks = (seg_chunks + 1) / 2;
    }
    c.seg_chunks = std::max(1, seg_chunks);
    c.segs_per_row = (c.chunks_per_row + c.seg_chunks - 1) / c.seg_chunks;
    c.smem_bytes = static_cast<int>(sizeof(float)) *
                   (B == 4 ? bd_smem_floats<4>() : B == 8 ? bd_smem_floats<8>() : B == 16 ? bd_smem_floats<16>()
                                                                                         : bd_smem_floats<32>());
    return true;
}

static int boxdit_run_any(const spd_plan* plan, int64_t n_dm, const float* plane, const float* mean, const float* sigma,
                          float* out_snr, int32_t* out_width, cudaStream_t stream, const float* sigma_w,
                          float* it_snr, int32_t* it_width, float threshold = 0.f, uint8_t* activity = nullptr);

int boxdit_run(const spd_plan* plan, int64_t n_dm, const float* plane, const float* mean, const float* sigma,
               float* out_snr, int32_t* out_width, cudaStream_t stream, const float* sigma_w, float threshold,
               uint8_t* activity) {
    return boxdit_run_any(plan, n_dm, plane, mean, sigma, out_snr, out_width, stream, sigma_w, nullptr, nullptr,
                          threshold, activity);
}

// Output separated by iteration (eq. 12): the levels' best keys go to their own decimated planes, concatenated
// in it_snr / it_width (layout of spd_run_iterations); whole planes only (n_dm = plan->n_dm).
int boxdit_run_iterations(const spd_plan* plan, const float* plane, const float* mean, const float* sigma,
                          float* it_snr, int32_t* it_width, cudaStream_t stream) {
    return boxdit_run_any(plan, plan->n_dm, plane, mean, sigma, nullptr, nullptr, stream, nullptr, it_snr, it_width);
}

static int boxdit_run_any(const spd_plan* plan, int64_t n_dm, const float* plane, const float* mean, const float* sigma,
                          float* out_snr, int32_t* out_width, cudaStream_t stream, const float* sigma_w,
                          float* it_snr, int32_t* it_width, float threshold, uint8_t* activity) {
    const BoxditConfig& c = plan->boxdit;
    BdParams prm = {};
    prm.activity = activity;
    // the tag replaces up to 8 low mantissa bits of a key (2^-15 relative): lower the threshold by more than that
    prm.thr_key = threshold - fabsf(threshold) * 4e-5f;
    if (activity) {
        const size_t bytes = (static_cast<size_t>(n_dm) * static_cast<size_t>(c.chunks_per_row) + 127) / 128 * 128;
        const cudaError_t em = cudaMemsetAsync(activity, 0, bytes, stream);
        if (em != cudaSuccess) return cuda_fail(em, "clearing the activity map");
    }
    prm.it_snr = it_snr;
    prm.it_width = it_width;
    if (it_snr) {
        long long off = 0;
        for (int i = 0; i < c.levels; ++i) {
            prm.it_off[i] = off;
            prm.it_npts[i] = (plan->n_t + (1ll << i) - 1) >> i;
            off += n_dm * prm.it_npts[i];
        }
    }
    prm.plane = plane;
    prm.mean = mean;
    prm.sigma = sigma;
    prm.sigma_w = sigma_w;
    prm.out_snr = out_snr;
    prm.out_width = out_width;
    prm.n_t = plan->n_t;
    prm.chunks_per_row = c.chunks_per_row;
    prm.segs_per_row = c.segs_per_row;
    prm.seg_chunks = c.seg_chunks;
    prm.warm_chunks = c.warm_chunks;
    prm.n_levels = c.levels;
    prm.n_w = static_cast<int>(plan->widths.size());
    prm.last_count = c.last_count;
    prm.l_max_total = plan->widths.back();
    prm.tag_mask = prm.n_w <= 128 ? ~127u : ~255u;
    const int64_t blocks = n_dm * c.segs_per_row;
    if (blocks > 0x7fffffffll) {
        set_error("plane too large for the BoxDIT kernel's grid");
        return SPD_ERR_INVALID_ARG;
    }
    switch (c.B) {
        case 4: return bd_launch<4>(prm, static_cast<unsigned>(blocks), stream);
        case 8: return bd_launch<8>(prm, static_cast<unsigned>(blocks), stream);
        case 16: return bd_launch<16>(prm, static_cast<unsigned>(blocks), stream);
        default: return bd_launch<32>(prm, static_cast<unsigned>(blocks), stream);
    }
}

}  // namespace spd
