// Streaming partial-sum tree for the IGRID depth-1 width set:
// widths 2^k (k = 0 .. LAST) and 3 * 2^m (m = 0 .. LAST-2), i.e. "L = sum a_k 2^(i-k)" of eq. (18)
// with one extra term (Table 1: 16 -> 16, 24), every width at
// every sample (reading A1).  26 widths up to 8192: 3.6 % mean loss on log-uniform pulse widths
// instead of the 7.4 % of the 14 widths 2^k.
//
// Non-power-of-two boxcars are built from two partial sums of the dyadic tree, never summed
// directly (eq. 18; SURVEY.md row a4  X_{a+b}[n] = P_a[n] + P_b[n+a]):
//
//     X_{3 * 2^m}[n] = P_m[n] + P_{m+1}[n + 2^m]
//
// The kernel is spd_tree.cu's (reverse-time streaming, float4 per thread x R rows, levels in
// registers / shared memory / delay registers by distance, tagged 3-input max; see there) with
// one more operand per level:
//   * m = 0, 1 (widths 3, 6): in registers from the three raw float4;
//   * m = 2 .. LT: P_{m+1}[n + 2^m] is read from the shared-memory buffer that exchange level
//     m+1 has just filled (one more 128-bit load per row and level, same barrier);
//   * m = LT+1: one extra exchange of P_{LT+2} (partner half a row away);
//   * m >= LT+2: P_{m+1} of the row 2^(m-LT-2) rows later is this step's new value of that
//     row, or - across the chunk boundary - the delay registers the next level keeps anyway.
#include <cuda_runtime.h>
#include <stdint.h>

#include <algorithm>

#include "spd_tree_common.cuh"

namespace spd {
namespace {

// Index in the ascending set 1, 2, 3, 4, 6, 8, 12, 16, 24, ...
constexpr int idx_pow2(int k) { return k == 0 ? 0 : 2 * k - 1; }
constexpr int idx_ig(int m) { return 2 * m + 2; }

// Scaled value with the inverted width index in the low mantissa bits; in the guarded variant
// element v of the float4 is valid iff WIDTH <= lim - v (reading A3).
template <int IDX, int WIDTH, bool FAST>
__device__ __forceinline__ float4 gkey(float4 p, float scale, int lim, uint32_t tm) {
    const float4 v = scale4(p, scale);
    float4 q = make_float4(pack1<IDX>(v.x, tm), pack1<IDX>(v.y, tm), pack1<IDX>(v.z, tm), pack1<IDX>(v.w, tm));
    if constexpr (!FAST) {
        const float ninf = __int_as_float(0xff800000);
        if (WIDTH > lim) q.x = ninf;
        if (WIDTH > lim - 1) q.y = ninf;
        if (WIDTH > lim - 2) q.z = ninf;
        if (WIDTH > lim - 3) q.w = ninf;
    }
    return q;
}
// SNR key of width 2^k (eq. 5: scale 2^(-k/2)) and of width 3 * 2^m (scale 2^(-m/2) / sqrt 3).
// SW: a measured sigma per width instead: cx.ls[width index] = 1 / sigma_{d, L}.
template <int k, bool FAST, bool SW>
__device__ __forceinline__ float4 kp(float4 p, int lim, const ChunkCtx& cx) {
    return gkey<idx_pow2(k), (1 << k), FAST>(p, SW ? cx.ls[idx_pow2(k)] : level_scale<k>(), lim, cx.tm);
}
template <int m, bool FAST, bool SW>
__device__ __forceinline__ float4 kg(float4 p, int lim, const ChunkCtx& cx) {
    return gkey<idx_ig(m), 3 * (1 << m), FAST>(p, SW ? cx.ls[idx_ig(m)] : level_scale<m>() * 0.57735026918962576451f, lim,
                                               cx.tm);
}

// Halo slots per parity: the exchange levels use d4 slots each (sum T - 2), the extra
// exchange T / 2 more.
template <int T>
constexpr int ig_halo_slots() {
    return 2 * T;
}

// Exchange levels k = 3 .. LT+1.  The buffer holds P_k: partner d4 slots later gives P_{k+1},
// partner d4 / 2 slots later gives width 3 * 2^(k-1) = P_{k-1}[n] + P_k[n + 2^(k-1)].
template <int T, int R, int K, bool FAST, bool SW, int k, int hoff>
__device__ __forceinline__ void ig_exchange_levels(float4 (&P)[R], float4 (&Pprev)[R], float4 (&best)[R],
                                                   const int (&lim)[R], float4* __restrict__ pp,
                                                   float4* __restrict__ hr, float4* __restrict__ hw, int& xsel,
                                                   const ChunkCtx& cx) {
    using G = Geo<T, R, K>;
    if constexpr (k <= G::LT + 1 && k + 1 <= G::LAST) {
        constexpr int d4 = (1 << k) / 4;
        constexpr int h4 = d4 / 2;
        const int tid = cx.tid;
        float4* const buf = pp + xsel * G::C4;
        xsel ^= 1;
#pragma unroll
        for (int r = 0; r < R; ++r) st_shared4(buf + tid + T * r, P[r]);
        if (tid < d4) hw[hoff + tid] = P[0];
        __syncthreads();
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const float4* s1 = buf + (tid + T * r + d4);
            const float4* s2 = buf + (tid + T * r + h4);
            if (r == R - 1 && tid + d4 >= T) s1 = hr + (hoff + tid + d4 - T);
            if (r == R - 1 && tid + h4 >= T) s2 = hr + (hoff + tid + h4 - T);
            const float4 now = add4(P[r], *s1);
            const float4 g = add4(Pprev[r], *s2);
            if (FAST || cx.do_out)
                best[r] = max4(best[r], kp<k + 1, FAST, SW>(now, lim[r], cx), kg<k - 1, FAST, SW>(g, lim[r], cx));
            Pprev[r] = P[r];
            P[r] = now;
        }
        ig_exchange_levels<T, R, K, FAST, SW, k + 1, hoff + d4>(P, Pprev, best, lim, pp, hr, hw, xsel, cx);
    } else if constexpr (G::J >= 1) {
        // extra exchange: P = P_{LT+2}, Pprev = P_{LT+1}; width 3 * 2^(LT+1) needs P_{LT+2} half a row later
        constexpr int h4 = T / 2;
        static_assert(hoff + h4 <= ig_halo_slots<T>(), "halo buffer overflow");
        const int tid = cx.tid;
        float4* const buf = pp + xsel * G::C4;
        xsel ^= 1;
#pragma unroll
        for (int r = 0; r < R; ++r) st_shared4(buf + tid + T * r, P[r]);
        if (tid < h4) hw[hoff + tid] = P[0];
        __syncthreads();
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const float4* s2 = buf + (tid + T * r + h4);
            if (r == R - 1 && tid + h4 >= T) s2 = hr + (hoff + tid + h4 - T);
            const float4 g = add4(Pprev[r], *s2);
            if (FAST || cx.do_out) best[r] = max4(best[r], kg<G::LT + 1, FAST, SW>(g, lim[r], cx));
        }
    }
}

// P_{k+1} of the row `row` (>= R: rows of earlier chunks) as kept by the delay registers of
// register level j1 = j + 1 (which stores its own inputs, i.e. level k+1 values).
template <int T, int R, int K, bool FAST, int PH, int j1>
__device__ __forceinline__ float4 ig_delayed(const float4 (&dl)[Geo<T, R, K>::ND + 1], int row_const) {
    // row_const is a compile-time constant after unrolling; written as a function of it
    using G = Geo<T, R, K>;
    constexpr int D1 = 1 << j1;   // partner distance of level j1 in rows
    constexpr int off1 = D1 - 1;  // its first delay register
    if constexpr (D1 < R) {
        return dl[off1 + (row_const - R)];  // first D1 rows of the previous chunk
    } else {
        constexpr int Q1 = D1 / R;  // FIFO depth in chunks
        const int age = row_const / R;  // chunks back (>= 1)
        const int rr = row_const % R;
        constexpr bool kSlotted = FAST && G::U >= Q1;
        // slotted: the chunk of age a was written at phase PH - a; canonical: newest at slot Q1 - 1
        const int slot = kSlotted ? (((PH - age) % Q1) + Q1) % Q1 : Q1 - age;
        return dl[off1 + slot * R + rr];
    }
}

// In-register levels j = 0 .. J-1 (own level k = LT + 2 + j, partner D = 2^j rows later).
template <int T, int R, int K, bool FAST, bool SW, int PH, int j>
__device__ __forceinline__ void ig_register_levels(float4 (&P)[R], float4 (&best)[R], const int (&lim)[R],
                                                   float4 (&dl)[Geo<T, R, K>::ND + 1], const ChunkCtx& cx) {
    using G = Geo<T, R, K>;
    if constexpr (j < G::J) {
        constexpr int D = 1 << j;
        constexpr int off = D - 1;
        constexpr int k = G::LT + 2 + j;
        float4 now[R];
        if constexpr (D < R) {
#pragma unroll
            for (int r = 0; r < R; ++r) now[r] = add4(P[r], r + D < R ? P[r + D] : dl[off + r + D - R]);
        } else {
            constexpr int Q = D / R;
            constexpr bool kSlotted = FAST && G::U >= Q;
            constexpr int slot = kSlotted ? (PH % Q) : 0;
#pragma unroll
            for (int r = 0; r < R; ++r) now[r] = add4(P[r], dl[off + slot * R + r]);
        }
        // width 3 * 2^k = P_k[row r] + P_{k+1}[row r + D]: exists while a next level does
        if constexpr (j + 1 < G::J) {
#pragma unroll
            for (int r = 0; r < R; ++r) {
                float4 nxt;
                if (r + D < R) {
                    nxt = now[r + D];
                } else {
                    nxt = ig_delayed<T, R, K, FAST, PH, j + 1>(dl, r + D);
                }
                const float4 g = add4(P[r], nxt);
                if (FAST || cx.do_out)
                    best[r] = max4(best[r], kp<k + 1, FAST, SW>(now[r], lim[r], cx), kg<k, FAST, SW>(g, lim[r], cx));
            }
        } else {
#pragma unroll
            for (int r = 0; r < R; ++r)
                if (FAST || cx.do_out) best[r] = max4(best[r], kp<k + 1, FAST, SW>(now[r], lim[r], cx));
        }
        // delay registers of this level take this chunk's inputs
        if constexpr (D < R) {
#pragma unroll
            for (int i = 0; i < D; ++i) dl[off + i] = P[i];
        } else {
            constexpr int Q = D / R;
            constexpr bool kSlotted = FAST && G::U >= Q;
            if constexpr (kSlotted) {
                constexpr int slot = PH % Q;
#pragma unroll
                for (int r = 0; r < R; ++r) dl[off + slot * R + r] = P[r];
            } else {
#pragma unroll
                for (int s = 0; s + 1 < Q; ++s) {
#pragma unroll
                    for (int r = 0; r < R; ++r) dl[off + s * R + r] = dl[off + (s + 1) * R + r];
                }
#pragma unroll
                for (int r = 0; r < R; ++r) dl[off + (Q - 1) * R + r] = P[r];
            }
        }
#pragma unroll
        for (int r = 0; r < R; ++r) P[r] = now[r];
        ig_register_levels<T, R, K, FAST, SW, PH, j + 1>(P, best, lim, dl, cx);
    }
}

// One streaming step (see tree_chunk in spd_tree.cu); needs K >= 5.
template <int T, int R, int K, bool FAST, int PH, bool SW>
__device__ __forceinline__ float ig_chunk(const float4* __restrict__ st4, float4* __restrict__ pp,
                                          float4* __restrict__ halo, int& xsel, int& hsel,
                                          float4 (&dl)[Geo<T, R, K>::ND + 1], const ChunkCtx& cx) {
    using G = Geo<T, R, K>;
    static_assert(K >= 5, "the IGRID tree needs max_width >= 16");
    const int tid = cx.tid;
    const float mu = cx.mu;
    const uint32_t tm = cx.tm;

    float4 P[R], Pprev[R], best[R];
    int lim[R];

    // ---- widths 1, 2, 3, 4, 6, 8 from three raw float4 ---------------------------------
#pragma unroll
    for (int r = 0; r < R; ++r) {
        if constexpr (FAST) {
            lim[r] = 1 << 30;
        } else {
            const long long left = cx.n_t - (cx.n0 + 4ll * (tid + T * r));
            lim[r] = left > (1ll << 30) ? (1 << 30) : (left < 0 ? 0 : static_cast<int>(left));
        }
        const float4 a = norm4(st4[tid + T * r], mu);
        const float4 b = norm4(st4[tid + T * r + 1], mu);
        const float4 c = norm4(st4[tid + T * r + 2], mu);
        const float s01 = a.x + a.y, s12 = a.y + a.z, s23 = a.z + a.w, s34 = a.w + b.x;
        const float s45 = b.x + b.y, s56 = b.y + b.z, s67 = b.z + b.w, s78 = b.w + c.x;
        const float s89 = c.x + c.y, s9a = c.y + c.z;
        const float q4567 = s45 + s67, q5678 = s56 + s78;
        const float4 p1 = make_float4(s01, s12, s23, s34);
        const float4 p2 = make_float4(s01 + s23, s12 + s34, s23 + s45, s34 + s56);
        const float4 p3 = make_float4(p2.x + q4567, p2.y + q5678, p2.z + (s67 + s89), p2.w + (s78 + s9a));
        // width 3 = x[n] + P_1[n+1]; width 6 = P_1[n] + P_2[n+2]
        const float4 x3 = make_float4(a.x + s12, a.y + s23, a.z + s34, a.w + s45);
        const float4 x6 = make_float4(s01 + p2.z, s12 + p2.w, s23 + q4567, s34 + q5678);
        if (FAST || cx.do_out) {
            float4 bb = max4(kp<0, FAST, SW>(a, lim[r], cx), kp<1, FAST, SW>(p1, lim[r], cx), kp<2, FAST, SW>(p2, lim[r], cx));
            bb = max4(bb, kp<3, FAST, SW>(p3, lim[r], cx), kg<0, FAST, SW>(x3, lim[r], cx));
            best[r] = max4(bb, kg<1, FAST, SW>(x6, lim[r], cx));
        }
        Pprev[r] = p2;
        P[r] = p3;
    }

    // ---- exchange levels (+ the extra one) ----------------------------------------------
    constexpr int HS = ig_halo_slots<T>();
    float4* const hr = halo + hsel * HS;
    float4* const hw = halo + (hsel ^ 1) * HS;
    hsel ^= 1;
    ig_exchange_levels<T, R, K, FAST, SW, 3, 0>(P, Pprev, best, lim, pp, hr, hw, xsel, cx);

    // ---- in-register levels ---------------------------------------------------------------
    ig_register_levels<T, R, K, FAST, SW, PH, 0>(P, best, lim, dl, cx);

    // ---- unpack and store -------------------------------------------------------------------
    float top = __int_as_float(0xff800000);
    if (FAST || cx.do_out) {
#pragma unroll
        for (int r = 0; r < R; ++r) {
            if (FAST || lim[r] > 0) {
                const float4 kq = best[r];
                top = fmax3(top, fmax3(kq.x, kq.y, kq.z), kq.w);
                const float4 y = scale4(make_float4(__uint_as_float(__float_as_uint(kq.x) & tm),
                                                    __uint_as_float(__float_as_uint(kq.y) & tm),
                                                    __uint_as_float(__float_as_uint(kq.z) & tm),
                                                    __uint_as_float(__float_as_uint(kq.w) & tm)),
                                        cx.inv);
                const int4 w = make_int4(static_cast<int>(~__float_as_uint(kq.x) & kCodeMask),
                                         static_cast<int>(~__float_as_uint(kq.y) & kCodeMask),
                                         static_cast<int>(~__float_as_uint(kq.z) & kCodeMask),
                                         static_cast<int>(~__float_as_uint(kq.w) & kCodeMask));
                const long long o = cx.n0 + 4ll * (tid + T * r);
                *reinterpret_cast<float4*>(cx.out_snr + o) = y;
                *reinterpret_cast<int4*>(cx.out_width + o) = w;
            }
        }
    }
    return top;
}

constexpr int ig_threads_for(int K) { return K <= 15 ? 128 : 256; }
constexpr int ig_rows_for(int) { return 4; }
// K <= 14: 3 blocks per SM (168 registers, no spills): 18.1 ms against 19.2 ms at 2 blocks (config-3 plane)
constexpr int ig_blocks_per_sm(int K) { return K <= 14 ? 3 : (K == 15 ? 2 : 1); }
// with a run-time scale per width (2K - 2 more registers) two blocks per SM up to K = 14
constexpr int ig_blocks_per_sm(int K, bool SW) { return (SW && K <= 14) ? 2 : ig_blocks_per_sm(K); }

template <int T, int R>
constexpr size_t ig_smem_bytes() {
    constexpr size_t C = 4 * T * R;
    return 2 * C * 4 + kStages * (C + 8) * 4 + 2 * ig_halo_slots<T>() * 16 + kStages * 8;
}

// Same streaming driver as spd_tree_kernel (segments, guarded steps, bulk-copy ring).
template <int T, int R, int K, bool SW>
__global__ void __launch_bounds__(T, ig_blocks_per_sm(K, SW)) spd_tree_ig_kernel(const TreeParams p) {
    using G = Geo<T, R, K>;
    constexpr int C = G::C;
    constexpr int M = 1 << (K - 1);
    constexpr int GUARD = M;  // widest window: 2^(K-1) > 3 * 2^(K-3)
    constexpr int HS = ig_halo_slots<T>();
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float4* const pp = reinterpret_cast<float4*>(smem_raw);
    float* const stages = reinterpret_cast<float*>(smem_raw + 2 * C * 4);
    float4* const halo = reinterpret_cast<float4*>(stages + kStages * (C + 8));
    uint64_t* const bars = reinterpret_cast<uint64_t*>(halo + 2 * HS);

    const int tid = threadIdx.x;
    const int d = blockIdx.x / p.segs_per_row;
    const int s = blockIdx.x - d * p.segs_per_row;
    const int c_lo = s * p.seg_chunks;
    const int c_hi = min(c_lo + p.seg_chunks, p.chunks_per_row);
    if (c_lo >= c_hi) return;
    const int c_top = min(c_hi + p.warm_chunks, p.chunks_per_row);
    const long long n_t = p.n_t;
    const int c_fast_end = n_t >= GUARD ? static_cast<int>((n_t - GUARD) / C) : 0;
    const int first_fast = max(c_lo, min(c_hi, c_fast_end));

    const float* __restrict__ row = p.plane + static_cast<long long>(d) * n_t;
    ChunkCtx cx;
    cx.mu = p.mean[d];
    const float sg = SW ? 1.0f : p.sigma[d];
    cx.inv = 1.0f / sg;
    if constexpr (SW) {
        // keys are SNRs already: 1 / sigma_{d, L} per width index, nothing left for the store
        const float* __restrict__ swr = p.sigma_w + static_cast<long long>(d) * (2 * K - 2);
#pragma unroll
        for (int k = 0; k < 2 * K - 2; ++k) cx.ls[k] = 1.0f / __ldg(swr + k);
    }
    cx.tm = p.tag_mask;
    cx.out_snr = p.out_snr + static_cast<long long>(d) * n_t;
    cx.out_width = p.out_width + static_cast<long long>(d) * n_t;
    cx.n_t = n_t;
    cx.tid = tid;
    uint8_t* const act = p.activity ? p.activity + static_cast<long long>(d) * p.chunks_per_row : nullptr;
    float thr_key = __int_as_float(0x7f800000);
    if (act) {
        const float t = p.threshold * sg;
        thr_key = t - fabsf(t) * 2e-6f;
    }

    for (int i = tid; i < 2 * HS; i += T) halo[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    if (tid == 0) {
#pragma unroll
        for (int i = 0; i < kStages; ++i) mbar_init(&bars[i], 1);
        fence_mbar_init();
    }
    float4 dl[G::ND + 1];
#pragma unroll
    for (int i = 0; i < G::ND + 1; ++i) dl[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    int xsel = 0, hsel = 0;
    __syncthreads();

    for (int c = c_top - 1; c >= first_fast; --c) {
        const long long n0 = static_cast<long long>(c) * C;
        {
            // n0 and n_t are multiples of 4: a float4 lies entirely inside or outside the row.  All of a thread's
            // 128-bit loads are issued before the first store (one memory latency per step, not one per element).
            constexpr int NV = (C + 8) / 4, NJ = (NV + T - 1) / T;
            const float4* const row4 = reinterpret_cast<const float4*>(row + n0);
            const float4 fill = make_float4(cx.mu, cx.mu, cx.mu, cx.mu);
            float4 v[NJ];
#pragma unroll
            for (int j = 0; j < NJ; ++j) {
                const int i = tid + T * j;
                v[j] = (i < NV && n0 + 4ll * i < n_t) ? __ldg(row4 + i) : fill;
            }
#pragma unroll
            for (int j = 0; j < NJ; ++j) {
                const int i = tid + T * j;
                if (i < NV) reinterpret_cast<float4*>(stages)[i] = v[j];
            }
        }
        __syncthreads();
        cx.n0 = n0;
        cx.do_out = c < c_hi;
        const float top = ig_chunk<T, R, K, false, 0, SW>(reinterpret_cast<const float4*>(stages), pp, halo, xsel, hsel,
                                                      dl, cx);
        if (act && cx.do_out && top >= thr_key) act[c] = 1;
        __syncthreads();
    }

    const int n_fast = first_fast - c_lo;
    if (n_fast <= 0) return;
    fence_proxy_async();
    __syncthreads();
    constexpr uint32_t kBytes = (C + 8) * 4;
    if (tid == 0) {
#pragma unroll
        for (int j = 0; j < kStages - 1; ++j) {
            if (j < n_fast) {
                mbar_arrive_expect_tx(&bars[j], kBytes);
                bulk_g2s(stages + j * (C + 8), row + static_cast<long long>(first_fast - 1 - j) * C, kBytes,
                         &bars[j]);
            }
        }
    }
    int stage = 0;
    uint32_t phase = 0;
    cx.do_out = true;
    int it = 0;
    while (it < n_fast) {
        static_phases<0, G::U>([&](auto ph) {
            if (it < n_fast) {
                if (tid == 0) {
                    const int nx = it + kStages - 1;
                    if (nx < n_fast) {
                        const int sx = stage == 0 ? kStages - 1 : stage - 1;
                        mbar_arrive_expect_tx(&bars[sx], kBytes);
                        bulk_g2s(stages + sx * (C + 8), row + static_cast<long long>(first_fast - 1 - nx) * C,
                                 kBytes, &bars[sx]);
                    }
                }
                mbar_wait(&bars[stage], phase);
                const int c = first_fast - 1 - it;
                cx.n0 = static_cast<long long>(c) * C;
                const float top = ig_chunk<T, R, K, true, decltype(ph)::value, SW>(
                    reinterpret_cast<const float4*>(stages + stage * (C + 8)), pp, halo, xsel, hsel, dl, cx);
                if (act && top >= thr_key) act[c] = 1;
                if (++stage == kStages) {
                    stage = 0;
                    phase ^= 1;
                }
                ++it;
            }
        });
    }
}

template <int T, int R, int K>
cudaError_t ig_prepare(TreeConfig& cfg) {
    cfg.smem_bytes = ig_smem_bytes<T, R>();
    cudaError_t e = cudaFuncSetAttribute(spd_tree_ig_kernel<T, R, K, false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         static_cast<int>(cfg.smem_bytes));
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(spd_tree_ig_kernel<T, R, K, true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 static_cast<int>(cfg.smem_bytes));
    if (e != cudaSuccess) return e;
    int nb = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, spd_tree_ig_kernel<T, R, K, false>, T, cfg.smem_bytes);
    if (e != cudaSuccess) return e;
    cfg.blocks_per_sm = nb;
    return cudaSuccess;
}

#define SPD_IG_CASES(OP) OP(5) OP(6) OP(7) OP(8) OP(9) OP(10) OP(11) OP(12) OP(13) OP(14) OP(15) OP(16)

}  // namespace

// widths == {2^k : k <= LAST} U {3 * 2^m : m <= LAST - 2} with LAST >= 4; returns K = LAST + 1 or 0.
int ig_applicable(const std::vector<int32_t>& widths, int64_t n_t) {
    if (n_t % 4 != 0 || widths.empty()) return 0;
    const int32_t top = widths.back();
    if (top < 16 || (top & (top - 1)) != 0) return 0;
    int last = 0;
    while ((1 << last) < top) ++last;
    if (last + 1 > kTreeMaxLevels) return 0;
    std::vector<int32_t> want;
    for (int k = 0; k <= last; ++k) want.push_back(1 << k);
    for (int m = 0; m <= last - 2; ++m) want.push_back(3 << m);
    std::sort(want.begin(), want.end());
    return want == widths ? last + 1 : 0;
}

int ig_configure(spd_plan* plan) {
    TreeConfig& cfg = plan->tree;
    cfg.T = ig_threads_for(cfg.K);
    cfg.chunk = 4 * cfg.T * ig_rows_for(cfg.K);
    cudaError_t e = cudaErrorInvalidValue;
#define SPD_PREP(KK) \
    if (cfg.K == KK) e = ig_prepare<ig_threads_for(KK), ig_rows_for(KK), KK>(cfg);
    SPD_IG_CASES(SPD_PREP)
#undef SPD_PREP
    if (e != cudaSuccess) return cuda_fail(e, "configuring the IGRID-tree kernel");
    if (cfg.blocks_per_sm < 1) {
        set_error("IGRID-tree kernel does not fit on this device (K=%d, smem=%zu)", cfg.K, cfg.smem_bytes);
        return SPD_ERR_CUDA;
    }
    return tree_configure_segments(plan);
}

int ig_run(const spd_plan* plan, int64_t n_dm, const float* plane, const float* mean, const float* sigma,
           float* out_snr, int32_t* out_width, float threshold, uint8_t* activity, cudaStream_t stream,
           const float* sigma_w) {
    const TreeConfig& cfg = plan->tree;
    TreeParams prm;
    prm.plane = plane;
    prm.mean = mean;
    prm.sigma = sigma;
    prm.sigma_w = sigma_w;  // [n_dm][2K - 2] or nullptr
    for (int k = 0; k < 16; ++k) prm.gmask[k] = 0u;
    prm.out_snr = out_snr;
    prm.out_width = out_width;
    prm.activity = activity;
    prm.threshold = threshold;
    prm.n_t = plan->n_t;
    prm.n_dm = n_dm;
    prm.chunks_per_row = cfg.chunks_per_row;
    prm.seg_chunks = cfg.seg_chunks;
    prm.segs_per_row = cfg.segs_per_row;
    prm.warm_chunks = cfg.warm_chunks;
    prm.tag_mask = ~kCodeMask;
    cudaError_t e = cudaSuccess;
    if (activity) {
        const size_t bytes = (static_cast<size_t>(n_dm) * cfg.chunks_per_row + 127) / 128 * 128;
        e = cudaMemsetAsync(activity, 0, bytes, stream);
        if (e != cudaSuccess) return cuda_fail(e, "clearing the activity map");
    }
    e = cudaErrorInvalidValue;
    const dim3 grid(static_cast<unsigned>(n_dm * cfg.segs_per_row));
#define SPD_LAUNCH(KK)                                                                                            \
    if (cfg.K == KK) {                                                                                            \
        if (sigma_w)                                                                                              \
            spd_tree_ig_kernel<ig_threads_for(KK), ig_rows_for(KK), KK, true>                                     \
                <<<grid, ig_threads_for(KK), cfg.smem_bytes, stream>>>(prm);                                      \
        else                                                                                                      \
            spd_tree_ig_kernel<ig_threads_for(KK), ig_rows_for(KK), KK, false>                                    \
                <<<grid, ig_threads_for(KK), cfg.smem_bytes, stream>>>(prm);                                      \
        e = cudaGetLastError();                                                                                   \
    }
    SPD_IG_CASES(SPD_LAUNCH)
#undef SPD_LAUNCH
    if (e != cudaSuccess) return cuda_fail(e, "launching the IGRID-tree kernel");
    return SPD_OK;
}

}  // namespace spd
