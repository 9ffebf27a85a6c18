// Dyadic partial-sum tree, streamed along each DM row.
//
// Width set {1, 2, 4, ..., 2^(K-1)} (the decimation-in-time set, Alg. 3)
// evaluated at EVERY sample (boxcar separation L_s = 1, reading A1).  Long boxcars are
// never summed directly: with P_k[n] = X_{2^k}[n] (eq. 2),
//
//     P_{k+1}[n] = P_k[n] + P_k[n + 2^k]                      (eq. 15/16 reuse)
//
// so every level costs one add per sample.  SNR_{2^k}[n] = P_k[n] / (sigma sqrt(2^k)) on
// mean-removed data (eq. 4, 5); Y = max_k, W = arg max_k (eq. 12,
// PAPER.md:183-185), smallest width winning exact ties.
//
// Design (B200, not the paper's P100/Titan V kernel):
//   * One block = one stream over a segment of one DM row, marching in REVERSE time in
//     chunks of C = 4*T*R samples (T threads, R "rows" of 4*T samples).  eq. (2) looks
//     forward in time, so in reverse time the partner P_k[n + 2^k] has always been computed
//     already; each level keeps a delay line instead of re-reading a (max_width - 1)-sample
//     halo per tile.  The halo is paid once per segment (warm-up chunks), not once per tile.
//   * Thread t owns, in each row, the 4 consecutive samples 4t..4t+3 (one float4).
//     Widths 2, 4, 8: in the thread's own registers from three float4 of raw samples (the
//     width-4 sums of the next float4 are recomputed rather than exchanged).
//     Levels 8 <= 2^k <= 2T: the partner belongs to another thread - exchanged through a
//     ping-pong shared-memory buffer with 128-bit accesses, one __syncthreads() each.
//     Levels 2^k >= 4T: the partner is the SAME thread's float4 1, 2, 4, ... rows later,
//     i.e. a register of this chunk or a delay register kept from the previous chunks.
//     The shared-memory data pipe is the binding unit (profiles/r01b_*), so T is as small
//     as the register file and the instruction cache allow (geometry table below).
//   * Delay lines deeper than one chunk are register FIFOs; the chunk loop is unrolled
//     over the FIFO depth so that the FIFO slot is a compile-time constant (no moves).
//   * Chunks are staged into shared memory by cp.async.bulk (TMA, 1-D) through a
//     3-deep mbarrier ring; results leave as 128-bit stores.
//   * SNR scale 2^(-k/2) is a compile-time constant (1/sigma is applied once per output
//     sample at the store); the width index rides in the 5 low mantissa bits of the SNR
//     being maximised (relative perturbation <= 2^-18, inside the 1e-4 tolerance), stored
//     inverted so that exact ties resolve to the smallest width; max is the 3-input FMNMX3.
//   * Row a8's threshold test is fused in: a chunk whose best SNR reaches the candidate
//     threshold sets one byte of the caller's activity map, so that the candidate kernel
//     only revisits those chunks (spd_candidates.cu).
//   * Row tails (valid-windows-only rule, reading A3) and warm-up chunks run in a
//     guarded variant of the same body; interior chunks run the unguarded one.
#include <cuda_runtime.h>
#include <stdint.h>

#include <algorithm>

#include "spd_tree_common.cuh"

namespace spd {
namespace {

// Keys of level k and the fold of a level pair: eq. (5)'s compile-time scale 2^(-k/2) (1 / sigma applied at
// the store), or - SW - a measured sigma per width: cx.ls[k] = 1 / sigma_{d, 2^k}.
template <int k, bool FAST, bool SW>
__device__ __forceinline__ float4 key_b(float4 p, int lim, const ChunkCtx& cx) {
    if constexpr (SW) {
        return keyx_rt<k, FAST>(p, lim, cx.tm, cx.ls[k]);
    } else {
        return keyx<k, FAST>(p, lim, cx.tm);
    }
}
template <int j, int K, bool FAST, bool SW>
__device__ __forceinline__ void fold_b(float4& best, float4 before, float4 now, int lim, const ChunkCtx& cx) {
    if constexpr (SW) {
        fold_rt<j, K, FAST>(best, before, now, lim, cx.tm, cx.ls);
    } else {
        fold<j, K, FAST>(best, before, now, lim, cx.tm);
    }
}

// Exchange levels k = 3 .. LT+1: P_{k+1}[n] = P_k[n] + P_k[n + 2^k], partner in another thread.
// hoff: halo slots used by the levels below (d4 slots each: the row-0 values that the next
// chunk's last row wraps into).
template <int T, int R, int K, bool FAST, bool SW, int k, int hoff>
__device__ __forceinline__ void exchange_levels(float4 (&P)[R], float4 (&best)[R], const int (&lim)[R],
                                                float4* __restrict__ pp, float4* __restrict__ hr,
                                                float4* __restrict__ hw, int& xsel, const ChunkCtx& cx) {
    using G = Geo<T, R, K>;
    if constexpr (k <= G::LT + 1 && k + 1 <= G::LAST) {
        constexpr int d4 = (1 << k) / 4;  // partner distance in float4
        static_assert(hoff + d4 <= T, "halo buffer overflow");
        const int tid = cx.tid;
        float4* const buf = pp + xsel * G::C4;
        xsel ^= 1;
#pragma unroll
        for (int r = 0; r < R; ++r) st_shared4(buf + tid + T * r, P[r]);
        if (tid < d4) hw[hoff + tid] = P[0];
        __syncthreads();
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const float4* src = buf + (tid + T * r + d4);
            if (r == R - 1 && tid + d4 >= T) src = hr + (hoff + tid + d4 - T);
            const float4 now = add4(P[r], *src);
            if (FAST || cx.do_out) fold_b<k + 1, K, FAST, SW>(best[r], P[r], now, lim[r], cx);
            P[r] = now;
        }
        exchange_levels<T, R, K, FAST, SW, k + 1, hoff + d4>(P, best, lim, pp, hr, hw, xsel, cx);
    }
}

// In-register levels j = 0 .. J-1: partner 2^j rows later in the same thread.  Delay
// registers of level j live at dl[2^j - 1 .. 2^(j+1) - 2].
template <int T, int R, int K, bool FAST, bool SW, int PH, int j>
__device__ __forceinline__ void register_levels(float4 (&P)[R], float4 (&best)[R], const int (&lim)[R],
                                                float4 (&dl)[Geo<T, R, K>::ND + 1], const ChunkCtx& cx) {
    using G = Geo<T, R, K>;
    if constexpr (j < G::J) {
        constexpr int D = 1 << j;   // partner distance in rows
        constexpr int off = D - 1;  // first delay register of this level
        constexpr int lvl = G::LT + 3 + j;
        float4 now[R];
        if constexpr (D < R) {
            // partner in this chunk, or among the first D rows of the previous chunk
#pragma unroll
            for (int r = 0; r < R; ++r) now[r] = add4(P[r], r + D < R ? P[r + D] : dl[off + r + D - R]);
#pragma unroll
            for (int i = 0; i < D; ++i) dl[off + i] = P[i];
        } else {
            // partner D / R chunks back: FIFO of Q chunks.  Unguarded steps use slot PH % Q
            // (the chunk loop is unrolled over the deepest FIFO); guarded steps keep the
            // FIFO in canonical order (slot 0 oldest) by moving registers.
            constexpr int Q = D / R;
            if constexpr (tree_tmem(K)) {
                // FIFO in tensor memory (K >= 15: the delay registers would otherwise cost 124 /
                // 252 registers per thread): slot = step mod depth as a run-time column offset,
                // one tcgen05.ld + tcgen05.st of R float4 per level.  Slots of the shallower FIFOs
                // come first: Q - 1 of them.
                static_assert(R == 8 || R == 4 || R == 2, "tensor-memory FIFOs move 2, 4 or 8 float4 per level");
                const uint32_t taddr = cx.tbase + 4u * R * static_cast<uint32_t>((Q - 1) + (cx.it & (Q - 1)));
                float4 old[R];
                if constexpr (R == 8) {
                    tmem_ld32(taddr, reinterpret_cast<float4(&)[8]>(old));
                    tmem_st32(taddr, reinterpret_cast<const float4(&)[8]>(P));
                } else if constexpr (R == 4) {
                    tmem_ld16(taddr, reinterpret_cast<float4(&)[4]>(old));
                    tmem_st16(taddr, reinterpret_cast<const float4(&)[4]>(P));
                } else {
                    tmem_ld8(taddr, reinterpret_cast<float4(&)[2]>(old));
                    tmem_st8(taddr, reinterpret_cast<const float4(&)[2]>(P));
                }
#pragma unroll
                for (int r = 0; r < R; ++r) now[r] = add4(P[r], old[r]);
            } else {
            constexpr bool kSlotted = FAST && G::U >= Q;  // slot known at compile time
            constexpr int slot = kSlotted ? (PH % Q) : 0;
#pragma unroll
            for (int r = 0; r < R; ++r) now[r] = add4(P[r], dl[off + slot * R + r]);
            if constexpr (kSlotted) {
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
        }
#pragma unroll
        for (int r = 0; r < R; ++r) {
            if (FAST || cx.do_out) fold_b<lvl, K, FAST, SW>(best[r], P[r], now[r], lim[r], cx);
            P[r] = now[r];
        }
        register_levels<T, R, K, FAST, SW, PH, j + 1>(P, best, lim, dl, cx);
    }
}

// One streaming step: the chunk staged at `st4` (C + 8 floats: the chunk and the first two
// float4 of the following chunk) -> Y, W for its C samples.  Returns the largest tagged,
// sigma-unscaled key of the chunk's samples owned by this thread (for the activity map).
template <int T, int R, int K, bool FAST, int PH, bool SW, bool U8>
__device__ __forceinline__ float tree_chunk(const float4* __restrict__ st4, float4* __restrict__ pp,
                                            float4* __restrict__ halo, int& xsel, int& hsel,
                                            float4 (&dl)[Geo<T, R, K>::ND + 1], const ChunkCtx& cx) {
    using G = Geo<T, R, K>;
    const int tid = cx.tid;
    const float mu = cx.mu;
    const uint32_t tm = cx.tm;

    float4 P[R], best[R];
    int lim[R];

    // ---- stage -> registers, remove the mean, levels 0..3 in the thread's own registers ----
#pragma unroll
    for (int r = 0; r < R; ++r) {
        if constexpr (FAST) {
            lim[r] = 1 << 30;
        } else {
            const long long left = cx.n_t - (cx.n0 + 4ll * (tid + T * r));
            lim[r] = left > (1ll << 30) ? (1 << 30) : (left < 0 ? 0 : static_cast<int>(left));
        }
        const float4 a = norm4(st4[tid + T * r], mu);
        if constexpr (K == 1) {
            P[r] = a;
            if (FAST || cx.do_out) best[r] = key_b<0, FAST, SW>(a, lim[r], cx);
        } else {
            const float4 b = norm4(st4[tid + T * r + 1], mu);
            const float s01 = a.x + a.y, s12 = a.y + a.z, s23 = a.z + a.w, s34 = a.w + b.x;
            const float4 p1 = make_float4(s01, s12, s23, s34);
            if constexpr (K == 2) {
                P[r] = p1;
                if (FAST || cx.do_out)
                    best[r] = max4(key_b<0, FAST, SW>(a, lim[r], cx), key_b<1, FAST, SW>(p1, lim[r], cx));
            } else {
                const float s45 = b.x + b.y, s56 = b.y + b.z;
                const float4 p2 = make_float4(s01 + s23, s12 + s34, s23 + s45, s34 + s56);
                if (FAST || cx.do_out)
                    best[r] = max4(key_b<0, FAST, SW>(a, lim[r], cx), key_b<1, FAST, SW>(p1, lim[r], cx),
                                   key_b<2, FAST, SW>(p2, lim[r], cx));
                if constexpr (K == 3) {
                    P[r] = p2;
                } else {
                    // Width 8 from a third float4 of raw samples: recomputing the width-4 sums of
                    // the next float4 here costs 8 adds and saves one whole shared-memory
                    // exchange (the L1/shared data pipe is the binding unit).
                    const float4 c = norm4(st4[tid + T * r + 2], mu);
                    const float s67 = b.z + b.w, s78 = b.w + c.x, s89 = c.x + c.y, s9a = c.y + c.z;
                    // packed adds of aligned pairs, same association as (s01 + s23) + (s45 + s67) ...
                    const float2 q2lo = __fadd2_rn(make_float2(s45, s56), make_float2(s67, s78));
                    const float2 q2hi = __fadd2_rn(make_float2(s67, s78), make_float2(s89, s9a));
                    const float2 p3lo = __fadd2_rn(make_float2(p2.x, p2.y), q2lo);
                    const float2 p3hi = __fadd2_rn(make_float2(p2.z, p2.w), q2hi);
                    const float4 p3 = make_float4(p3lo.x, p3lo.y, p3hi.x, p3hi.y);
                    if (FAST || cx.do_out) fold_b<3, K, FAST, SW>(best[r], p2, p3, lim[r], cx);
                    P[r] = p3;
                }
            }
        }
    }

    // ---- exchange levels: 8 <= 2^k <= 2T ----------------------------------------------
    float4* const hr = halo + hsel * T;        // written by the previous (later-in-time) chunk
    float4* const hw = halo + (hsel ^ 1) * T;  // read by the next chunk
    hsel ^= 1;
    exchange_levels<T, R, K, FAST, SW, 3, 0>(P, best, lim, pp, hr, hw, xsel, cx);

    // ---- in-register levels: partner 1, 2, 4, ... rows later (same thread) -------------
    register_levels<T, R, K, FAST, SW, PH, 0>(P, best, lim, dl, cx);

    // ---- unpack and store: Y = key (code bits cleared) / sigma, W = inverted code ---------------------------
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
                if constexpr (U8) {
                    // the four low bytes of the keys into one word (3 PRMT), inverted and masked at once
                    const uint32_t t = __byte_perm(__float_as_uint(kq.x), __float_as_uint(kq.y), 0x0040);
                    const uint32_t u = __byte_perm(__float_as_uint(kq.z), __float_as_uint(kq.w), 0x4000);
                    const uint32_t packed = ~__byte_perm(t, u, 0x7610) & 0x1f1f1f1fu;
                    *reinterpret_cast<uint32_t*>(reinterpret_cast<uint8_t*>(cx.out_width) + o) = packed;
                } else {
                    *reinterpret_cast<int4*>(cx.out_width + o) = w;
                }
            }
        }
    }
    if constexpr (tree_tmem(K)) tmem_wait_st();
    // With no exchange level there is no barrier inside the step: add the one that
    // orders this step's stage reads before the next refill of the stage.
    if constexpr (G::LAST < 4) __syncthreads();
    return top;
}

// Threads per block T, rows per chunk R and resident blocks per SM, per depth K (measured
// sweeps in DESIGN.md "Tuning log").  K <= 14: T = 128, R = 4, 3 blocks (165 registers, no
// spills): 11.5 ms on config 3.  T = 64 (one exchange level fewer) ties at 11.7 ms once its
// chunk loop is not unrolled past the instruction cache, T = 256 (one more) is at 13.4 ms.
// K = 15, 16 keep their delay FIFOs in tensor memory: 4 and 2 blocks of 128 threads per SM.
constexpr int tree_threads_for(int) { return 128; }
// K = 16: eight rows per chunk (4096 samples, 255 registers, two blocks per SM) - half the barriers per sample of
// four rows: config 4 in 7.23 ms against 7.35 ms
constexpr int tree_rows_for(int K) { return K == 16 ? 8 : 4; }
constexpr int tree_blocks_per_sm(int K) { return K <= 14 ? 3 : (K == 15 ? 4 : 2); }
// Tensor-memory columns a block allocates for its FIFOs (K >= 15): 4 R columns per FIFO slot,
// 2^JF - 1 slots, rounded up to a power of two.
template <int T, int R, int K>
constexpr int tree_tmem_cols() {
    using G = Geo<T, R, K>;
    constexpr int LR = ilog2(R);
    constexpr int JF = G::J > LR ? G::J - LR : 0;
    // warps w and w + 4 share a lane quarter: every set of 128 threads has its own columns
    constexpr int need = (T / 128) * 4 * R * ((1 << JF) - 1);
    return need <= 32 ? 32 : need <= 64 ? 64 : need <= 128 ? 128 : need <= 256 ? 256 : 512;
}

template <int T, int R, int K>
constexpr size_t tree_smem_bytes() {
    constexpr size_t C = 4 * T * R;
    return 2 * C * 4 + kStages * (C + 8) * 4 + 2 * T * 16 + kStages * 8 + 16;
}

template <int T, int R, int K, bool SW, bool U8>
__global__ void __launch_bounds__(T, tree_blocks_per_sm(K)) spd_tree_kernel(const TreeParams p) {
    using G = Geo<T, R, K>;
    constexpr int C = G::C;
    constexpr int M = 1 << (K - 1);
    constexpr int GUARD = M > 8 ? M : 8;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float4* const pp = reinterpret_cast<float4*>(smem_raw);
    float* const stages = reinterpret_cast<float*>(smem_raw + 2 * C * 4);
    float4* const halo = reinterpret_cast<float4*>(stages + kStages * (C + 8));
    uint64_t* const bars = reinterpret_cast<uint64_t*>(halo + 2 * T);
    uint32_t* const tslot = reinterpret_cast<uint32_t*>(bars + kStages);
    constexpr int kTmemCols = tree_tmem_cols<T, R, K>();

    const int tid = threadIdx.x;
    const int d = blockIdx.x / p.segs_per_row;
    const int s = blockIdx.x - d * p.segs_per_row;
    const int c_lo = s * p.seg_chunks;
    const int c_hi = min(c_lo + p.seg_chunks, p.chunks_per_row);
    if (c_lo >= c_hi) return;
    const int c_top = min(c_hi + p.warm_chunks, p.chunks_per_row);
    const long long n_t = p.n_t;
    // chunk c runs unguarded iff (c + 1) * C + GUARD <= n_t
    const int c_fast_end = n_t >= GUARD ? static_cast<int>((n_t - GUARD) / C) : 0;
    const int first_fast = max(c_lo, min(c_hi, c_fast_end));  // chunks [c_lo, first_fast) are fast

    const float* __restrict__ row = p.plane + static_cast<long long>(d) * n_t;
    ChunkCtx cx;
    cx.mu = p.mean[d];
    const float sg = SW ? 1.0f : p.sigma[d];
    cx.inv = 1.0f / sg;
    if constexpr (SW) {
        // keys are SNRs already: 1 / sigma_{d, 2^k} per level, nothing left for the store
        const float* __restrict__ swr = p.sigma_w + static_cast<long long>(d) * K;
#pragma unroll
        for (int k = 0; k < K; ++k) cx.ls[k] = 1.0f / __ldg(swr + k);
    }
    cx.tm = p.tag_mask;
    cx.out_snr = p.out_snr + static_cast<long long>(d) * n_t;
    // a uint8 plane advances by n_t bytes per row: n_t / 4 int32 (n_t % 4 == 0 on this path)
    cx.out_width = p.out_width + static_cast<long long>(d) * (U8 ? n_t / 4 : n_t);
    cx.n_t = n_t;
    cx.tid = tid;
    // Activity threshold on the sigma-unscaled key: Y = key / sigma >= thr  <=  key >= thr * sigma
    // lowered by a few ulp so that rounding can only add chunks to the map, never drop one.
    uint8_t* const act = p.activity ? p.activity + static_cast<long long>(d) * p.chunks_per_row : nullptr;
    float thr_key = __int_as_float(0x7f800000);
    if (act) {
        const float t = p.threshold * sg;
        thr_key = t - fabsf(t) * 2e-6f;
    }

    for (int i = tid; i < 2 * T; i += T) halo[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    if (tid == 0) {
#pragma unroll
        for (int i = 0; i < kStages; ++i) mbar_init(&bars[i], 1);
        fence_mbar_init();
    }
    float4 dl[G::ND + 1];
#pragma unroll
    for (int i = 0; i < G::ND + 1; ++i) dl[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    int xsel = 0, hsel = 0;
    cx.tbase = 0;
    cx.it = 0;
    if constexpr (tree_tmem(K)) {
        if (tid < 32) tmem_alloc<kTmemCols>(tslot);
        tmem_fence_before_sync();
        __syncthreads();
        tmem_fence_after_sync();
        constexpr int kSetCols = kTmemCols / (T / 128);  // columns of one set of 128 threads
        // this warp's lane quarter, and the columns of its set of 128 threads
        cx.tbase = *tslot + (static_cast<uint32_t>((tid >> 5) & 3) << 21) + static_cast<uint32_t>(tid >> 7) * kSetCols;
        const float4 zero[2] = {make_float4(0.f, 0.f, 0.f, 0.f), make_float4(0.f, 0.f, 0.f, 0.f)};
#pragma unroll
        for (int col = 0; col < kSetCols; col += 8) tmem_st8(cx.tbase + col, zero);
        tmem_wait_st();
    } else {
        __syncthreads();
    }

    // ---- guarded steps: warm-up chunks of an interior segment, then the row tail -----
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
        const float top = tree_chunk<T, R, K, false, 0, SW, U8>(reinterpret_cast<const float4*>(stages), pp, halo,
                                                                xsel, hsel, dl, cx);
        if (act && cx.do_out && top >= thr_key) act[c] = 1;
        ++cx.it;
        __syncthreads();
    }

    // ---- unguarded steps: bulk-copy ring ----------------------------------------------
    const int n_fast = first_fast - c_lo;
    if (n_fast > 0) {
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
        // tensor-memory FIFOs take their slot at run time: two steps per trip only to overlap them
        static_phases<0, (tree_tmem(K) ? (R >= 8 ? 1 : 2) : G::U)>([&](auto ph) {
            if (it < n_fast) {
                if (tid == 0) {
                    const int nx = it + kStages - 1;
                    if (nx < n_fast) {
                        const int sx = stage == 0 ? kStages - 1 : stage - 1;  // (it + kStages - 1) % kStages
                        mbar_arrive_expect_tx(&bars[sx], kBytes);
                        bulk_g2s(stages + sx * (C + 8), row + static_cast<long long>(first_fast - 1 - nx) * C,
                                 kBytes, &bars[sx]);
                    }
                }
                mbar_wait(&bars[stage], phase);
                const int c = first_fast - 1 - it;
                cx.n0 = static_cast<long long>(c) * C;
                const float top = tree_chunk<T, R, K, true, decltype(ph)::value, SW, U8>(
                    reinterpret_cast<const float4*>(stages + stage * (C + 8)), pp, halo, xsel, hsel, dl, cx);
                if (act && top >= thr_key) act[c] = 1;
                if (++stage == kStages) {
                    stage = 0;
                    phase ^= 1;
                }
                ++it;
                ++cx.it;
            }
        });
    }
    }
    if constexpr (tree_tmem(K)) {
        tmem_fence_before_sync();
        __syncthreads();
        if (tid < 32) tmem_dealloc<kTmemCols>(*tslot);
    }
}

// Variants: 0 = eq. (5) scale, int32 index; 1 = measured sigma per width (spd_run_sigma_w); 2 = uint8 index
// (SPD_FLAG_WIDTH_U8).  1 and 2 are instantiated where this kernel is the plan's default (K <= 8, K >= 15).
constexpr bool tree_has_variants(int K) { return K <= 8 || K >= 15; }

template <int T, int R, int K>
cudaError_t launch_tree(const TreeConfig& cfg, const TreeParams& prm, int64_t n_dm, int variant, cudaStream_t stream) {
    const dim3 grid(static_cast<unsigned>(n_dm * cfg.segs_per_row));
    if (variant == 0) {
        spd_tree_kernel<T, R, K, false, false><<<grid, T, cfg.smem_bytes, stream>>>(prm);
    } else if constexpr (tree_has_variants(K)) {
        if (variant == 1)
            spd_tree_kernel<T, R, K, true, false><<<grid, T, cfg.smem_bytes, stream>>>(prm);
        else
            spd_tree_kernel<T, R, K, false, true><<<grid, T, cfg.smem_bytes, stream>>>(prm);
    } else {
        return cudaErrorNotSupported;
    }
    return cudaGetLastError();
}

template <typename Kern>
cudaError_t prepare_kernel(Kern kern, int T, size_t smem, int* nb) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem));
    if (e != cudaSuccess) return e;
    return cudaOccupancyMaxActiveBlocksPerMultiprocessor(nb, kern, T, smem);
}

template <int T, int R, int K>
cudaError_t prepare_tree(TreeConfig& cfg) {
    cfg.smem_bytes = tree_smem_bytes<T, R, K>();
    int nb = 0;
    cudaError_t e = prepare_kernel(spd_tree_kernel<T, R, K, false, false>, T, cfg.smem_bytes, &nb);
    if (e != cudaSuccess) return e;
    if constexpr (tree_tmem(K)) {
        // no more resident blocks than tensor memory has columns for (a block that cannot
        // allocate would spin): pad the shared-memory request until the occupancy fits
        const int max_blocks = 512 / tree_tmem_cols<T, R, K>();
        while (nb > max_blocks && cfg.smem_bytes < (200u << 10)) {
            cfg.smem_bytes += 4096;
            e = prepare_kernel(spd_tree_kernel<T, R, K, false, false>, T, cfg.smem_bytes, &nb);
            if (e != cudaSuccess) return e;
        }
    }
    if constexpr (tree_has_variants(K)) {
        // the variants use a few more registers: never more resident blocks than the plain kernel
        int nv = 0;
        if ((e = prepare_kernel(spd_tree_kernel<T, R, K, true, false>, T, cfg.smem_bytes, &nv)) != cudaSuccess) return e;
        if ((e = prepare_kernel(spd_tree_kernel<T, R, K, false, true>, T, cfg.smem_bytes, &nv)) != cudaSuccess) return e;
    }
    cfg.blocks_per_sm = nb;
    return cudaSuccess;
}

#define SPD_TREE_CASES(OP) \
    OP(1)                  \
    OP(2)                  \
    OP(3)                  \
    OP(4)                  \
    OP(5)                  \
    OP(6)                  \
    OP(7)                  \
    OP(8)                  \
    OP(9)                  \
    OP(10)                 \
    OP(11)                 \
    OP(12)                 \
    OP(13)                 \
    OP(14)                 \
    OP(15)                 \
    OP(16)

}  // namespace

bool tree_applicable(const std::vector<int32_t>& widths, int64_t n_t) {
    const int K = static_cast<int>(widths.size());
    if (K < 1 || K > kTreeMaxLevels) return false;
    for (int k = 0; k < K; ++k)
        if (widths[k] != (1 << k)) return false;
    if (n_t % 4 != 0) return false;  // 16-byte row alignment for the bulk copies
    return true;
}

int tree_configure(spd_plan* plan) {
    TreeConfig& cfg = plan->tree;
    cfg.K = static_cast<int>(plan->widths.size());
    if (ws_applicable(cfg.K, plan->flags)) return ws_configure(plan);
    cfg.kind = 0;
    cfg.T = tree_threads_for(cfg.K);
    cfg.chunk = 4 * cfg.T * tree_rows_for(cfg.K);
    cudaError_t e = cudaErrorInvalidValue;
#define SPD_PREP(KK) \
    if (cfg.K == KK) e = prepare_tree<tree_threads_for(KK), tree_rows_for(KK), KK>(cfg);
    SPD_TREE_CASES(SPD_PREP)
#undef SPD_PREP
    if (e != cudaSuccess) return cuda_fail(e, "configuring the dyadic-tree kernel");
    if (cfg.blocks_per_sm < 1) {
        set_error("dyadic-tree kernel does not fit on this device (K=%d, smem=%zu)", cfg.K, cfg.smem_bytes);
        return SPD_ERR_CUDA;
    }
    return tree_configure_segments(plan);
}

// Chunks, look-ahead and segments per row from cfg.K, cfg.chunk and cfg.blocks_per_sm
// (shared with the IGRID tree, spd_tree_ig.cu).
int tree_configure_segments(spd_plan* plan) {
    TreeConfig& cfg = plan->tree;
    const int64_t C = cfg.chunk;
    const int64_t M = int64_t(1) << (cfg.K - 1);
    cfg.chunks_per_row = static_cast<int>((plan->n_t + C - 1) / C);
    cfg.warm_chunks = cfg.K >= 2 ? static_cast<int>((M - 1 + C - 1) / C) : 0;
    // Segments: enough independent streams to fill and balance the machine, each long
    // enough that replaying its look-ahead (warm_chunks) stays a few per cent.
    const int64_t slots = int64_t(plan->sm_count) * cfg.blocks_per_sm;
    int64_t segs = 1;
    const int64_t min_seg_chunks = std::max<int64_t>(16 * cfg.warm_chunks, 8);
    if (plan->segs_option > 0) {  // SPD_OPT_SEGMENTS_PER_ROW
        segs = plan->segs_option;
    } else {
        while (plan->n_dm * segs < 8 * slots && (cfg.chunks_per_row + 2 * segs - 1) / (2 * segs) >= min_seg_chunks)
            segs *= 2;
    }
    segs = std::min<int64_t>(segs, cfg.chunks_per_row);
    cfg.seg_chunks = static_cast<int>((cfg.chunks_per_row + segs - 1) / segs);
    cfg.segs_per_row = static_cast<int>((cfg.chunks_per_row + cfg.seg_chunks - 1) / cfg.seg_chunks);
    if (plan->n_dm * cfg.segs_per_row > 0x7fffffffll) {
        set_error("grid too large");
        return SPD_ERR_INVALID_ARG;
    }
    return SPD_OK;
}

int tree_run(const spd_plan* plan, int64_t n_dm, const float* plane, const float* mean, const float* sigma,
             float* out_snr, void* out_width, float threshold, uint8_t* activity, cudaStream_t stream,
             const float* sigma_w) {
    const TreeConfig& cfg = plan->tree;
    if (cfg.kind == 1)
        return ws_run(plan, n_dm, plane, mean, sigma, out_snr, out_width, threshold, activity, stream, sigma_w);
    const int variant = sigma_w ? 1 : (plan->width_bytes == 1 ? 2 : 0);
    if (variant != 0 && !tree_has_variants(cfg.K)) {
        set_error("the block-per-stream kernel forced by SPD_FLAG_BLOCK_TREE has no sigma-per-width / uint8 variant "
                  "for %d widths", cfg.K);
        return SPD_ERR_INVALID_ARG;
    }
    TreeParams prm;
    prm.plane = plane;
    prm.mean = mean;
    prm.sigma = sigma;
    prm.sigma_w = sigma_w;
    for (int k = 0; k < 16; ++k) prm.gmask[k] = 0u;
    prm.out_snr = out_snr;
    prm.out_width = static_cast<int32_t*>(out_width);
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
        // the map is padded to a multiple of 128 bytes; the padding is cleared too
        const size_t bytes = (static_cast<size_t>(n_dm) * cfg.chunks_per_row + 127) / 128 * 128;
        e = cudaMemsetAsync(activity, 0, bytes, stream);
        if (e != cudaSuccess) return cuda_fail(e, "clearing the activity map");
    }
    e = cudaErrorInvalidValue;
#define SPD_LAUNCH(KK) \
    if (cfg.K == KK) e = launch_tree<tree_threads_for(KK), tree_rows_for(KK), KK>(cfg, prm, n_dm, variant, stream);
    SPD_TREE_CASES(SPD_LAUNCH)
#undef SPD_LAUNCH
    if (e != cudaSuccess) return cuda_fail(e, "launching the dyadic-tree kernel");
    return SPD_OK;
}

}  // namespace spd
