// Dyadic partial-sum tree, one WARP per stream, for
// 9 <= K <= 14 widths {1, 2, ..., 2^(K-1)}.
//
// Same arithmetic as spd_tree.cu (eq. 2, 4, 5, 12 and the reuse of eq. 15/16:
// P_{k+1}[n] = P_k[n] + P_k[n + 2^k]), different
// decomposition.  In spd_tree.cu a block of 4 warps shares one stream, so every level whose
// partner lies in another thread costs a block barrier.  Here every warp streams its own piece
// of the plane in reverse time and nothing is shared between warps: no block barrier at all.
//
//   * A step is R = 4 "rows" of 128 samples; lane l owns the float4 4l..4l+3 of every row.
//   * Widths 2, 4, 8: in the lane's registers from three raw float4 (as spd_tree.cu).
//   * Partner 8, 16, 32, 64 samples later = 2, 4, 8, 16 lanes later ("lane levels"): through a
//     warp-private shared-memory buffer ordered by __syncwarp (one 128-bit store and load per
//     float4; shuffles would take eight instructions, and the issue slots are what binds).
//     A lane that runs off its row continues in the next row, which is adjacent in the buffer;
//     the last row continues in the first row of the previous step (4 float4 kept, stored
//     behind the rows).
//   * Partner 128 * 2^j samples later = the same lane, 2^j rows later ("row levels"): a
//     register of this step or of the previous step (7 float4 kept), or - 2, 4, 8 steps back -
//     a FIFO.
//   * The FIFOs (14 x 4 float4 per lane for K = 14: the 28 KB of delay state that forces
//     spd_tree.cu to spread a stream over 128 threads) live in TENSOR MEMORY: each warp owns
//     32 lanes x 224 columns, written with tcgen05.st and read with tcgen05.ld (32x32b.x16:
//     one instruction moves the 4 float4 of a level), slot = step mod depth as a run-time
//     column offset - no unrolling over FIFO phases, no register rotation.  TMEM is used as
//     plain per-lane scratch; there is no MMA anywhere (streaming reduction, not a contraction).
//   * Raw samples arrive by 1-D cp.async.bulk through a 4-stage mbarrier ring PER WARP.
//   * SNR scale, width tag, 3-input max, threshold flag, guarded tail steps: as spd_tree.cu;
//     look-ahead steps of a piece that starts inside a row compute the sums only.
//   * Work split: the steps of the plane, in row-major order, are cut into one piece per
//     resident warp (148 SMs x 8), so all warps finish together and a piece replays look-ahead
//     once (for the one row part that stops short of its row's end).
//
// One block of 8 warps per SM (2 warps per lane quarter of TMEM, 2 x 224 <= 512 columns).
// Measured on config 3: 10.7 ms against 11.4 ms of spd_tree.cu.
#include <cuda_runtime.h>
#include <stdint.h>

#include <algorithm>

#pragma once
#include "spd_tree_common.cuh"

namespace spd {
namespace {

constexpr int kWsWarps = 8;                 // streams per block
constexpr int kWsRows = 4;                  // rows of 128 samples per step (8: 32 KB loop body, slower - DESIGN.md 10b)
constexpr int kWsStep = 128 * kWsRows;      // samples per step
constexpr int kWsStage = kWsStep + 8;       // floats per stage: the step + two float4 of look-ahead
constexpr int kWsMinK = 9, kWsMaxK = 14;  // K = 8: the block kernel is 2 % faster (measured)
// Activity map: one byte per kWsActSteps steps (2048 samples, the block kernel's granularity:
// finer flags only lengthen the candidate kernel's scan of the map).
constexpr int kWsActSteps = 2048 / kWsStep;
constexpr int kWsStages = 4;                // bulk-copy ring depth per warp (3 and 6 measure the same)
constexpr int kWsUnroll = 2;                // steps per trip of the main loop (3: past the instruction cache)

template <int K>
struct WsGeo {
    static constexpr int LAST = K - 1;
    // row levels j = 0 .. J-1: partner 2^j rows later, level 7+j -> level 8+j
    static constexpr int J = imax(0, LAST - 7);
    // partner 1, 2 or 4 rows later: inside this step or the previous one (R = 4: 4 rows = one step back): registers
    static constexpr int JNMAX = 3;
    static constexpr int JN = J < JNMAX ? J : JNMAX;
    static constexpr int NEAR = (1 << JN) - 1;  // float4 kept from the previous step
    static constexpr int JF = J - JN;           // FIFO levels i < JF: partner Q0 * 2^i steps back
    static constexpr int Q0 = (1 << JNMAX) / kWsRows;  // steps back of the first FIFO level
    static constexpr int COLS = 4 * kWsRows * Q0 * ((1 << JF) - 1);  // TMEM columns per warp
};

// One level's rows of a step (kWsRows float4 per lane) <-> 4 * kWsRows columns.
__device__ __forceinline__ void tmem_ld_rows(uint32_t taddr, float4 (&v)[kWsRows]) { tmem_ld16(taddr, v); }
__device__ __forceinline__ void tmem_st_rows(uint32_t taddr, const float4 (&v)[kWsRows]) { tmem_st16(taddr, v); }


// Lane levels k = 3 .. 6: P_{k+1}[n] = P_k[n] + P_k[n + 2^k], partner 2^k / 4 lanes later; the
// lanes that run off a row continue in the next row, the last row in the first row of the
// previous (later-in-time) step, kept in hs[k - 3].
// The exchange goes through a warp-private shared-memory buffer (one 128-bit store and load per
// float4 and level, ordered by __syncwarp: two instructions where shuffles take eight - measured
// 11.37 against 11.86 ms; the L1 data pipe has the room, the issue slots do not).  Two buffers
// alternate between levels.
constexpr int kWsXBuf = (kWsRows + 1) * 32;  // float4 per exchange buffer: R rows + the kept row

// Keys of level k: eq. (5)'s compile-time scale 2^(-k/2) (1 / sigma applied at the store), or a measured
// sigma per width (SW).
template <int k, bool FAST, bool SW>
__device__ __forceinline__ float4 key_sw(float4 p, int lim, const ChunkCtx& cx) {
    if constexpr (SW) {
        return keyx_rt<k, FAST>(p, lim, cx.tm, cx.ls[k]);
    } else {
        return keyx<k, FAST>(p, lim, cx.tm);
    }
}
// Grid plans (row f2, reading A16): level k counts only at samples that are multiples of its separation
// gmask[k] + 1 (a power of two).  nb = index of the float4's first sample (a multiple of 4), so of the
// four samples x is on the grid iff nb & gmask == 0, z iff the separation is 1 or 2, y and w iff it is 1.
template <int k>
__device__ __forceinline__ float4 grid_mask(float4 q, uint32_t nb, const ChunkCtx& cx) {
    const uint32_t m = cx.gmask[k];
    const float ninf = __int_as_float(0xff800000);
    if ((nb & m) != 0u) q.x = ninf;
    if (m != 0u) {
        q.y = ninf;
        q.w = ninf;
    }
    if (m > 1u) q.z = ninf;
    return q;
}
// One level of a grid plan folded into best.  A level whose separation is 4 or more has at most the FIRST
// sample of a float4 on its grid: only that key is formed - one multiply, one tag, one select, one max instead
// of the eight instructions of a full float4 - which is where the paper's grids save their work (PAPER.md:201,
// 311: "wider pulses ... at every D^(i) point").  Separations do not decrease with the width, so these are the
// levels k >= KX for some KX, a template parameter of the kernel (the host picks the smallest instantiated
// value that is not below the plan's); the levels below take the full float4 with the off-grid elements masked,
// which is right for any separation.
constexpr int kWsNoGrid = 99;
template <int k, int KX, bool FAST, bool SW>
__device__ __forceinline__ void grid_level(float4& best, float4 p, int lim, uint32_t nb, const ChunkCtx& cx) {
    const uint32_t m = cx.gmask[k];
    if constexpr (k >= KX) {
        float v = SW ? p.x * cx.ls[k] : p.x * level_scale<k>();
        v = pack1<k>(v, cx.tm);
        const float ninf = __int_as_float(0xff800000);
        bool off = (nb & m) != 0u;
        if constexpr (!FAST) off = off || (1 << k) > lim;
        best.x = fmaxf(best.x, off ? ninf : v);
    } else {
        best = max4(best, grid_mask<k>(key_sw<k, FAST, SW>(p, lim, cx), nb, cx));
    }
}

template <int j, int K, bool FAST, bool SW, int KX>
__device__ __forceinline__ void fold_sw(float4& best, float4 before, float4 now, int lim, uint32_t nb,
                                        const ChunkCtx& cx) {
    constexpr bool GR = KX != kWsNoGrid;
    if constexpr (j >= 3) {
        if constexpr (GR) {
            if constexpr ((j & 1) == 0) {
                grid_level<j - 1, KX, FAST, SW>(best, before, lim, nb, cx);
                grid_level<j, KX, FAST, SW>(best, now, lim, nb, cx);
            } else if constexpr (j == K - 1) {
                grid_level<j, KX, FAST, SW>(best, now, lim, nb, cx);
            }
        } else if constexpr ((j & 1) == 0) {
            best = max4(best, key_sw<j - 1, FAST, SW>(before, lim, cx), key_sw<j, FAST, SW>(now, lim, cx));
        } else if constexpr (j == K - 1) {
            best = max4(best, key_sw<j, FAST, SW>(now, lim, cx));
        }
    }
}

// Step modes: 0 = guarded (row tail: windows checked against the end of the row, output if
// cx.do_out), 1 = interior step with output, 2 = interior look-ahead step (sums only).
template <int MODE>
__device__ __forceinline__ bool wants_out(const ChunkCtx& cx) {
    if constexpr (MODE == 1) {
        return true;
    } else if constexpr (MODE == 2) {
        return false;
    } else {
        return cx.do_out;
    }
}

template <int K, int MODE, bool SW, int KX, int k>
__device__ __forceinline__ void lane_levels(float4 (&P)[kWsRows], float4 (&best)[kWsRows],
                                            const int (&lim)[kWsRows], const uint32_t (&nb)[kWsRows], float4 (&hs)[4],
                                            float4* __restrict__ xb,
                                            int lane, const ChunkCtx& cx) {
    constexpr int R = kWsRows;
    if constexpr (k <= 6 && k + 1 <= WsGeo<K>::LAST) {
        constexpr int d4 = (1 << k) / 4;
        float4 partner[R];
        float4* const buf = xb + (k & 1) * kWsXBuf + lane;
#pragma unroll
        for (int r = 0; r < R; ++r) st_shared4(buf + 32 * r, P[r]);
        st_shared4(buf + 32 * R, hs[k - 3]);
        __syncwarp();
#pragma unroll
        for (int r = 0; r < R; ++r) partner[r] = buf[32 * r + d4];
        hs[k - 3] = P[0];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const float4 now = add4(P[r], partner[r]);
            if (wants_out<MODE>(cx)) fold_sw<k + 1, K, (MODE != 0), SW, KX>(best[r], P[r], now, lim[r], nb[r], cx);
            P[r] = now;
        }
        lane_levels<K, MODE, SW, KX, k + 1>(P, best, lim, nb, hs, xb, lane, cx);
    }
}

// Row levels j < JN: partner 2^j rows later, in this step or among the first rows of the
// previous step (nr[2^j - 1 .. 2^(j+1) - 2]).
template <int K, int MODE, bool SW, int KX, int j>
__device__ __forceinline__ void near_levels(float4 (&P)[kWsRows], float4 (&best)[kWsRows],
                                            const int (&lim)[kWsRows], const uint32_t (&nb)[kWsRows],
                                            float4 (&nr)[WsGeo<K>::NEAR + 1], const ChunkCtx& cx) {
    constexpr int R = kWsRows;
    if constexpr (j < WsGeo<K>::JN) {
        constexpr int D = 1 << j;
        constexpr int off = D - 1;
        constexpr int lvl = 8 + j;  // level produced
        float4 now[R];
#pragma unroll
        for (int r = 0; r < R; ++r) now[r] = add4(P[r], r + D < R ? P[r + D] : nr[off + r + D - R]);
#pragma unroll
        for (int i = 0; i < D; ++i) nr[off + i] = P[i];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            if (wants_out<MODE>(cx)) fold_sw<lvl, K, (MODE != 0), SW, KX>(best[r], P[r], now[r], lim[r], nb[r], cx);
            P[r] = now[r];
        }
        near_levels<K, MODE, SW, KX, j + 1>(P, best, lim, nb, nr, cx);
    }
}

// FIFO levels i < JF: partner 2^i steps back, same lane, same row: tensor memory.
template <int K, int MODE, bool SW, int KX, int i>
__device__ __forceinline__ void fifo_levels(float4 (&P)[kWsRows], float4 (&best)[kWsRows],
                                            const int (&lim)[kWsRows], const uint32_t (&nb)[kWsRows], uint32_t tbase,
                                            int it, const ChunkCtx& cx) {
    constexpr int R = kWsRows;
    if constexpr (i < WsGeo<K>::JF) {
        constexpr int Q = WsGeo<K>::Q0 << i;     // FIFO depth in steps
        constexpr int lvl = 8 + WsGeo<K>::JN + i;  // level produced
        constexpr int first = WsGeo<K>::Q0 * ((1 << i) - 1);  // slots of the levels below
        const uint32_t taddr = tbase + 4u * R * static_cast<uint32_t>(first + (it & (Q - 1)));
        float4 old[R];
        tmem_ld_rows(taddr, old);
        tmem_st_rows(taddr, P);
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const float4 now = add4(P[r], old[r]);
            if (wants_out<MODE>(cx)) fold_sw<lvl, K, (MODE != 0), SW, KX>(best[r], P[r], now, lim[r], nb[r], cx);
            P[r] = now;
        }
        fifo_levels<K, MODE, SW, KX, i + 1>(P, best, lim, nb, tbase, it, cx);
    }
}

template <int MODE, bool GR, bool U8>
__device__ __forceinline__ float ws_store(const float4 (&best)[kWsRows], const int (&lim)[kWsRows], int lane,
                                          const ChunkCtx& cx);

// One step of one warp: the kWsStage floats at st4 -> Y, W of its kWsStep samples.
template <int K, int MODE, bool SW, int KX, bool U8>
__device__ __forceinline__ float ws_step(const float4* __restrict__ st4, float4 (&hs)[4],
                                         float4 (&nr)[WsGeo<K>::NEAR + 1], float4* __restrict__ xb, uint32_t tbase,
                                         int it, int lane, const ChunkCtx& cx) {
    constexpr int R = kWsRows;
    constexpr bool GR = KX != kWsNoGrid;
    const float mu = cx.mu;
    float4 P[R], best[R];
    int lim[R];
    uint32_t nb[R];  // index of each float4's first sample (low 32 bits; grid plans only)
#pragma unroll
    for (int r = 0; r < R; ++r) {
        nb[r] = static_cast<uint32_t>(cx.n0) + 4u * static_cast<uint32_t>(lane + 32 * r);
        if constexpr (MODE != 0) {
            lim[r] = 1 << 30;
        } else {
            const long long left = cx.n_t - (cx.n0 + 4ll * (lane + 32 * r));
            lim[r] = left > (1ll << 30) ? (1 << 30) : (left < 0 ? 0 : static_cast<int>(left));
        }
        // widths 1, 2, 4, 8 from three raw float4 (eq. 2 on mean-removed samples)
        const float4 a = norm4(st4[lane + 32 * r], mu);
        const float4 b = norm4(st4[lane + 32 * r + 1], mu);
        const float4 c = norm4(st4[lane + 32 * r + 2], mu);
        const float s01 = a.x + a.y, s12 = a.y + a.z, s23 = a.z + a.w, s34 = a.w + b.x;
        const float s45 = b.x + b.y, s56 = b.y + b.z, s67 = b.z + b.w, s78 = b.w + c.x;
        const float s89 = c.x + c.y, s9a = c.y + c.z;
        const float4 p1 = make_float4(s01, s12, s23, s34);
        // widths 4 and 8 as packed adds of aligned pairs of the width-2 sums: the same additions in
        // the same association as (s01 + s23) + (s45 + s67) ..., 6 FADD2 for 12 FADD
        const float2 u01 = make_float2(s01, s12), u23 = make_float2(s23, s34), u45 = make_float2(s45, s56),
                     u67 = make_float2(s67, s78), u89 = make_float2(s89, s9a);
        const float2 p2lo = __fadd2_rn(u01, u23), p2hi = __fadd2_rn(u23, u45);
        const float2 q2lo = __fadd2_rn(u45, u67), q2hi = __fadd2_rn(u67, u89);
        const float2 p3lo = __fadd2_rn(p2lo, q2lo), p3hi = __fadd2_rn(p2hi, q2hi);
        const float4 p2 = make_float4(p2lo.x, p2lo.y, p2hi.x, p2hi.y);
        const float4 p3 = make_float4(p3lo.x, p3lo.y, p3hi.x, p3hi.y);
        if (wants_out<MODE>(cx)) {
            constexpr bool F = MODE != 0;
            if constexpr (GR) {
                best[r] = grid_mask<0>(key_sw<0, F, SW>(a, lim[r], cx), nb[r], cx);
                grid_level<1, KX, F, SW>(best[r], p1, lim[r], nb[r], cx);
                grid_level<2, KX, F, SW>(best[r], p2, lim[r], nb[r], cx);
            } else {
                best[r] = max4(key_sw<0, F, SW>(a, lim[r], cx), key_sw<1, F, SW>(p1, lim[r], cx),
                               key_sw<2, F, SW>(p2, lim[r], cx));
            }
            fold_sw<3, K, F, SW, KX>(best[r], p2, p3, lim[r], nb[r], cx);
        }
        P[r] = p3;
    }
    lane_levels<K, MODE, SW, KX, 3>(P, best, lim, nb, hs, xb, lane, cx);
    near_levels<K, MODE, SW, KX, 0>(P, best, lim, nb, nr, cx);
    fifo_levels<K, MODE, SW, KX, 0>(P, best, lim, nb, tbase, it, cx);
    if constexpr (WsGeo<K>::JF > 0) tmem_wait_st();

    return ws_store<MODE, GR, U8>(best, lim, lane, cx);
}

// ------------------------------------------------------------------------------------------------------------
// IGRID depth-1 width set (eq. 18 / Table 1): widths 2^k (k <= LAST) and 3 * 2^m (m <= LAST - 2),
// every extra width from two partial sums of the same tree: X_{3 * 2^m}[n] = P_m[n] +
// P_{m+1}[n + 2^m].  P_{m+1} half a partner distance away is read from where the tree keeps it anyway: the
// exchange buffer level m+1 has just filled (lane levels; one more exchange for P_7), this step's rows or the
// rows the next level keeps (row levels), the next level's FIFO in tensor memory at half its depth.
// Width indices in the ascending set 1, 2, 3, 4, 6, 8, 12, 16, 24, ...
// ------------------------------------------------------------------------------------------------------------
constexpr int idx_pow2(int k) { return k == 0 ? 0 : 2 * k - 1; }
constexpr int idx_ig(int m) { return 2 * m + 2; }
template <int m>
__device__ __forceinline__ constexpr float ig_scale() {  // 1 / sqrt(3 * 2^m)
    return level_scale<m>() * 0.57735026918962576451f;
}

// Key of one width (index IDX, WIDTH samples, on the grid of level LVL) over a float4.
template <int IDX, int WIDTH, bool FAST, bool SW>
__device__ __forceinline__ float4 ig_key(float4 p, float scale, int lim, const ChunkCtx& cx) {
    const float4 v = (IDX == 0 && !SW) ? p : scale4(p, SW ? cx.ls[IDX] : scale);  // width 1: scale 1
    float4 q = make_float4(pack1<IDX>(v.x, cx.tm), pack1<IDX>(v.y, cx.tm), pack1<IDX>(v.z, cx.tm), pack1<IDX>(v.w, cx.tm));
    if constexpr (!FAST) {
        const float ninf = __int_as_float(0xff800000);
        if (WIDTH > lim) q.x = ninf;
        if (WIDTH > lim - 1) q.y = ninf;
        if (WIDTH > lim - 2) q.z = ninf;
        if (WIDTH > lim - 3) q.w = ninf;
    }
    return q;
}
__device__ __forceinline__ float4 mask_to_grid(float4 q, uint32_t nb, uint32_t m) {
    const float ninf = __int_as_float(0xff800000);
    if ((nb & m) != 0u) q.x = ninf;
    if (m != 0u) {
        q.y = ninf;
        q.w = ninf;
    }
    if (m > 1u) q.z = ninf;
    return q;
}
// One width of a grid plan folded into best (see grid_level): LVL is the level whose separation applies.
template <int IDX, int WIDTH, int LVL, int KX, bool FAST, bool SW>
__device__ __forceinline__ void ig_grid_fold(float4& best, float4 p, float scale, int lim, uint32_t nb,
                                             const ChunkCtx& cx) {
    const uint32_t m = cx.gmask[LVL];
    if constexpr (LVL >= KX) {
        float v = p.x * (SW ? cx.ls[IDX] : scale);
        v = pack1<IDX>(v, cx.tm);
        const float ninf = __int_as_float(0xff800000);
        bool off = (nb & m) != 0u;
        if constexpr (!FAST) off = off || WIDTH > lim;
        best.x = fmaxf(best.x, off ? ninf : v);
    } else {
        best = max4(best, mask_to_grid(ig_key<IDX, WIDTH, FAST, SW>(p, scale, lim, cx), nb, m));
    }
}
// Width 2^k (sum pk) and width 3 * 2^m (sum gm; m < 0: none) folded into best.
template <int k, int m, int KX, bool FAST, bool SW>
__device__ __forceinline__ void ig_fold(float4& best, float4 pk, float4 gm, int lim, uint32_t nb, const ChunkCtx& cx) {
    constexpr bool GR = KX != kWsNoGrid;
    if constexpr (GR) {
        ig_grid_fold<idx_pow2(k), (1 << k), k, KX, FAST, SW>(best, pk, level_scale<k>(), lim, nb, cx);
        if constexpr (m >= 0)  // the widths of an octave share its separation: level m + 1
            ig_grid_fold<idx_ig(m), 3 * (1 << m), m + 1, KX, FAST, SW>(best, gm, ig_scale<m>(), lim, nb, cx);
    } else if constexpr (m >= 0) {
        best = max4(best, ig_key<idx_pow2(k), (1 << k), FAST, SW>(pk, level_scale<k>(), lim, cx),
                    ig_key<idx_ig(m), 3 * (1 << m), FAST, SW>(gm, ig_scale<m>(), lim, cx));
    } else {
        best = max4(best, ig_key<idx_pow2(k), (1 << k), FAST, SW>(pk, level_scale<k>(), lim, cx));
    }
}

// Width 3 * 2^m alone.
template <int m, int KX, bool FAST, bool SW>
__device__ __forceinline__ void ig_fold_one(float4& best, float4 gm, int lim, uint32_t nb, const ChunkCtx& cx) {
    if constexpr (KX != kWsNoGrid) {
        ig_grid_fold<idx_ig(m), 3 * (1 << m), m + 1, KX, FAST, SW>(best, gm, ig_scale<m>(), lim, nb, cx);
    } else {
        best = max4(best, ig_key<idx_ig(m), 3 * (1 << m), FAST, SW>(gm, ig_scale<m>(), lim, cx));
    }
}

// Lane levels k = 3 .. 6 with the extra width 3 * 2^(k-1) = P_{k-1}[n] + P_k[n + 2^(k-1)], and - k = 7 - the one
// more exchange of P_7 for width 192 = P_6[n] + P_7[n + 64].
template <int K, int MODE, bool SW, int KX, int k>
__device__ __forceinline__ void ig_lane_levels(float4 (&P)[kWsRows], float4 (&Pprev)[kWsRows], float4 (&best)[kWsRows],
                                               const int (&lim)[kWsRows], const uint32_t (&nb)[kWsRows], float4 (&hs)[5],
                                               float4* __restrict__ xb, int lane, const ChunkCtx& cx) {
    constexpr int R = kWsRows;
    constexpr int LAST = WsGeo<K>::LAST;
    if constexpr (k <= 6) {
        constexpr int d4 = (1 << k) / 4;
        float4* const buf = xb + (k & 1) * kWsXBuf + lane;
#pragma unroll
        for (int r = 0; r < R; ++r) st_shared4(buf + 32 * r, P[r]);
        st_shared4(buf + 32 * R, hs[k - 3]);
        __syncwarp();
        hs[k - 3] = P[0];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const float4 now = add4(P[r], buf[32 * r + d4]);
            if (wants_out<MODE>(cx)) {
                const float4 g = add4(Pprev[r], buf[32 * r + d4 / 2]);
                ig_fold<k + 1, k - 1, KX, (MODE != 0), SW>(best[r], now, g, lim[r], nb[r], cx);
            }
            Pprev[r] = P[r];
            P[r] = now;
        }
        ig_lane_levels<K, MODE, SW, KX, k + 1>(P, Pprev, best, lim, nb, hs, xb, lane, cx);
    } else if constexpr (8 <= LAST) {  // width 192 exists
        if (wants_out<MODE>(cx)) {
            float4* const buf = xb + (k & 1) * kWsXBuf + lane;
#pragma unroll
            for (int r = 0; r < R; ++r) st_shared4(buf + 32 * r, P[r]);
            st_shared4(buf + 32 * R, hs[4]);
            __syncwarp();
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const float4 g = add4(Pprev[r], buf[32 * r + 16]);
                ig_fold_one<6, KX, (MODE != 0), SW>(best[r], g, lim[r], nb[r], cx);
            }
        }
        hs[4] = P[0];
    }
}

// Row levels j < JN with the extra width 3 * 2^(7+j) = P_{7+j}[row r] + P_{8+j}[row r + 2^j]: this step's new
// value of that row, or the previous step's, which the next level keeps (nr) or - last near level - has stored
// in its FIFO one step ago.
template <int K, int MODE, bool SW, int KX, int j>
__device__ __forceinline__ void ig_near_levels(float4 (&P)[kWsRows], float4 (&best)[kWsRows], const int (&lim)[kWsRows],
                                               const uint32_t (&nb)[kWsRows], float4 (&nr)[WsGeo<K>::NEAR + 1],
                                               uint32_t tbase, int it, const ChunkCtx& cx) {
    using G = WsGeo<K>;
    constexpr int R = kWsRows;
    if constexpr (j < G::JN) {
        constexpr int D = 1 << j;
        constexpr int off = D - 1;
        constexpr int k = 7 + j;                       // level of P
        constexpr bool kHasIg = k + 2 <= G::LAST;      // width 3 * 2^k exists
        float4 now[R];
#pragma unroll
        for (int r = 0; r < R; ++r) now[r] = add4(P[r], r + D < R ? P[r + D] : nr[off + r + D - R]);
        if (wants_out<MODE>(cx)) {
            if constexpr (kHasIg) {
                float4 prev[R];  // P_{k+1} of the previous step's rows 0 .. D-1 (only those are used)
                if constexpr (j + 1 < G::JN) {
#pragma unroll
                    for (int i = 0; i < D; ++i) prev[i] = nr[2 * D - 1 + i];
                } else {  // the first FIFO level stored them one step ago
                    static_assert(G::JF >= 1, "a next level exists");
                    constexpr int Q = G::Q0;
                    tmem_ld_rows(tbase + 4u * R * static_cast<uint32_t>((it - 1) & (Q - 1)), prev);
                }
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const float4 g = add4(P[r], r + D < R ? now[r + D] : prev[r + D - R]);
                    ig_fold<k + 1, k, KX, (MODE != 0), SW>(best[r], now[r], g, lim[r], nb[r], cx);
                }
            } else {
#pragma unroll
                for (int r = 0; r < R; ++r) ig_fold<k + 1, -1, KX, (MODE != 0), SW>(best[r], now[r], now[r], lim[r], nb[r], cx);
            }
        }
#pragma unroll
        for (int i = 0; i < D; ++i) nr[off + i] = P[i];
#pragma unroll
        for (int r = 0; r < R; ++r) P[r] = now[r];
        ig_near_levels<K, MODE, SW, KX, j + 1>(P, best, lim, nb, nr, tbase, it, cx);
    }
}

// FIFO levels i < JF with the extra width 3 * 2^(10+i) = P_{10+i}[n] + P_{11+i}[n + 2^(10+i)]: the next level's
// FIFO (twice as deep) holds P_{11+i} of Q steps ago.
template <int K, int MODE, bool SW, int KX, int i>
__device__ __forceinline__ void ig_fifo_levels(float4 (&P)[kWsRows], float4 (&best)[kWsRows], const int (&lim)[kWsRows],
                                               const uint32_t (&nb)[kWsRows], uint32_t tbase, int it, const ChunkCtx& cx) {
    using G = WsGeo<K>;
    constexpr int R = kWsRows;
    if constexpr (i < G::JF) {
        constexpr int Q = G::Q0 << i;
        constexpr int k = 7 + G::JN + i;               // level of P
        constexpr int first = G::Q0 * ((1 << i) - 1);
        constexpr bool kHasIg = i + 1 < G::JF;
        const uint32_t taddr = tbase + 4u * R * static_cast<uint32_t>(first + (it & (Q - 1)));
        float4 old[R];
        tmem_ld_rows(taddr, old);
        tmem_st_rows(taddr, P);
        float4 half[R];
        if constexpr (kHasIg) {
            if (wants_out<MODE>(cx)) {
                constexpr int first2 = G::Q0 * ((2 << i) - 1);
                tmem_ld_rows(tbase + 4u * R * static_cast<uint32_t>(first2 + ((it - Q) & (2 * Q - 1))), half);
            }
        }
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const float4 now = add4(P[r], old[r]);
            if (wants_out<MODE>(cx)) {
                if constexpr (kHasIg) {
                    const float4 g = add4(P[r], half[r]);
                    ig_fold<k + 1, k, KX, (MODE != 0), SW>(best[r], now, g, lim[r], nb[r], cx);
                } else {
                    ig_fold<k + 1, -1, KX, (MODE != 0), SW>(best[r], now, now, lim[r], nb[r], cx);
                }
            }
            P[r] = now;
        }
        ig_fifo_levels<K, MODE, SW, KX, i + 1>(P, best, lim, nb, tbase, it, cx);
    }
}

// Store of one step's results (shared by both width families).
template <int MODE, bool GR, bool U8>
__device__ __forceinline__ float ws_store(const float4 (&best)[kWsRows], const int (&lim)[kWsRows], int lane,
                                          const ChunkCtx& cx) {
    constexpr int R = kWsRows;
    float top = __int_as_float(0xff800000);
    if (wants_out<MODE>(cx)) {
#pragma unroll
        for (int r = 0; r < R; ++r) {
            if (MODE != 0 || lim[r] > 0) {
                const float4 kq = best[r];
                top = fmax3(top, fmax3(kq.x, kq.y, kq.z), kq.w);
                // Y keeps the 5 tag bits of the key: clearing them would perturb the value by up to
                // 31 ulp as well (same bound) and costs four more ALU-pipe ops.
                const float4 y = scale4(kq, cx.inv);
                const long long o = cx.n0 + 4ll * (lane + 32 * r);
                *reinterpret_cast<float4*>(cx.out_snr + o) = y;
                if constexpr (U8) {
                    // the four low bytes of the keys into one word (3 PRMT), inverted and masked at once
                    const uint32_t t = __byte_perm(__float_as_uint(kq.x), __float_as_uint(kq.y), 0x0040);
                    const uint32_t u = __byte_perm(__float_as_uint(kq.z), __float_as_uint(kq.w), 0x4000);
                    const uint32_t packed = ~__byte_perm(t, u, 0x7610) & 0x1f1f1f1fu;
                    *reinterpret_cast<uint32_t*>(reinterpret_cast<uint8_t*>(cx.out_width) + o) = packed;
                } else {
                    int4 wv = make_int4(static_cast<int>(~__float_as_uint(kq.x) & kCodeMask),
                                        static_cast<int>(~__float_as_uint(kq.y) & kCodeMask),
                                        static_cast<int>(~__float_as_uint(kq.z) & kCodeMask),
                                        static_cast<int>(~__float_as_uint(kq.w) & kCodeMask));
                    if constexpr (GR) {  // on no width's grid: -inf / -1 (reading A16)
                        const float ninf = __int_as_float(0xff800000);
                        if (kq.x == ninf) wv.x = -1;
                        if (kq.y == ninf) wv.y = -1;
                        if (kq.z == ninf) wv.z = -1;
                        if (kq.w == ninf) wv.w = -1;
                    }
                    *reinterpret_cast<int4*>(cx.out_width + o) = wv;
                }
            }
        }
    }
    return top;
}

// One step of one warp for the IGRID depth-1 width set.
template <int K, int MODE, bool SW, int KX, bool U8>
__device__ __forceinline__ float ws_step_ig(const float4* __restrict__ st4, float4 (&hs)[5],
                                            float4 (&nr)[WsGeo<K>::NEAR + 1], float4* __restrict__ xb, uint32_t tbase,
                                            int it, int lane, const ChunkCtx& cx) {
    constexpr int R = kWsRows;
    constexpr bool GR = KX != kWsNoGrid;
    constexpr bool F = MODE != 0;
    const float mu = cx.mu;
    float4 P[R], Pprev[R], best[R];
    int lim[R];
    uint32_t nb[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        nb[r] = static_cast<uint32_t>(cx.n0) + 4u * static_cast<uint32_t>(lane + 32 * r);
        if constexpr (MODE != 0) {
            lim[r] = 1 << 30;
        } else {
            const long long left = cx.n_t - (cx.n0 + 4ll * (lane + 32 * r));
            lim[r] = left > (1ll << 30) ? (1 << 30) : (left < 0 ? 0 : static_cast<int>(left));
        }
        // widths 1, 2, 3, 4, 6, 8 from three raw float4
        const float4 a = norm4(st4[lane + 32 * r], mu);
        const float4 b = norm4(st4[lane + 32 * r + 1], mu);
        const float4 c = norm4(st4[lane + 32 * r + 2], mu);
        const float s01 = a.x + a.y, s12 = a.y + a.z, s23 = a.z + a.w, s34 = a.w + b.x;
        const float s45 = b.x + b.y, s56 = b.y + b.z, s67 = b.z + b.w, s78 = b.w + c.x;
        const float s89 = c.x + c.y, s9a = c.y + c.z;
        const float4 p1 = make_float4(s01, s12, s23, s34);
        const float2 u01 = make_float2(s01, s12), u23 = make_float2(s23, s34), u45 = make_float2(s45, s56),
                     u67 = make_float2(s67, s78), u89 = make_float2(s89, s9a);
        const float2 p2lo = __fadd2_rn(u01, u23), p2hi = __fadd2_rn(u23, u45);
        const float2 q2lo = __fadd2_rn(u45, u67), q2hi = __fadd2_rn(u67, u89);
        const float2 p3lo = __fadd2_rn(p2lo, q2lo), p3hi = __fadd2_rn(p2hi, q2hi);
        const float4 p2 = make_float4(p2lo.x, p2lo.y, p2hi.x, p2hi.y);
        const float4 p3 = make_float4(p3lo.x, p3lo.y, p3hi.x, p3hi.y);
        if (wants_out<MODE>(cx)) {
            // width 3 = x[n] + P_1[n+1]; width 6 = P_1[n] + P_2[n+2]
            const float4 x3 = make_float4(a.x + s12, a.y + s23, a.z + s34, a.w + s45);
            const float2 x6lo = __fadd2_rn(u01, p2hi), x6hi = __fadd2_rn(u23, q2lo);
            const float4 x6 = make_float4(x6lo.x, x6lo.y, x6hi.x, x6hi.y);
            if constexpr (GR) {
                best[r] = mask_to_grid(ig_key<0, 1, F, SW>(a, 1.0f, lim[r], cx), nb[r], cx.gmask[0]);
                ig_fold<1, 0, KX, F, SW>(best[r], p1, x3, lim[r], nb[r], cx);
            } else {
                best[r] = max4(ig_key<0, 1, F, SW>(a, 1.0f, lim[r], cx), ig_key<idx_pow2(1), 2, F, SW>(p1, level_scale<1>(), lim[r], cx),
                               ig_key<idx_ig(0), 3, F, SW>(x3, ig_scale<0>(), lim[r], cx));
            }
            ig_fold<2, 1, KX, F, SW>(best[r], p2, x6, lim[r], nb[r], cx);
            ig_fold<3, -1, KX, F, SW>(best[r], p3, p3, lim[r], nb[r], cx);
        }
        Pprev[r] = p2;
        P[r] = p3;
    }
    ig_lane_levels<K, MODE, SW, KX, 3>(P, Pprev, best, lim, nb, hs, xb, lane, cx);
    ig_near_levels<K, MODE, SW, KX, 0>(P, best, lim, nb, nr, tbase, it, cx);
    ig_fifo_levels<K, MODE, SW, KX, 0>(P, best, lim, nb, tbase, it, cx);
    if constexpr (WsGeo<K>::JF > 0) tmem_wait_st();
    return ws_store<MODE, GR, U8>(best, lim, lane, cx);
}

// One step for either width family.
template <int K, int MODE, bool SW, int KX, bool U8, bool IG, int NH>
__device__ __forceinline__ float ws_any_step(const float4* __restrict__ st4, float4 (&hs)[NH],
                                             float4 (&nr)[WsGeo<K>::NEAR + 1], float4* __restrict__ xb, uint32_t tbase,
                                             int it, int lane, const ChunkCtx& cx) {
    if constexpr (IG) {
        return ws_step_ig<K, MODE, SW, KX, U8>(st4, hs, nr, xb, tbase, it, lane, cx);
    } else {
        return ws_step<K, MODE, SW, KX, U8>(st4, hs, nr, xb, tbase, it, lane, cx);
    }
}

constexpr size_t kWsStagesBytes = static_cast<size_t>(kWsWarps) * kWsStages * kWsStage * 4;
constexpr size_t kWsXBytes = static_cast<size_t>(kWsWarps) * 2 * kWsXBuf * 16;
constexpr size_t ws_smem_bytes() { return kWsStagesBytes + kWsXBytes + kWsWarps * kWsStages * 8 + 16; }

template <int K, bool SW, int KX, bool U8, bool IG>
__global__ void __launch_bounds__(32 * kWsWarps, 1) spd_tree_ws_kernel(const TreeParams p, const int n_pieces) {
    using G = WsGeo<K>;
    constexpr bool GR = KX != kWsNoGrid;
    constexpr int S = kWsStep;
    constexpr int M = 1 << (K - 1);
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    float* const stages = reinterpret_cast<float*>(smem_raw) + warp * kWsStages * kWsStage;
    float4* const xb = reinterpret_cast<float4*>(smem_raw + kWsStagesBytes) + warp * 2 * kWsXBuf;
    uint64_t* const bars = reinterpret_cast<uint64_t*>(smem_raw + kWsStagesBytes + kWsXBytes) + warp * kWsStages;
    uint32_t* const tslot =
        reinterpret_cast<uint32_t*>(smem_raw + kWsStagesBytes + kWsXBytes + kWsWarps * kWsStages * 8);

    if (lane == 0) {
#pragma unroll
        for (int i = 0; i < kWsStages; ++i) mbar_init(&bars[i], 1);
        fence_mbar_init();
    }
    uint32_t tbase = 0;
    if constexpr (G::COLS > 0) {
        if (warp == 0) tmem_alloc<512>(tslot);
        tmem_fence_before_sync();
        __syncthreads();
        tmem_fence_after_sync();
        // this warp's lane quarter, and its half of the columns
        tbase = *tslot + (static_cast<uint32_t>(warp & 3) << 21) + static_cast<uint32_t>(warp >> 2) * 256u;
    } else {
        __syncthreads();
    }

    const long long n_t = p.n_t;
    // step c runs unguarded iff (c + 1) * S + max(M, 8) <= n_t
    const int c_fast_end = n_t >= M ? static_cast<int>((n_t - M) / S) : 0;
    ChunkCtx cx;
    cx.tm = p.tag_mask;
    if constexpr (GR) {
#pragma unroll
        for (int k = 0; k < K; ++k) cx.gmask[k] = p.gmask[k];
    }
    cx.n_t = n_t;
    cx.tid = lane;
    int stage = 0;
    uint32_t phase = 0;
    constexpr uint32_t kBytes = kWsStage * 4;

    // A piece is a run of p.seg_chunks steps.  segs_per_row > 0: pieces are the segments of the
    // rows (piece = row * segs_per_row + segment).  segs_per_row == 0: pieces partition the
    // plane's steps in row-major order and may span several rows; every row part inside a
    // piece is one stream (only a part that stops short of its row's end replays look-ahead).
    const long long cpr = p.chunks_per_row;
    for (int piece = blockIdx.x * kWsWarps + warp; piece < n_pieces; piece += gridDim.x * kWsWarps) {
        long long lin_lo, lin_hi;  // steps [lin_lo, lin_hi) of the plane, row-major
        if (p.segs_per_row > 0) {
            const int d0 = piece / p.segs_per_row;
            const int s0 = piece - d0 * p.segs_per_row;
            lin_lo = d0 * cpr + static_cast<long long>(s0) * p.seg_chunks;
            lin_hi = min(lin_lo + p.seg_chunks, (d0 + 1) * cpr);
        } else {
            lin_lo = static_cast<long long>(piece) * p.seg_chunks;
            lin_hi = min(lin_lo + p.seg_chunks, cpr * p.n_dm);
        }
      while (lin_hi > lin_lo) {
        const int d = static_cast<int>((lin_hi - 1) / cpr);
        const long long row_lo = d * cpr;
        const int c_hi = static_cast<int>(lin_hi - row_lo);
        const int c_lo = static_cast<int>(max(lin_lo, row_lo) - row_lo);
        lin_hi = row_lo + c_lo;
        const int c_top = min(c_hi + p.warm_chunks, p.chunks_per_row);
        // steps [c_lo, ring_top) are interior: bulk-copy ring; those >= c_hi are look-ahead only
        const int ring_top = max(c_lo, min(c_top, c_fast_end));

        const float* __restrict__ row = p.plane + static_cast<long long>(d) * n_t;
        cx.mu = p.mean[d];
        const float sg = SW ? 1.0f : p.sigma[d];
        cx.inv = 1.0f / sg;
        if constexpr (SW) {
            // keys are SNRs already: 1 / sigma_{d, 2^k} per level, nothing left for the store
            constexpr int NW = IG ? 2 * K - 2 : K;  // widths of the plan: one scale per width index
            const float* __restrict__ swr = p.sigma_w + static_cast<long long>(d) * NW;
#pragma unroll
            for (int k = 0; k < NW; ++k) cx.ls[k] = 1.0f / __ldg(swr + k);
            cx.inv = 1.0f;
        }
        cx.out_snr = p.out_snr + static_cast<long long>(d) * n_t;
        // a uint8 plane advances by n_t bytes per row: n_t / 4 int32 (n_t % 4 == 0 on this path)
        cx.out_width = p.out_width + static_cast<long long>(d) * (U8 ? n_t / 4 : n_t);
        uint8_t* const act =
            p.activity ? p.activity + static_cast<long long>(d) * ((p.chunks_per_row + kWsActSteps - 1) / kWsActSteps)
                       : nullptr;
        float thr_key = __int_as_float(0x7f800000);
        if (act) {
            const float t = SW ? p.threshold : p.threshold * sg;
            thr_key = t - fabsf(t) * 2e-6f;
        }

        float4 hs[IG ? 5 : 4], nr[G::NEAR + 1];
#pragma unroll
        for (int i = 0; i < (IG ? 5 : 4); ++i) hs[i] = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
        for (int i = 0; i < G::NEAR + 1; ++i) nr[i] = make_float4(0.f, 0.f, 0.f, 0.f);
        if constexpr (G::COLS > 0) {
            float4 zero[kWsRows];
#pragma unroll
            for (int i = 0; i < kWsRows; ++i) zero[i] = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
            for (int col = 0; col < G::COLS; col += 4 * kWsRows) tmem_st_rows(tbase + col, zero);
            tmem_wait_st();
        }
        int it = 0;

        // ---- guarded steps: the row tail (windows may cross the end of the row) ------------
        float* const gbuf = stages + stage * kWsStage;
        for (int c = c_top - 1; c >= ring_top; --c, ++it) {
            const long long n0 = static_cast<long long>(c) * S;
            // n0 and n_t are multiples of 4: a float4 lies entirely inside or outside the row
            const float4* const row4 = reinterpret_cast<const float4*>(row + n0);
            const float4 fill = make_float4(cx.mu, cx.mu, cx.mu, cx.mu);
#pragma unroll
            for (int j = 0; j < (kWsStage / 4 + 31) / 32; ++j) {
                const int i = lane + 32 * j;
                if (i < kWsStage / 4)
                    reinterpret_cast<float4*>(gbuf)[i] = n0 + 4ll * i < n_t ? __ldg(row4 + i) : fill;
            }
            __syncwarp();
            cx.n0 = n0;
            cx.do_out = c < c_hi;
            const float top = ws_any_step<K, 0, SW, KX, U8, IG>(reinterpret_cast<const float4*>(gbuf), hs, nr, xb, tbase, it, lane, cx);
            if (act && cx.do_out && top >= thr_key) act[c / kWsActSteps] = 1;
            __syncwarp();
        }

        // ---- interior steps: this warp's bulk-copy ring ------------------------------------
        const int n_ring = ring_top - c_lo;
        if (n_ring <= 0) continue;  // next row part of the piece
        fence_proxy_async();
        __syncwarp();
        if (lane == 0) {
            int sx = stage;
#pragma unroll
            for (int j = 0; j < kWsStages - 1; ++j) {
                if (j < n_ring) {
                    mbar_arrive_expect_tx(&bars[sx], kBytes);
                    bulk_g2s(stages + sx * kWsStage, row + static_cast<long long>(ring_top - 1 - j) * S, kBytes,
                             &bars[sx]);
                }
                sx = sx + 1 == kWsStages ? 0 : sx + 1;
            }
        }
        // refill the stage read one step ago with the step kWsStages - 1 ahead, wait for this one
        auto ring_next = [&](int f) {
            __syncwarp();  // every lane has finished reading the stage that is refilled now
            if (lane == 0) {
                const int nx = f + kWsStages - 1;
                if (nx < n_ring) {
                    const int sx = stage == 0 ? kWsStages - 1 : stage - 1;  // (stage + kWsStages - 1) % kWsStages
                    mbar_arrive_expect_tx(&bars[sx], kBytes);
                    bulk_g2s(stages + sx * kWsStage, row + static_cast<long long>(ring_top - 1 - nx) * S, kBytes,
                             &bars[sx]);
                }
            }
            mbar_wait(&bars[stage], phase);
        };
        auto ring_done = [&]() {
            if (++stage == kWsStages) {
                stage = 0;
                phase ^= 1;
            }
        };
        const int n_warm = max(0, ring_top - c_hi);  // look-ahead steps first: sums only
        int f = 0;
        for (; f < n_warm; ++f, ++it) {
            ring_next(f);
            cx.n0 = static_cast<long long>(ring_top - 1 - f) * S;
            ws_any_step<K, 2, SW, KX, U8, IG>(reinterpret_cast<const float4*>(stages + stage * kWsStage), hs, nr, xb, tbase, it, lane, cx);
            ring_done();
        }
        // Two steps per loop trip: the values kept from one step to the next (hs, nr: 11 float4)
        // alternate between two register sets instead of being moved, and the first levels of a
        // step overlap the last levels of the one before (10.70 -> 10.26 ms on config 3; x3: see DESIGN).
        // the all-masked grid body and the IGRID body are larger: one step per trip keeps the loop in the instruction cache
        constexpr int kTrip = ((GR && KX > 6) || IG) ? 1 : kWsUnroll;
#pragma unroll kTrip
        for (; f < n_ring; ++f, ++it) {
            ring_next(f);
            const int c = ring_top - 1 - f;
            cx.n0 = static_cast<long long>(c) * S;
            const float top = ws_any_step<K, 1, SW, KX, U8, IG>(reinterpret_cast<const float4*>(stages + stage * kWsStage), hs, nr, xb,
                                            tbase, it, lane, cx);
            if (act && top >= thr_key) act[c / kWsActSteps] = 1;
            ring_done();
        }
      }
    }

    if constexpr (G::COLS > 0) {
        tmem_fence_before_sync();
        __syncthreads();
        if (warp == 0) tmem_dealloc<512>(*tslot);
    }
}


// ---- host side, shared by spd_tree_ws.cu (widths 2^k) and spd_tree_ws_ig.cu (IGRID depth 1) ----------------

// Instantiated values of KX for grid plans: the first level whose keys are formed for the first sample of a
// float4 only (separation >= 4).  2: Alg. 3's DIT (width 2^k every 2^k-th sample); 4, 6: widths on four and
// sixteen layers; kWsNoGrid - 1: every level masked (any separations).
constexpr int kWsGridKx[4] = {2, 4, 6, kWsNoGrid - 1};

template <int K, bool IG>
cudaError_t ws_prepare(int smem) {
    const auto attr = cudaFuncAttributeMaxDynamicSharedMemorySize;
    cudaError_t e = cudaFuncSetAttribute(spd_tree_ws_kernel<K, false, kWsNoGrid, false, IG>, attr, smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(spd_tree_ws_kernel<K, true, kWsNoGrid, false, IG>, attr, smem);
    if constexpr (!IG) {
        if (e == cudaSuccess) e = cudaFuncSetAttribute(spd_tree_ws_kernel<K, false, kWsNoGrid, true, IG>, attr, smem);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(spd_tree_ws_kernel<K, false, kWsGridKx[0], false, IG>, attr, smem);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(spd_tree_ws_kernel<K, false, kWsGridKx[2], false, IG>, attr, smem);
    }
    if (e == cudaSuccess) e = cudaFuncSetAttribute(spd_tree_ws_kernel<K, false, kWsGridKx[1], false, IG>, attr, smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(spd_tree_ws_kernel<K, false, kWsGridKx[3], false, IG>, attr, smem);
    return e;
}

// variant: 0 plain, 1 sigma per width, 2 uint8 index, 3 + i: grid plan with threshold kWsGridKx[i]
// (the IGRID family instantiates 0, 1, 4 and 6)
template <int K, bool IG>
cudaError_t ws_launch(int variant, dim3 grid, size_t sm, cudaStream_t stream, const TreeParams& prm, int np) {
    const int T = 32 * kWsWarps;
    switch (variant) {
        case 0: spd_tree_ws_kernel<K, false, kWsNoGrid, false, IG><<<grid, T, sm, stream>>>(prm, np); break;
        case 1: spd_tree_ws_kernel<K, true, kWsNoGrid, false, IG><<<grid, T, sm, stream>>>(prm, np); break;
        case 4: spd_tree_ws_kernel<K, false, kWsGridKx[1], false, IG><<<grid, T, sm, stream>>>(prm, np); break;
        case 6: spd_tree_ws_kernel<K, false, kWsGridKx[3], false, IG><<<grid, T, sm, stream>>>(prm, np); break;
        default:
            if constexpr (!IG) {
                if (variant == 2) { spd_tree_ws_kernel<K, false, kWsNoGrid, true, IG><<<grid, T, sm, stream>>>(prm, np); break; }
                if (variant == 3) { spd_tree_ws_kernel<K, false, kWsGridKx[0], false, IG><<<grid, T, sm, stream>>>(prm, np); break; }
                if (variant == 5) { spd_tree_ws_kernel<K, false, kWsGridKx[2], false, IG><<<grid, T, sm, stream>>>(prm, np); break; }
            }
            return cudaErrorNotSupported;
    }
    return cudaGetLastError();
}

#define SPD_WS_CASES(OP) OP(9) OP(10) OP(11) OP(12) OP(13) OP(14)

// Pieces of a launch over n_dm rows: steps per piece and number of pieces.
inline void ws_pieces(const spd_plan* plan, int64_t n_dm, int* piece_chunks, int64_t* n_pieces) {
    const TreeConfig& cfg = plan->tree;
    if (cfg.segs_per_row > 0) {
        *piece_chunks = cfg.seg_chunks;
        *n_pieces = n_dm * cfg.segs_per_row;
        return;
    }
    const int64_t total = n_dm * cfg.chunks_per_row;
    const int64_t slots = int64_t(plan->sm_count) * kWsWarps;
    // a piece no shorter than a few look-aheads, so that replaying one stays cheap
    const int64_t min_len = std::max<int64_t>(8, 4 * int64_t(cfg.warm_chunks));
    const int64_t want = std::max<int64_t>(1, std::min<int64_t>(slots, total / min_len));
    const int64_t len = std::min<int64_t>((total + want - 1) / want, 0x3fffffff);
    *piece_chunks = static_cast<int>(len);
    *n_pieces = (total + len - 1) / len;
}

// plan->tree.K (levels) must be set; IG: the plan's widths are the IGRID depth-1 set over those levels.
template <bool IG>
int ws_configure_t(spd_plan* plan) {
    TreeConfig& cfg = plan->tree;
    cfg.kind = 1;
    cfg.ig = IG;
    cfg.T = 32 * kWsWarps;
    cfg.chunk = kWsStep;
    cfg.act_block = kWsStep * kWsActSteps;
    cfg.blocks_per_sm = 1;
    cfg.smem_bytes = ws_smem_bytes();
    cudaError_t e = cudaErrorInvalidValue;
#define SPD_PREP(KK) \
    if (cfg.K == KK) e = ws_prepare<KK, IG>(static_cast<int>(cfg.smem_bytes));
    SPD_WS_CASES(SPD_PREP)
#undef SPD_PREP
    if (e != cudaSuccess) return cuda_fail(e, "configuring the warp-stream tree kernel");

    const int64_t S = kWsStep;
    const int64_t M = int64_t(1) << (cfg.K - 1);
    cfg.chunks_per_row = static_cast<int>((plan->n_t + S - 1) / S);
    cfg.warm_chunks = static_cast<int>((M - 1 + S - 1) / S);
    // Work split.  Default: the steps of the plane, in row-major order, are cut into one piece
    // per resident warp (sm_count * 8), so every warp does the same number of steps and only
    // the one row part per piece that stops short of its row's end replays look-ahead.
    // SPD_OPT_SEGMENTS_PER_ROW = s: every row cut into s equal segments instead.
    cfg.segs_per_row = 0;
    cfg.seg_chunks = 0;  // per launch (depends on the rows of the launch): ws_pieces()
    if (plan->segs_option > 0) {
        const int64_t segs = std::min<int64_t>(plan->segs_option, cfg.chunks_per_row);
        cfg.seg_chunks = static_cast<int>((cfg.chunks_per_row + segs - 1) / segs);
        cfg.segs_per_row = static_cast<int>((cfg.chunks_per_row + cfg.seg_chunks - 1) / cfg.seg_chunks);
        if (plan->n_dm * cfg.segs_per_row > 0x7fffffffll) {
            set_error("too many streams");
            return SPD_ERR_INVALID_ARG;
        }
    }
    return SPD_OK;
}

template <bool IG>
int ws_run_t(const spd_plan* plan, int64_t n_dm, const float* plane, const float* mean, const float* sigma,
             float* out_snr, void* out_width, float threshold, uint8_t* activity, cudaStream_t stream,
             const float* sigma_w) {
    const TreeConfig& cfg = plan->tree;
    TreeParams prm;
    prm.plane = plane;
    prm.mean = mean;
    prm.sigma = sigma;
    prm.sigma_w = sigma_w;
    prm.out_snr = out_snr;
    prm.out_width = static_cast<int32_t*>(out_width);
    prm.activity = activity;
    prm.threshold = threshold;
    int piece_chunks = 0;
    int64_t n_pieces = 0;
    ws_pieces(plan, n_dm, &piece_chunks, &n_pieces);
    if (n_pieces > 0x7fffffffll) {
        set_error("too many pieces");
        return SPD_ERR_INVALID_ARG;
    }
    prm.n_t = plan->n_t;
    prm.n_dm = n_dm;
    prm.chunks_per_row = cfg.chunks_per_row;
    prm.seg_chunks = piece_chunks;
    prm.segs_per_row = cfg.segs_per_row;
    prm.warm_chunks = cfg.warm_chunks;
    prm.tag_mask = ~kCodeMask;
    // separation of level k = that of width 2^k (IGRID family: the widths of an octave share it, checked at plan
    // creation)
    const bool grid = !plan->separations.empty();
    for (int k = 0; k < 16; ++k) {
        const int wi = IG ? (k == 0 ? 0 : 2 * k - 1) : k;
        prm.gmask[k] = (grid && k < cfg.K) ? static_cast<uint32_t>(plan->separations[wi] - 1) : 0u;
    }
    if (activity) {
        const size_t bytes = (static_cast<size_t>(n_dm) * static_cast<size_t>(activity_per_row(plan)) + 127) / 128 * 128;
        const cudaError_t em = cudaMemsetAsync(activity, 0, bytes, stream);
        if (em != cudaSuccess) return cuda_fail(em, "clearing the activity map");
    }
    const int64_t blocks = std::min<int64_t>(plan->sm_count, (n_pieces + kWsWarps - 1) / kWsWarps);
    const dim3 grid_dim(static_cast<unsigned>(std::max<int64_t>(1, blocks)));
    const bool u8 = plan->width_bytes == 1;
    if ((u8 || sigma_w) && grid) {
        set_error("a grid plan on the tree kernel runs with eq. (5)'s sqrt(width) and an int32 width index");
        return SPD_ERR_INVALID_ARG;
    }
    int variant = sigma_w ? 1 : (u8 ? 2 : 0);
    if (grid) {
        // the first level with a separation of 4 or more, rounded up to an instantiated threshold
        int kx = cfg.K;
        for (int k = cfg.K - 1; k >= 0 && prm.gmask[k] >= 3u; --k) kx = k;
        if constexpr (IG)
            variant = kx <= kWsGridKx[1] ? 4 : 6;
        else
            variant = kx <= kWsGridKx[0] ? 3 : (kx <= kWsGridKx[1] ? 4 : (kx <= kWsGridKx[2] ? 5 : 6));
    }
    cudaError_t e = cudaErrorInvalidValue;
#define SPD_LAUNCH(KK) \
    if (cfg.K == KK) e = ws_launch<KK, IG>(variant, grid_dim, cfg.smem_bytes, stream, prm, static_cast<int>(n_pieces));
    SPD_WS_CASES(SPD_LAUNCH)
#undef SPD_LAUNCH
    if (e != cudaSuccess) return cuda_fail(e, "launching the warp-stream tree kernel");
    return SPD_OK;
}

}  // namespace
}  // namespace spd
