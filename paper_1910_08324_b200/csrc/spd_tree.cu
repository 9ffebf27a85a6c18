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
//     chunks of C = 16*T samples.  eq. (2) looks forward in time, so in reverse time the
//     partner P_k[n + 2^k] has always been computed already; each level keeps a delay
//     line instead of re-reading a (max_width - 1)-sample halo per tile.  The halo is
//     paid once per segment (warm-up chunks), not once per tile.
//   * Thread t owns, in each of the chunk's 4 "rows" of 4*T samples, the 4 consecutive
//     samples 4t..4t+3 (one float4).  Widths 2, 4, 8: in the thread's own registers from
//     three float4 of raw samples (the width-4 sums of the next float4 are recomputed
//     rather than exchanged).  Levels 8 <= 2^k <= 2T: the partner belongs to another thread - exchanged through
//     a ping-pong shared-memory buffer with 128-bit accesses, one __syncthreads() each.
//     Levels 2^k >= 4T: the partner is the SAME thread's float4 1, 2, 4 or 8 rows later,
//     i.e. a register of this chunk or a delay register kept from the previous chunks.
//   * Chunks are staged into shared memory by cp.async.bulk (TMA, 1-D) through a
//     3-deep mbarrier ring; results leave as 128-bit streaming stores.
//   * SNR scale 2^(-k/2) is a compile-time constant (data are divided by sigma on load);
//     the width index rides in the 5 low mantissa bits of the SNR being maximised
//     (relative perturbation <= 2^-18, inside the 1e-4 tolerance), stored inverted so
//     that exact ties resolve to the smallest width; max is the 3-input FMNMX3.
//   * Row tails (valid-windows-only rule, reading A3) and warm-up chunks run in a
//     guarded variant of the same body; interior chunks run the unguarded one.
#include <cuda_runtime.h>
#include <stdint.h>

#include <algorithm>
#include <cstdlib>

#include "spd_internal.h"

namespace spd {
namespace {

struct TreeParams {
    const float* plane;
    const float* mean;
    const float* sigma;
    float* out_snr;
    int32_t* out_width;
    long long n_t;
    int chunks_per_row;
    int seg_chunks;
    int segs_per_row;
    int warm_chunks;
    // ~kCodeMask, passed at run time on purpose: as a compile-time constant the tag
    // (v & mask) | code has two immediates and costs two LOP3 per value instead of one.
    uint32_t tag_mask;
};

// ------------------------------------------------------------------------------------
// PTX helpers: mbarrier + 1-D bulk copy (TMA), 3-input max.
// ------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n"
        " .reg .pred p;\n"
        " mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        " selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    while (!mbar_try_wait(bar, parity)) {
    }
}
__device__ __forceinline__ void bulk_g2s(void* dst_smem, const void* src_gmem, uint32_t bytes, uint64_t* bar) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
            smem_u32(dst_smem)),
        "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
        : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }

__device__ __forceinline__ float fmax3(float a, float b, float c) {
    float d;
    asm("max.f32 %0, %1, %2, %3;" : "=f"(d) : "f"(a), "f"(b), "f"(c));
    return d;
}

// ------------------------------------------------------------------------------------
// float4 arithmetic on the packed FP32x2 pipe.
// ------------------------------------------------------------------------------------
__device__ __forceinline__ float4 add4(float4 a, float4 b) {
    const float2 lo = __fadd2_rn(make_float2(a.x, a.y), make_float2(b.x, b.y));
    const float2 hi = __fadd2_rn(make_float2(a.z, a.w), make_float2(b.z, b.w));
    return make_float4(lo.x, lo.y, hi.x, hi.y);
}
__device__ __forceinline__ float4 scale4(float4 a, float c) {
    const float2 cc = make_float2(c, c);
    const float2 lo = __fmul2_rn(make_float2(a.x, a.y), cc);
    const float2 hi = __fmul2_rn(make_float2(a.z, a.w), cc);
    return make_float4(lo.x, lo.y, hi.x, hi.y);
}
// x - mu (eq. 4 numerator per sample; exact-ish, no cancellation later).  The division by
// sigma is applied once per output sample at the store, not per input sample here.
__device__ __forceinline__ float4 norm4(float4 a, float mu) {
    const float2 m = make_float2(-mu, -mu);
    const float2 lo = __fadd2_rn(make_float2(a.x, a.y), m);
    const float2 hi = __fadd2_rn(make_float2(a.z, a.w), m);
    return make_float4(lo.x, lo.y, hi.x, hi.y);
}

// 2^(-k/2): SNR scale of width 2^k on unit-variance data (eq. 5).
template <int k>
__device__ __forceinline__ constexpr float level_scale() {
    return ((k & 1) ? 0.70710678118654752440f : 1.0f) / static_cast<float>(1 << (k / 2));
}

constexpr uint32_t kCodeBits = 5;
constexpr uint32_t kCodeMask = (1u << kCodeBits) - 1u;

// SNR of level k with the inverted width index in the low mantissa bits.
template <int k>
__device__ __forceinline__ float pack1(float v, uint32_t tm) {
    return __uint_as_float((__float_as_uint(v) & tm) | (kCodeMask - static_cast<uint32_t>(k)));
}
template <int k>
__device__ __forceinline__ float4 key4(float4 p, uint32_t tm) {
    const float4 v = scale4(p, level_scale<k>());
    return make_float4(pack1<k>(v.x, tm), pack1<k>(v.y, tm), pack1<k>(v.z, tm), pack1<k>(v.w, tm));
}
// Guarded variant: element v of the float4 is valid iff 2^k <= lim - v (reading A3).
template <int k>
__device__ __forceinline__ float4 key4_masked(float4 p, int lim, uint32_t tm) {
    float4 q = key4<k>(p, tm);
    const int w = 1 << k;
    const float ninf = __int_as_float(0xff800000);
    if (w > lim) q.x = ninf;
    if (w > lim - 1) q.y = ninf;
    if (w > lim - 2) q.z = ninf;
    if (w > lim - 3) q.w = ninf;
    return q;
}
__device__ __forceinline__ float4 max4(float4 a, float4 b) {
    return make_float4(fmaxf(a.x, b.x), fmaxf(a.y, b.y), fmaxf(a.z, b.z), fmaxf(a.w, b.w));
}
__device__ __forceinline__ float4 max4(float4 a, float4 b, float4 c) {
    return make_float4(fmax3(a.x, b.x, c.x), fmax3(a.y, b.y, c.y), fmax3(a.z, b.z, c.z), fmax3(a.w, b.w, c.w));
}

template <int k, bool FAST>
__device__ __forceinline__ float4 keyx(float4 p, int lim, uint32_t tm) {
    if constexpr (FAST) {
        return key4<k>(p, tm);
    } else {
        return key4_masked<k>(p, lim, tm);
    }
}

// Fold the SNR of level j (just produced as `now` from `before` = level j-1) into best.
// Levels 0..2 are folded by the caller; above, levels are folded in pairs (j-1, j) when
// j is even so that one FMNMX3 serves two widths; a trailing odd level is folded alone.
template <int j, int K, bool FAST>
__device__ __forceinline__ void fold(float4& best, float4 before, float4 now, int lim, uint32_t tm) {
    if constexpr (j >= 3) {
        if constexpr ((j & 1) == 0) {
            best = max4(best, keyx<j - 1, FAST>(before, lim, tm), keyx<j, FAST>(now, lim, tm));
        } else if constexpr (j == K - 1) {
            best = max4(best, keyx<j, FAST>(now, lim, tm));
        }
    }
}

constexpr int ilog2(int v) { return v <= 1 ? 0 : 1 + ilog2(v / 2); }

// Delay registers of the in-register levels: the first rows of the previous chunks.
struct Delay {
    float4 a;     // row offset 1
    float4 b[2];  // row offset 2
    float4 c[4];  // row offset 4 (= previous chunk)
    float4 d0[4]; // row offset 8: two chunks ago
    float4 d1[4]; //               previous chunk
};

// One streaming step: the chunk staged at `st4` (C + 8 floats: the chunk and the first two
// float4 of the following chunk) -> Y, W for its C samples.
template <int T, int K, bool FAST>
__device__ __forceinline__ void tree_chunk(const float4* __restrict__ st4, float4* __restrict__ pp,
                                           float4* __restrict__ halo, int& xsel, int& hsel, Delay& dl,
                                           const float mu, const float inv, const uint32_t tm,
                                           float* __restrict__ out_snr,
                                           int32_t* __restrict__ out_width, const long long n0,
                                           const long long n_t, const bool do_out, const int tid) {
    constexpr int R = kRowsPerChunk;
    constexpr int LT = ilog2(T);
    constexpr int C4 = R * T;  // float4 per chunk
    constexpr int LAST = K - 1;

    float4 P[R], best[R];
    int lim[R];

    // ---- stage -> registers, remove the mean, levels 0..3 in the thread's own registers ----
#pragma unroll
    for (int r = 0; r < R; ++r) {
        if constexpr (FAST) {
            lim[r] = 1 << 30;
        } else {
            const long long left = n_t - (n0 + 4ll * (tid + T * r));
            lim[r] = left > (1ll << 30) ? (1 << 30) : (left < 0 ? 0 : static_cast<int>(left));
        }
        const float4 a = norm4(st4[tid + T * r], mu);
        if constexpr (K == 1) {
            P[r] = a;
            if (FAST || do_out) best[r] = keyx<0, FAST>(a, lim[r], tm);
        } else {
            const float4 b = norm4(st4[tid + T * r + 1], mu);
            const float s01 = a.x + a.y, s12 = a.y + a.z, s23 = a.z + a.w, s34 = a.w + b.x;
            const float4 p1 = make_float4(s01, s12, s23, s34);
            if constexpr (K == 2) {
                P[r] = p1;
                if (FAST || do_out) best[r] = max4(keyx<0, FAST>(a, lim[r], tm), keyx<1, FAST>(p1, lim[r], tm));
            } else {
                const float s45 = b.x + b.y, s56 = b.y + b.z;
                const float4 p2 = make_float4(s01 + s23, s12 + s34, s23 + s45, s34 + s56);
                if (FAST || do_out)
                    best[r] = max4(keyx<0, FAST>(a, lim[r], tm), keyx<1, FAST>(p1, lim[r], tm), keyx<2, FAST>(p2, lim[r], tm));
                if constexpr (K == 3) {
                    P[r] = p2;
                } else {
                    // Width 8 from a third float4 of raw samples: recomputing the width-4 sums of
                    // the next float4 here costs 8 adds on an idle pipe and saves one whole
                    // shared-memory exchange (the L1/shared data pipe is the binding unit).
                    const float4 c = norm4(st4[tid + T * r + 2], mu);
                    const float s67 = b.z + b.w, s78 = b.w + c.x, s89 = c.x + c.y, s9a = c.y + c.z;
                    const float4 p3 = make_float4((s01 + s23) + (s45 + s67), (s12 + s34) + (s56 + s78),
                                                  (s23 + s45) + (s67 + s89), (s34 + s56) + (s78 + s9a));
                    if (FAST || do_out) fold<3, K, FAST>(best[r], p2, p3, lim[r], tm);
                    P[r] = p3;
                }
            }
        }
    }

    // ---- exchange levels: P_{k+1}[n] = P_k[n] + P_k[n + 2^k], 8 <= 2^k <= 2T -----------
    float4* const hr = halo + hsel * T;        // written by the previous (later-in-time) chunk
    float4* const hw = halo + (hsel ^ 1) * T;  // read by the next chunk
    hsel ^= 1;
#pragma unroll
    for (int k = 3; k <= LT + 1; ++k) {
        if (k + 1 <= LAST) {
            const int d4 = (1 << k) / 4;  // partner distance in float4
            const int hoff = d4 - 2;      // sum of the halo sizes of the levels below
            float4* const buf = pp + xsel * C4;
            xsel ^= 1;
#pragma unroll
            for (int r = 0; r < R; ++r) buf[tid + T * r] = P[r];
            if (tid < d4) hw[hoff + tid] = P[0];
            __syncthreads();
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const float4* src = buf + (tid + T * r + d4);
                if (r == R - 1 && tid + d4 >= T) src = hr + (hoff + tid + d4 - T);
                const float4 now = add4(P[r], *src);
                if (FAST || do_out) {
                    switch (k) {  // k is a compile-time constant after unrolling
                        case 3: fold<4, K, FAST>(best[r], P[r], now, lim[r], tm); break;
                        case 4: fold<5, K, FAST>(best[r], P[r], now, lim[r], tm); break;
                        case 5: fold<6, K, FAST>(best[r], P[r], now, lim[r], tm); break;
                        case 6: fold<7, K, FAST>(best[r], P[r], now, lim[r], tm); break;
                        case 7: fold<8, K, FAST>(best[r], P[r], now, lim[r], tm); break;
                        case 8: fold<9, K, FAST>(best[r], P[r], now, lim[r], tm); break;
                        case 9: fold<10, K, FAST>(best[r], P[r], now, lim[r], tm); break;
                        case 10: fold<11, K, FAST>(best[r], P[r], now, lim[r], tm); break;
                        default: break;
                    }
                }
                P[r] = now;
            }
        }
    }

    // ---- in-register levels: partner 1, 2, 4, 8 rows later (same thread) --------------
    if constexpr (LAST >= LT + 3) {
        float4 now[R];
#pragma unroll
        for (int r = 0; r < R; ++r) now[r] = add4(P[r], r + 1 < R ? P[r + 1] : dl.a);
        dl.a = P[0];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            if (FAST || do_out) fold<LT + 3, K, FAST>(best[r], P[r], now[r], lim[r], tm);
            P[r] = now[r];
        }
    }
    if constexpr (LAST >= LT + 4) {
        float4 now[R];
#pragma unroll
        for (int r = 0; r < R; ++r) now[r] = add4(P[r], r + 2 < R ? P[r + 2] : dl.b[r + 2 - R]);
        dl.b[0] = P[0];
        dl.b[1] = P[1];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            if (FAST || do_out) fold<LT + 4, K, FAST>(best[r], P[r], now[r], lim[r], tm);
            P[r] = now[r];
        }
    }
    if constexpr (LAST >= LT + 5) {
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const float4 now = add4(P[r], dl.c[r]);
            dl.c[r] = P[r];
            if (FAST || do_out) fold<LT + 5, K, FAST>(best[r], P[r], now, lim[r], tm);
            P[r] = now;
        }
    }
    if constexpr (LAST >= LT + 6) {
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const float4 now = add4(P[r], dl.d0[r]);
            dl.d0[r] = dl.d1[r];
            dl.d1[r] = P[r];
            if (FAST || do_out) fold<LT + 6, K, FAST>(best[r], P[r], now, lim[r], tm);
            P[r] = now;
        }
    }

    // ---- unpack and store: Y = key with the code bits cleared, W = inverted code --------
    if (FAST || do_out) {
#pragma unroll
        for (int r = 0; r < R; ++r) {
            if (FAST || lim[r] > 0) {
                const uint32_t kx = __float_as_uint(best[r].x), ky = __float_as_uint(best[r].y);
                const uint32_t kz = __float_as_uint(best[r].z), kw = __float_as_uint(best[r].w);
                const float4 y = make_float4(__uint_as_float(kx & tm) * inv, __uint_as_float(ky & tm) * inv,
                                             __uint_as_float(kz & tm) * inv, __uint_as_float(kw & tm) * inv);
                const int4 w = make_int4(static_cast<int>(~kx & kCodeMask), static_cast<int>(~ky & kCodeMask),
                                         static_cast<int>(~kz & kCodeMask), static_cast<int>(~kw & kCodeMask));
                const long long o = n0 + 4ll * (tid + T * r);
                __stcs(reinterpret_cast<float4*>(out_snr + o), y);
                __stcs(reinterpret_cast<int4*>(out_width + o), w);
            }
        }
    }
    // With no exchange level there is no barrier inside the step: add the one that
    // orders this step's stage reads before the next refill of the stage.
    if constexpr (LAST < 4) __syncthreads();
}

// Resident blocks per SM for T = 128.  3 (168 registers per thread, no spills) measured 3 %
// faster than 4 (128 registers, 11 spilled delay registers): the kernel is bound by the
// L1/shared data pipe, not by occupancy (profiles/r01b_*).
#ifndef SPD_TREE_BPS128
#define SPD_TREE_BPS128 3
#endif
constexpr int tree_blocks_per_sm(int T) { return T == 128 ? SPD_TREE_BPS128 : (T == 256 ? 2 : 1); }

template <int T>
constexpr size_t tree_smem_bytes() {
    constexpr size_t C = 16 * T;
    return 2 * C * 4 + kStages * (C + 8) * 4 + 2 * T * 16 + kStages * 8;
}

template <int T, int K>
__global__ void __launch_bounds__(T, tree_blocks_per_sm(T)) spd_tree_kernel(const TreeParams p) {
    constexpr int C = 16 * T;
    constexpr int M = 1 << (K - 1);
    constexpr int GUARD = M > 8 ? M : 8;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float4* const pp = reinterpret_cast<float4*>(smem_raw);
    float* const stages = reinterpret_cast<float*>(smem_raw + 2 * C * 4);
    float4* const halo = reinterpret_cast<float4*>(stages + kStages * (C + 8));
    uint64_t* const bars = reinterpret_cast<uint64_t*>(halo + 2 * T);

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
    float* __restrict__ out_snr = p.out_snr + static_cast<long long>(d) * n_t;
    int32_t* __restrict__ out_width = p.out_width + static_cast<long long>(d) * n_t;
    const float mu = p.mean[d];
    const float inv = 1.0f / p.sigma[d];
    const uint32_t tm = p.tag_mask;

    for (int i = tid; i < 2 * T; i += T) halo[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    if (tid == 0) {
#pragma unroll
        for (int i = 0; i < kStages; ++i) mbar_init(&bars[i], 1);
        fence_mbar_init();
    }
    Delay dl;
    {
        const float4 z = make_float4(0.f, 0.f, 0.f, 0.f);
        dl.a = z;
        dl.b[0] = dl.b[1] = z;
#pragma unroll
        for (int r = 0; r < 4; ++r) dl.c[r] = dl.d0[r] = dl.d1[r] = z;
    }
    int xsel = 0, hsel = 0;
    __syncthreads();

    // ---- guarded steps: warm-up chunks of an interior segment, then the row tail -----
    for (int c = c_top - 1; c >= first_fast; --c) {
        const long long n0 = static_cast<long long>(c) * C;
        for (int i = tid; i < C + 8; i += T) {
            const long long n = n0 + i;
            stages[i] = n < n_t ? __ldg(row + n) : mu;
        }
        __syncthreads();
        tree_chunk<T, K, false>(reinterpret_cast<const float4*>(stages), pp, halo, xsel, hsel, dl, mu, inv, tm,
                                out_snr, out_width, n0, n_t, c < c_hi, tid);
        __syncthreads();
    }

    // ---- unguarded steps: bulk-copy ring ----------------------------------------------
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
    for (int it = 0; it < n_fast; ++it) {
        if (tid == 0) {
            const int nx = it + kStages - 1;
            if (nx < n_fast) {
                const int sx = stage == 0 ? kStages - 1 : stage - 1;  // (it + kStages - 1) % kStages
                mbar_arrive_expect_tx(&bars[sx], kBytes);
                bulk_g2s(stages + sx * (C + 8), row + static_cast<long long>(first_fast - 1 - nx) * C, kBytes,
                         &bars[sx]);
            }
        }
        mbar_wait(&bars[stage], phase);
        const long long n0 = static_cast<long long>(first_fast - 1 - it) * C;
        tree_chunk<T, K, true>(reinterpret_cast<const float4*>(stages + stage * (C + 8)), pp, halo, xsel, hsel,
                               dl, mu, inv, tm, out_snr, out_width, n0, n_t, true, tid);
        if (++stage == kStages) {
            stage = 0;
            phase ^= 1;
        }
    }
}

template <int T, int K>
cudaError_t launch_tree(const TreeConfig& cfg, const TreeParams& prm, int64_t n_dm, cudaStream_t stream) {
    const dim3 grid(static_cast<unsigned>(n_dm * cfg.segs_per_row));
    spd_tree_kernel<T, K><<<grid, T, cfg.smem_bytes, stream>>>(prm);
    return cudaGetLastError();
}

template <int T, int K>
cudaError_t prepare_tree(TreeConfig& cfg) {
    cfg.smem_bytes = tree_smem_bytes<T>();
    if (const char* env = std::getenv("SPD_TREE_PAD_SMEM")) cfg.smem_bytes += static_cast<size_t>(std::atoll(env));
    cudaError_t e = cudaFuncSetAttribute(spd_tree_kernel<T, K>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         static_cast<int>(cfg.smem_bytes));
    if (e != cudaSuccess) return e;
    int nb = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, spd_tree_kernel<T, K>, T, cfg.smem_bytes);
    if (e != cudaSuccess) return e;
    cfg.blocks_per_sm = nb;
    return cudaSuccess;
}

#define SPD_TREE_CASES(OP)      \
    OP(128, 1)                  \
    OP(128, 2)                  \
    OP(128, 3)                  \
    OP(128, 4)                  \
    OP(128, 5)                  \
    OP(128, 6)                  \
    OP(128, 7)                  \
    OP(128, 8)                  \
    OP(128, 9)                  \
    OP(128, 10)                 \
    OP(128, 11)                 \
    OP(128, 12)                 \
    OP(128, 13)                 \
    OP(128, 14)                 \
    OP(256, 15)                 \
    OP(512, 16)

constexpr int tree_threads_for(int K) { return K <= 14 ? 128 : (K == 15 ? 256 : 512); }

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
    cfg.T = tree_threads_for(cfg.K);
    cfg.chunk = 16 * cfg.T;
    cudaError_t e = cudaErrorInvalidValue;
#define SPD_PREP(TT, KK) \
    if (cfg.K == KK) e = prepare_tree<TT, KK>(cfg);
    SPD_TREE_CASES(SPD_PREP)
#undef SPD_PREP
    if (e != cudaSuccess) return cuda_fail(e, "configuring the dyadic-tree kernel");
    if (cfg.blocks_per_sm < 1) {
        set_error("dyadic-tree kernel does not fit on this device (K=%d, smem=%zu)", cfg.K, cfg.smem_bytes);
        return SPD_ERR_CUDA;
    }
    const int64_t C = cfg.chunk;
    const int64_t M = int64_t(1) << (cfg.K - 1);
    cfg.chunks_per_row = static_cast<int>((plan->n_t + C - 1) / C);
    cfg.warm_chunks = cfg.K >= 2 ? static_cast<int>((M - 1 + C - 1) / C) : 0;
    // Segments: enough independent streams to fill and balance the machine, each long
    // enough that replaying its look-ahead (warm_chunks) stays a few per cent.
    const int64_t slots = int64_t(plan->sm_count) * cfg.blocks_per_sm;
    int64_t segs = 1;
    const int64_t min_seg_chunks = std::max<int64_t>(16 * cfg.warm_chunks, 8);
    if (const char* env = std::getenv("SPD_SEGS_PER_ROW")) {
        segs = std::max<int64_t>(1, std::atoll(env));
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
             float* out_snr, int32_t* out_width, cudaStream_t stream) {
    const TreeConfig& cfg = plan->tree;
    TreeParams prm;
    prm.plane = plane;
    prm.mean = mean;
    prm.sigma = sigma;
    prm.out_snr = out_snr;
    prm.out_width = out_width;
    prm.n_t = plan->n_t;
    prm.chunks_per_row = cfg.chunks_per_row;
    prm.seg_chunks = cfg.seg_chunks;
    prm.segs_per_row = cfg.segs_per_row;
    prm.warm_chunks = cfg.warm_chunks;
    prm.tag_mask = ~kCodeMask;
    cudaError_t e = cudaErrorInvalidValue;
#define SPD_LAUNCH(TT, KK) \
    if (cfg.K == KK) e = launch_tree<TT, KK>(cfg, prm, n_dm, stream);
    SPD_TREE_CASES(SPD_LAUNCH)
#undef SPD_LAUNCH
    if (e != cudaSuccess) return cuda_fail(e, "launching the dyadic-tree kernel");
    return SPD_OK;
}

}  // namespace spd
