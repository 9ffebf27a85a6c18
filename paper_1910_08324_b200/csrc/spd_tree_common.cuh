// Shared by the streaming-tree kernels (spd_tree.cu: widths 2^k; spd_tree_ig.cu: widths 2^k and
// 3 * 2^m): launch parameters, PTX helpers (mbarrier, 1-D bulk copy, 3-input max), packed
// float4 arithmetic, width-index tags, geometry.  Internal to libspd_b200.so.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include <type_traits>

#include "spd_internal.h"

namespace spd {
namespace {

struct TreeParams {
    const float* plane;
    const float* mean;
    const float* sigma;
    float* out_snr;
    int32_t* out_width;
    uint32_t gmask[16];    // grid plans: separation of level k minus one (a power of two minus one); else unused
    const float* sigma_w;  // nullptr, or [n_dm][K] measured standard deviation per width (warp-stream kernel)
    uint8_t* activity;  // [n_dm][chunks_per_row] or nullptr
    float threshold;    // candidate threshold in SNR units (used only with activity)
    long long n_t;
    long long n_dm;  // rows of this launch (warp-stream kernel: pieces may span rows)
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
// Tensor memory as per-lane scratch (delay lines; no MMA anywhere): a warp reaches the 32
// lanes of its quarter (warp index mod 4), thread i lane i, with the 32x32b shapes below.
// ------------------------------------------------------------------------------------
// Allocation by one whole warp of the block: COLS = 32, 64, 128, 256 or 512 columns of all 128
// lanes; the base address lands in *slot (shared memory).  Freed by the same warp at the end.
template <int COLS>
__device__ __forceinline__ void tmem_alloc(uint32_t* slot) {
    static_assert(COLS == 32 || COLS == 64 || COLS == 128 || COLS == 256 || COLS == 512, "tmem columns");
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(slot)), "n"(COLS)
                 : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
template <int COLS>
__device__ __forceinline__ void tmem_dealloc(uint32_t base) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(base), "n"(COLS) : "memory");
}
__device__ __forceinline__ void tmem_fence_before_sync() {
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
}
__device__ __forceinline__ void tmem_fence_after_sync() {
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
}
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

// 8 float4 per lane <- 32 consecutive columns of the warp's lanes; complete on return.
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, float4 (&v)[8]) {
    uint32_t r[32];
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];\n"
        "tcgen05.wait::ld.sync.aligned;"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
          "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]),
          "=r"(r[16]), "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]),
          "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
        : "r"(taddr)
        : "memory");
#pragma unroll
    for (int i = 0; i < 8; ++i)
        v[i] = make_float4(__uint_as_float(r[4 * i]), __uint_as_float(r[4 * i + 1]), __uint_as_float(r[4 * i + 2]),
                           __uint_as_float(r[4 * i + 3]));
}
__device__ __forceinline__ void tmem_st32(uint32_t taddr, const float4 (&v)[8]) {
    uint32_t r[32];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        r[4 * i] = __float_as_uint(v[i].x);
        r[4 * i + 1] = __float_as_uint(v[i].y);
        r[4 * i + 2] = __float_as_uint(v[i].z);
        r[4 * i + 3] = __float_as_uint(v[i].w);
    }
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], "
        "{%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, "
        "%17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31, %32};" ::"r"(taddr),
        "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]), "r"(r[9]),
        "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15]), "r"(r[16]), "r"(r[17]), "r"(r[18]),
        "r"(r[19]), "r"(r[20]), "r"(r[21]), "r"(r[22]), "r"(r[23]), "r"(r[24]), "r"(r[25]), "r"(r[26]), "r"(r[27]),
        "r"(r[28]), "r"(r[29]), "r"(r[30]), "r"(r[31])
        : "memory");
}

__device__ __forceinline__ void tmem_ld8(uint32_t taddr, float4 (&v)[2]) {
    uint32_t r[8];
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];\n"
        "tcgen05.wait::ld.sync.aligned;"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
        : "r"(taddr)
        : "memory");
#pragma unroll
    for (int i = 0; i < 2; ++i)
        v[i] = make_float4(__uint_as_float(r[4 * i]), __uint_as_float(r[4 * i + 1]), __uint_as_float(r[4 * i + 2]),
                           __uint_as_float(r[4 * i + 3]));
}
__device__ __forceinline__ void tmem_st8(uint32_t taddr, const float4 (&v)[2]) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"r"(taddr),
                 "r"(__float_as_uint(v[0].x)), "r"(__float_as_uint(v[0].y)), "r"(__float_as_uint(v[0].z)),
                 "r"(__float_as_uint(v[0].w)), "r"(__float_as_uint(v[1].x)), "r"(__float_as_uint(v[1].y)),
                 "r"(__float_as_uint(v[1].z)), "r"(__float_as_uint(v[1].w))
                 : "memory");
}
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, float4 (&v)[4]) {
    uint32_t r[16];
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];\n"
        "tcgen05.wait::ld.sync.aligned;"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
          "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
        : "r"(taddr)
        : "memory");
#pragma unroll
    for (int i = 0; i < 4; ++i)
        v[i] = make_float4(__uint_as_float(r[4 * i]), __uint_as_float(r[4 * i + 1]), __uint_as_float(r[4 * i + 2]),
                           __uint_as_float(r[4 * i + 3]));
}
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const float4 (&v)[4]) {
    uint32_t r[16];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        r[4 * i] = __float_as_uint(v[i].x);
        r[4 * i + 1] = __float_as_uint(v[i].y);
        r[4 * i + 2] = __float_as_uint(v[i].z);
        r[4 * i + 3] = __float_as_uint(v[i].w);
    }
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], "
        "{%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};" ::"r"(taddr),
        "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]), "r"(r[9]),
        "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15])
        : "memory");
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
// x - mu (eq. 4 numerator per sample; sums of mean-free data never cancel later).  The
// division by sigma is applied once per output sample at the store, not per input sample.
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
    const float4 v = k == 0 ? p : scale4(p, level_scale<k>());  // x * 1.0f is not folded by the compiler
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

// Run-time scale per level (a measured standard deviation per width, instead of
// eq. (5)'s 2^(-k/2) / sigma): ls[k] = 1 / sigma_{d, 2^k}, the same tag and max.
template <int k, bool FAST>
__device__ __forceinline__ float4 keyx_rt(float4 p, int lim, uint32_t tm, float s) {
    const float4 v = scale4(p, s);
    float4 q = make_float4(pack1<k>(v.x, tm), pack1<k>(v.y, tm), pack1<k>(v.z, tm), pack1<k>(v.w, tm));
    if constexpr (!FAST) {
        const int w = 1 << k;
        const float ninf = __int_as_float(0xff800000);
        if (w > lim) q.x = ninf;
        if (w > lim - 1) q.y = ninf;
        if (w > lim - 2) q.z = ninf;
        if (w > lim - 3) q.w = ninf;
    }
    return q;
}
template <int j, int K, bool FAST>
__device__ __forceinline__ void fold_rt(float4& best, float4 before, float4 now, int lim, uint32_t tm,
                                        const float (&ls)[32]) {
    if constexpr (j >= 3) {
        if constexpr ((j & 1) == 0) {
            best = max4(best, keyx_rt<j - 1, FAST>(before, lim, tm, ls[j - 1]), keyx_rt<j, FAST>(now, lim, tm, ls[j]));
        } else if constexpr (j == K - 1) {
            best = max4(best, keyx_rt<j, FAST>(now, lim, tm, ls[j]));
        }
    }
}

// Shared-memory store of a float4, issued as two 64-bit halves in PTX.  The sums are produced
// by packed FADD2 into register PAIRS; written as one 128-bit store the allocator spends up to
// four register moves per store on forming an aligned QUAD.  ptxas re-merges the halves into
// one STS.128 but no longer needs the moves (7 -> 2 moves per sample).
__device__ __forceinline__ void st_shared4(float4* dst, float4 v) {
    const uint32_t a = smem_u32(dst);
    asm volatile("st.shared.v2.f32 [%0], {%1, %2};" ::"r"(a), "f"(v.x), "f"(v.y) : "memory");
    asm volatile("st.shared.v2.f32 [%0+8], {%1, %2};" ::"r"(a), "f"(v.z), "f"(v.w) : "memory");
}

// The chunk loop is unrolled over the delay FIFOs up to this factor: a FIFO no deeper than
// the unroll gets a compile-time slot (no register moves), a deeper one is rotated by moves.
// Code size grows with the factor; past the instruction cache the kernel stalls on fetch
// (T = 64, R = 4 unrolled x4: smsp stall_no_instruction 2.6 per issue).
constexpr int kTreeMaxUnroll = 2;
// Block-per-stream dyadic kernel (spd_tree.cu): delay FIFOs in tensor memory from this depth on.
constexpr bool tree_tmem(int K) { return K >= 15; }
constexpr int tree_max_unroll(int K) { return K == 16 ? 4 : kTreeMaxUnroll; }

constexpr int ilog2(int v) { return v <= 1 ? 0 : 1 + ilog2(v / 2); }
constexpr int imax(int a, int b) { return a > b ? a : b; }

// Geometry of one kernel instantiation.
template <int T, int R, int K>
struct Geo {
    static constexpr int LT = ilog2(T);
    static constexpr int C4 = R * T;   // float4 per chunk
    static constexpr int C = 4 * C4;   // samples per chunk
    static constexpr int LAST = K - 1;  // highest level: width 2^LAST
    // In-register levels j = 0 .. J-1: partner 2^j rows later, produces level LT + 3 + j.
    static constexpr int J = imax(0, LAST - LT - 2);
    static constexpr int ND = (1 << J) - 1;  // float4 of delay registers: sum of 2^j
    // Depth, in chunks, of the deepest delay FIFO = unroll factor of the chunk loop.
    static constexpr int TOPQ = J > 0 ? imax(1, (1 << (J - 1)) / R) : 1;
    static constexpr int U = TOPQ < tree_max_unroll(K) ? TOPQ : tree_max_unroll(K);
};

struct ChunkCtx {
    float mu, inv;
    uint32_t tm;
    float* __restrict__ out_snr;
    int32_t* __restrict__ out_width;
    long long n0, n_t;
    bool do_out;
    int tid;
    uint32_t gmask[16];  // boxcar separation per level minus one (kernels instantiated for a grid plan)
    float ls[32];    // run-time scale per width index (kernels instantiated for a sigma per width)
    uint32_t tbase;  // tensor-memory base of this thread's delay FIFOs (kernels that keep them there)
    int it;          // steps done on this stream (FIFO slot = it mod depth)
};

// Compile-time loop over the phases of the unrolled chunk loop.
template <int PH, int U, typename F>
__device__ __forceinline__ void static_phases(F&& f) {
    if constexpr (PH < U) {
        f(std::integral_constant<int, PH>{});
        static_phases<PH + 1, U>(f);
    }
}


}  // namespace
}  // namespace spd
