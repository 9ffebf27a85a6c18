// tag_variants.cu - register-only microbenchmark: can the width tag of a key leave the half-rate ALU pipe?
// (per key the tree kernels spend one LOP3 - (v & mask) | code - and half an FMNMX3 there.)
//
// Not part of libspd_b200.so (the build compiles csrc/*.cu only).  Build and run on a B200:
//
//     nvcc -O3 -std=c++17 -gencode arch=compute_100a,code=sm_100a -o tag_variants tag_variants.cu && ./tag_variants
//
// Variants of the per-level mix (per float4 and level: 2 FADD2 for the sum, then scale + tag + 3-input maximum):
//   LOP3     key = (p * s + C0') & mask | code        FFMA2 + 2 LOP3 per pair of values (today's cost)
//   FMA tag  t = p * s + C1 rounds the scaled value to 16 ulp of C0's binade (C1's binade is 16 times coarser),
//            key = t + (C0 - C1 + code * ulp) is exact: FFMA2 + FADD2 per pair, nothing on the ALU pipe.
//            A FIXED-POINT key: SNR quantum 16 ulp of C0's binade, and the value must stay inside one binade
//            ([32, 64) here: SNR in [-4, 28)) - the price that keeps this out of the library.
//   IMAD     t = sat(p * s' + c) in [0, 1], key = bits(t) * 16 + code, unsigned 3-input maximum.
// MASK selects, per level, which of the first two is used.
#include <cstdint>
#include <cstdio>
#include <cuda_runtime.h>

__device__ __forceinline__ float fmax3(float a, float b, float c) {
    float d;
    asm volatile("max.f32 %0, %1, %2, %3;" : "=f"(d) : "f"(a), "f"(b), "f"(c));
    return d;
}
__device__ __forceinline__ float4 add4(float4 a, float4 b) {
    const float2 lo = __fadd2_rn(make_float2(a.x, a.y), make_float2(b.x, b.y));
    const float2 hi = __fadd2_rn(make_float2(a.z, a.w), make_float2(b.z, b.w));
    return make_float4(lo.x, lo.y, hi.x, hi.y);
}
__device__ __forceinline__ float4 fma4(float4 p, float s, float c) {
    const float2 ss = make_float2(s, s), cc = make_float2(c, c);
    const float2 lo = __ffma2_rn(make_float2(p.x, p.y), ss, cc);
    const float2 hi = __ffma2_rn(make_float2(p.z, p.w), ss, cc);
    return make_float4(lo.x, lo.y, hi.x, hi.y);
}
__device__ __forceinline__ float4 addc4(float4 p, float c) {
    const float2 cc = make_float2(c, c);
    const float2 lo = __fadd2_rn(make_float2(p.x, p.y), cc);
    const float2 hi = __fadd2_rn(make_float2(p.z, p.w), cc);
    return make_float4(lo.x, lo.y, hi.x, hi.y);
}
__device__ __forceinline__ float tagf(float v, uint32_t tm, uint32_t code) {
    return __uint_as_float((__float_as_uint(v) & tm) | code);
}
__device__ __forceinline__ float4 tag4(float4 a, uint32_t tm, uint32_t code) {
    return make_float4(tagf(a.x, tm, code), tagf(a.y, tm, code), tagf(a.z, tm, code), tagf(a.w, tm, code));
}
constexpr float kC0 = 36.0f;             // keys live in [32, 64): SNR + 36
constexpr float kU0 = 1.0f / 262144.0f;  // ulp of [32, 64) = 2^-18
constexpr float kC1 = 1536.0f;           // a coarser binade for the rounding step (timing only: 32 times coarser)

template <uint32_t MASK, bool SCALAR>
__device__ __forceinline__ float4 key(float4 p, int lv, float s, uint32_t tm) {
    const uint32_t code = 15u - lv;
    if ((MASK >> lv) & 1u) {
        const float D = (kC0 - kC1) + code * kU0;
        if (SCALAR) {
            const float4 t = make_float4(fmaf(p.x, s, kC1), fmaf(p.y, s, kC1), fmaf(p.z, s, kC1), fmaf(p.w, s, kC1));
            return make_float4(t.x + D, t.y + D, t.z + D, t.w + D);
        }
        return addc4(fma4(p, s, kC1), D);
    }
    const float Cb = kC0 + 8 * kU0;
    if (SCALAR) {
        const float4 t = make_float4(fmaf(p.x, s, Cb), fmaf(p.y, s, Cb), fmaf(p.z, s, Cb), fmaf(p.w, s, Cb));
        return tag4(t, tm, code);
    }
    return tag4(fma4(p, s, Cb), tm, code);
}
__device__ constexpr float kScale[14] = {1.f, 0.70710678f, 0.5f, 0.35355339f, 0.25f, 0.17677670f, 0.125f,
                                         0.088388348f, 0.0625f, 0.044194174f, 0.03125f, 0.022097087f, 0.015625f,
                                         0.011048543f};
template <uint32_t MASK, bool SCALAR>
__global__ void __launch_bounds__(256) mix_kernel(float* out, uint32_t tm, int iters) {
    float4 P[4], Q[4], best[4];
    for (int r = 0; r < 4; ++r) {
        P[r] = make_float4(threadIdx.x + r, 1.f, 2.f, 3.f);
        Q[r] = make_float4(0.5f, threadIdx.x * 0.25f, 2.f, r);
        best[r] = make_float4(-1e30f, -1e30f, -1e30f, -1e30f);
    }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int lv = 0; lv < 14; lv += 2) {
#pragma unroll
            for (int r = 0; r < 4; ++r) {
                const float4 n1 = add4(P[r], Q[r]);
                const float4 n2 = add4(n1, Q[(r + 1) & 3]);
                const float4 a = key<MASK, SCALAR>(n1, lv, kScale[lv], tm);
                const float4 b = key<MASK, SCALAR>(n2, lv + 1, kScale[lv + 1], tm);
                best[r] = make_float4(fmax3(best[r].x, a.x, b.x), fmax3(best[r].y, a.y, b.y),
                                      fmax3(best[r].z, a.z, b.z), fmax3(best[r].w, a.w, b.w));
                Q[r] = P[r];
                P[r] = n2;
            }
        }
    }
    float s = 0.f;
    for (int r = 0; r < 4; ++r) s += best[r].x + best[r].y + best[r].z + best[r].w + P[r].x;
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}
__global__ void __launch_bounds__(256) mix_imad_kernel(float* out, float cc, uint32_t sixteen, int iters) {
    float4 P[4], Q[4];
    uint4 best[4];
    for (int r = 0; r < 4; ++r) {
        P[r] = make_float4(threadIdx.x + r, 1.f, 2.f, 3.f);
        Q[r] = make_float4(0.5f, threadIdx.x * 0.25f, 2.f, r);
        best[r] = make_uint4(0, 0, 0, 0);
    }
    auto k1 = [&](float p, float s, uint32_t code) {
        float t;
        asm("fma.rn.sat.f32 %0, %1, %2, %3;" : "=f"(t) : "f"(p), "f"(s * (1.0f / 4096.0f)), "f"(cc));
        uint32_t k;
        asm("mad.lo.u32 %0, %1, %2, %3;" : "=r"(k) : "r"(__float_as_uint(t)), "r"(sixteen), "r"(code));
        return k;
    };
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int lv = 0; lv < 14; lv += 2) {
#pragma unroll
            for (int r = 0; r < 4; ++r) {
                const float4 n1 = add4(P[r], Q[r]);
                const float4 n2 = add4(n1, Q[(r + 1) & 3]);
                const uint32_t ca = 15u - lv, cb = 14u - lv;
                best[r].x = max(best[r].x, max(k1(n1.x, kScale[lv], ca), k1(n2.x, kScale[lv + 1], cb)));
                best[r].y = max(best[r].y, max(k1(n1.y, kScale[lv], ca), k1(n2.y, kScale[lv + 1], cb)));
                best[r].z = max(best[r].z, max(k1(n1.z, kScale[lv], ca), k1(n2.z, kScale[lv + 1], cb)));
                best[r].w = max(best[r].w, max(k1(n1.w, kScale[lv], ca), k1(n2.w, kScale[lv + 1], cb)));
                Q[r] = P[r];
                P[r] = n2;
            }
        }
    }
    float s = 0.f;
    for (int r = 0; r < 4; ++r) s += float(best[r].x + best[r].y + best[r].z + best[r].w) + P[r].x;
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}
static double sm_clock_hz() {
    int khz = 0;
    cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, 0);
    return khz * 1e3;
}
template <typename F>
static void run(const char* name, F launch) {
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const int iters = 20000;
    for (int bps = 1; bps <= 2; ++bps) {
        launch(bps, 10);
        cudaEventRecord(e0);
        launch(bps, iters);
        cudaEventRecord(e1);
        cudaEventSynchronize(e1);
        float ms;
        cudaEventElapsedTime(&ms, e0, e1);
        printf("%-52s %2d warps per SM: %.2f clk per float4-level per sub-partition\n", name, 8 * bps,
               ms * 1e-3 * sm_clock_hz() / (14.0 * 4 * iters * (8 * bps) / 4));
    }
}
int main() {
    float* out;
    cudaMalloc(&out, 148 * 3 * 256 * 4);
    const uint32_t tm = 0xfffffff0u;
#define MIX(MASK, SC, NAME) run(NAME, [&](int bps, int it) { mix_kernel<MASK, SC><<<148 * bps, 256>>>(out, tm, it); })
    MIX(0x0000u, false, "FFMA2+LOP3 all levels (today's cost)");
    MIX(0x3fffu, false, "FFMA2+FADD2 all levels");
    MIX(0x2aaau, false, "FFMA2+FADD2 odd levels, LOP3 even (1/2)");
    MIX(0x2492u, false, "FFMA2+FADD2 on 5 of 14 levels (lv%3==1)");
    MIX(0x36dbu, false, "FFMA2+FADD2 on 10 of 14 levels (lv%3!=2)");
    MIX(0x3fffu, true, "scalar FFMA+FADD all levels");
    MIX(0x2aaau, true, "scalar FFMA+FADD odd levels, LOP3 even");
    run("FFMA.SAT + IMAD + unsigned max all levels",
        [&](int bps, int it) { mix_imad_kernel<<<148 * bps, 256>>>(out, 0.001953125f, 16u, it); });
    cudaDeviceSynchronize();
    printf("%s\n", cudaGetErrorString(cudaGetLastError()));
    return 0;
}
