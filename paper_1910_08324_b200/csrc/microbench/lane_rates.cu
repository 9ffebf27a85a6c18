// lane_rates.cu - register-only microbenchmarks behind the "ALU-pipe roofline" of DESIGN.md sec. 7b.
//
// Not part of libspd_b200.so (the build compiles csrc/*.cu only).  Build and run on a B200:
//
//     nvcc -O3 -std=c++17 -gencode arch=compute_100a,code=sm_100a -o lane_rates lane_rates.cu && ./lane_rates
//
// Part 1: reciprocal throughput (clocks per warp instruction per SM sub-partition) of the instruction kinds
// the tree kernels are made of, 16 independent chains per thread, 16 warps per SM.
// Part 2: the per-level instruction mix of the kernels - per float4 and level: 2 FADD2 (the partial sum),
// 2 FMUL2 (the sqrt(width) scale), 4 LOP3 (the width tag), 2 FMNMX3 (the running maximum over two levels) -
// and variants of it, in clocks per float4-level per sub-partition.  LOP3 and FMNMX3 share the half-rate ALU
// pipe (two clocks each: 12 clocks for the mix), the packed FP32 instructions the FMA pipe (two clocks each:
// 8.2 clocks); the two pipes overlap only in part: the mix measures 15.9 clocks whatever the number of resident
// warps, 15.5 without the multiplies (the ALU pipe binds) and 10.2-10.8 without the tags.
#include <cstdint>
#include <cstdio>
#include <cuda_runtime.h>

__device__ __forceinline__ float fmax3(float a, float b, float c) {
    float d;
    asm volatile("max.f32 %0, %1, %2, %3;" : "=f"(d) : "f"(a), "f"(b), "f"(c));
    return d;
}

template <int OP>
__global__ void __launch_bounds__(256) rate_kernel(float* out, unsigned tm, float c0, int iters) {
    float v[16];
    for (int i = 0; i < 16; ++i) v[i] = threadIdx.x * 0.001f + i;
    const float w = c0 + threadIdx.x;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 16; ++i) {
            if (OP == 0) v[i] = fmax3(v[i], v[(i + 1) & 15], w);
            if (OP == 1) asm volatile("max.f32 %0, %0, %1;" : "+f"(v[i]) : "f"(w));
            if (OP == 2) asm volatile("max.f32 %0, %0, %1;" : "+f"(v[i]) : "f"(v[(i + 5) & 15]));
            if (OP == 3) { unsigned u = __float_as_uint(v[i]); asm volatile("lop3.b32 %0, %0, %1, 17, 0xec;" : "+r"(u) : "r"(tm)); v[i] = __uint_as_float(u); }
            if (OP == 4) asm volatile("add.f32 %0, %0, %1;" : "+f"(v[i]) : "f"(v[(i + 5) & 15]));
            if (OP == 5) asm volatile("mul.f32 %0, %0, 0f3F3504F3;" : "+f"(v[i]));
            if (OP == 6) { unsigned u = __float_as_uint(v[i]); asm volatile("add.u32 %0, %0, %1;" : "+r"(u) : "r"(__float_as_uint(v[(i + 5) & 15]))); v[i] = __uint_as_float(u); }
            if (OP == 7) { unsigned u = __float_as_uint(v[i]); asm volatile("prmt.b32 %0, %0, %1, 0x3214;" : "+r"(u) : "r"(tm)); v[i] = __uint_as_float(u); }
            if (OP == 8) { unsigned u = __float_as_uint(v[i]); asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(u) : "r"(tm), "r"(__float_as_uint(w))); v[i] = __uint_as_float(u); }
        }
        if (OP == 9 || OP == 10) {
#pragma unroll
            for (int i = 0; i < 16; i += 2) {
                float2 a = make_float2(v[i], v[i + 1]);
                if (OP == 9) a = __fadd2_rn(a, make_float2(w, w));
                if (OP == 10) a = __fmul2_rn(a, make_float2(0.70710678f, 0.70710678f));
                v[i] = a.x;
                v[i + 1] = a.y;
            }
        }
    }
    float s = 0.f;
    for (int i = 0; i < 16; ++i) s += v[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

static double sm_clock_hz() {
    int khz = 0;
    cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, 0);
    return khz * 1e3;
}

template <int OP>
static void rate(const char* name, int per_iter) {
    float* out;
    cudaMalloc(&out, 148 * 2 * 256 * 4);
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const int iters = 100000;
    rate_kernel<OP><<<148 * 2, 256>>>(out, 0xffffffe0u, 1.0f, 10);
    cudaEventRecord(e0);
    rate_kernel<OP><<<148 * 2, 256>>>(out, 0xffffffe0u, 1.0f, iters);
    cudaEventRecord(e1);
    cudaEventSynchronize(e1);
    float ms;
    cudaEventElapsedTime(&ms, e0, e1);
    printf("%-34s %.2f clk per warp instruction per sub-partition\n", name, ms * 1e-3 * sm_clock_hz() / (double(per_iter) * iters * 16 / 4));
    cudaFree(out);
}

template <bool PK>
__device__ __forceinline__ float4 add4(float4 a, float4 b) {
    if (PK) {
        const float2 lo = __fadd2_rn(make_float2(a.x, a.y), make_float2(b.x, b.y));
        const float2 hi = __fadd2_rn(make_float2(a.z, a.w), make_float2(b.z, b.w));
        return make_float4(lo.x, lo.y, hi.x, hi.y);
    }
    return make_float4(a.x + b.x, a.y + b.y, a.z + b.z, a.w + b.w);
}
template <bool PK>
__device__ __forceinline__ float4 mul4(float4 p, float c) {
    if (PK) {
        const float2 cc = make_float2(c, c);
        const float2 lo = __fmul2_rn(make_float2(p.x, p.y), cc);
        const float2 hi = __fmul2_rn(make_float2(p.z, p.w), cc);
        return make_float4(lo.x, lo.y, hi.x, hi.y);
    }
    return make_float4(p.x * c, p.y * c, p.z * c, p.w * c);
}
__device__ __forceinline__ float tag(float v, uint32_t tm, uint32_t code) {
    return __uint_as_float((__float_as_uint(v) & tm) | code);
}
// PK: packed adds and multiplies; TAG: width tags; MUL: the scale multiply; the running maximum is always the 3-input one.
template <bool PK, bool TAG, bool MUL>
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
                const float4 n1 = add4<PK>(P[r], Q[r]);
                const float4 n2 = add4<PK>(n1, Q[(r + 1) & 3]);
                float4 a = n1, b = n2;
                if (MUL) {
                    a = mul4<PK>(n1, 0.70710678f);
                    b = mul4<PK>(n2, 0.5f);
                }
                if (TAG) {
                    a = make_float4(tag(a.x, tm, 31u - lv), tag(a.y, tm, 31u - lv), tag(a.z, tm, 31u - lv), tag(a.w, tm, 31u - lv));
                    b = make_float4(tag(b.x, tm, 30u - lv), tag(b.y, tm, 30u - lv), tag(b.z, tm, 30u - lv), tag(b.w, tm, 30u - lv));
                }
                best[r] = make_float4(fmax3(best[r].x, a.x, b.x), fmax3(best[r].y, a.y, b.y), fmax3(best[r].z, a.z, b.z),
                                      fmax3(best[r].w, a.w, b.w));
                Q[r] = P[r];
                P[r] = n2;
            }
        }
    }
    float s = 0.f;
    for (int r = 0; r < 4; ++r) s += best[r].x + best[r].y + best[r].z + best[r].w + P[r].x;
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}
template <bool PK, bool TAG, bool MUL>
static void mix(const char* name) {
    float* out;
    cudaMalloc(&out, 148 * 3 * 256 * 4);
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const int iters = 20000;
    for (int bps = 1; bps <= 3; ++bps) {
        mix_kernel<PK, TAG, MUL><<<148 * bps, 256>>>(out, 0xffffffe0u, 10);
        cudaEventRecord(e0);
        mix_kernel<PK, TAG, MUL><<<148 * bps, 256>>>(out, 0xffffffe0u, iters);
        cudaEventRecord(e1);
        cudaEventSynchronize(e1);
        float ms;
        cudaEventElapsedTime(&ms, e0, e1);
        printf("%-44s %2d warps per SM: %.2f clk per float4-level per sub-partition\n", name, 8 * bps,
               ms * 1e-3 * sm_clock_hz() / (14.0 * 4 * iters * (8 * bps) / 4));
    }
    cudaFree(out);
}

int main() {
    printf("SM clock used for the conversion: %.0f MHz (cudaDevAttrClockRate)\n", sm_clock_hz() / 1e6);
    rate<0>("FMNMX3 (max of three)", 16);
    rate<1>("FMNMX, one operand reused", 16);
    rate<2>("FMNMX, two fresh registers", 16);
    rate<3>("LOP3 (v & mask) | imm", 16);
    rate<4>("FADD, two fresh registers", 16);
    rate<5>("FMUL by an immediate", 16);
    rate<6>("IADD, two fresh registers", 16);
    rate<7>("PRMT", 16);
    rate<8>("IMAD", 16);
    rate<9>("FADD2 (packed pair)", 8);
    rate<10>("FMUL2 by an immediate (packed pair)", 8);
    mix<true, true, true>("FADD2 FMUL2 LOP3 FMNMX3 (the kernels' mix)");
    mix<true, false, true>("FADD2 FMUL2      FMNMX3 (no tags)");
    mix<true, true, false>("FADD2       LOP3 FMNMX3 (no multiplies)");
    mix<false, true, true>("FADD  FMUL  LOP3 FMNMX3 (scalar FP32)");
    return 0;
}
