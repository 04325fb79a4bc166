// probe_fma_peak.cu -- standalone microbenchmark behind the ALU roofline peak of DESIGN.md section 6 (not part of libadock.so):
// FFMA2-only, FFMA-only and mixed dependent chains; reports FMA lanes per clock and SM.  profiles/r01d_fma_peak.md
#include <cstdio>
#include <cuda_runtime.h>
typedef unsigned long long u64;
__device__ __forceinline__ u64 fma2(u64 a, u64 b, u64 c) { u64 d; asm volatile("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d; }
__device__ __forceinline__ float fma1(float a, float b, float c) { float d; asm volatile("fma.rn.f32 %0, %1, %2, %3;" : "=f"(d) : "f"(a), "f"(b), "f"(c)); return d; }
template <int NP, int NS>   // NP packed chains, NS scalar chains per thread
__global__ void k(float* out, int iters, float seed) {
    u64 p[NP > 0 ? NP : 1]; float s[NS > 0 ? NS : 1];
    for (int i = 0; i < NP; ++i) p[i] = (u64)__float_as_uint(seed + i) | ((u64)__float_as_uint(seed - i) << 32);
    for (int i = 0; i < NS; ++i) s[i] = seed * (i + 1);
    const u64 a = (u64)__float_as_uint(0.999f) | ((u64)__float_as_uint(1.001f) << 32), b = (u64)__float_as_uint(1e-3f) | ((u64)__float_as_uint(-1e-3f) << 32);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 4; ++r) {
#pragma unroll
            for (int i = 0; i < NP; ++i) p[i] = fma2(p[i], a, b);
#pragma unroll
            for (int i = 0; i < NS; ++i) s[i] = fma1(s[i], 0.999f, 1e-3f);
        }
    }
    float acc = 0;
    for (int i = 0; i < NP; ++i) acc += __uint_as_float((unsigned)p[i]) + __uint_as_float((unsigned)(p[i] >> 32));
    for (int i = 0; i < NS; ++i) acc += s[i];
    if (acc == 12345.678f) out[0] = acc;
}
template <int NP, int NS>
void run(const char* name, int warps_per_sm) {
    float* d; cudaMalloc(&d, 4);
    int sms; cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, 0);
    int clk; cudaDeviceGetAttribute(&clk, cudaDevAttrClockRate, 0);
    const int iters = 20000;
    dim3 grid(sms), block(32 * warps_per_sm);
    k<NP, NS><<<grid, block>>>(d, 100, 1.0f);
    cudaEvent_t a, b; cudaEventCreate(&a); cudaEventCreate(&b);
    cudaEventRecord(a);
    k<NP, NS><<<grid, block>>>(d, iters, 1.0f);
    cudaEventRecord(b); cudaEventSynchronize(b);
    float ms; cudaEventElapsedTime(&ms, a, b);
    const double lanes = (double)sms * warps_per_sm * 32 * iters * 4 * (2.0 * NP + NS);
    const double cycles = ms * 1e-3 * clk * 1e3;
    printf("%-28s warps/SM %2d: %.3f ms  %.1f FMA lanes/clk/SM  (%.1f TFLOP/s)\n", name, warps_per_sm, ms, lanes / cycles / sms, 2 * lanes / (ms * 1e-3) / 1e12);
    cudaFree(d);
}
int main() {
    for (int w : {8, 16, 32}) {
        if (w == 8) { run<8, 0>("FFMA2 x8", 8); run<0, 8>("FFMA x8", 8); run<4, 8>("FFMA2 x4 + FFMA x8", 8); run<8, 8>("FFMA2 x8 + FFMA x8", 8); run<8, 4>("FFMA2 x8 + FFMA x4", 8); }
        if (w == 16) { run<8, 0>("FFMA2 x8", 16); run<0, 8>("FFMA x8", 16); run<4, 8>("FFMA2 x4 + FFMA x8", 16); run<8, 8>("FFMA2 x8 + FFMA x8", 16); }
        if (w == 32) { run<8, 0>("FFMA2 x8", 32); run<0, 8>("FFMA x8", 32); run<4, 8>("FFMA2 x4 + FFMA x8", 32); }
    }
    return 0;
}
