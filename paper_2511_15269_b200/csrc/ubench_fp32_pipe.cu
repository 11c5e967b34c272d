// ubench_fp32_pipe.cu -- stand-alone micro-benchmark of the FP32 pipe of one B200 for the instruction mixes of the P2P kernel
// (p2p_fast.cu): scalar FFMA, packed FFMA2 / FADD2 / FMUL2, MUFU.RSQ and the FSETP/FSEL mask, registers only, 1..8 warps per
// scheduler.  It backs the FP32 peak used as roofline denominator (148 SM x 128 lanes x 2 flop x clock)
// and the "what binds the P2P" paragraph there.  Build and run:  python -m paper_2511_15269_b200.build --ubench &&
// paper_2511_15269_b200/ubench_fp32_pipe      (results: profiles/r01_fp32_pipe_microbench.md)
#include <cstdio>
#include <cuda_runtime.h>
typedef unsigned long long u64;
__device__ __forceinline__ u64 fma2(u64 a, u64 b, u64 c) { u64 r; asm volatile("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }
__device__ __forceinline__ u64 add2(u64 a, u64 b) { u64 r; asm volatile("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ u64 mul2(u64 a, u64 b) { u64 r; asm volatile("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ float fma1(float a, float b, float c) { float r; asm volatile("fma.rn.f32 %0, %1, %2, %3;" : "=f"(r) : "f"(a), "f"(b), "f"(c)); return r; }
__device__ __forceinline__ float rsq(float x) { float r; asm volatile("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ u64 pk(float lo, float hi) { u64 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ void upk(u64 v, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }

// MODE 0: 8 independent FFMA2 chains; 1: 16 scalar FFMA chains; 2: 8 FFMA2 + 8 FFMA interleaved; 3: 8 FFMA2 + 2 MUFU per 8; 4: FADD2 only
// 5: 8 FFMA2 + 4 MUFU + 4 FSEL-ish (p2p-like ratios: 13 packed : 2 mufu : 4 alu)
template <int MODE>
__global__ void k(float* out, int iters, float s) {
    u64 a[8], x[8], y[8]; float b[16];
    for (int i = 0; i < 8; ++i) { x[i] = pk(s + threadIdx.x * 0.25f + i, s - i); y[i] = pk(s * (i + 1) + threadIdx.x, s * 2 * i - threadIdx.x); }
    for (int i = 0; i < 8; ++i) a[i] = pk(threadIdx.x + i, threadIdx.x - i);
    for (int i = 0; i < 16; ++i) b[i] = threadIdx.x * 0.5f + i;
    const u64 m = pk(s, s * 0.5f), c = pk(0.25f, 0.125f);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            if (MODE == 0) {
#pragma unroll
                for (int i = 0; i < 8; ++i) a[i] = fma2(a[i], m, c);
            } else if (MODE == 1) {
#pragma unroll
                for (int i = 0; i < 16; ++i) b[i] = fma1(b[i], s, 0.25f);
            } else if (MODE == 2) {
#pragma unroll
                for (int i = 0; i < 8; ++i) { a[i] = fma2(a[i], m, c); b[i] = fma1(b[i], s, 0.25f); }
            } else if (MODE == 3) {
#pragma unroll
                for (int i = 0; i < 8; ++i) { a[i] = fma2(a[i], m, c); if (i % 4 == 0) b[i] = rsq(b[i]); }
            } else if (MODE == 4) {
#pragma unroll
                for (int i = 0; i < 8; ++i) a[i] = add2(a[i], m);
            } else if (MODE == 6) {
#pragma unroll
                for (int i = 0; i < 8; ++i) a[i] = mul2(a[i], m);
            } else if (MODE == 7) {  // p2p mix: 4 add2, 4 mul2, 5 fma2
#pragma unroll
                for (int i = 0; i < 4; ++i) a[i] = add2(a[i], m);
#pragma unroll
                for (int i = 0; i < 4; ++i) a[4 + i] = mul2(a[4 + i], m);
#pragma unroll
                for (int i = 0; i < 5; ++i) a[i] = fma2(a[i], m, c);
            } else if (MODE == 8) {  // three distinct register pairs per instruction (register-file bandwidth)
#pragma unroll
                for (int i = 0; i < 8; ++i) a[i] = fma2(x[i], y[i], a[i]);
            } else if (MODE == 5) {
#pragma unroll
                for (int i = 0; i < 13; ++i) a[i % 8] = fma2(a[i % 8], m, c);
                b[0] = rsq(b[0]); b[1] = rsq(b[1]);
                b[2] = b[0] >= 1e-38f ? b[2] : 0.f; b[3] = b[1] >= 1e-38f ? b[3] : 0.f;
            }
        }
    }
    float r = 0;
    for (int i = 0; i < 8; ++i) { float p0, p1; upk(a[i], p0, p1); r += p0 + p1; upk(x[i], p0, p1); r += p0 + p1; upk(y[i], p0, p1); r += p0 + p1; }
    for (int i = 0; i < 16; ++i) r += b[i];
    if (r == 12345.678f) out[0] = r;
}
template <int MODE>
void run(const char* name, double lane_ops_per_iter_thread, int wps) {
    float* d; cudaMalloc(&d, 4);
    const int iters = 4096;
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    int blocks = 148 * wps / 4 * 4;  // 128-thread CTAs: wps*4 warps per SM => wps*... keep simple: CTAs per SM = wps
    k<MODE><<<148 * wps, 128>>>(d, 16, 1.0001f);
    cudaEventRecord(e0);
    k<MODE><<<148 * wps, 128>>>(d, iters, 1.0001f);
    cudaEventRecord(e1); cudaEventSynchronize(e1);
    float ms; cudaEventElapsedTime(&ms, e0, e1);
    double ops = (double)148 * wps * 128 * iters * 4 * lane_ops_per_iter_thread;
    printf("%-40s warps/SMSP %d: %.3f ms, %.1f lane-ops/clk/SM (peak 128) at 1965 MHz\n", name, wps, ms, ops / (ms * 1e-3) / 1.965e9 / 148);
    (void)blocks;
}
int main() {
    for (int wps : {1, 2, 4, 8}) {
        run<0>("FFMA2 x8 chains", 16, wps);
        run<1>("FFMA x16 chains", 16, wps);
        run<2>("FFMA2 x8 + FFMA x8", 24, wps);
        run<3>("FFMA2 x8 + 2 MUFU", 16, wps);
        run<4>("FADD2 x8", 16, wps);
        run<5>("13 FFMA2 + 2 MUFU + 2 FSETP/FSEL", 26, wps);
        run<6>("FMUL2 x8", 16, wps);
        run<7>("4 FADD2 + 4 FMUL2 + 5 FFMA2", 26, wps);
        run<8>("FFMA2 a=x*y+a, 3 distinct pairs", 16, wps);
    }
    return 0;
}
