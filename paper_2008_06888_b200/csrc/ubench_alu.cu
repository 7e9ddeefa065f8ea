// ubench_alu.cu -- instruction-throughput probe behind DESIGN.md's ALU roofline (not part of
// libttn.so): per-SM issue rate of the candidate max / add instructions of the max-plus gate on
// sm_100a.  Build and run (profiles/r01_ubench.md):
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o ubench_alu paper_2008_06888_b200/csrc/ubench_alu.cu && ./ubench_alu
// The "FMNMX" line alone is not meaningful (ptxas folds the idempotent second max); the FMNMX
// rate is read from the two "gate" lines (2 FMNMX per 3 resp. 4 instructions).
#include <cstdio>
#include <cuda_runtime.h>
#include <cuda_fp16.h>
#define N 32
#define ITERS 2000
template <int OP> __device__ __forceinline__ void step(float (&v)[N], unsigned (&u)[N], float m, unsigned mu) {
#pragma unroll
    for (int j = 0; j < N; j += 2) {
        if (OP == 0) { v[j] = fmaxf(v[j], v[j+1]); v[j+1] = fmaxf(v[j+1], m); }                       // FMNMX only
        if (OP == 1) { v[j] = v[j] + m; v[j+1] = v[j+1] + m; }                                        // FADD
        if (OP == 2) { asm("{.reg .b64 a,b,c; mov.b64 a,{%0,%1}; mov.b64 b,{%2,%2}; add.f32x2 c,a,b; mov.b64 {%0,%1},c;}" : "+f"(v[j]), "+f"(v[j+1]) : "f"(m)); } // FADD2
        if (OP == 3) { float t0, t1; asm("{.reg .b64 a,b,c; mov.b64 a,{%2,%3}; mov.b64 b,{%4,%4}; add.f32x2 c,a,b; mov.b64 {%0,%1},c;}" : "=f"(t0), "=f"(t1) : "f"(v[j]), "f"(v[j+1]), "f"(m));
                       v[j] = fmaxf(v[j], t1); v[j+1] = fmaxf(v[j+1], t0); }                          // gate: 2 FMNMX + 1 FADD2
        if (OP == 4) { asm("max.s32 %0,%0,%1;" : "+r"(u[j]) : "r"(u[j+1])); asm("max.s32 %0,%0,%1;" : "+r"(u[j+1]) : "r"(mu)); }   // IMNMX
        if (OP == 5) { asm("max.s16x2 %0,%0,%1;" : "+r"(u[j]) : "r"(u[j+1])); asm("max.s16x2 %0,%0,%1;" : "+r"(u[j+1]) : "r"(mu)); }
        if (OP == 6) { asm("max.f16x2 %0,%0,%1;" : "+r"(u[j]) : "r"(u[j+1])); asm("max.f16x2 %0,%0,%1;" : "+r"(u[j+1]) : "r"(mu)); }
        if (OP == 7) { asm("max.f32 %0,%0,%1,%2;" : "+f"(v[j]) : "f"(v[j+1]), "f"(m)); asm("max.f32 %0,%0,%1,%2;" : "+f"(v[j+1]) : "f"(m), "f"(v[j])); }  // FMNMX3
        if (OP == 8) { u[j] = __viaddmax_s32(u[j+1], mu, u[j]); u[j+1] = __viaddmax_s32(u[j], mu, u[j+1]); }
        if (OP == 9) { u[j] = __viaddmax_s16x2(u[j+1], mu, u[j]); u[j+1] = __viaddmax_s16x2(u[j], mu, u[j+1]); }
        if (OP == 10) { asm("add.f16x2 %0,%0,%1;" : "+r"(u[j]) : "r"(mu)); asm("add.f16x2 %0,%0,%1;" : "+r"(u[j+1]) : "r"(mu)); }
        if (OP == 11) { unsigned t; asm("add.f16x2 %0,%1,%2;" : "=r"(t) : "r"(u[j+1]), "r"(mu)); asm("max.f16x2 %0,%0,%1;" : "+r"(u[j]) : "r"(t));
                        asm("add.f16x2 %0,%1,%2;" : "=r"(t) : "r"(u[j]), "r"(mu)); asm("max.f16x2 %0,%0,%1;" : "+r"(u[j+1]) : "r"(t)); }   // half2 gate
        if (OP == 12) { unsigned t; asm("add.s16x2 %0,%1,%2;" : "=r"(t) : "r"(u[j+1]), "r"(mu)); asm("max.s16x2 %0,%0,%1;" : "+r"(u[j]) : "r"(t));
                        asm("add.s16x2 %0,%1,%2;" : "=r"(t) : "r"(u[j]), "r"(mu)); asm("max.s16x2 %0,%0,%1;" : "+r"(u[j+1]) : "r"(t)); }
        if (OP == 13) { float t = v[j+1] + m; v[j] = fmaxf(v[j], t); t = v[j] + m; v[j+1] = fmaxf(v[j+1], t); }  // scalar FADD + FMNMX
        if (OP == 14) { v[j] = fmaf(v[j], 1.0f, m); v[j+1] = fmaf(v[j+1], m, v[j]); }                  // FFMA
        if (OP == 15) { asm("max.bf16x2 %0,%0,%1;" : "+r"(u[j]) : "r"(u[j+1])); asm("max.bf16x2 %0,%0,%1;" : "+r"(u[j+1]) : "r"(mu)); }
    }
}
template <int OP> __global__ void __launch_bounds__(1024) k(float* out, float m, unsigned mu, long long* cyc) {
    float v[N]; unsigned u[N];
#pragma unroll
    for (int j = 0; j < N; ++j) { v[j] = threadIdx.x * 0.001f + j; u[j] = threadIdx.x * 7 + j; }
    __syncthreads();
    long long t0 = clock64();
    for (int it = 0; it < ITERS; ++it) step<OP>(v, u, m, mu);
    long long t1 = clock64();
    float s = 0; unsigned su = 0;
#pragma unroll
    for (int j = 0; j < N; ++j) { s += v[j]; su += u[j]; }
    out[blockIdx.x * blockDim.x + threadIdx.x] = s + su;
    if (threadIdx.x == 0) cyc[blockIdx.x] = t1 - t0;
}
template <int OP> void run(const char* name, int ops_per_pair, int elems_per_op, float* out, long long* cyc) {
    for (int threads : {128, 256, 512, 1024}) {
        k<OP><<<148, threads>>>(out, 0.5f, 3u, cyc);
        cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
        cudaEventRecord(e0);
        k<OP><<<148, threads>>>(out, 0.5f, 3u, cyc);
        cudaEventRecord(e1); cudaDeviceSynchronize();
        float ms; cudaEventElapsedTime(&ms, e0, e1);
        long long h[148]; cudaMemcpy(h, cyc, sizeof h, cudaMemcpyDeviceToHost);
        double c = 0; for (int i = 0; i < 148; ++i) c += h[i]; c /= 148;
        double instr = (double)ITERS * (N / 2) * ops_per_pair * threads;   // thread-instr per SM
        printf("%-28s threads=%4d  %.1f thread-instr/clk/SM  (%.1f elem-ops/clk/SM)  %.3f ms  err=%s\n", name, threads, instr / c,
               instr / c * elems_per_op, ms, cudaGetErrorString(cudaGetLastError()));
    }
}
int main() {
    float* out; long long* cyc; cudaMalloc(&out, 148 * 1024 * 4); cudaMalloc(&cyc, 148 * 8);
    run<0>("FMNMX", 2, 1, out, cyc);
    run<1>("FADD", 2, 1, out, cyc);
    run<2>("FADD2", 1, 2, out, cyc);
    run<14>("FFMA", 2, 1, out, cyc);
    run<3>("gate 2FMNMX+FADD2", 3, 1, out, cyc);
    run<13>("gate 2FMNMX+2FADD", 4, 1, out, cyc);
    run<4>("IMNMX s32", 2, 1, out, cyc);
    run<5>("max.s16x2", 2, 2, out, cyc);
    run<6>("max.f16x2", 2, 2, out, cyc);
    run<15>("max.bf16x2", 2, 2, out, cyc);
    run<7>("FMNMX3", 2, 1, out, cyc);
    run<8>("viaddmax s32", 2, 1, out, cyc);
    run<9>("viaddmax s16x2", 2, 2, out, cyc);
    run<10>("add.f16x2", 2, 2, out, cyc);
    run<11>("gate f16x2 (add+max)x2", 4, 2, out, cyc);
    run<12>("gate s16x2 (add+max)x2", 4, 2, out, cyc);
    return 0;
}
