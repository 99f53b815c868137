// mm_ubench_rf.cu -- stand-alone microbenchmark: the 6-FMA stencil update of an 8-cell patch with 48 distinct
// coefficient registers, i.e. the level loop of mm_coef.cuh without its shuffles.  Measures the issue rate of FFMAs
// whose three source registers are all distinct -- (A) accumulator-stationary source order (what the kernel does),
// (B) x-stationary order (each value feeds its five accumulators back to back, so ptxas can flag operand reuse),
// (C) packed FFMA2 -- to show the register-file operand bandwidth that bounds the level loop.  Not part of libmm.so.
//   nvcc -O3 -gencode arch=compute_100a,code=sm_100a -o mm_ubench_rf paper_1908_04279_b200/csrc/mm_ubench_rf.cu && ./mm_ubench_rf
// Results: profiles/r01e_README.md.
#include <cstdio>
#include <cuda_runtime.h>
#define ITERS 2048
template <int ORDER> __global__ void __launch_bounds__(256, 1) kern(float *out, const float *cin, long long *clk)
{
    float c[6][8], x[8], r[8];
    for (int k = 0; k < 6; k++) for (int i = 0; i < 8; i++) c[k][i] = cin[(k * 8 + i) * 32 + (threadIdx.x & 31)];
    for (int i = 0; i < 8; i++) { x[i] = threadIdx.x + i; r[i] = i; }
    long long t0 = clock64();
#pragma unroll 1
    for (int it = 0; it < ITERS; it++) {
        float n[8];
        if (ORDER == 0) {
#pragma unroll
            for (int i = 0; i < 8; i++) {
                float a = fmaf(c[0][i], x[i], 1.0f);
                a = fmaf(c[1][i], x[(i + 1) & 7], a);
                a = fmaf(c[2][i], x[(i + 7) & 7], a);
                a = fmaf(c[3][i], x[(i + 2) & 7], a);
                a = fmaf(c[4][i], x[(i + 6) & 7], a);
                n[i] = fmaf(c[5][i], r[i], a);
            }
        } else if (ORDER == 2) {
            // packed: pairs (2p, 2p+1); shifted pairs s[p] = (x[2p+1], x[2p+2]) serve both misaligned neighbours
            float2 sh[4];
#pragma unroll
            for (int p = 0; p < 4; p++) sh[p] = make_float2(x[2 * p + 1], x[(2 * p + 2) & 7]);
#pragma unroll
            for (int p = 0; p < 4; p++) {
                const int i = 2 * p;
                float2 a = __ffma2_rn(make_float2(c[0][i], c[0][i + 1]), make_float2(x[i], x[i + 1]), make_float2(1.0f, 1.0f));
                a = __ffma2_rn(make_float2(c[1][i], c[1][i + 1]), sh[p], a);
                a = __ffma2_rn(make_float2(c[2][i], c[2][i + 1]), sh[(p + 3) & 3], a);
                a = __ffma2_rn(make_float2(c[3][i], c[3][i + 1]), make_float2(x[(i + 2) & 7], x[(i + 3) & 7]), a);
                a = __ffma2_rn(make_float2(c[4][i], c[4][i + 1]), make_float2(x[(i + 6) & 7], x[(i + 7) & 7]), a);
                a = __ffma2_rn(make_float2(c[5][i], c[5][i + 1]), make_float2(r[i], r[i + 1]), a);
                n[i] = a.x; n[i + 1] = a.y;
            }
        } else {
#pragma unroll
            for (int i = 0; i < 8; i++) n[i] = fmaf(c[5][i], r[i], 1.0f);
#pragma unroll
            for (int j = 0; j < 8; j++) {   // x[j] feeds five accumulators back to back
                n[j] = fmaf(c[0][j], x[j], n[j]);
                n[(j + 7) & 7] = fmaf(c[1][(j + 7) & 7], x[j], n[(j + 7) & 7]);
                n[(j + 1) & 7] = fmaf(c[2][(j + 1) & 7], x[j], n[(j + 1) & 7]);
                n[(j + 6) & 7] = fmaf(c[3][(j + 6) & 7], x[j], n[(j + 6) & 7]);
                n[(j + 2) & 7] = fmaf(c[4][(j + 2) & 7], x[j], n[(j + 2) & 7]);
            }
        }
#pragma unroll
        for (int i = 0; i < 8; i++) { r[i] = x[i]; x[i] = n[i]; }
    }
    long long t1 = clock64();
    float s = 0; for (int i = 0; i < 8; i++) s += x[i] + r[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
    if (threadIdx.x == 0 && blockIdx.x == 0) *clk = t1 - t0;
}
template <int ORDER> void run(const char *name)
{
    float *out, *cin; long long *clk; cudaMalloc(&out, 148 * 1024 * 4); cudaMalloc(&cin, 48 * 32 * 4); cudaMalloc(&clk, 8);
    float h[48 * 32]; for (int i = 0; i < 48 * 32; i++) h[i] = 0.1f + 1e-3f * (i % 97);
    cudaMemcpy(cin, h, sizeof h, cudaMemcpyHostToDevice);
    for (int threads : {128, 256}) {
        kern<ORDER><<<148, threads>>>(out, cin, clk); cudaDeviceSynchronize();
        long long c; cudaMemcpy(&c, clk, 8, cudaMemcpyDeviceToHost);
        printf("%s warps/SM=%d: %.3f FFMA/clk/SM (48 FFMA per iteration per warp, %lld clk / %d iterations)\n", name, threads / 32,
               48.0 * ITERS * (threads / 32) / c, c, ITERS);
    }
}
int main() { run<0>("acc-stationary"); run<1>("x-stationary  "); run<2>("packed acc-st "); return 0; }
