// mm_ubench.cu -- stand-alone microbenchmark behind the arithmetic choices of mm_coef.cuh: issue throughput of the
// candidate instructions on sm_100a, in warp-instructions per clock per SM (register-only, 8 independent chains per
// thread, one CTA per SM, 4/8/16/32 warps).  Not part of libmm.so.  Results: profiles/r01b_ubench.txt.
//   nvcc -O3 -gencode arch=compute_100a,code=sm_100a -o mm_ubench paper_1908_04279_b200/csrc/mm_ubench.cu && ./mm_ubench
#include <cstdio>
#include <cstdint>
#include <cuda_runtime.h>
#define ITERS 4096
#define ILP 8
template <int OP> __device__ __forceinline__ void op(float (&x)[ILP], float a, float b, unsigned long long (&y)[ILP], unsigned long long A2, unsigned long long B2, double (&d)[ILP], double da, double db)
{
#pragma unroll
    for (int i = 0; i < ILP; i++) {
        if (OP == 0) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(x[i]) : "f"(a), "f"(b));
        if (OP == 1) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(y[i]) : "l"(A2), "l"(B2));
        if (OP == 2) asm volatile("add.f32 %0, %0, %1;" : "+f"(x[i]) : "f"(a));
        if (OP == 3) asm volatile("add.rn.f32x2 %0, %0, %1;" : "+l"(y[i]) : "l"(A2));
        if (OP == 4) asm volatile("max.f32 %0, %0, %1;" : "+f"(x[i]) : "f"(a));
        if (OP == 5) asm volatile("{.reg .pred p; setp.lt.f32 p, %0, %1; selp.f32 %0, %2, %0, p;}" : "+f"(x[i]) : "f"(a), "f"(b));
        if (OP == 6) asm volatile("{.reg .b32 t; mov.b32 t, %0; lop3.b32 t, t, %1, %2, 0x96; mov.b32 %0, t;}" : "+f"(x[i]) : "r"(__float_as_int(a)), "r"(__float_as_int(b)));
        if (OP == 7) asm volatile("fma.rn.f64 %0, %0, %1, %2;" : "+d"(d[i]) : "d"(da), "d"(db));
        if (OP == 8) asm volatile("add.f64 %0, %0, %1;" : "+d"(d[i]) : "d"(da));
        if (OP == 9) asm volatile("{.reg .pred p; setp.lt.f64 p, %0, %1; selp.f64 %0, %2, %0, p;}" : "+d"(d[i]) : "d"(da), "d"(db));
        if (OP == 10) asm volatile("shfl.sync.down.b32 %0, %0, 1, 0x1f, 0xffffffff;" : "+f"(x[i]));
        if (OP == 11) { asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(x[i]) : "f"(a), "f"(b)); asm volatile("max.f32 %0, %0, %1;" : "+f"(x[i]) : "f"(a)); }
        if (OP == 12) asm volatile("mul.rn.f32x2 %0, %0, %1;" : "+l"(y[i]) : "l"(A2));
        if (OP == 13) asm volatile("mul.f32 %0, %0, %1;" : "+f"(x[i]) : "f"(a));
        if (OP == 14) asm volatile("max.f64 %0, %0, %1;" : "+d"(d[i]) : "d"(da));
        if (OP == 15) asm volatile("mul.f64 %0, %0, %1;" : "+d"(d[i]) : "d"(da));
        if (OP == 16) { asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(y[i]) : "l"(A2), "l"(B2)); asm volatile("max.f32 %0, %0, %1;" : "+f"(x[i]) : "f"(a)); }
        if (OP == 17) { asm volatile("fma.rn.f64 %0, %0, %1, %2;" : "+d"(d[i]) : "d"(da), "d"(db)); asm volatile("max.f32 %0, %0, %1;" : "+f"(x[i]) : "f"(a)); asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(x[(i+1)%ILP]) : "f"(a), "f"(b));}
    }
}
template <int OP> __global__ void kern(float *out, float a, float b, double da, double db, long long *clk)
{
    float x[ILP]; unsigned long long y[ILP]; double d[ILP];
    for (int i = 0; i < ILP; i++) { x[i] = threadIdx.x + i; y[i] = threadIdx.x * 77 + i; d[i] = threadIdx.x + i; }
    unsigned long long A2 = ((unsigned long long)__float_as_uint(a) << 32) | __float_as_uint(a), B2 = ((unsigned long long)__float_as_uint(b) << 32) | __float_as_uint(b);
    long long t0 = clock64();
    for (int it = 0; it < ITERS; it++) op<OP>(x, a, b, y, A2, B2, d, da, db);
    long long t1 = clock64();
    float s = 0; for (int i = 0; i < ILP; i++) s += x[i] + (float)y[i] + (float)d[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
    if (threadIdx.x == 0 && blockIdx.x == 0) *clk = t1 - t0;
}
template <int OP> void run(const char *name, int nper)
{
    float *out; long long *clk; cudaMalloc(&out, 148 * 1024 * 4 * 2); cudaMalloc(&clk, 8);
    for (int threads : {128, 256, 512, 1024}) {
        kern<OP><<<148, threads>>>(out, 1.0001f, 0.5f, 1.0001, 0.5, clk);
        cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
        cudaEventRecord(e0); kern<OP><<<148, threads>>>(out, 1.0001f, 0.5f, 1.0001, 0.5, clk); cudaEventRecord(e1); cudaEventSynchronize(e1);
        float ms; cudaEventElapsedTime(&ms, e0, e1); long long c; cudaMemcpy(&c, clk, 8, cudaMemcpyDeviceToHost);
        double winst = (double)ITERS * ILP * nper * (threads / 32);
        printf("%-22s warps/SM=%2d  %.3f warp-inst/clk/SM (clk)  %.1f G warp-inst/s chip\n", name, threads / 32, winst / c, winst * 148 / (ms * 1e6));
    }
    cudaFree(out); cudaFree(clk);
}
int main()
{
    run<0>("FFMA", 1); run<1>("FFMA2", 1); run<2>("FADD", 1); run<3>("FADD2", 1); run<13>("FMUL", 1); run<12>("FMUL2", 1); run<4>("FMNMX", 1); run<5>("FSETP+FSEL", 2); run<6>("LOP3", 1);
    run<7>("DFMA", 1); run<8>("DADD", 1); run<15>("DMUL", 1); run<9>("DSETP+2SEL", 3); run<14>("DMNMX", 1); run<10>("SHFL", 1); run<11>("FFMA+FMNMX", 2); run<16>("FFMA2+FMNMX", 2); run<17>("DFMA+FMNMX+FFMA", 3);
    return 0;
}
