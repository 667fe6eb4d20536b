// fp64_pipe_bench.cu -- microbenchmark behind the ALU roofline of DESIGN.md section 6: throughput of
// DFMA / DADD / DMUL / DSETP / fmin-fmax on the fp64 pipe, dependent-issue latencies, and the
// accuracy of the production reciprocal / rsqrt (hydro_math_fast.cuh) against the IEEE results.
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -std=c++17 -o fp64_pipe_bench fp64_pipe_bench.cu
// Not part of the library; results of round 1 are in profiles/r1_fp64_pipe_microbench.md.
#include <cstdio>
#include <cmath>
#include <cuda_runtime.h>
#include "../hydro_math_fast.cuh"
using namespace hyd;

template <int OP> __global__ void tput(double *out, int iters, double s)
{
    double a0 = threadIdx.x * 1e-3 + 1.0, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6, a7 = a0 + 7;
    const double m = s, c = 1e-9;
    int p = 0;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            if (OP == 0) { a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c); a4 = fma(a4, m, c); a5 = fma(a5, m, c); a6 = fma(a6, m, c); a7 = fma(a7, m, c); }
            if (OP == 1) { a0 = a0 + c; a1 = a1 + c; a2 = a2 + c; a3 = a3 + c; a4 = a4 + c; a5 = a5 + c; a6 = a6 + c; a7 = a7 + c; }
            if (OP == 2) { a0 = a0 * m; a1 = a1 * m; a2 = a2 * m; a3 = a3 * m; a4 = a4 * m; a5 = a5 * m; a6 = a6 * m; a7 = a7 * m; }
            if (OP == 3) { p += (a0 < m + u) + (a1 < m + u) + (a2 < m + u) + (a3 < m + u) + (a4 < m + u) + (a5 < m + u) + (a6 < m + u) + (a7 < m + u); }
            if (OP == 4) { a0 = fmin(a0, m + u); a1 = fmax(a1, m + u); a2 = fmin(a2, m - u); a3 = fmax(a3, m - u); a4 = fmin(a4, m + 2 * u); a5 = fmax(a5, m + 2 * u); a6 = fmin(a6, m - 2 * u); a7 = fmax(a7, m - 2 * u); }
        }
    }
    out[blockIdx.x * blockDim.x + threadIdx.x] = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7 + p;
}

__global__ void acc(double *res, int n)
{
    double e_rcp = 0, e_rsq = 0, e_rsq1 = 0, e_rcp1 = 0;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        // x spans many binades and mantissas
        const double x = exp2((i % 61) - 30.0) * (1.0 + (double)((i * 2654435761u) & 0xffffff) / 16777216.0 + 1e-9 * i);
        const double r0 = 1.0 / x, q0 = 1.0 / sqrt(x);   // reference (IEEE divide/sqrt)
        const double r2 = fast::rcp(x), q2 = fast::rsqrt(x);
        double y; asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
        double e = fma(-x, y, 1.0); double r1 = fma(y, e, y);      // one Newton step
        double z; asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(z) : "d"(x));
        e = fma(-x, z * z, 1.0); double p = fma(0.375, e, 0.5); double q1 = fma(z, p * e, z);
        const double ulp_r = fabs(r0) * 2.220446049250313e-16, ulp_q = fabs(q0) * 2.220446049250313e-16;
        e_rcp = fmax(e_rcp, fabs(r2 - r0) / ulp_r); e_rcp1 = fmax(e_rcp1, fabs(r1 - r0) / ulp_r);
        // q0 is itself double-rounded; compare in higher precision through x*q*q - 1
        e_rsq = fmax(e_rsq, fabs(fma(x * q2, q2, -1.0)) / 2.220446049250313e-16);
        e_rsq1 = fmax(e_rsq1, fabs(fma(x * q1, q1, -1.0)) / 2.220446049250313e-16);
        (void)ulp_q;
    }
    atomicMax((unsigned long long *)&res[0], (unsigned long long)__double_as_longlong(e_rcp));
    atomicMax((unsigned long long *)&res[1], (unsigned long long)__double_as_longlong(e_rcp1));
    atomicMax((unsigned long long *)&res[2], (unsigned long long)__double_as_longlong(e_rsq));
    atomicMax((unsigned long long *)&res[3], (unsigned long long)__double_as_longlong(e_rsq1));
}

__global__ void lat_dfma(double *out, int iters, double m, long long *cyc)
{
    double a = threadIdx.x + 1.0; const double c = 1e-9;
    long long t0 = clock64();
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 16; ++u) a = fma(a, m, c);
    }
    long long t1 = clock64();
    out[threadIdx.x] = a; if (threadIdx.x == 0) cyc[0] = t1 - t0;
}
__global__ void lat_dadd(double *out, int iters, double m, long long *cyc)
{
    double a = threadIdx.x + 1.0;
    long long t0 = clock64();
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 16; ++u) a = a + m;
    }
    long long t1 = clock64();
    out[threadIdx.x] = a; if (threadIdx.x == 0) cyc[0] = t1 - t0;
}
__global__ void lat_sel(double *out, int iters, double m, long long *cyc)
{
    double a = threadIdx.x + 1.0;
    long long t0 = clock64();
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 16; ++u) { a = (a < m) ? a + 1.0 : a - 1.0; }   // DSETP -> (DADD both) -> FSEL chain
    }
    long long t1 = clock64();
    out[threadIdx.x] = a; if (threadIdx.x == 0) cyc[0] = t1 - t0;
}
__global__ void lat_mufu(double *out, int iters, double m, long long *cyc)
{
    double a = threadIdx.x + 1.5;
    long long t0 = clock64();
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 16; ++u) { double y; asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(a)); a = y; }
    }
    long long t1 = clock64();
    out[threadIdx.x] = a; if (threadIdx.x == 0) cyc[0] = t1 - t0;
}
// two warps per SMSP, one doing DFMA chain and one doing integer: can they co-issue at full rate?
__global__ void mix(double *out, int iters, double m, long long *cyc)
{
    const int w = threadIdx.x >> 5;
    double a0 = threadIdx.x + 1.0, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3; const double c = 1e-9;
    int i0 = threadIdx.x, i1 = i0 + 1, i2 = i0 + 2, i3 = i0 + 3;
    long long t0 = clock64();
    if ((w >> 2) & 1) {
        for (int i = 0; i < iters; ++i) {
#pragma unroll
            for (int u = 0; u < 8; ++u) { i0 = i0 * 3 + i1; i1 = i1 * 5 + i2; i2 = i2 * 7 + i3; i3 = i3 * 9 + i0; }
        }
    } else {
        for (int i = 0; i < iters; ++i) {
#pragma unroll
            for (int u = 0; u < 8; ++u) { a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c); }
        }
    }
    long long t1 = clock64();
    out[threadIdx.x] = a0 + a1 + a2 + a3 + i0 + i1 + i2 + i3; if ((threadIdx.x & 31) == 0) cyc[w] = t1 - t0;
}
int main()
{
    double *out; cudaMalloc(&out, 148 * 8 * 256 * sizeof(double));
    cudaEvent_t a, b; cudaEventCreate(&a); cudaEventCreate(&b);
    const char *names[] = {"DFMA", "DADD", "DMUL", "DSETP", "DMNMX(fmin/fmax)"};
    for (int op = 0; op < 5; ++op) {
        for (int wps : {4, 8, 16}) {          // warps per SM via blocks of 256 x (wps/8)... use 1 block/SM of wps*32 threads
            const int iters = 4000, blocks = 148, threads = wps * 32;
            float ms = 0;
            for (int rep = 0; rep < 3; ++rep) {
                cudaEventRecord(a);
                if (op == 0) tput<0><<<blocks, threads>>>(out, iters, 1.0000001);
                if (op == 1) tput<1><<<blocks, threads>>>(out, iters, 1.0000001);
                if (op == 2) tput<2><<<blocks, threads>>>(out, iters, 1.0000001);
                if (op == 3) tput<3><<<blocks, threads>>>(out, iters, 1.0000001);
                if (op == 4) tput<4><<<blocks, threads>>>(out, iters, 1.0000001);
                cudaEventRecord(b); cudaEventSynchronize(b); cudaEventElapsedTime(&ms, a, b);
            }
            const double inst = (double)blocks * threads * iters * 64.0;    // thread-instructions
            printf("%-18s warps/SM=%2d  %.3f ms  %.2f T thread-inst/s  = %.1f lanes/clk/SM @1.965GHz\n", names[op], wps, ms,
                   inst / ms * 1e-9, inst / (ms * 1e-3) / 148 / 1.965e9);
        }
    }
    double *res; cudaMalloc(&res, 4 * sizeof(double)); cudaMemset(res, 0, 32);
    acc<<<296, 256>>>(res, 1 << 26);
    double h[4]; cudaMemcpy(h, res, 32, cudaMemcpyDeviceToHost);
    printf("max err: rcp(production: seed + one third-order step) %.3f ulp, rcp(1 NR) %.3g ulp, rsqrt(3rd+NR) %.3f (x q^2-1)/eps, rsqrt(3rd only) %.3f\n", h[0], h[1], h[2], h[3]);
    {
        long long *cyc, h[64]; cudaMalloc(&cyc, 64 * 8);
        const int iters = 2000;
    lat_dfma<<<1, 32>>>(out, iters, 1.0000001, cyc); cudaMemcpy(h, cyc, 8, cudaMemcpyDeviceToHost);
    printf("DFMA dependent latency: %.2f cycles\n", (double)h[0] / (iters * 16));
    lat_dadd<<<1, 32>>>(out, iters, 1.0000001, cyc); cudaMemcpy(h, cyc, 8, cudaMemcpyDeviceToHost);
    printf("DADD dependent latency: %.2f cycles\n", (double)h[0] / (iters * 16));
    lat_sel<<<1, 32>>>(out, iters, 1e300, cyc); cudaMemcpy(h, cyc, 8, cudaMemcpyDeviceToHost);
    printf("DSETP+DADD+FSEL chain per step: %.2f cycles\n", (double)h[0] / (iters * 16));
    lat_mufu<<<1, 32>>>(out, iters, 1.0, cyc); cudaMemcpy(h, cyc, 8, cudaMemcpyDeviceToHost);
    printf("MUFU.RCP64H dependent latency: %.2f cycles\n", (double)h[0] / (iters * 16));
    mix<<<1, 256>>>(out, iters, 1.0000001, cyc); cudaMemcpy(h, cyc, 64, cudaMemcpyDeviceToHost);
    printf("mix: fp64 warps (4 DFMA chains x 8 x iters = %d instr): %lld cycles ; int warps (%d IMAD): %lld cycles\n", iters * 32, h[0], iters * 32, h[4]);
    mix<<<1, 128>>>(out, iters, 1.0000001, cyc); cudaMemcpy(h, cyc, 64, cudaMemcpyDeviceToHost);
    printf("fp64 warps alone: %lld cycles\n", h[0]);
    }
    printf("%s\n", cudaGetErrorString(cudaGetLastError()));
    return 0;
}
