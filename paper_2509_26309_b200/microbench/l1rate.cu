// l1rate.cu -- microbenchmark behind DESIGN.md section 5 ("what bounds cfg4 and cfg5"); not part of libtbpm.so.
//   nvcc -O3 -gencode arch=compute_100a,code=sm_100a -o l1rate paper_2509_26309_b200/microbench/l1rate.cu && ./l1rate
// How fast does one SM's L1/LSU accept 128-byte line requests, for (A) one warp-wide 256-bit load touching 8 lines,
// (B) eight 256-bit loads with 4 active lanes each (1 line per instruction), (C) two 128-bit loads (4 lines each)?
// Data is L2-resident (buffer 48 MB, each block strides so that L1 rarely hits), gather-like row addressing.
#include <cstdio>
#include <cuda_runtime.h>
__device__ __forceinline__ void ld256(double (&a)[4], const double *p)
{
    asm volatile("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(a[0]), "=d"(a[1]), "=d"(a[2]), "=d"(a[3]) : "l"(p));
}
__device__ __forceinline__ void ld256_if(double (&a)[4], const double *p, bool on)
{
    asm volatile("{\n.reg .pred q;\nsetp.ne.b32 q, %5, 0;\n@q ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];\n}" : "+d"(a[0]), "+d"(a[1]), "+d"(a[2]), "+d"(a[3]) : "l"(p), "r"((int)on));
}
__device__ __forceinline__ void ld128(double (&a)[2], const double *p)
{
    asm volatile("ld.global.nc.v2.f64 {%0,%1}, [%2];" : "=d"(a[0]), "=d"(a[1]) : "l"(p));
}
// rows of 128 B; a warp works on 8 rows per step; each step gathers G = 8 "neighbour" rows per row at pseudo-random offsets
template <int MODE>
__global__ void __launch_bounds__(512, 1) k(const double *buf, long n_rows, int steps, double *out)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int sub = lane >> 2, q = lane & 3;
    double acc = 0;
    long base = ((long)blockIdx.x * 16 + warp) * 8;
    for (int s = 0; s < steps; ++s) {
        double x[8][4];
#pragma unroll
        for (int g = 0; g < 8; ++g) { x[g][0] = x[g][1] = x[g][2] = x[g][3] = 0; }
#pragma unroll
        for (int g = 0; g < 8; ++g) {
            const long r = (base + sub + (long)g * 4099 * 8 + (long)s * 148 * 16 * 8) % n_rows;
            const double *p = buf + r * 16 + q * 4;
            if (MODE == 0) ld256(x[g], p);
            else if (MODE == 1) {
#pragma unroll
                for (int j = 0; j < 8; ++j) ld256_if(x[g], p, sub == j);
            } else {
                double a[2], b[2];
                ld128(a, p); ld128(b, p + 2);
                x[g][0] = a[0]; x[g][1] = a[1]; x[g][2] = b[0]; x[g][3] = b[1];
            }
        }
#pragma unroll
        for (int g = 0; g < 8; ++g) acc += x[g][0] + x[g][1] + x[g][2] + x[g][3];
    }
    if (acc == 1.2345) out[0] = acc;
}
int main()
{
    int sms; cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, 0);
    const long n_rows = 48l * 1024 * 1024 / 128;
    double *buf, *out; cudaMalloc(&buf, n_rows * 128); cudaMalloc(&out, 8); cudaMemset(buf, 0, n_rows * 128);
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int steps = 2000;
    for (int mode = 0; mode < 3; ++mode)
        for (int rep = 0; rep < 3; ++rep) {
            cudaEventRecord(e0);
            if (mode == 0) k<0><<<sms, 512>>>(buf, n_rows, steps, out);
            if (mode == 1) k<1><<<sms, 512>>>(buf, n_rows, steps, out);
            if (mode == 2) k<2><<<sms, 512>>>(buf, n_rows, steps, out);
            cudaEventRecord(e1); cudaEventSynchronize(e1);
            float ms; cudaEventElapsedTime(&ms, e0, e1);
            const double lines = (double)sms * 16 * steps * 8 * 8;            // 128-byte lines requested
            if (rep == 2) printf("mode %d: %.3f ms, %.2f TB/s, %.2f ns per line per SM (%.2f cycles at 1.9 GHz)\n", mode, ms,
                                 lines * 128 / ms / 1e9, ms * 1e6 / (lines / sms), ms * 1e6 / (lines / sms) * 1.9);
        }
    printf("%s\n", cudaGetErrorString(cudaGetLastError()));
    return 0;
}
