// fp64_pipe_bench.cu -- stand-alone micro-benchmark of the FP64 pipe of sm_100a: scalar DFMA against the FP64 tensor
// instruction (mma.sync.m8n8k4.f64 -> DMMA.8x8x4).  Not part of libtrimeg.so; evidence for DESIGN.md section 6 ("what was
// measured and not built: the mode sum as a GEMM") and profiles/r02_mode_loop.md.
//   nvcc -O3 -std=c++17 -gencode arch=compute_100a,code=sm_100a -o fp64_pipe_bench fp64_pipe_bench.cu && ./fp64_pipe_bench
// Questions: (1) what does DMMA reach, with how many warps and independent accumulator tiles; (2) does it care whether its
// A / B fragments change from instruction to instruction (the operand port that limits DFMA); (3) is it a pipe of its own
// (DMMA and DFMA streams of one warp add up) or the FP64 pipe (they share).
#include <cstdio>
#include <cuda_runtime.h>

__device__ __forceinline__ void dmma884(double &d0, double &d1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

template <int NACC>
__global__ void __launch_bounds__(512, 1) k_dfma(double *out, int iters, double a, double b)
{
    double acc[NACC];
#pragma unroll
    for (int i = 0; i < NACC; ++i) acc[i] = threadIdx.x + i;
#pragma unroll 1
    for (int it = 0; it < iters; ++it)
#pragma unroll
        for (int r = 0; r < 4; ++r)
#pragma unroll
            for (int i = 0; i < NACC; ++i) acc[i] = fma(acc[i], a, b);
    double s = 0;
#pragma unroll
    for (int i = 0; i < NACC; ++i) s += acc[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// NT independent 8 x 8 accumulator tiles; A / B fragments fixed (FRESH = 0) or different registers in every instruction (1)
template <int NT, int FRESH>
__global__ void __launch_bounds__(512, 1) k_dmma(double *out, int iters, double a0, double b0)
{
    double d0[NT], d1[NT], a[NT], b[NT];
#pragma unroll
    for (int i = 0; i < NT; ++i) { d0[i] = threadIdx.x + i; d1[i] = i; a[i] = a0 + i * 1e-9 * threadIdx.x; b[i] = b0 - i * 1e-9 * threadIdx.x; }
#pragma unroll 1
    for (int it = 0; it < iters; ++it)
#pragma unroll
        for (int r = 0; r < 4; ++r)
#pragma unroll
            for (int i = 0; i < NT; ++i) dmma884(d0[i], d1[i], FRESH ? a[(i + r) % NT] : a[0], FRESH ? b[(i + 2 * r) % NT] : b[0]);
    double s = 0;
#pragma unroll
    for (int i = 0; i < NT; ++i) s += d0[i] + d1[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// NT DMMA tiles and NF DFMA chains per round in one warp
template <int NT, int NF>
__global__ void __launch_bounds__(512, 1) k_mixed(double *out, int iters, double a0, double b0)
{
    double d0[NT], d1[NT], acc[NF];
#pragma unroll
    for (int i = 0; i < NT; ++i) { d0[i] = threadIdx.x + i; d1[i] = i; }
#pragma unroll
    for (int i = 0; i < NF; ++i) acc[i] = threadIdx.x - i;
#pragma unroll 1
    for (int it = 0; it < iters; ++it)
#pragma unroll
        for (int r = 0; r < 4; ++r) {
#pragma unroll
            for (int i = 0; i < NT; ++i) dmma884(d0[i], d1[i], a0, b0);
#pragma unroll
            for (int i = 0; i < NF; ++i) acc[i] = fma(acc[i], a0, b0);
        }
    double s = 0;
#pragma unroll
    for (int i = 0; i < NT; ++i) s += d0[i] + d1[i];
#pragma unroll
    for (int i = 0; i < NF; ++i) s += acc[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

template <typename F>
float time_it(F f)
{
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    f();
    float best = 1e30f;
    for (int r = 0; r < 3; ++r) {
        cudaEventRecord(e0); f(); cudaEventRecord(e1); cudaEventSynchronize(e1);
        float ms; cudaEventElapsedTime(&ms, e0, e1); if (ms < best) best = ms;
    }
    return best;
}

int main()
{
    const int grid = 148 * 4, iters = 4000;
    double *out;
    if (cudaMalloc(&out, sizeof(double) * grid * 512) != cudaSuccess) { printf("no device\n"); return 1; }
    for (int threads : {128, 256, 512}) {                   // 1, 2, 4 warps per scheduler
        const double warps = grid * threads / 32.0;
        float ms;
        ms = time_it([&] { k_dfma<8><<<grid, threads>>>(out, iters, 1.0000001, 1e-9); });
        printf("%3d threads  DFMA, 8 chains, constant a and b       %8.3f ms  %6.2f TFLOP/s\n", threads, ms, warps * 32 * iters * 4.0 * 8 * 2 / ms * 1e-9);
        ms = time_it([&] { k_dmma<8, 0><<<grid, threads>>>(out, iters, 1.0000001, 1e-9); });
        printf("%3d threads  DMMA 8x8x4, 8 tiles, fixed fragments   %8.3f ms  %6.2f TFLOP/s\n", threads, ms, warps * iters * 4.0 * 8 * 512 / ms * 1e-9);
        ms = time_it([&] { k_dmma<8, 1><<<grid, threads>>>(out, iters, 1.0000001, 1e-9); });
        printf("%3d threads  DMMA 8x8x4, 8 tiles, fresh fragments   %8.3f ms  %6.2f TFLOP/s\n", threads, ms, warps * iters * 4.0 * 8 * 512 / ms * 1e-9);
        ms = time_it([&] { k_dmma<2, 0><<<grid, threads>>>(out, iters, 1.0000001, 1e-9); });
        printf("%3d threads  DMMA 8x8x4, 2 tiles                    %8.3f ms  %6.2f TFLOP/s\n", threads, ms, warps * iters * 4.0 * 2 * 512 / ms * 1e-9);
        ms = time_it([&] { k_mixed<4, 32><<<grid, threads>>>(out, iters, 1.0000001, 1e-9); });
        printf("%3d threads  4 DMMA + 32 DFMA per round             %8.3f ms  %6.2f TFLOP/s (both)\n", threads, ms, warps * iters * 4.0 * (4 * 512 + 32 * 64) / ms * 1e-9);
    }
    cudaDeviceSynchronize();
    printf("%s\n", cudaGetErrorString(cudaGetLastError()));
    return 0;
}
