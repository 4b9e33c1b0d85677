// modeloop_bench.cu -- stand-alone micro-benchmark of the mode loop (row a3) in its source forms: coefficient records in
// shared memory, nothing else in the kernel.  Not part of libtrimeg.so; evidence for DESIGN.md section 6 and
// profiles/r02_mode_loop.md.
//   nvcc -O3 -std=c++17 -gencode arch=compute_100a,code=sm_100a -o modeloop_bench modeloop_bench.cu && ./modeloop_bench
//   cuobjdump -sass modeloop_bench | python sass_census.py - k_                     (operand census of the loops)
// Forms: A  two markers per thread, every coefficient loaded once for both (trimeg_multi.cuh, the WCACHE kernel);
//        B  the same source with one marker per thread, two passes;
//        C  one marker per evaluation in two phases separated by a branch (trimeg_lane.cuh, the LANE kernel), two passes.
#include <cstdio>
#include <vector>
#include "trimeg_multi.cuh"
#include "trimeg_lane.cuh"
using namespace trimeg;
constexpr int NMODES = 16;
constexpr int REC = NMODES * NCOEF + 3;

#define SETUP                                                                                        \
    extern __shared__ double2 sh[];                                                                  \
    double *st = reinterpret_cast<double *>(sh + 8 * REC);                                           \
    for (int k = threadIdx.x; k < 8 * REC; k += blockDim.x) sh[k] = rec_g[k];                        \
    for (int p = 0; p < 2; ++p) {                                                                    \
        st[(p * 3 + 0) * 512 + threadIdx.x] = in[threadIdx.x * 2 + p];                               \
        st[(p * 3 + 1) * 512 + threadIdx.x] = in[1100 + threadIdx.x * 2 + p];                        \
        st[(p * 3 + 2) * 512 + threadIdx.x] = in[2200 + threadIdx.x * 2 + p];                        \
    }                                                                                                \
    __syncthreads();                                                                                 \
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;                                         \
    const double2 *c0 = sh + ((w + lane / 8) & 7) * REC;                                             \
    double acc = 0.0;

template <int THREADS>
__global__ void __launch_bounds__(THREADS, 1) k_A(const double2 *rec_g, const double *in, double *out, int iters, FieldDev F, int zero)
{
    SETUP
    double xi[2], eta[2], phi[2], f[2], fx[2], fe[2], fp[2];
    for (int p = 0; p < 2; ++p) { xi[p] = st[(p * 3 + 0) * 512 + threadIdx.x]; eta[p] = st[(p * 3 + 1) * 512 + threadIdx.x]; phi[p] = st[(p * 3 + 2) * 512 + threadIdx.x]; }
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
        double Er[2], Ei[2], Dr[2], Di[2];
        for (int p = 0; p < 2; ++p) { Er[p] = 1.0; Ei[p] = 0.0; Dr[p] = phi[p]; Di[p] = 1.0 - phi[p]; }
        gather_modes_impl<2, false, true>(F, c0, xi, eta, phi, Er, Ei, Dr, Di, f, fx, fe, fp);
        for (int p = 0; p < 2; ++p) { acc += f[p] + fx[p] + fe[p] + fp[p]; xi[p] += 1e-9 * f[p]; }
    }
    out[blockIdx.x * blockDim.x + threadIdx.x] = acc + zero;
}

template <int THREADS>
__global__ void __launch_bounds__(THREADS, 1) k_B(const double2 *rec_g, const double *in, double *out, int iters, FieldDev F, int zero)
{
    SETUP
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll 1
        for (int p = 0; p < 2; ++p) {
            double xi[1], eta[1], phi[1], f[1], fx[1], fe[1], fp[1], Er[1] = {1.0}, Ei[1] = {0.0}, Dr[1], Di[1];
            xi[0] = st[(p * 3 + 0) * 512 + threadIdx.x]; eta[0] = st[(p * 3 + 1) * 512 + threadIdx.x]; phi[0] = st[(p * 3 + 2) * 512 + threadIdx.x];
            Dr[0] = phi[0]; Di[0] = 1.0 - phi[0];
            gather_modes_impl<1, false, true>(F, c0, xi, eta, phi, Er, Ei, Dr, Di, f, fx, fe, fp);
            acc += f[0] + fx[0] + fe[0] + fp[0];
            st[(p * 3 + 0) * 512 + threadIdx.x] = xi[0] + 1e-9 * f[0];
        }
    }
    out[blockIdx.x * blockDim.x + threadIdx.x] = acc + zero;
}

template <int THREADS>
__global__ void __launch_bounds__(THREADS, 1) k_C(const double2 *rec_g, const double *in, double *out, int iters, FieldDev F, int zero)
{
    SETUP
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
#pragma unroll 1
        for (int p = 0; p < 2; ++p) {
            const double xi = st[(p * 3 + 0) * 512 + threadIdx.x], eta = st[(p * 3 + 1) * 512 + threadIdx.x], phi = st[(p * 3 + 2) * 512 + threadIdx.x];
            double Er = 1.0, Ei = 0.0, Dr = phi, Di = 1.0 - phi, f = 0, fx = 0, fe = 0, fp = 0, nn = 1.0;
            const double2 *c = c0;
#pragma unroll 1
            for (int m = 0; m < F.n_modes; ++m, c += NCOEF) {
                double pr, pi, pxr, pxi, per, pei;
                eval_quintic_2ph(c, xi, eta, zero + m, pr, pi, pxr, pxi, per, pei);
                f = fma(pr, Er, fma(-pi, Ei, f));
                fx = fma(pxr, Er, fma(-pxi, Ei, fx));
                fe = fma(per, Er, fma(-pei, Ei, fe));
                fp = fma(-nn, fma(pi, Er, pr * Ei), fp);
                const double tr = fma(Er, Dr, -Ei * Di);
                Ei = fma(Er, Di, Ei * Dr);
                Er = tr;
                nn += 2.0;
            }
            acc += f + fx + fe + fp;
            st[(p * 3 + 0) * 512 + threadIdx.x] = xi + 1e-9 * f;
        }
    }
    out[blockIdx.x * blockDim.x + threadIdx.x] = acc;
}

__global__ void __launch_bounds__(256) k_dfma_peak(double *out, double a, double b)
{
    double acc[8];
    for (int k = 0; k < 8; ++k) acc[k] = (double)(threadIdx.x + k);
#pragma unroll 4
    for (int it = 0; it < 4096; ++it)
#pragma unroll
        for (int k = 0; k < 8; ++k) acc[k] = fma(acc[k], a, b);
    double s = 0;
    for (int k = 0; k < 8; ++k) s += acc[k];
    if (s == 123.456) out[0] = s;
}

template <typename K>
void run(const char *name, K kern, int threads, const double2 *rec, const double *in, double *out, FieldDev F, double clock_ghz)
{
    const size_t smem = 227 * 1024;
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    const int iters = 200, blocks = 148 * 4;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    float best = 1e30f;
    for (int rep = 0; rep < 4; ++rep) {
        cudaEventRecord(e0);
        kern<<<blocks, threads, smem>>>(rec, in, out, iters, F, 0);
        cudaEventRecord(e1); cudaEventSynchronize(e1);
        float ms;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best) best = ms;
    }
    const double evals = 2.0 * threads * blocks * (double)iters * NMODES;      // marker-mode evaluations
    const double tf = evals * 170.0 / (best * 1e-3) * 1e-12;
    const double cyc = best * 1e-3 * clock_ghz * 1e9 / (evals / (148.0 * 4 * 32));
    printf("%-34s %3d threads: %7.3f ms  %6.2f TFLOP/s (170 flops per marker and mode)  %6.1f cycles of a scheduler per warp-wide marker-mode  %s\n",
           name, threads, best, tf, cyc, cudaGetErrorString(cudaGetLastError()));
}

int main()
{
    std::vector<double2> hrec(8 * REC);
    for (size_t k = 0; k < hrec.size(); ++k) { hrec[k].x = 1e-3 * ((k * 7919) % 1000) / 1000.0; hrec[k].y = 1e-3 * ((k * 104729) % 1000) / 1000.0; }
    std::vector<double> hin(4096);
    for (size_t k = 0; k < hin.size(); ++k) hin[k] = 0.1 + 0.3 * ((k * 31) % 97) / 97.0;
    double2 *rec; double *in, *out;
    cudaMalloc(&rec, hrec.size() * sizeof(double2)); cudaMalloc(&in, hin.size() * 8); cudaMalloc(&out, 148 * 4 * 512 * 8);
    cudaMemcpy(rec, hrec.data(), hrec.size() * sizeof(double2), cudaMemcpyHostToDevice);
    cudaMemcpy(in, hin.data(), hin.size() * 8, cudaMemcpyHostToDevice);
    FieldDev F; F.n_modes = NMODES; F.coef = nullptr; F.mode_n = nullptr; F.n_first = 1; F.n_step = 2; F.is_ap = 1;
    int khz = 0; cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, 0);
    const double ghz = khz * 1e-6;
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    float best = 1e30f;
    for (int rep = 0; rep < 4; ++rep) {
        cudaEventRecord(e0); k_dfma_peak<<<148 * 32, 256>>>(out, 0.999999, 1e-9); cudaEventRecord(e1); cudaEventSynchronize(e1);
        float ms; cudaEventElapsedTime(&ms, e0, e1); if (rep > 0 && ms < best) best = ms;
    }
    printf("DFMA peak %.2f TFLOP/s at %.3f GHz\n", 2.0 * 4096 * 8 * 256.0 * 148 * 32 / (best * 1e-3) * 1e-12, ghz);
    run("A  two markers per thread", k_A<384>, 384, rec, in, out, F, ghz);
    run("A  two markers per thread", k_A<512>, 512, rec, in, out, F, ghz);
    run("B  one marker, two passes", k_B<384>, 384, rec, in, out, F, ghz);
    run("B  one marker, two passes", k_B<512>, 512, rec, in, out, F, ghz);
    run("C  one marker, two phases", k_C<384>, 384, rec, in, out, F, ghz);
    run("C  one marker, two phases", k_C<512>, 512, rec, in, out, F, ghz);
    return 0;
}
