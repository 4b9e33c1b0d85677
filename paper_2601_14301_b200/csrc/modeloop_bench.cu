// modeloop_bench.cu -- stand-alone micro-benchmark of the mode loop (row a3) in its source forms: coefficient records in
// shared memory, nothing else in the kernel.  Not part of libtrimeg.so; evidence for DESIGN.md section 6 and
// profiles/r02_mode_loop.md.
//   nvcc -O3 -std=c++17 -gencode arch=compute_100a,code=sm_100a -o modeloop_bench modeloop_bench.cu && ./modeloop_bench
//   cuobjdump -sass modeloop_bench | python sass_census.py - k_                     (operand census of the loops)
// Forms: A  two markers per thread, every coefficient loaded once for both (trimeg_multi.cuh; the WCACHE kernel until the
//           lane pairs replaced it);
//        B  the same source with one marker per thread, two passes;
//        C  one marker per evaluation in two phases separated by a branch (trimeg_lane.cuh: both push kernels), two passes;
//        G  two markers per thread, every coefficient loaded once into registers, one basic block per marker and half
//           record (measured, not taken: faster than A with three warps per scheduler, slower with one, slower in the kernel).
// Second part: what a warp-wide 16-byte shared-memory load costs as a function of WHICH lanes read the same record
// (k_C with a lane -> record pattern; wavefronts per load from
//   ncu --metrics l1tex__data_pipe_lsu_wavefronts_mem_shared.sum,smsp__sass_inst_executed_op_shared_ld.sum -k regex:k_C ./modeloop_bench).
#include <cstdio>
#include <vector>
#include "trimeg_multi.cuh"
#include "trimeg_lane.cuh"
using namespace trimeg;
constexpr int NMODES = 16;
constexpr int REC = NMODES * NCOEF + 3;

// lane -> record (0..7) patterns of the shared-memory study
template <int PAT>
__device__ __forceinline__ int pattern_rec(int lane, int w)
{
    switch (PAT) {
    case 0: return w & 7;                                                   // one record per warp
    case 1: return (w + lane / 8) & 7;                                      // four records, one per quarter-warp (default of forms A-G)
    case 2: return lane & 7;                                                // eight records, lane l -> record l mod 8
    case 3: return (w + (lane & 1)) & 7;                                    // two records, lanes alternate
    case 4: return lane < 20 ? 0 : lane < 26 ? 1 : lane < 30 ? 2 : 3;       // runs of 20, 6, 4, 2 lanes (even starts)
    case 5: return (lane & 15) >> 1;                                        // lane pairs, eight records per half-warp
    case 6: return (((lane & 15) >> 2) << 1) | (lane & 1);                  // [0 1 0 1 2 3 2 3 ...]
    case 7: return lane == 2 ? 1 : lane == 5 ? 2 : 0;                       // two single lanes on records of their own
    case 8: return lane == 0 ? 1 : lane == 4 ? 2 : lane == 8 ? 3 : 0;       // [1 0 0 0 2 0 0 0 3 0 0 0 0 ...]
    case 9: return ((lane * 5 + 3) & 15) % 3;                               // three records, interleaved
    default: return lane < 16 ? 0 : (lane & 3);                             // half-warp 0 on one record, half-warp 1 on four, interleaved
    }
}

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
    const double2 *c0 = sh + pattern_rec<PAT>(lane, w) * REC;                                             \
    double acc = 0.0;

template <int THREADS, int PAT = 1>
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

template <int THREADS, int PAT = 1>
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

template <int THREADS, int PAT = 1>
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

// ---- form G: rows eta^JHI..eta^JLO of one marker from coefficients in registers (operations and order of eval_quintic_multi)
template <int JHI, int JLO>
__device__ __forceinline__ void g_rows(const double2 (&cc)[NCOEF], double xi, double eta, double &pr, double &pi, double &pxr,
                                       double &pxi, double &per, double &pei)
{
#pragma unroll
    for (int j = JHI; j >= JLO; --j) {
        const int n = 5 - j;
        double ar = 0.0, ai = 0.0, dr = 0.0, di = 0.0;
#pragma unroll
        for (int i = n; i >= 0; --i) {
            const double2 c = cc[kidx(i, j)];
            if (i == n) { ar = c.x; ai = c.y; }
            else {
                if (i == n - 1) { dr = ar; di = ai; }
                else { dr = fma(dr, xi, ar); di = fma(di, xi, ai); }
                ar = fma(ar, xi, c.x); ai = fma(ai, xi, c.y);
            }
        }
        if (j == 5) { pr = ar; pi = ai; }
        else {
            if (j == 4) { per = pr; pei = pi; pxr = dr; pxi = di; }
            else {
                per = fma(per, eta, pr); pei = fma(pei, eta, pi);
                pxr = fma(pxr, eta, dr); pxi = fma(pxi, eta, di);
            }
            pr = fma(pr, eta, ar); pi = fma(pi, eta, ai);
        }
    }
}

template <int THREADS, int JSPLIT, int PAT = 1>
__global__ void __launch_bounds__(THREADS, 1) k_G(const double2 *rec_g, const double *in, double *out, int iters, FieldDev F, int zero)
{
    SETUP
    double xi[2], eta[2], phi[2];
    for (int p = 0; p < 2; ++p) { xi[p] = st[(p * 3 + 0) * 512 + threadIdx.x]; eta[p] = st[(p * 3 + 1) * 512 + threadIdx.x]; phi[p] = st[(p * 3 + 2) * 512 + threadIdx.x]; }
    const int zero2 = zero * (int)blockDim.x;
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
        double Er[2], Ei[2], Dr[2], Di[2], f[2], fx[2], fe[2], fp[2];
        for (int p = 0; p < 2; ++p) { Er[p] = 1.0; Ei[p] = 0.0; Dr[p] = phi[p]; Di[p] = 1.0 - phi[p]; f[p] = fx[p] = fe[p] = fp[p] = 0.0; }
        double nn = 1.0;
        const double2 *c = c0;
#pragma unroll 1
        for (int m = 0; m < F.n_modes; ++m, c += NCOEF) {
            double pr[2] = {0, 0}, pi[2] = {0, 0}, pxr[2] = {0, 0}, pxi[2] = {0, 0}, per[2] = {0, 0}, pei[2] = {0, 0};
            double2 cc[NCOEF];
#pragma unroll
            for (int k = 0; k < NCOEF; ++k) cc[k] = c[k];
            const int op0 = m + zero, op1 = m ^ zero2;                  // >= 0, opaque, unrelated for the compiler
            if (op0 >= 0) g_rows<5, JSPLIT>(cc, xi[0], eta[0], pr[0], pi[0], pxr[0], pxi[0], per[0], pei[0]);
            if (op1 >= 0) g_rows<5, JSPLIT>(cc, xi[1], eta[1], pr[1], pi[1], pxr[1], pxi[1], per[1], pei[1]);
            if (op1 >= -1) g_rows<JSPLIT - 1, 0>(cc, xi[0], eta[0], pr[0], pi[0], pxr[0], pxi[0], per[0], pei[0]);
            if (op0 >= -1) g_rows<JSPLIT - 1, 0>(cc, xi[1], eta[1], pr[1], pi[1], pxr[1], pxi[1], per[1], pei[1]);
#pragma unroll
            for (int p = 0; p < 2; ++p) {
                f[p] = fma(pr[p], Er[p], fma(-pi[p], Ei[p], f[p]));
                fx[p] = fma(pxr[p], Er[p], fma(-pxi[p], Ei[p], fx[p]));
                fe[p] = fma(per[p], Er[p], fma(-pei[p], Ei[p], fe[p]));
                fp[p] = fma(-nn, fma(pi[p], Er[p], pr[p] * Ei[p]), fp[p]);
                const double tr = fma(Er[p], Dr[p], -Ei[p] * Di[p]);
                Ei[p] = fma(Er[p], Di[p], Ei[p] * Dr[p]);
                Er[p] = tr;
            }
            nn += 2.0;
        }
        for (int p = 0; p < 2; ++p) { acc += f[p] + fx[p] + fe[p] + fp[p]; xi[p] += 1e-9 * f[p]; }
    }
    out[blockIdx.x * blockDim.x + threadIdx.x] = acc + zero;
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
    printf("%-44s %3d threads: %7.3f ms  %6.2f TFLOP/s (170 flops per marker and mode)  %6.1f cycles of a scheduler per warp-wide marker-mode  %s\n",
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
    run("G  two markers, marker blocks", k_G<384, 2>, 384, rec, in, out, F, ghz);
    printf("-- one and two warps per scheduler (the push kernel's warps are not all in the mode loop at once)\n");
    run("A  two markers per thread", k_A<128>, 128, rec, in, out, F, ghz);
    run("A  two markers per thread", k_A<256>, 256, rec, in, out, F, ghz);
    run("C  one marker, two phases", k_C<128>, 128, rec, in, out, F, ghz);
    run("C  one marker, two phases", k_C<256>, 256, rec, in, out, F, ghz);
    run("G  two markers, marker blocks", k_G<128, 2>, 128, rec, in, out, F, ghz);
    run("G  two markers, marker blocks", k_G<256, 2>, 256, rec, in, out, F, ghz);
    printf("-- form C, which lanes read the same record (16-byte shared-memory loads)\n");
    run("C  pattern 0: one record per warp", k_C<384, 0>, 384, rec, in, out, F, ghz);
    run("C  pattern 2: lane l -> record l mod 8", k_C<384, 2>, 384, rec, in, out, F, ghz);
    run("C  pattern 3: two records, alternating", k_C<384, 3>, 384, rec, in, out, F, ghz);
    run("C  pattern 4: runs of 20, 6, 4, 2 lanes", k_C<384, 4>, 384, rec, in, out, F, ghz);
    run("C  pattern 5: lane pairs, 8 per half-warp", k_C<384, 5>, 384, rec, in, out, F, ghz);
    run("C  pattern 6: [0 1 0 1 2 3 2 3 ...]", k_C<384, 6>, 384, rec, in, out, F, ghz);
    run("C  pattern 7: two single lanes", k_C<384, 7>, 384, rec, in, out, F, ghz);
    run("C  pattern 8: [1 0 0 0 2 0 0 0 3 0 ...]", k_C<384, 8>, 384, rec, in, out, F, ghz);
    run("C  pattern 9: three records interleaved", k_C<384, 9>, 384, rec, in, out, F, ghz);
    run("C  pattern 10: one half-warp on four", k_C<384, 10>, 384, rec, in, out, F, ghz);
    return 0;
}
