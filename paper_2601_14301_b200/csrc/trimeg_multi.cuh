// trimeg_multi.cuh -- row a3 for P markers of ONE triangle per thread: every coefficient is loaded
// once and feeds P Horner recurrences from a register.  The many-mode push kernel ran on this form
// until the lane pairs of trimeg_push_wcache.cu (one marker per lane and evaluation, two lanes on one
// record) replaced it; it is kept as form A of the mode-loop study (modeloop_bench.cu,
// profiles/r02_mode_loop.md) and is not part of libtrimeg.so any more.
// The arithmetic of every marker (order of operations, fused multiply-adds) is that of
// eval_quintic() / gather() in trimeg_device.cuh.
#pragma once
#include "trimeg_device.cuh"

namespace trimeg {

// P markers, one triangle: complex quintic and its xi / eta derivatives by bivariate Horner
// (same operation order per marker as eval_quintic), every coefficient loaded once.
template <int P, bool GLOBAL>
__device__ __forceinline__ void eval_quintic_multi(const double2 *__restrict__ c, const double (&xi)[P],
                                                   const double (&eta)[P], double (&pr)[P], double (&pi)[P],
                                                   double (&pxr)[P], double (&pxi)[P], double (&per)[P],
                                                   double (&pei)[P])
{
    double ar[P], ai[P], dr[P], di[P];
#pragma unroll
    for (int j = 5; j >= 0; --j) {
        const int n = 5 - j;
#pragma unroll
        for (int i = n; i >= 0; --i) {
            const double2 cc = GLOBAL ? __ldg(c + kidx(i, j)) : c[kidx(i, j)];
#pragma unroll
            for (int p = 0; p < P; ++p) {
                if (i == n) { ar[p] = cc.x; ai[p] = cc.y; dr[p] = 0.0; di[p] = 0.0; }
                else {
                    if (i == n - 1) { dr[p] = ar[p]; di[p] = ai[p]; }
                    else { dr[p] = fma(dr[p], xi[p], ar[p]); di[p] = fma(di[p], xi[p], ai[p]); }
                    ar[p] = fma(ar[p], xi[p], cc.x); ai[p] = fma(ai[p], xi[p], cc.y);
                }
            }
        }
#pragma unroll
        for (int p = 0; p < P; ++p) {
            if (j == 5) { pr[p] = ar[p]; pi[p] = ai[p]; }
            else {
                if (j == 4) { per[p] = pr[p]; pei[p] = pi[p]; pxr[p] = dr[p]; pxi[p] = di[p]; }
                else {
                    per[p] = fma(per[p], eta[p], pr[p]); pei[p] = fma(pei[p], eta[p], pi[p]);
                    pxr[p] = fma(pxr[p], eta[p], dr[p]); pxi[p] = fma(pxi[p], eta[p], di[p]);
                }
                pr[p] = fma(pr[p], eta[p], ar[p]); pi[p] = fma(pi[p], eta[p], ai[p]);
            }
        }
    }
}

// The same for a mode with n = 0, whose imaginary part never reaches the result (reading G15): real parts only,
// half the arithmetic.  The real chains are those of eval_quintic_multi, operation for operation.
template <int P, bool GLOBAL>
__device__ __forceinline__ void eval_quintic_multi_real(const double2 *__restrict__ c, const double (&xi)[P],
                                                        const double (&eta)[P], double (&pr)[P], double (&pxr)[P],
                                                        double (&per)[P])
{
    double ar[P], dr[P];
#pragma unroll
    for (int j = 5; j >= 0; --j) {
        const int n = 5 - j;
#pragma unroll
        for (int i = n; i >= 0; --i) {
            const double cx = GLOBAL ? __ldg(&c[kidx(i, j)].x) : c[kidx(i, j)].x;
#pragma unroll
            for (int p = 0; p < P; ++p) {
                if (i == n) { ar[p] = cx; dr[p] = 0.0; }
                else {
                    if (i == n - 1) dr[p] = ar[p];
                    else dr[p] = fma(dr[p], xi[p], ar[p]);
                    ar[p] = fma(ar[p], xi[p], cx);
                }
            }
        }
#pragma unroll
        for (int p = 0; p < P; ++p) {
            if (j == 5) pr[p] = ar[p];
            else {
                if (j == 4) { per[p] = pr[p]; pxr[p] = dr[p]; }
                else { per[p] = fma(per[p], eta[p], pr[p]); pxr[p] = fma(pxr[p], eta[p], dr[p]); }
                pr[p] = fma(pr[p], eta[p], ar[p]);
            }
        }
    }
}

// Toroidal factors of P markers: E = e^{i n_first phi}, D = e^{i n_step phi} (arithmetic progression of
// mode numbers; else E is recomputed per mode inside gather_modes).
template <int P>
__device__ __forceinline__ void gather_phases(const FieldDev &F, const double (&phi)[P], double (&Er)[P], double (&Ei)[P],
                                              double (&Dr)[P], double (&Di)[P])
{
#pragma unroll
    for (int p = 0; p < P; ++p) {
        Er[p] = 1.0; Ei[p] = 0.0; Dr[p] = 1.0; Di[p] = 0.0;
        if (F.is_ap) {
            if (F.n_first != 0) sincos((double)F.n_first * phi[p], &Ei[p], &Er[p]);
            if (F.n_modes > 1) sincos((double)F.n_step * phi[p], &Di[p], &Dr[p]);
        }
    }
}

// dphi, d/dxi, d/deta, d/dphi for P markers of one triangle whose record [n_modes][21] starts at c
// (same formulas as gather()); GLOBAL: c is global memory (read-only path), else shared memory
template <int P, bool GLOBAL, bool AP>
__device__ __forceinline__ void gather_modes_impl(const FieldDev &F, const double2 *c, const double (&xi)[P],
                                                  const double (&eta)[P], const double (&phi)[P], double (&Er)[P],
                                                  double (&Ei)[P], const double (&Dr)[P], const double (&Di)[P],
                                                  double (&f)[P], double (&fx)[P], double (&fe)[P], double (&fp)[P])
{
#pragma unroll
    for (int p = 0; p < P; ++p) f[p] = fx[p] = fe[p] = fp[p] = 0.0;
    double nn = (double)F.n_first;
    const double dn = (double)F.n_step;
    const int n_modes = F.n_modes;
    int m = 0;
    if (n_modes > 0 && (AP ? F.n_first : __ldg(F.mode_n)) == 0) {      // leading n = 0 mode: E = 1, Re(P) is all that counts
        double pr[P], pxr[P], per[P];
        eval_quintic_multi_real<P, GLOBAL>(c, xi, eta, pr, pxr, per);
#pragma unroll
        for (int p = 0; p < P; ++p) {
            f[p] = pr[p]; fx[p] = pxr[p]; fe[p] = per[p];
            if (AP) { Er[p] = Dr[p]; Ei[p] = Di[p]; }                   // E_{dn} = 1 * D, exactly
        }
        if (AP) nn += dn;
        m = 1; c += NCOEF;
    }
#pragma unroll 1
    for (; m < n_modes; ++m, c += NCOEF) {
        if (!AP) {
            nn = (double)__ldg(F.mode_n + m);
#pragma unroll
            for (int p = 0; p < P; ++p) sincos(nn * phi[p], &Ei[p], &Er[p]);
        }
        double pr[P], pi[P], pxr[P], pxi[P], per[P], pei[P];
        eval_quintic_multi<P, GLOBAL>(c, xi, eta, pr, pi, pxr, pxi, per, pei);
#pragma unroll
        for (int p = 0; p < P; ++p) {
            f[p] = fma(pr[p], Er[p], fma(-pi[p], Ei[p], f[p]));
            fx[p] = fma(pxr[p], Er[p], fma(-pxi[p], Ei[p], fx[p]));
            fe[p] = fma(per[p], Er[p], fma(-pei[p], Ei[p], fe[p]));
            fp[p] = fma(-nn, fma(pi[p], Er[p], pr[p] * Ei[p]), fp[p]);          // Re(i n P E)
            if (AP) {                                                           // E_{n + dn} = E_n E_dn
                const double tr = fma(Er[p], Dr[p], -Ei[p] * Di[p]);
                Ei[p] = fma(Er[p], Di[p], Ei[p] * Dr[p]);
                Er[p] = tr;
            }
        }
        if (AP) nn += dn;
    }
}

// dphi, d/dxi, d/deta, d/dphi for P markers of one triangle whose record [n_modes][21] starts at c
// (same formulas as gather()); GLOBAL: c is global memory (read-only path), else shared memory.
// Two copies of the loop, so that the mode loop itself is free of the is_ap branch.
template <int P, bool GLOBAL>
__device__ __forceinline__ void gather_modes(const FieldDev &F, const double2 *c, const double (&xi)[P], const double (&eta)[P],
                                             const double (&phi)[P], double (&Er)[P], double (&Ei)[P], const double (&Dr)[P],
                                             const double (&Di)[P], double (&f)[P], double (&fx)[P], double (&fe)[P],
                                             double (&fp)[P])
{
    if (F.is_ap) gather_modes_impl<P, GLOBAL, true>(F, c, xi, eta, phi, Er, Ei, Dr, Di, f, fx, fe, fp);
    else gather_modes_impl<P, GLOBAL, false>(F, c, xi, eta, phi, Er, Ei, Dr, Di, f, fx, fe, fp);
}

template <int P, bool GLOBAL>
__device__ __forceinline__ void gather_multi(const FieldDev &F, const double2 *c, const double (&xi)[P], const double (&eta)[P],
                                             const double (&phi)[P], double (&f)[P], double (&fx)[P], double (&fe)[P],
                                             double (&fp)[P])
{
    double Er[P], Ei[P], Dr[P], Di[P];
    gather_phases<P>(F, phi, Er, Ei, Dr, Di);
    gather_modes<P, GLOBAL>(F, c, xi, eta, phi, Er, Ei, Dr, Di, f, fx, fe, fp);
}

}  // namespace trimeg
