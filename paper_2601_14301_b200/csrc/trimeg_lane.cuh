// trimeg_lane.cuh -- row a3 for ONE marker per lane, written for the FP64 pipe's operand port.
//
// On sm_100 the FP64 pipe reads one 64-bit register operand per cycle: a DFMA costs max(2, number of source registers
// that do not come out of the operand-reuse cache) cycles, and the reuse cache serves an operand only to the NEXT
// instruction of the same warp in the same operand slot.  A Horner step a <- a x + c has three register operands; it runs at
// the pipe's rate of one per 2 cycles only inside a run of instructions that share the multiplier x.  ptxas sets the
// .reuse flags such an order allows, but its scheduler interleaves everything that is independent (the xi-Horners of one
// marker with those of another, and with the eta-Horner), which leaves 2.5-2.65 cycles per DFMA
// (profiles/r02_mode_loop.md).  The source form here gives it nothing to interleave:
//   * one marker per evaluation (no second marker whose chains alternate with the first's);
//   * two phases: first every Horner in xi -- A_j(xi) and A_j'(xi) for the six powers of eta, 50 DFMAs that all have xi as
//     their multiplier --, then the Horner in eta for P, dP/dxi, dP/deta, 26 DFMAs that all have eta;
//   * the phases sit in different basic blocks: a branch on a condition the compiler cannot see through (always taken)
//     separates them, and its dead side reads every phase-one result, so that phase one cannot sink into the branch.
// The operations on every value, and their order, are those of eval_quintic() / gather() in trimeg_device.cuh: the
// results are bit-identical.
#pragma once
#include "trimeg_device.cuh"

namespace trimeg {

// opaque: any int >= 0 that the compiler cannot bound (mode index + a run-time zero)
__device__ __forceinline__ void eval_quintic_2ph(const double2 *__restrict__ c, double xi, double eta, int opaque,
                                                 double &pr, double &pi, double &pxr, double &pxi, double &per, double &pei)
{
    double Ar[6], Ai[6], Dr[6], Di[6];
#pragma unroll
    for (int j = 5; j >= 0; --j) {                       // phase 1: A_j(xi) = sum_i c_ij xi^i and A_j'(xi)
        const int n = 5 - j;
        double ar = 0.0, ai = 0.0, dr = 0.0, di = 0.0;
#pragma unroll
        for (int i = n; i >= 0; --i) {
            const double2 cc = c[kidx(i, j)];
            if (i == n) { ar = cc.x; ai = cc.y; }
            else {
                if (i == n - 1) { dr = ar; di = ai; }
                else { dr = fma(dr, xi, ar); di = fma(di, xi, ai); }
                ar = fma(ar, xi, cc.x); ai = fma(ai, xi, cc.y);
            }
        }
        Ar[j] = ar; Ai[j] = ai; Dr[j] = dr; Di[j] = di;
    }
    if (opaque >= 0) {                                   // phase 2: Horner in eta (always taken)
        double qr = Ar[5], qi = Ai[5], er = 0.0, ei = 0.0, xr = Dr[4], xm = Di[4];
#pragma unroll
        for (int j = 4; j >= 0; --j) {
            if (j == 4) { er = qr; ei = qi; }
            else {
                er = fma(er, eta, qr); ei = fma(ei, eta, qi);
                xr = fma(xr, eta, Dr[j]); xm = fma(xm, eta, Di[j]);
            }
            qr = fma(qr, eta, Ar[j]); qi = fma(qi, eta, Ai[j]);
        }
        pr = qr; pi = qi; pxr = xr; pxi = xm; per = er; pei = ei;
    } else {                                             // never taken: keeps phase 1 in front of the branch
        double s = 0.0;
#pragma unroll
        for (int j = 0; j < 6; ++j) s += (Ar[j] + Ai[j]) + (Dr[j] + Di[j]);
        pr = pi = pxr = pxi = per = pei = s;
    }
}

// a mode with n = 0: only Re(P) reaches the result (reading G15): the real chains alone
__device__ __forceinline__ void eval_quintic_real_2ph(const double2 *__restrict__ c, double xi, double eta, int opaque,
                                                      double &pr, double &pxr, double &per)
{
    double Ar[6], Dr[6];
#pragma unroll
    for (int j = 5; j >= 0; --j) {
        const int n = 5 - j;
        double ar = 0.0, dr = 0.0;
#pragma unroll
        for (int i = n; i >= 0; --i) {
            const double cx = c[kidx(i, j)].x;
            if (i == n) ar = cx;
            else {
                if (i == n - 1) dr = ar;
                else dr = fma(dr, xi, ar);
                ar = fma(ar, xi, cx);
            }
        }
        Ar[j] = ar; Dr[j] = dr;
    }
    if (opaque >= 0) {
        double qr = Ar[5], er = 0.0, xr = Dr[4];
#pragma unroll
        for (int j = 4; j >= 0; --j) {
            if (j == 4) er = qr;
            else { er = fma(er, eta, qr); xr = fma(xr, eta, Dr[j]); }
            qr = fma(qr, eta, Ar[j]);
        }
        pr = qr; pxr = xr; per = er;
    } else {
        double s = 0.0;
#pragma unroll
        for (int j = 0; j < 6; ++j) s += Ar[j] + Dr[j];
        pr = pxr = per = s;
    }
}

// dphi, d/dxi, d/deta, d/dphi of one marker from the record [n_modes][21] at c (shared memory): the formulas, the
// toroidal factors and the order of the accumulation are those of gather() in trimeg_device.cuh.  zero: a run-time 0.
template <bool AP>
__device__ __forceinline__ void gather_lane_impl(const FieldDev &F, const double2 *c, double xi, double eta, double phi,
                                                 int zero, double &f, double &fx, double &fe, double &fp)
{
    f = fx = fe = fp = 0.0;
    double Er = 1.0, Ei = 0.0, Dr = 1.0, Di = 0.0;
    if (AP) {
        if (F.n_first != 0) sincos((double)F.n_first * phi, &Ei, &Er);
        if (F.n_modes > 1) sincos((double)F.n_step * phi, &Di, &Dr);
    }
    double nn = (double)F.n_first;
    const double dn = (double)F.n_step;
    const int n_modes = F.n_modes;
    int m = 0;
    if (n_modes > 0 && (AP ? F.n_first : __ldg(F.mode_n)) == 0) {      // leading n = 0 mode: E = 1, Re(P) is all that counts
        eval_quintic_real_2ph(c, xi, eta, zero, f, fx, fe);
        if (AP) { Er = Dr; Ei = Di; nn += dn; }                        // E_{dn} = 1 * D, exactly
        m = 1; c += NCOEF;
    }
#pragma unroll 1
    for (int left = n_modes - m; left > 0; --left, c += NCOEF) {      // counts down: the loop test needs no bound from the constant bank
        if (!AP) { nn = (double)__ldg(F.mode_n + (n_modes - left)); sincos(nn * phi, &Ei, &Er); }
        double pr, pi, pxr, pxi, per, pei;
        eval_quintic_2ph(c, xi, eta, left + zero, pr, pi, pxr, pxi, per, pei);
        f = fma(pr, Er, fma(-pi, Ei, f));
        fx = fma(pxr, Er, fma(-pxi, Ei, fx));
        fe = fma(per, Er, fma(-pei, Ei, fe));
        fp = fma(-nn, fma(pi, Er, pr * Ei), fp);                       // Re(i n P E)
        if (AP) {                                                      // E_{n + dn} = E_n E_dn
            const double tr = fma(Er, Dr, -Ei * Di);
            Ei = fma(Er, Di, Ei * Dr);
            Er = tr;
            nn += dn;
        }
    }
}

// ---- row f3: the field on cubic B-spline toroidal planes.  Two planes take the places of the real and the imaginary part
// of a complex mode: one two-phase evaluation per pair of planes, (j0-1, j0) and (j0+1, j0+2), each plane a real record
// of 21 doubles (8-byte shared-memory loads: planes are 21 doubles apart, markers of one triangle on different planes
// read different banks).  Per-plane chains and the order of the four weighted sums are those of gather().
__device__ __forceinline__ void eval_quintic_2ph_pair(const double *__restrict__ c0, const double *__restrict__ c1, double xi,
                                                      double eta, int opaque, double &pr, double &pi, double &pxr, double &pxi,
                                                      double &per, double &pei)
{
    double Ar[6], Ai[6], Dr[6], Di[6];
#pragma unroll
    for (int j = 5; j >= 0; --j) {
        const int n = 5 - j;
        double ar = 0.0, ai = 0.0, dr = 0.0, di = 0.0;
#pragma unroll
        for (int i = n; i >= 0; --i) {
            const double cx = c0[kidx(i, j)], cy = c1[kidx(i, j)];
            if (i == n) { ar = cx; ai = cy; }
            else {
                if (i == n - 1) { dr = ar; di = ai; }
                else { dr = fma(dr, xi, ar); di = fma(di, xi, ai); }
                ar = fma(ar, xi, cx); ai = fma(ai, xi, cy);
            }
        }
        Ar[j] = ar; Ai[j] = ai; Dr[j] = dr; Di[j] = di;
    }
    if (opaque >= 0) {
        double qr = Ar[5], qi = Ai[5], er = 0.0, ei = 0.0, xr = Dr[4], xm = Di[4];
#pragma unroll
        for (int j = 4; j >= 0; --j) {
            if (j == 4) { er = qr; ei = qi; }
            else {
                er = fma(er, eta, qr); ei = fma(ei, eta, qi);
                xr = fma(xr, eta, Dr[j]); xm = fma(xm, eta, Di[j]);
            }
            qr = fma(qr, eta, Ar[j]); qi = fma(qi, eta, Ai[j]);
        }
        pr = qr; pi = qi; pxr = xr; pxi = xm; per = er; pei = ei;
    } else {
        double s = 0.0;
#pragma unroll
        for (int j = 0; j < 6; ++j) s += (Ar[j] + Ai[j]) + (Dr[j] + Di[j]);
        pr = pi = pxr = pxi = per = pei = s;
    }
}

__device__ __forceinline__ void gather_lane_spline(const FieldDev &F, const double *rec, double xi, double eta, double phi,
                                                   int zero, double &f, double &fx, double &fe, double &fp)
{
    const SplineW s = spline_weights(F.n_phi, F.inv_h, phi);
    const int ja = (s.j0 == 0) ? F.n_phi - 1 : s.j0 - 1;
    const int jc = (s.j0 + 1 == F.n_phi) ? 0 : s.j0 + 1;
    const int jd = (jc + 1 == F.n_phi) ? 0 : jc + 1;
    double pr, pi, pxr, pxi, per, pei;
    eval_quintic_2ph_pair(rec + ja * NCOEF, rec + s.j0 * NCOEF, xi, eta, s.j0 + zero, pr, pi, pxr, pxi, per, pei);
    f = s.N[0] * pr; fx = s.N[0] * pxr; fe = s.N[0] * per; fp = s.D[0] * pr;
    f = fma(s.N[1], pi, f); fx = fma(s.N[1], pxi, fx); fe = fma(s.N[1], pei, fe); fp = fma(s.D[1], pi, fp);
    eval_quintic_2ph_pair(rec + jc * NCOEF, rec + jd * NCOEF, xi, eta, jd + zero, pr, pi, pxr, pxi, per, pei);
    f = fma(s.N[2], pr, f); fx = fma(s.N[2], pxr, fx); fe = fma(s.N[2], per, fe); fp = fma(s.D[2], pr, fp);
    f = fma(s.N[3], pi, f); fx = fma(s.N[3], pxi, fx); fe = fma(s.N[3], pei, fe); fp = fma(s.D[3], pi, fp);
}

// length of a triangle's record in 16-byte units, and where it starts in the global table (harmonic or B-spline field)
__device__ __host__ __forceinline__ int lane_rec_len(const FieldDev &F) { return TRIMEG_HAS_SPL(F) ? F.n_phi * NCOEF / 2 : F.n_modes * NCOEF; }
__device__ __forceinline__ const double2 *lane_rec_src(const FieldDev &F, int t)
{
    return TRIMEG_HAS_SPL(F) ? reinterpret_cast<const double2 *>(F.spl + (size_t)t * F.n_phi * NCOEF) : F.coef + (size_t)t * F.n_modes * NCOEF;
}

// harmonic field only (the gather-alone kernel is never launched on a B-spline field)
__device__ __forceinline__ void gather_lane_harmonic(const FieldDev &F, const double2 *c, double xi, double eta, double phi, int zero,
                                                     double &f, double &fx, double &fe, double &fp)
{
    if (F.is_ap) gather_lane_impl<true>(F, c, xi, eta, phi, zero, f, fx, fe, fp);
    else gather_lane_impl<false>(F, c, xi, eta, phi, zero, f, fx, fe, fp);
}

__device__ __forceinline__ void gather_lane(const FieldDev &F, const double2 *c, double xi, double eta, double phi, int zero,
                                            double &f, double &fx, double &fe, double &fp)
{
    if (TRIMEG_HAS_SPL(F)) { gather_lane_spline(F, reinterpret_cast<const double *>(c), xi, eta, phi, zero, f, fx, fe, fp); return; }
    if (F.is_ap) gather_lane_impl<true>(F, c, xi, eta, phi, zero, f, fx, fe, fp);
    else gather_lane_impl<false>(F, c, xi, eta, phi, zero, f, fx, fe, fp);
}

}  // namespace trimeg
