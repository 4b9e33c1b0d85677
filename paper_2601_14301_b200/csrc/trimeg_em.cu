// trimeg_em.cu -- row f2 of DESIGN.md section 1: the electromagnetic terms of the thesis's push kernel and its pullback kernel.
//
// K1: one right-hand-side evaluation per marker with the three perturbed fields of the mixed-variable
// scheme -- dPhi, dA^s (symplectic part), dA^h (Hamiltonian part), dA_par = dA^s + dA^h (A.1) -- all on the
// same C1 x toroidal-harmonic basis: locate -> three gathers -> equilibrium -> b* (A.7-A.9) -> A.10-A.17 with the ideal
// Ohm's law substituted (reading G26) -> weight rate at v_par = u_par - (q/m) dA^h.  The marker's velocity coordinate is
// u_par.  K2: the pullback of u_par and w, one gather of dA^h per marker.
// One thread per marker; the three tables are read through L1 (the lanes of a warp of cell-sorted markers read the same
// records).  Fields whose table was not uploaded are identically zero.
#include "trimeg_internal.h"

namespace trimeg {

namespace {

struct Fld3 { FieldVal phi, as, ah; };

// O9 of the oracle, operation for operation up to the table-seeded reciprocals of trimeg_device.cuh
__device__ __forceinline__ Rates rhs_point_em(const PhysDev &p, double R, double Z, double upar, double mu, double w, const Fld3 &F)
{
    if (TRIMEG_HAS_EQTAB(p)) return rhs_from_eq<true>(p, eq_table(p.eq, R, Z), R, upar, mu, w, F.phi, F.as, F.ah);
    if (TRIMEG_IS_REDUCED(p)) return rhs_point_reduced<true>(p, R, Z, upar, mu, w, F.phi, F.as, F.ah);   // row f4, A.19-A.29
    const double x = R - p.R0;
    const double s = fma(x, x, Z * Z);
    const double qb = fma(p.qs, s, p.q0);
    const double iq = rcp_fast(qb);
    const double iq2 = iq * iq;
    const double g = fma(s, iq2, p.R0sq);
    const double gs = iq2 * fma(s * p.m2qs, iq, 1.0);
    const double isg = rsqrt_fast(g);
    const double sg = g * isg;
    const double ig = isg * isg;
    const double h = iq * isg;
    const double hs = -h * fma(0.5 * gs, ig, p.qs * iq);
    const double iR = rcp_fast(R);
    const double u = p.B0 * iR;
    const double B = u * sg;
    const double iB = (R * p.invB0) * isg;
    const double uq = u * iq;
    const double bR = -Z * h, bZ = x * h, bphi = p.R0 * isg;
    const double gsi = gs * isg;
    const double ug = u * gsi;
    const double dBdZ = ug * Z;
    const double dBdR = fma(ug, x, -(B * iR));
    const double dc = -(p.R0 * gsi) * ig;
    const double curlR = -dc * Z;
    const double curlZ = fma(dc, x, bphi * iR);
    const double curlP = -2.0 * fma(s, hs, h);
    const double ev = p.eps * upar;
    const double Bsp = fma(ev, fma(bR, curlR, fma(bZ, curlZ, bphi * curlP)), B);
    const double iBsp = rcp_fast(Bsp);
    const double k = ev * iBsp;
    const double lead = (p.eom_variant == 1) ? B * iBsp : 1.0;
    const double b0R = fma(lead, bR, k * curlR), b0Z = fma(lead, bZ, k * curlZ), b0P = fma(lead, bphi, k * curlP);   // A.4-A.6
    const double CE = p.rho0B0 * iBsp;
    const double Cd = ((p.eps * mu) * iB) * iBsp;
    // b* = b0* + C_E grad(dA^s) x b (A.7-A.9); (grad f)_phi = (1/R) d f/d phi
    const double AsP = F.as.fphi * iR, AhP = F.ah.fphi * iR, PhP = F.phi.fphi * iR;
    const double bsR = fma(CE, fma(bZ, AsP, -bphi * F.as.fZ), b0R);
    const double bsZ = fma(CE, fma(bphi, F.as.fR, -bR * AsP), b0Z);
    const double bsP = fma(CE, fma(bR, F.as.fZ, -bZ * F.as.fR), b0P);
    // grad-B drift (A.10-A.12; sign of A.11 as reading G1), equilibrium part
    const double CdBphi = Cd * (u * p.R0);
    const double Rmu = CdBphi * dBdZ, Zmu = -CdBphi * dBdR;
    const double Pmu_R = (Cd * uq) * fma(x, dBdR, Z * dBdZ);          // R phidot_mu
    const double R0dot = fma(b0R, upar, Rmu), Z0dot = fma(b0Z, upar, Zmu), P0 = fma(b0P, upar, Pmu_R);
    const double u0dot = -mu * fma(b0R, dBdR, b0Z * dBdZ);
    // perturbed part: dG = dPhi - u_par (dA^s + dA^h) (A.14-A.16)
    const double GR = fma(-upar, F.as.fR + F.ah.fR, F.phi.fR), GZ = fma(-upar, F.as.fZ + F.ah.fZ, F.phi.fZ);
    const double GP = fma(-upar, AsP + AhP, PhP);
    const double qA = p.qom * F.ah.f;
    const double dRdot = fma(CE, fma(bphi, GZ, -bZ * GP), -qA * bsR);
    const double dZdot = fma(CE, fma(-bphi, GR, bR * GP), -qA * bsZ);
    const double dP = fma(CE, fma(bZ, GR, -bR * GZ), -qA * bsP);      // R dphidot
    // A.17 with Ohm's law: -(q/m) [ (b* - b).grad dPhi - u_par b*.grad dA^h ] - (v_mu . grad) dA^s
    const double t1 = fma(bsR - bR, F.phi.fR, fma(bsZ - bZ, F.phi.fZ, (bsP - bphi) * PhP));
    const double t2 = fma(bsR, F.ah.fR, fma(bsZ, F.ah.fZ, bsP * AhP));
    const double dudot = fma(-p.qom, fma(-upar, t2, t1), -fma(Rmu, F.as.fR, fma(Zmu, F.as.fZ, Pmu_R * AsP)));
    // weight rate at the physical velocity
    const double vpar = upar - qA;
    const double ir = (s > 1e-300) ? rsqrt_fast(s) : 0.0;
    const double drdot = fma(dRdot, x, dZdot * Z) * ir;
    const double en = fma(vpar * vpar, p.invT, fma(mu * B, p.invT2, -1.5));
    const double L = fma(drdot, -fma(en, p.kappa_T, p.kappa_n),
                         fma(-(mu * p.invT2), fma(dRdot, dBdR, dZdot * dBdZ), -(vpar * p.invT2) * dudot));
    Rates o;
    o.R = R0dot + dRdot;
    o.Z = Z0dot + dZdot;
    o.phi = iR * (P0 + dP);
    o.vpar = u0dot + dudot;
    o.w = (p.weight_mode == 0) ? (w - 1.0) * L : -L;
    return o;
}

__device__ __forceinline__ FieldVal gather_or_zero(const FieldDev &F, const double2 *table, int t, const Bary &b, double phi)
{
    FieldVal v;
    v.f = v.fR = v.fZ = v.fphi = 0.0;
    if (table == nullptr || F.n_modes == 0) return v;
    FieldDev G = F;
    G.coef = table;
    return gather(G, t, b, phi);
}

__global__ void __launch_bounds__(128) rhs_em_kernel(MeshDev M, FieldDev F, const double2 *tab_as, const double2 *tab_ah, PhysDev P,
                                                     trimeg_markers m, size_t n, double *__restrict__ dR, double *__restrict__ dZ,
                                                     double *__restrict__ dP, double *__restrict__ dU, double *__restrict__ dW)
{
    const size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n) return;
    Rates k;
    k.R = k.Z = k.phi = k.vpar = k.w = 0.0;
    const int hint = m.cell ? m.cell[p] : -1;
    Bary b;
    int moved = 0;
    const double R = m.R[p], Z = m.Z[p];
    const int t = locate(M, R, Z, hint, b, moved);
    if (t >= 0) {
        const double phi = m.phi[p];
        Fld3 f;
        f.phi = gather_or_zero(F, F.coef, t, b, phi);
        f.as = gather_or_zero(F, tab_as, t, b, phi);
        f.ah = gather_or_zero(F, tab_ah, t, b, phi);
        k = rhs_point_em(P, R, Z, m.vpar[p], m.mu[p], m.w[p], f);
    }
    dR[p] = k.R; dZ[p] = k.Z; dP[p] = k.phi; dU[p] = k.vpar; dW[p] = k.w;
}

// K2: u_new = u_old - (q/m) dA^h;  w_new = w_old - (2 q/T) u_new dA^h (1 - w_old)  [weight_mode 1: x 1]  (O10, readings G7, G27)
__global__ void __launch_bounds__(256) pullback_kernel(MeshDev M, FieldDev F, const double2 *tab_ah, PhysDev P, trimeg_markers m, size_t n)
{
    const size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n) return;
    const int hint = m.cell[p];
    if (hint < 0) return;                                // flagged: left untouched
    Bary b;
    int moved = 0;
    const int t = locate(M, m.R[p], m.Z[p], hint, b, moved);
    if (t < 0) return;
    const double Ah = gather_or_zero(F, tab_ah, t, b, m.phi[p]).f;
    const double w0 = m.w[p];
    const double unew = m.vpar[p] - P.qom * Ah;
    const double fac = (P.weight_mode == 0) ? (1.0 - w0) : 1.0;
    m.w[p] = w0 - (P.qom * P.invT2) * unew * Ah * fac;
    m.vpar[p] = unew;
}

}  // namespace

#ifdef TRIMEG_CORE_ONLY
cudaError_t launch_rhs_em_core(trimeg_ctx *c, const trimeg_markers &m, size_t n, double *dR, double *dZ, double *dP, double *dU, double *dW,
                               cudaStream_t s)
#else
cudaError_t launch_rhs_em(trimeg_ctx *c, const trimeg_markers &m, size_t n, double *dR, double *dZ, double *dP, double *dU, double *dW,
                          cudaStream_t s)
#endif
{
    if (n == 0) return cudaSuccess;
#ifndef TRIMEG_CORE_ONLY
    if (core_case(c)) return launch_rhs_em_core(c, m, n, dR, dZ, dP, dU, dW, s);   // the same kernel without the branches of row f4
#endif
    rhs_em_kernel<<<(unsigned)((n + 127) / 128), 128, 0, s>>>(c->mesh, c->field, c->d_coef_aux[0], c->d_coef_aux[1], c->phys, m, n, dR, dZ, dP,
                                                             dU, dW);
    c->n_launches++;
    return cudaGetLastError();
}

#ifndef TRIMEG_CORE_ONLY
cudaError_t launch_pullback(trimeg_ctx *c, const trimeg_markers &m, size_t n, cudaStream_t s)
{
    if (n == 0 || c->d_coef_aux[1] == nullptr) return cudaSuccess;       // no dA^h: nothing to pull back
    pullback_kernel<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(c->mesh, c->field, c->d_coef_aux[1], c->phys, m, n);
    c->n_launches++;
    return cudaGetLastError();
}

#endif

}  // namespace trimeg
