// trimeg_device.cuh -- device-side building blocks of the marker push (sm_100a, fp64).
//
// Rows of DESIGN.md §1: a2 locator, a3 field gather, a4 equilibrium, a5 RHS assembly.
// Citations: PAPER.md:<line> = /root/reference/PAPER.md; readings G*/L*/O* = DESIGN.md §3.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace trimeg {

constexpr int NCOEF = 21;
// A candidate triangle is accepted without looking at any other one only if the marker is
// inside it by this margin in barycentric units (rule L3).  Rounding errors of the test are
// <~ 1e-13 even on the thinnest axis-fan triangles, so a triangle passing with this margin is
// the only one whose contains() test can pass.
constexpr double LOC_TAU = 1e-9;
constexpr int LOC_MAX_HOPS = 8;

struct MeshDev {
    int n_r, n_theta, n_tri;
    const double *geom;     // [n_tri][6]  R_v0, Z_v0, xi_R, xi_Z, eta_R, eta_Z
    const double *r_nodes;  // [n_r + 1]
    double Rax, Zax;        // axis vertex
    double rin2;            // squared inscribed radius of the outer polygon (gap rule, O3)
    // row f4, unstructured triangulation (n_r == 0): neighbour table and the thesis's box grid
    const int *nbr;         // [n_tri][3] triangle across the edge where barycentric coordinate 0 / 1 / 2 vanishes, -1 = boundary
    const int *box_off;     // [nbx * nby + 1]
    const int *box_tri;     // triangles whose (inflated) bounding box overlaps the box, ascending
    int nbx, nby;
    double bx0, bz0, inv_bdx, inv_bdz;
};
constexpr double LOC_GAP_TOL = 1e-12;   // reading G31
// A translation unit compiled with TRIMEG_CORE_ONLY (trimeg_push_*_core.cu) holds the hot kernels for the core case alone --
// ring x sector mesh, harmonic field, rigorous equations -- without the branches of rows f3 / f4 (they cost 0.9 % of the push
// although never taken: code size and register allocation); the launchers pick it when the context is in that case.
// TRIMEG_SPLINE_ONLY (trimeg_push_lane_spline.cu): the same for row f3 -- ring x sector mesh, field on B-spline planes,
// rigorous equations, analytic equilibrium (the general build of the lane kernel spills with row f4's branches in it).
#if defined(TRIMEG_CORE_ONLY)
#define TRIMEG_HAS_SPL(F) false
#define TRIMEG_IS_REDUCED(p) false
#define TRIMEG_IS_UNS(M) false
#define TRIMEG_HAS_EQTAB(p) false
#elif defined(TRIMEG_SPLINE_ONLY)
#define TRIMEG_HAS_SPL(F) true
#define TRIMEG_IS_REDUCED(p) false
#define TRIMEG_IS_UNS(M) false
#define TRIMEG_HAS_EQTAB(p) false
#else
#define TRIMEG_HAS_EQTAB(p) ((p).eq != nullptr)
#define TRIMEG_HAS_SPL(F) ((F).n_phi > 0)
#define TRIMEG_IS_REDUCED(p) ((p).eom_variant == 2)
#define TRIMEG_IS_UNS(M) ((M).n_r == 0)
#endif

struct FieldDev {
    int n_modes;
    const double2 *coef;    // [n_tri][n_modes][21] (re, im)
    const int *mode_n;      // [n_modes] (device)
    int n_first, n_step;    // arithmetic progression n_k = n_first + k n_step if is_ap
    int is_ap;
    // row f3: cubic B-spline toroidal basis.  n_phi > 0: the field is
    // sum_j N_j(phi) P_j(xi, eta) on n_phi uniform periodic planes (then n_modes == 0)
    int n_phi;
    const double *spl;      // [n_tri][n_phi][21] real
    double inv_h;           // n_phi / (2 pi)
};

struct PhysDev {
    double R0, B0, invB0, q0, qs;   // qs = q2 / a^2 = d q / d s,  s = r^2
    double eps;                     // (m_s/q_s) rho_0 B_0  (reading G23)
    double rho0B0;                  // numerator of C_E
    double qom;                     // q_s / m_s
    double invT, kappa_n, kappa_T;
    double R0sq, m2qs, invT2;       // R0^2, -2 qs, 2 / T
    int eom_variant, weight_mode;
    // row f4: equilibrium from cubic-B-spline tables of psi(R, Z) and F(psi) (reading G32), a
    // descriptor in device memory (kept out of the kernel parameters: the hot kernels' code does not change with it);
    // NULL: the analytic circular equilibrium above
    const struct EqTabDev *eq;
};
struct EqTabDev {
    int eq_nR, eq_nZ, eq_nF;
    double eq_Ra, eq_Za, eq_ihR, eq_ihZ, eq_pa, eq_ihp;   // first knot positions, reciprocal spacings
    const double *eq_C, *eq_D;      // [nR][nZ], [nF] coefficients
};

// --------------------------------------------------------------------------- a2 locator
// contains() of PAPER.md:291 in local coordinates, every operation individually rounded
// in the fixed order of reading O3 / rule L2 (no fused multiply-add).
struct Bary {
    double xi, eta, l0;
    double xR, xZ, eR, eZ;   // xi_R, xi_Z, eta_R, eta_Z of the triangle
};

__device__ __forceinline__ Bary bary_rn(const MeshDev &M, int t, double R, double Z)
{
    const double2 *g = reinterpret_cast<const double2 *>(M.geom + 6 * (size_t)t);
    const double2 v0 = __ldg(g), gx = __ldg(g + 1), ge = __ldg(g + 2);
    Bary b;
    const double dx = __dsub_rn(R, v0.x), dz = __dsub_rn(Z, v0.y);
    b.xi = __dadd_rn(__dmul_rn(gx.x, dx), __dmul_rn(gx.y, dz));
    b.eta = __dadd_rn(__dmul_rn(ge.x, dx), __dmul_rn(ge.y, dz));
    b.l0 = __dsub_rn(__dsub_rn(1.0, b.xi), b.eta);
    b.xR = gx.x; b.xZ = gx.y; b.eR = ge.x; b.eZ = ge.y;
    return b;
}

// Triangle across the edge on which barycentric coordinate `which` vanishes
// (0: lambda0, 1: xi, 2: eta); -1 = across the outer boundary.  Closed form on the
// ring x sector numbering (O1).
__device__ __forceinline__ int neighbour(const MeshDev &M, int t, int which)
{
    if (TRIMEG_IS_UNS(M)) return __ldg(M.nbr + 3 * (size_t)t + which);
    const int nth = M.n_theta;
    if (t < nth) {                                   // axis fan, sector j = t
        if (which == 0) return nth + 2 * t + 1;      // outer chord -> ring 1, k = 1
        if (which == 1) return (t + 1 == nth) ? 0 : t + 1;
        return (t == 0) ? nth - 1 : t - 1;
    }
    const int u = t - nth, k = u & 1, c = u >> 1;
    const int i = c / nth + 1, j = c - (i - 1) * nth;
    if (k == 0) {                                    // (v(i,j), v(i+1,j), v(i+1,j+1))
        if (which == 0) return (i + 1 <= M.n_r - 1) ? nth + 2 * (i * nth + j) + 1 : -1;
        if (which == 1) return t + 1;
        const int jm = (j == 0) ? nth - 1 : j - 1;
        return nth + 2 * ((i - 1) * nth + jm) + 1;
    }
    // k == 1: (v(i,j), v(i+1,j+1), v(i,j+1))
    if (which == 0) { const int jp = (j + 1 == nth) ? 0 : j + 1; return nth + 2 * ((i - 1) * nth + jp); }
    if (which == 1) return (i >= 2) ? nth + 2 * ((i - 2) * nth + j) : j;
    return t - 1;
}

// (r, theta) ring / sector guess: only ever selects CANDIDATES (rule L1).
static __device__ __noinline__ void ring_sector_guess(const MeshDev &M, double R, double Z, int &i0, int &j0)
{
    const double x = R - M.Rax, z = Z - M.Zax;
    const double r = sqrt(x * x + z * z);
    double th = atan2(z, x);
    if (th < 0.0) th += 6.283185307179586476925286766559;
    int lo = 0, hi = M.n_r;                          // largest i with r_nodes[i] <= r
    while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (__ldg(M.r_nodes + mid) <= r) lo = mid; else hi = mid; }
    i0 = lo;
    double jf = floor(th * (double)M.n_theta * 0.15915494309189533576888376337251);
    if (!(jf >= 0.0 && jf < (double)M.n_theta)) jf = 0.0;
    j0 = (int)jf;
}

// Unstructured mesh: the box of the point, its triangles in ascending order, first one whose test passes; if none passes
// the one with the largest smallest barycentric coordinate when that is >= -LOC_GAP_TOL (reading G31).  Same decisions as
// the rule over all triangles: every triangle that can pass (or come within the gap tolerance) at a point of the box is
// in the box's list (bounding boxes inflated by 1e-6 of the box size).
static __device__ __noinline__ int locate_box(const MeshDev &M, double R, double Z, Bary &out)
{
    const double fx = floor((R - M.bx0) * M.inv_bdx), fz = floor((Z - M.bz0) * M.inv_bdz);
    if (!(fx >= -1.0 && fx <= (double)M.nbx && fz >= -1.0 && fz <= (double)M.nby)) return -1;      // also NaN
    int i = (int)fx, j = (int)fz;
    i = max(0, min(M.nbx - 1, i)); j = max(0, min(M.nby - 1, j));
    const int b = j * M.nbx + i;
    const int q0 = __ldg(M.box_off + b), q1 = __ldg(M.box_off + b + 1);
    int gap_best = -1;
    double gap_m = -INFINITY;
    Bary gb;
    gb.xi = gb.eta = gb.l0 = gb.xR = gb.xZ = gb.eR = gb.eZ = 0.0;
#pragma unroll 1
    for (int q = q0; q < q1; ++q) {
        const int t = __ldg(M.box_tri + q);
        const Bary bb = bary_rn(M, t, R, Z);
        if (bb.xi >= 0.0 && bb.eta >= 0.0 && bb.l0 >= 0.0) { out = bb; return t; }
        const double m = fmin(fmin(bb.xi, bb.eta), bb.l0);
        if (m > gap_m) { gap_m = m; gap_best = t; gb = bb; }
    }
    if (gap_best >= 0 && gap_m >= -LOC_GAP_TOL) { out = gb; return gap_best; }
    return -1;
}

// The complete rule of reading O3 on the 3x3 cell neighbourhood of the guess: lowest t whose
// test passes; if none passes, the gap rule.  Same decisions as a brute-force search.
static __device__ __noinline__ int locate_full(const MeshDev &M, double R, double Z, Bary &out)
{
    if (TRIMEG_IS_UNS(M)) return locate_box(M, R, Z, out);
    int i0, j0;
    ring_sector_guess(M, R, Z, i0, j0);
    int best = -1, gap_best = -1;
    double gap_m = -INFINITY;
    Bary bb, gb;
    bb.xi = bb.eta = bb.l0 = bb.xR = bb.xZ = bb.eR = bb.eZ = 0.0;
    gb = bb;
    for (int ii = i0 - 1; ii <= i0 + 1; ++ii) {
        if (ii < 0 || ii > M.n_r - 1) continue;
        for (int dj = -1; dj <= 1; ++dj) {
            int jj = j0 + dj;
            if (jj < 0) jj += M.n_theta;
            if (jj >= M.n_theta) jj -= M.n_theta;
            const int base = (ii == 0) ? jj : M.n_theta + 2 * ((ii - 1) * M.n_theta + jj);
            const int cnt = (ii == 0) ? 1 : 2;
            for (int k = 0; k < cnt; ++k) {
                const int t = base + k;
                const Bary b = bary_rn(M, t, R, Z);
                const double m = fmin(fmin(b.xi, b.eta), b.l0);
                if (b.xi >= 0.0 && b.eta >= 0.0 && b.l0 >= 0.0) {
                    if (best < 0 || t < best) { best = t; bb = b; }
                }
                if (m > gap_m || (m == gap_m && t < gap_best)) { gap_m = m; gap_best = t; gb = b; }
            }
        }
    }
    if (best >= 0) { out = bb; return best; }
    const double x = __dsub_rn(R, M.Rax), z = __dsub_rn(Z, M.Zax);
    const double s = __dadd_rn(__dmul_rn(x, x), __dmul_rn(z, z));
    if (s < M.rin2) { out = gb; return gap_best; }
    return -1;
}

// Locator used on the hot path: hinted triangle first, then a walk across the violated
// edge (closed-form neighbours), complete rule only for markers within LOC_TAU of an edge.
// Returns the triangle or -1 (outside the outer polygon); `moved` is set when the hint was left.
__device__ __forceinline__ int locate(const MeshDev &M, double R, double Z, int hint, Bary &out, int &moved)
{
    int t = hint;
    if (t < 0 || t >= M.n_tri) {
        if (TRIMEG_IS_UNS(M)) { moved = 1; return locate_full(M, R, Z, out); }
        int i0, j0;
        ring_sector_guess(M, R, Z, i0, j0);
        if (i0 > M.n_r - 1) i0 = M.n_r - 1;
        t = (i0 == 0) ? j0 : M.n_theta + 2 * ((i0 - 1) * M.n_theta + j0);
    }
#pragma unroll 1
    for (int hop = 0; hop < LOC_MAX_HOPS; ++hop) {
        const Bary b = bary_rn(M, t, R, Z);
        const double m = fmin(fmin(b.xi, b.eta), b.l0);
        if (m > LOC_TAU) { out = b; return t; }
        if (!(m < -LOC_TAU)) break;                   // within TAU of an edge (or NaN): full rule
        const int which = (b.l0 <= b.xi && b.l0 <= b.eta) ? 0 : ((b.xi <= b.eta) ? 1 : 2);
        const int tn = neighbour(M, t, which);
        moved = 1;
        if (tn < 0) return -1;                        // beyond an outer chord by a clear margin
        t = tn;
    }
    moved = 1;
    return locate_full(M, R, Z, out);
}

// --------------------------------------------------------------------------- a3 gather
// One toroidal mode: complex quintic P and its xi / eta derivatives by bivariate Horner with
// the product rule (76 real FMAs), coefficients degree-major k(i,j) = d(d+1)/2 + j, d = i+j.
struct Cplx { double re, im; };

__device__ __forceinline__ constexpr int kidx(int i, int j) { return (i + j) * (i + j + 1) / 2 + j; }

__device__ __forceinline__ void eval_quintic(const double2 *__restrict__ c, double xi, double eta,
                                             Cplx &P, Cplx &Px, Cplx &Pe)
{
    double pr = 0.0, pi = 0.0, pxr = 0.0, pxi = 0.0, per = 0.0, pei = 0.0;
#pragma unroll
    for (int j = 5; j >= 0; --j) {
        // A_j(xi) = sum_i c_ij xi^i and A_j'(xi), i = 0 .. 5-j
        const int n = 5 - j;
        double2 top = __ldg(c + kidx(n, j));
        double ar = top.x, ai = top.y, dr = 0.0, di = 0.0;
#pragma unroll
        for (int i = n - 1; i >= 0; --i) {
            const double2 cc = __ldg(c + kidx(i, j));
            if (i == n - 1) { dr = ar; di = ai; }
            else { dr = fma(dr, xi, ar); di = fma(di, xi, ai); }
            ar = fma(ar, xi, cc.x); ai = fma(ai, xi, cc.y);
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
    P.re = pr; P.im = pi; Px.re = pxr; Px.im = pxi; Pe.re = per; Pe.im = pei;
}

// A real quintic (the real chains of eval_quintic alone), coefficient k at c[k * STRIDE].
template <int STRIDE>
__device__ __forceinline__ void eval_quintic_real_s(const double *__restrict__ c, double xi, double eta,
                                                    double &P, double &Px, double &Pe)
{
    double pr = 0.0, pxr = 0.0, per = 0.0;
#pragma unroll
    for (int j = 5; j >= 0; --j) {
        const int n = 5 - j;
        double ar = __ldg(c + STRIDE * kidx(n, j)), dr = 0.0;
#pragma unroll
        for (int i = n - 1; i >= 0; --i) {
            const double cx = __ldg(c + STRIDE * kidx(i, j));
            if (i == n - 1) dr = ar;
            else dr = fma(dr, xi, ar);
            ar = fma(ar, xi, cx);
        }
        if (j == 5) pr = ar;
        else {
            if (j == 4) { per = pr; pxr = dr; }
            else { per = fma(per, eta, pr); pxr = fma(pxr, eta, dr); }
            pr = fma(pr, eta, ar);
        }
    }
    P = pr; Px = pxr; Pe = per;
}
// A mode with n = 0: only Re(P) reaches the result (reading G15).
__device__ __forceinline__ void eval_quintic_real(const double2 *__restrict__ c, double xi, double eta,
                                                  double &P, double &Px, double &Pe)
{
    eval_quintic_real_s<2>(reinterpret_cast<const double *>(c), xi, eta, P, Px, Pe);
}

// Row f3: the four cubic B-splines that are non-zero at phi (reading G28: N_j(phi) = beta(phi/h - j), h = 2 pi/n_phi,
// periodic in j) and their phi-derivatives.  With x = phi/h, j0 = floor(x), t = x - j0 in [0, 1):
//   planes j0-1, j0, j0+1, j0+2 carry beta(t+1), beta(t), beta(t-1), beta(t-2).
struct SplineW { int j0; double N[4], D[4]; };
__device__ __forceinline__ SplineW spline_weights(int n_phi, double inv_h, double phi)
{
    SplineW s;
    const double x = phi * inv_h;
    const double fl = floor(x);
    const double t = x - fl, u = 1.0 - t;
    const double np = (double)n_phi;
    s.j0 = (int)(fl - np * floor(fl / np));
    if (s.j0 >= n_phi) s.j0 -= n_phi;                      // fl / np rounded up to an integer
    if (s.j0 < 0) s.j0 += n_phi;
    const double t2 = t * t, u2 = u * u;
    s.N[0] = u2 * u * (1.0 / 6.0);
    s.N[1] = fma(t2, fma(0.5, t, -1.0), 2.0 / 3.0);
    s.N[2] = fma(u2, fma(0.5, u, -1.0), 2.0 / 3.0);
    s.N[3] = t2 * t * (1.0 / 6.0);
    s.D[0] = -0.5 * u2 * inv_h;
    s.D[1] = t * fma(1.5, t, -2.0) * inv_h;
    s.D[2] = -u * fma(1.5, u, -2.0) * inv_h;
    s.D[3] = 0.5 * t2 * inv_h;
    return s;
}

struct FieldVal { double f, fR, fZ, fphi; };   // dphi, d/dR, d/dZ, d/dphi

// dphi = sum_n Re(P_n E_n), E_n = e^{i n phi}; no factor 2, Im of n = 0 ignored (G15).
__device__ __forceinline__ FieldVal gather(const FieldDev &F, int t, const Bary &b, double phi)
{
    double f = 0.0, fx = 0.0, fe = 0.0, fp = 0.0;
    if (TRIMEG_HAS_SPL(F)) {
        const SplineW s = spline_weights(F.n_phi, F.inv_h, phi);
        const double *base = F.spl + (size_t)t * F.n_phi * NCOEF;
        int j = (s.j0 == 0) ? F.n_phi - 1 : s.j0 - 1;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            double P, Px, Pe;
            eval_quintic_real_s<1>(base + j * NCOEF, b.xi, b.eta, P, Px, Pe);
            f = fma(s.N[k], P, f); fx = fma(s.N[k], Px, fx); fe = fma(s.N[k], Pe, fe); fp = fma(s.D[k], P, fp);
            j = (j + 1 == F.n_phi) ? 0 : j + 1;
        }
    } else if (F.n_modes > 0) {
        const double2 *c = F.coef + (size_t)t * F.n_modes * NCOEF;
        double Er, Ei, Dr = 1.0, Di = 0.0;
        if (F.is_ap) {
            if (F.n_first == 0) { Er = 1.0; Ei = 0.0; }
            else sincos((double)F.n_first * phi, &Ei, &Er);
            if (F.n_modes > 1) sincos((double)F.n_step * phi, &Di, &Dr);
        } else { Er = 1.0; Ei = 0.0; }
        double nn = (double)F.n_first;
        int m = 0;
        if ((F.is_ap ? F.n_first : __ldg(F.mode_n)) == 0) {      // leading n = 0 mode: E = 1, real part only
            eval_quintic_real(c, b.xi, b.eta, f, fx, fe);
            if (F.is_ap) { Er = Dr; Ei = Di; nn += (double)F.n_step; }
            m = 1; c += NCOEF;
        }
#pragma unroll 1
        for (; m < F.n_modes; ++m, c += NCOEF) {
            if (!F.is_ap) { nn = (double)__ldg(F.mode_n + m); sincos(nn * phi, &Ei, &Er); }
            Cplx P, Px, Pe;
            eval_quintic(c, b.xi, b.eta, P, Px, Pe);
            f = fma(P.re, Er, fma(-P.im, Ei, f));
            fx = fma(Px.re, Er, fma(-Px.im, Ei, fx));
            fe = fma(Pe.re, Er, fma(-Pe.im, Ei, fe));
            fp = fma(-nn, fma(P.im, Er, P.re * Ei), fp);          // Re(i n P E)
            if (F.is_ap) {                                        // E_{n + dn} = E_n E_dn
                const double tr = fma(Er, Dr, -Ei * Di);
                Ei = fma(Er, Di, Ei * Dr);
                Er = tr;
                nn += (double)F.n_step;
            }
        }
    }
    FieldVal v;
    v.f = f;
    v.fR = fma(b.xR, fx, b.eR * fe);
    v.fZ = fma(b.xZ, fx, b.eZ * fe);
    v.fphi = fp;
    return v;
}

// ------------------------------------------------------------------- a4 + a5 equilibrium, RHS
// Reciprocal and reciprocal square root without the IEEE division sequence: the hardware's 20-bit table seed
// (MUFU.RCP64H / MUFU.RSQ64H, which runs beside the FP64 pipe) and ONE third-order correction step
// (2^-20 -> 2^-60 relative), branch-free: 3 (5) FP64 instructions instead of ~12 with a slow-path test.  The result is
// within ~1.5 ulp of the exact value (parity bar 1e-12).  Arguments are normal positive numbers here (R, q, g, B*_par, s).
__device__ __forceinline__ double rcp_fast(double x)
{
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double e = fma(-x, y, 1.0);
    return fma(y, fma(e, e, e), y);                      // y (1 + e + e^2)
}
__device__ __forceinline__ double rsqrt_fast(double x)
{
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double e = fma(-(x * y), y, 1.0);
    return fma(y, e * fma(0.375, e, 0.5), y);            // y (1 + e/2 + 3 e^2/8)
}

// Analytic circular equilibrium: psi' = B0 r / q(r), F = B0 R0 (G11), B = grad psi x grad phi
// + F grad phi; b0* (A.4-A.6), equilibrium drifts (A.10-A.13, sign of
// A.11 per G1), E x B and parallel acceleration (A.14-A.17 with dA = 0, G3), weight rate from
// d ln f_M/dt (kappa_X along -rhat, G6/G10).
struct Rates { double R, Z, phi, vpar, w; };

// ---- row f4: tabulated equilibrium.  psi(R, Z) = sum C[i][j] beta((R - Ra)/hR - i) beta((Z - Za)/hZ - j), F(psi) likewise in one
// dimension; B_R = -psi_Z/R, B_Z = psi_R/R, B_phi = F/R; |B|, grad B, b and curl b from the first and second
// derivatives by the quotient rule.  The sixteen (four) non-zero terms; the caller guarantees that the mesh lies where the
// 4 x 4 stencil is inside the table (checked at upload); the F index is clamped (the end pieces extend as cubics).
struct EqVal { double B, BR, BZ, BP, bR, bZ, bphi, dBdR, dBdZ, curlR, curlZ, curlP, psiR, psiZ; };

__device__ __forceinline__ void bspl4(double t, double ih, double N[4], double D1[4], double D2[4])
{
    const double u = 1.0 - t, t2 = t * t, u2 = u * u;
    N[0] = u2 * u * (1.0 / 6.0); N[1] = fma(t2, fma(0.5, t, -1.0), 2.0 / 3.0); N[2] = fma(u2, fma(0.5, u, -1.0), 2.0 / 3.0); N[3] = t2 * t * (1.0 / 6.0);
    D1[0] = -0.5 * u2 * ih; D1[1] = t * fma(1.5, t, -2.0) * ih; D1[2] = -u * fma(1.5, u, -2.0) * ih; D1[3] = 0.5 * t2 * ih;
    const double ih2 = ih * ih;
    D2[0] = u * ih2; D2[1] = fma(3.0, t, -2.0) * ih2; D2[2] = fma(3.0, u, -2.0) * ih2; D2[3] = t * ih2;
}

static __device__ __noinline__ EqVal eq_table(const EqTabDev *__restrict__ q, double R, double Z)
{
    const EqTabDev p = *q;
    const double xr = (R - p.eq_Ra) * p.eq_ihR, xz = (Z - p.eq_Za) * p.eq_ihZ;
    const double fr = floor(xr), fz = floor(xz);
    int i0 = (int)fr, j0 = (int)fz;
    i0 = max(1, min(p.eq_nR - 3, i0)); j0 = max(1, min(p.eq_nZ - 3, j0));
    double NR[4], DR[4], ER[4], NZ[4], DZ[4], EZ[4];
    bspl4(xr - (double)i0, p.eq_ihR, NR, DR, ER);
    bspl4(xz - (double)j0, p.eq_ihZ, NZ, DZ, EZ);
    double psi = 0.0, pR = 0.0, pZ = 0.0, pRR = 0.0, pRZ = 0.0, pZZ = 0.0;
#pragma unroll
    for (int a = 0; a < 4; ++a) {
        const double *row = p.eq_C + (size_t)(i0 - 1 + a) * p.eq_nZ + (j0 - 1);
        double s0 = 0.0, s1 = 0.0, s2 = 0.0;             // sum over Z of the row with beta, beta', beta''
#pragma unroll
        for (int b = 0; b < 4; ++b) {
            const double c = __ldg(row + b);
            s0 = fma(c, NZ[b], s0); s1 = fma(c, DZ[b], s1); s2 = fma(c, EZ[b], s2);
        }
        psi = fma(NR[a], s0, psi); pR = fma(DR[a], s0, pR); pRR = fma(ER[a], s0, pRR);
        pZ = fma(NR[a], s1, pZ); pRZ = fma(DR[a], s1, pRZ); pZZ = fma(NR[a], s2, pZZ);
    }
    const double xp = (psi - p.eq_pa) * p.eq_ihp;
    int k0 = (int)floor(xp);
    k0 = max(1, min(p.eq_nF - 3, k0));
    double NF[4], DF[4], EF[4];
    bspl4(xp - (double)k0, p.eq_ihp, NF, DF, EF);
    double F = 0.0, Fp = 0.0;
#pragma unroll
    for (int k = 0; k < 4; ++k) { const double d = __ldg(p.eq_D + k0 - 1 + k); F = fma(d, NF[k], F); Fp = fma(d, DF[k], Fp); }
    const double iR = 1.0 / R, iR2 = iR * iR;
    EqVal e;
    e.BR = -pZ * iR; e.BZ = pR * iR; e.BP = F * iR;
    const double BR_R = fma(-pRZ, iR, pZ * iR2), BR_Z = -pZZ * iR;
    const double BZ_R = fma(pRR, iR, -pR * iR2), BZ_Z = pRZ * iR;
    const double BP_R = fma(Fp * pR, iR, -F * iR2), BP_Z = Fp * pZ * iR;
    e.B = sqrt(fma(e.BR, e.BR, fma(e.BZ, e.BZ, e.BP * e.BP)));
    const double iB = 1.0 / e.B;
    e.dBdR = fma(e.BR, BR_R, fma(e.BZ, BZ_R, e.BP * BP_R)) * iB;
    e.dBdZ = fma(e.BR, BR_Z, fma(e.BZ, BZ_Z, e.BP * BP_Z)) * iB;
    e.bR = e.BR * iB; e.bZ = e.BZ * iB; e.bphi = e.BP * iB;
    const double dbR_dZ = fma(-e.bR, e.dBdZ, BR_Z) * iB, dbZ_dR = fma(-e.bZ, e.dBdR, BZ_R) * iB;
    const double dbP_dR = fma(-e.bphi, e.dBdR, BP_R) * iB, dbP_dZ = fma(-e.bphi, e.dBdZ, BP_Z) * iB;
    e.curlR = -dbP_dZ;                                   // brackets of A.4-A.6
    e.curlZ = fma(e.bphi, iR, dbP_dR);
    e.curlP = dbR_dZ - dbZ_dR;
    e.psiR = pR; e.psiZ = pZ;
    return e;
}

// The equations of every variant on a general equilibrium value, as the oracle states them (O6, O9, O12): rigorous (0, 1) and
// reduced (2), electrostatic (EM = false: A.17 / A.28 with dA = 0) and electromagnetic under the ideal Ohm's law.  The
// profile gradients act along grad psi (reading G32).
template <bool EM>
__device__ __forceinline__ Rates rhs_from_eq(const PhysDev &p, const EqVal &e, double R, double upar, double mu, double w,
                                             const FieldVal &Phi, const FieldVal &As, const FieldVal &Ah)
{
    const double iR = 1.0 / R;
    const bool reduced = p.eom_variant == 2;
    const double iB = 1.0 / e.B;
    const double ev = p.eps * upar;
    const double Bsp = reduced ? e.B : fma(ev, fma(e.bR, e.curlR, fma(e.bZ, e.curlZ, e.bphi * e.curlP)), e.B);
    const double iBsp = 1.0 / Bsp;
    const double k = reduced ? 0.0 : ev * iBsp;
    const double lead = (p.eom_variant == 1) ? e.B * iBsp : 1.0;
    const double b0R = fma(lead, e.bR, k * e.curlR), b0Z = fma(lead, e.bZ, k * e.curlZ), b0P = fma(lead, e.bphi, k * e.curlP);
    const double CE = p.rho0B0 * iBsp;
    // drift coefficient: rigorous eps mu/(B B*par), reduced eps (u^2 + mu B)/B^3
    const double Cmu = reduced ? p.eps * mu * iB * iB : p.eps * mu * iB * iBsp;
    const double Cd = reduced ? p.eps * fma(upar, upar, mu * e.B) * iB * iB * iB : Cmu;
    const double xR = e.BP * e.dBdZ, xZ = -e.BP * e.dBdR, xP = fma(e.BZ, e.dBdR, -e.BR * e.dBdZ);   // B x grad B
    const double R0dot = fma(b0R, upar, Cd * xR), Z0dot = fma(b0Z, upar, Cd * xZ), P0 = fma(b0P, upar, Cd * xP);
    const double u0dot = -mu * fma(b0R, e.dBdR, b0Z * e.dBdZ);
    const double PhP = Phi.fphi * iR;
    double dRdot, dZdot, dP, dudot, vpar = upar;
    if (EM) {
        const double AsP = As.fphi * iR, AhP = Ah.fphi * iR;
        const double bsR = reduced ? e.bR : fma(CE, fma(e.bZ, AsP, -e.bphi * As.fZ), b0R);      // b* (A.7-A.9); reduced: b
        const double bsZ = reduced ? e.bZ : fma(CE, fma(e.bphi, As.fR, -e.bR * AsP), b0Z);
        const double bsP = reduced ? e.bphi : fma(CE, fma(e.bR, As.fZ, -e.bZ * As.fR), b0P);
        const double GR = fma(-upar, As.fR + Ah.fR, Phi.fR), GZ = fma(-upar, As.fZ + Ah.fZ, Phi.fZ), GP = fma(-upar, AsP + AhP, PhP);
        const double qA = p.qom * Ah.f;
        dRdot = fma(CE, fma(e.bphi, GZ, -e.bZ * GP), -qA * bsR);
        dZdot = fma(CE, fma(-e.bphi, GR, e.bR * GP), -qA * bsZ);
        dP = fma(CE, fma(e.bZ, GR, -e.bR * GZ), -qA * bsP);
        const double t1 = reduced ? 0.0 : fma(bsR - e.bR, Phi.fR, fma(bsZ - e.bZ, Phi.fZ, (bsP - e.bphi) * PhP));
        const double t2 = fma(bsR, Ah.fR, fma(bsZ, Ah.fZ, bsP * AhP));
        dudot = fma(-p.qom, fma(-upar, t2, t1), -Cmu * fma(xR, As.fR, fma(xZ, As.fZ, xP * AsP)));
        vpar = upar - qA;
    } else {
        dRdot = CE * fma(e.bphi, Phi.fZ, -e.bZ * PhP);
        dZdot = CE * fma(-e.bphi, Phi.fR, e.bR * PhP);
        dP = CE * fma(e.bZ, Phi.fR, -e.bR * Phi.fZ);
        dudot = -p.qom * fma(b0R, Phi.fR, fma(b0Z, Phi.fZ, b0P * PhP));
    }
    const double g2 = fma(e.psiR, e.psiR, e.psiZ * e.psiZ);
    const double drdot = (g2 > 0.0) ? fma(dRdot, e.psiR, dZdot * e.psiZ) * rsqrt(g2) : 0.0;
    const double en = fma(vpar * vpar, p.invT, fma(mu * e.B, p.invT2, -1.5));
    const double L = fma(drdot, -fma(en, p.kappa_T, p.kappa_n),
                         fma(-(mu * p.invT2), fma(dRdot, e.dBdR, dZdot * e.dBdZ), -(vpar * p.invT2) * dudot));
    Rates o;
    o.R = R0dot + dRdot;
    o.Z = Z0dot + dZdot;
    o.phi = iR * (P0 + dP);
    o.vpar = u0dot + dudot;
    o.w = (p.weight_mode == 0) ? (w - 1.0) * L : -L;
    return o;
}

// Row f4, eom_variant 2: the reduced equations A.19-A.29 ("only the dominant terms ... replacing b* with b",
// PAPER.md:1276-1307; readings G29, G30): R0dot = u b + C_d B x grad B with C_d = eps (u^2 + mu B)/B^3, u0dot = -mu b.grad B,
// dRdot = C_E b x grad(dG) - (q/m) dA^h b with C_E = rho_0 B_0/B, dudot = -(q/m)[b.grad dPhi - u b.grad dA^h] - v_mu.grad dA^s
// (A.28); EM = true: dA^s, dA^h present and the parallel electric field cancelled by the ideal Ohm's law (A.29).
template <bool EM>
__device__ __forceinline__ Rates rhs_point_reduced(const PhysDev &p, double R, double Z, double upar, double mu, double w,
                                                   const FieldVal &Phi, const FieldVal &As, const FieldVal &Ah)
{
    const double x = R - p.R0;
    const double s = fma(x, x, Z * Z);
    const double qb = fma(p.qs, s, p.q0);
    const double iq = rcp_fast(qb);
    const double iq2 = iq * iq;
    const double g = fma(s, iq2, p.R0sq);
    const double gs = iq2 * fma(s * p.m2qs, iq, 1.0);
    const double isg = rsqrt_fast(g);
    const double sg = g * isg;
    const double h = iq * isg;
    const double iR = rcp_fast(R);
    const double u = p.B0 * iR;
    const double B = u * sg;
    const double iB = (R * p.invB0) * isg;
    const double uq = u * iq;                            // B_Z = uq x, B_R = -uq Z
    const double bR = -Z * h, bZ = x * h, bphi = p.R0 * isg;
    const double ug = u * (gs * isg);
    const double dBdZ = ug * Z;
    const double dBdR = fma(ug, x, -(B * iR));
    const double iB2 = iB * iB;
    const double eB3 = p.eps * (iB2 * iB);               // (m/q) rho_0 B_0 / B^3
    const double Cd = eB3 * fma(upar, upar, mu * B);
    const double CE = p.rho0B0 * iB;
    const double Bphi = u * p.R0;
    const double xR = Bphi * dBdZ, xZ = -Bphi * dBdR;    // (B x grad B)_R, _Z
    const double xP = uq * fma(x, dBdR, Z * dBdZ);       // (B x grad B)_phi = B_Z dB/dR - B_R dB/dZ
    const double R0dot = fma(bR, upar, Cd * xR);         // A.19
    const double Z0dot = fma(bZ, upar, Cd * xZ);         // A.20
    const double P0 = fma(bphi, upar, Cd * xP);          // A.21 (times R)
    const double u0dot = -mu * fma(bR, dBdR, bZ * dBdZ); // A.22 (G29)
    const double PhP = Phi.fphi * iR;
    double dRdot, dZdot, dP, dudot, vpar;
    if (EM) {
        const double AsP = As.fphi * iR, AhP = Ah.fphi * iR;
        const double GR = fma(-upar, As.fR + Ah.fR, Phi.fR), GZ = fma(-upar, As.fZ + Ah.fZ, Phi.fZ);
        const double GP = fma(-upar, AsP + AhP, PhP);
        const double qA = p.qom * Ah.f;
        dRdot = fma(CE, fma(bphi, GZ, -bZ * GP), -qA * bR);          // A.24
        dZdot = fma(CE, fma(-bphi, GR, bR * GP), -qA * bZ);          // A.25
        dP = fma(CE, fma(bZ, GR, -bR * GZ), -qA * bphi);             // A.26 (times R)
        const double Cmu = eB3 * (mu * B);
        const double t2 = fma(bR, Ah.fR, fma(bZ, Ah.fZ, bphi * AhP));
        dudot = fma(p.qom * upar, t2, -Cmu * fma(xR, As.fR, fma(xZ, As.fZ, xP * AsP)));   // A.29
        vpar = upar - qA;
    } else {
        dRdot = CE * fma(bphi, Phi.fZ, -bZ * PhP);
        dZdot = CE * fma(-bphi, Phi.fR, bR * PhP);
        dP = CE * fma(bZ, Phi.fR, -bR * Phi.fZ);
        dudot = -p.qom * fma(bR, Phi.fR, fma(bZ, Phi.fZ, bphi * PhP));                    // A.28, dA = 0
        vpar = upar;
    }
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

__device__ __forceinline__ Rates rhs_point(const PhysDev &p, double R, double Z, double vpar, double mu,
                                           double w, const FieldVal &fld)
{
    if (TRIMEG_HAS_EQTAB(p)) return rhs_from_eq<false>(p, eq_table(p.eq, R, Z), R, vpar, mu, w, fld, fld, fld);
    if (TRIMEG_IS_REDUCED(p)) return rhs_point_reduced<false>(p, R, Z, vpar, mu, w, fld, fld, fld);
    const double x = R - p.R0;
    const double s = fma(x, x, Z * Z);
    const double qb = fma(p.qs, s, p.q0);
    const double iq = rcp_fast(qb);
    const double iq2 = iq * iq;
    const double g = fma(s, iq2, p.R0sq);
    const double gs = iq2 * fma(s * p.m2qs, iq, 1.0);    // dg/ds = 1/q^2 - 2 s q_s/q^3
    const double isg = rsqrt_fast(g);
    const double sg = g * isg;
    const double ig = isg * isg;
    const double h = iq * isg;
    const double hs = -h * fma(0.5 * gs, ig, p.qs * iq);
    const double iR = rcp_fast(R);
    const double u = p.B0 * iR;                          // B0 / R
    const double B = u * sg;
    const double iB = (R * p.invB0) * isg;
    const double uq = u * iq;                            // B_Z = uq x, B_R = -uq Z
    const double bR = -Z * h, bZ = x * h, bphi = p.R0 * isg;
    const double gsi = gs * isg;
    const double ug = u * gsi;
    const double dBdZ = ug * Z;
    const double dBdR = fma(ug, x, -(B * iR));
    const double dc = -(p.R0 * gsi) * ig;                // d b_phi / d s * 2 ... times x or Z
    const double curlR = -dc * Z;                        // -(d b_phi/dZ)
    const double curlZ = fma(dc, x, bphi * iR);          //  d b_phi/dR + b_phi/R
    const double curlP = -2.0 * fma(s, hs, h);           //  d b_R/dZ - d b_Z/dR
    const double bcurlb = fma(bR, curlR, fma(bZ, curlZ, bphi * curlP));
    const double ev = p.eps * vpar;
    const double Bsp = fma(ev, bcurlb, B);               // B*_par
    const double iBsp = rcp_fast(Bsp);
    const double k = ev * iBsp;
    double b0R, b0Z, b0P;
    if (p.eom_variant == 1) {
        const double lead = B * iBsp;
        b0R = fma(lead, bR, k * curlR); b0Z = fma(lead, bZ, k * curlZ); b0P = fma(lead, bphi, k * curlP);
    } else {
        b0R = fma(k, curlR, bR); b0Z = fma(k, curlZ, bZ); b0P = fma(k, curlP, bphi);
    }
    const double Cd = ((p.eps * mu) * iB) * iBsp;
    const double CE = p.rho0B0 * iBsp;
    const double CdBphi = Cd * (u * p.R0);
    const double R0dot = fma(b0R, vpar, CdBphi * dBdZ);
    const double Z0dot = fma(b0Z, vpar, -CdBphi * dBdR);
    const double P0 = fma(b0P, vpar, (Cd * uq) * fma(x, dBdR, Z * dBdZ));     // R dphi/dt, equilibrium part (B_Z dB/dR - B_R dB/dZ = uq (x dB/dR + Z dB/dZ))
    const double v0dot = -mu * fma(b0R, dBdR, b0Z * dBdZ);
    const double fP_R = fld.fphi * iR;                   // (1/R) d dphi / d phi
    const double dRdot = CE * fma(bphi, fld.fZ, -bZ * fP_R);
    const double dZdot = CE * fma(-bphi, fld.fR, bR * fP_R);
    const double dP = fma(bZ, fld.fR, -bR * fld.fZ);     // R dphi/dt / C_E, perturbed part
    const double dvdot = -p.qom * fma(b0R, fld.fR, fma(b0Z, fld.fZ, b0P * fP_R));
    const double ir = (s > 1e-300) ? rsqrt_fast(s) : 0.0;
    const double drdot = fma(dRdot, x, dZdot * Z) * ir;
    const double en = fma(vpar * vpar, p.invT, fma(mu * B, p.invT2, -1.5));
    const double L = fma(drdot, -fma(en, p.kappa_T, p.kappa_n),
                         fma(-(mu * p.invT2), fma(dRdot, dBdR, dZdot * dBdZ), -(vpar * p.invT2) * dvdot));
    Rates o;
    o.R = R0dot + dRdot;
    o.Z = Z0dot + dZdot;
    o.phi = iR * fma(CE, dP, P0);
    o.vpar = v0dot + dvdot;
    o.w = (p.weight_mode == 0) ? (w - 1.0) * L : -L;
    return o;
}

}  // namespace trimeg
