/*
 * trimeg_oracle.c -- CPU ORACLE for the TRIMEG marker-push hot path.
 *
 * THIS FILE IS TEST INFRASTRUCTURE.  It is a plain, slow, fp64 restatement of
 * what the path computes, written from the paper (/root/reference/PAPER.md,
 * cited below as PAPER.md:<line>) and from the readings fixed in SURVEY.md
 * §8(c) / DESIGN.md §3.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may call it.  It shares NO code,
 * header, table or helper with the CUDA library (paper_2601_14301_b200/csrc);
 * the only thing both consume is the seeded input generator
 * (paper_2601_14301_b200/inputs.py), which holds no method arithmetic.
 *
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC (see oracle/build.py).
 * -ffp-contract=off is part of the definition of the locator (rule L2): every
 * operation of inside() is individually rounded, in the order written here.
 *
 * Parity unpinned (defined by SURVEY.md, not by the paper): the form of the
 * weight equation (G7) and the profile-gradient conventions (G10).  Everything
 * else is pinned by tests/test_oracle_*.py against closed forms, invariants,
 * finite differences and brute force.
 *
 * What is computed, in the paper's order (push kernel):
 *   O1 mesh            ring x sector triangulation, local coordinates (xi, eta)
 *                      with vertices at (0,0),(1,0),(0,1)
 *   O2 Bell expansion  18 nodal DOFs (6 per vertex)  -> 21 monomial coefficients
 *                      of the quintic
 *   O3 locator         brute force and the O(1) candidate search
 *                      with contains()
 *   O4 gather (g2p)    dphi, d/dR, d/dZ, d/dphi at the marker PAPER.md:235, 604
 *   O5 equilibrium     B = grad psi x grad phi + F grad phi PAPER.md:1156-1164
 *   O6 RHS             A.4-A.6, A.10-A.17 (dA = 0), d ln f_M/dt
 *                                                     PAPER.md:1204-1269
 *   O7 RK4             classic 4-stage integrator
 *   O8 scatter (p2g)   projection of the marker weights onto the same basis: the adjoint of O4
 *                                                           PAPER.md:232, 249
 *   O9 EM RHS          one right-hand side with dA^s, dA^h (mixed variables): A.7-A.9, A.14-A.17 with the
 *                      ideal Ohm's law substituted
 *   O10 pullback       u_par, w after the pullback transformation
 *   O11 spline basis   the thesis's own toroidal discretisation: cubic B-splines in phi instead of harmonics
 *                                                           PAPER.md:223, 365-368
 *   O13 general mesh   unstructured triangulation with the thesis's box-grid locator
 *   O14 tabulated eq.  equilibrium from cubic-B-spline tables of psi(R, Z) and F(psi)
 *   O12 reduced model  eom_variant 2: the "dominant terms" equations A.19-A.29 (b* -> b)
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_NCOEF 21
#define ORC_TWO_PI 6.283185307179586476925286766559

typedef struct {
    double R0, a, B0, q0, q2;      /* circular equilibrium, q(r) = q0 + q2 (r/a)^2 */
    double rho0, qs_over_ms;       /* rho_0, q_s/m_s               */
    double T, kappa_n, kappa_T;    /* Tbar, log-gradients (1/length) */
    int eom_variant;               /* 0 = b0* as printed (A.4-A.6); 1 = (B/B*par) b + ... (reading G2); 2 = reduced model A.19-A.29 (O12) */
    int weight_mode;               /* 0: wdot = -(1-w) L ; 1: wdot = -L (reading G7) */
} orc_params;

struct orc_eqtab;
typedef struct {
    int n_r, n_theta, n_vert, n_tri;
    double *r_nodes;               /* n_r + 1 */
    double *Rv, *Zv;               /* n_vert  */
    int *tri;                      /* [n_tri][3] vertex ids, counter-clockwise */
    double *geom;                  /* [n_tri][6] R_v0, Z_v0, xi_R, xi_Z, eta_R, eta_Z */
    double rin2;                   /* squared inscribed radius of the outer polygon */
    orc_params p;
    int n_modes;
    int *mode_n;                   /* toroidal mode numbers n (Def. 19) */
    double *coef;                  /* [n_tri][n_modes][21][2] (re, im) */
    double **basis;                /* O8: per triangle, lazily, [21][18] monomial coefficients of the 18 basis functions */
    double *coef_aux[2];           /* O9/O10: dA^s (0) and dA^h (1), same layout and mode list as coef; NULL = identically zero */
    /* O13: unstructured mesh (n_r == 0): box grid of PAPER.md:261-291, 602 in CSR form */
    int nbx, nby;                  /* boxes in R and Z */
    double bx0, bz0, bdx, bdz;     /* lower-left corner of the grid, box sizes */
    int *box_off, *box_tri;        /* [nbx*nby + 1], triangle lists (ascending) */
    struct orc_eqtab *eq;          /* O14: tabulated (psi, F) equilibrium, NULL = the analytic circular one */
    int n_phi;                     /* O11: > 0 = the field is Y = sum_j N_j(phi) P_j(xi, eta) on n_phi toroidal planes */
    double *coef_spl;              /* [n_tri][n_phi][21] real monomial coefficients, one quintic per triangle and plane */
} orc_ctx;

/* ------------------------------------------------------------------ O1 mesh */
static int vid(const orc_ctx *c, int i, int j)
{ /* v(i,j) = 1 + (i-1) n_theta + (j mod n_theta), i = 1..n_r */
    int jj = ((j % c->n_theta) + c->n_theta) % c->n_theta;
    return 1 + (i - 1) * c->n_theta + jj;
}

orc_ctx *orc_create(int n_r, int n_theta, const double *r_nodes,
                    const double *Rv, const double *Zv, const orc_params *p)
{
    if (n_r < 2 || n_theta < 3) return NULL;
    orc_ctx *c = (orc_ctx *)calloc(1, sizeof(orc_ctx));
    c->n_r = n_r; c->n_theta = n_theta;
    c->n_vert = 1 + n_r * n_theta;
    c->n_tri = (2 * n_r - 1) * n_theta;
    c->p = *p;
    c->r_nodes = (double *)malloc(sizeof(double) * (n_r + 1));
    memcpy(c->r_nodes, r_nodes, sizeof(double) * (n_r + 1));
    c->Rv = (double *)malloc(sizeof(double) * c->n_vert);
    c->Zv = (double *)malloc(sizeof(double) * c->n_vert);
    memcpy(c->Rv, Rv, sizeof(double) * c->n_vert);
    memcpy(c->Zv, Zv, sizeof(double) * c->n_vert);
    c->tri = (int *)malloc(sizeof(int) * 3 * c->n_tri);
    c->geom = (double *)malloc(sizeof(double) * 6 * c->n_tri);
    /* fan: t = j : (axis, v(1,j), v(1,j+1)) */
    for (int j = 0; j < n_theta; ++j) {
        int *t = c->tri + 3 * j;
        t[0] = 0; t[1] = vid(c, 1, j); t[2] = vid(c, 1, j + 1);
    }
    /* rings i = 1..n_r-1, two triangles per ring-sector quad */
    for (int i = 1; i <= n_r - 1; ++i)
        for (int j = 0; j < n_theta; ++j) {
            int base = n_theta + 2 * ((i - 1) * n_theta + j);
            int *t0 = c->tri + 3 * base, *t1 = c->tri + 3 * (base + 1);
            t0[0] = vid(c, i, j); t0[1] = vid(c, i + 1, j);     t0[2] = vid(c, i + 1, j + 1);
            t1[0] = vid(c, i, j); t1[1] = vid(c, i + 1, j + 1); t1[2] = vid(c, i, j + 1);
        }
    /* local coordinates: vertices map to (xi,eta) = (0,0),(1,0),(0,1) */
    for (int t = 0; t < c->n_tri; ++t) {
        const int *v = c->tri + 3 * t;
        double R0 = c->Rv[v[0]], Z0 = c->Zv[v[0]];
        double e1R = c->Rv[v[1]] - R0, e1Z = c->Zv[v[1]] - Z0;
        double e2R = c->Rv[v[2]] - R0, e2Z = c->Zv[v[2]] - Z0;
        double D = e1R * e2Z - e2R * e1Z;
        double *g = c->geom + 6 * t;
        g[0] = R0; g[1] = Z0;
        g[2] = e2Z / D;      /* xi_R  */
        g[3] = -e2R / D;     /* xi_Z  */
        g[4] = -e1Z / D;     /* eta_R */
        g[5] = e1R / D;      /* eta_Z */
    }
    /* inscribed radius of the outer polygon = distance axis -> midpoint of an outer chord */
    {
        int va = vid(c, n_r, 0), vb = vid(c, n_r, 1);
        double mx = 0.5 * (c->Rv[va] + c->Rv[vb]) - c->Rv[0];
        double mz = 0.5 * (c->Zv[va] + c->Zv[vb]) - c->Zv[0];
        c->rin2 = mx * mx + mz * mz;
    }
    return c;
}

void orc_destroy(orc_ctx *c);
void orc_set_equilibrium_table(orc_ctx *c, int nR, int nZ, double Ra, double Za, double hR, double hZ, const double *C,
                               int nF, double pa, double hp, const double *D);
static int inside(const orc_ctx *c, int t, double R, double Z, double *xi, double *eta, double *lam0);
static double min3(double a, double b, double c);
/* ------------------------------------------------- O13 unstructured mesh + box-grid locator */
/* "An intermediate grid ... of bounding boxes, where each element is itself a vector storing all the triangular elements that
 * overlap with the corresponding box"; the search discretises the particle position to a box "in O(1) time" and loops over
 * the box's triangles calling the inside-triangle test until one contains the particle.
 * Triangles: any conforming triangulation, vertices counter-clockwise (a clockwise triple is turned).  Lists are ascending in
 * t, so the first hit is the lowest index (reading O3 as on the structured mesh).  A triangle is entered in every box its
 * bounding box, inflated by 1e-6 of the box size, overlaps.  Reading G31 (no passage fixes what happens on an edge where
 * rounding fails both neighbours' tests): if no triangle of the box passes, the one with the largest smallest barycentric
 * coordinate is taken when that coordinate is >= -1e-12, else the marker is outside (-1).  The definition the grid is pinned
 * against is the same rule over ALL triangles (orc_locate_brute). */
#define ORC_GAP_TOL 1e-12
orc_ctx *orc_create_unstructured(int n_vert, const double *Rv, const double *Zv, int n_tri, const int *tri, int nbx, int nby,
                                 const orc_params *p)
{
    if (n_vert < 3 || n_tri < 1 || nbx < 1 || nby < 1) return NULL;
    orc_ctx *c = (orc_ctx *)calloc(1, sizeof(orc_ctx));
    c->n_r = 0; c->n_theta = 0; c->n_vert = n_vert; c->n_tri = n_tri; c->p = *p;
    c->Rv = (double *)malloc(sizeof(double) * n_vert); c->Zv = (double *)malloc(sizeof(double) * n_vert);
    memcpy(c->Rv, Rv, sizeof(double) * n_vert); memcpy(c->Zv, Zv, sizeof(double) * n_vert);
    c->tri = (int *)malloc(sizeof(int) * 3 * n_tri);
    memcpy(c->tri, tri, sizeof(int) * 3 * n_tri);
    c->geom = (double *)malloc(sizeof(double) * 6 * n_tri);
    double lo[2] = {INFINITY, INFINITY}, hi[2] = {-INFINITY, -INFINITY};
    for (int v = 0; v < n_vert; ++v) {
        if (Rv[v] < lo[0]) lo[0] = Rv[v];
        if (Rv[v] > hi[0]) hi[0] = Rv[v];
        if (Zv[v] < lo[1]) lo[1] = Zv[v];
        if (Zv[v] > hi[1]) hi[1] = Zv[v];
    }
    for (int t = 0; t < n_tri; ++t) {
        int *v = c->tri + 3 * t;
        for (int q = 0; q < 3; ++q) if (v[q] < 0 || v[q] >= n_vert) { orc_destroy(c); return NULL; }
        double e1R = Rv[v[1]] - Rv[v[0]], e1Z = Zv[v[1]] - Zv[v[0]], e2R = Rv[v[2]] - Rv[v[0]], e2Z = Zv[v[2]] - Zv[v[0]];
        double D = e1R * e2Z - e2R * e1Z;
        if (D == 0.0) { orc_destroy(c); return NULL; }
        if (D < 0.0) { int tmp = v[1]; v[1] = v[2]; v[2] = tmp; double a = e1R, b = e1Z; e1R = e2R; e1Z = e2Z; e2R = a; e2Z = b; D = -D; }
        double *g = c->geom + 6 * t;
        g[0] = Rv[v[0]]; g[1] = Zv[v[0]];
        g[2] = e2Z / D; g[3] = -e2R / D; g[4] = -e1Z / D; g[5] = e1R / D;
    }
    c->nbx = nbx; c->nby = nby;
    c->bx0 = lo[0]; c->bz0 = lo[1];
    c->bdx = (hi[0] - lo[0]) / nbx; c->bdz = (hi[1] - lo[1]) / nby;
    const int nb = nbx * nby;
    c->box_off = (int *)calloc((size_t)nb + 1, sizeof(int));
    for (int pass = 0; pass < 2; ++pass) {              /* count, then fill; t ascending keeps every list sorted */
        int *fill = (pass == 1) ? (int *)calloc((size_t)nb, sizeof(int)) : NULL;
        for (int t = 0; t < n_tri; ++t) {
            const int *v = c->tri + 3 * t;
            double tl[2] = {INFINITY, INFINITY}, th[2] = {-INFINITY, -INFINITY};
            for (int q = 0; q < 3; ++q) {
                if (Rv[v[q]] < tl[0]) tl[0] = Rv[v[q]];
                if (Rv[v[q]] > th[0]) th[0] = Rv[v[q]];
                if (Zv[v[q]] < tl[1]) tl[1] = Zv[v[q]];
                if (Zv[v[q]] > th[1]) th[1] = Zv[v[q]];
            }
            int i0 = (int)floor((tl[0] - c->bx0) / c->bdx - 1e-6), i1 = (int)floor((th[0] - c->bx0) / c->bdx + 1e-6);
            int j0 = (int)floor((tl[1] - c->bz0) / c->bdz - 1e-6), j1 = (int)floor((th[1] - c->bz0) / c->bdz + 1e-6);
            if (i0 < 0) i0 = 0;
            if (j0 < 0) j0 = 0;
            if (i1 > nbx - 1) i1 = nbx - 1;
            if (j1 > nby - 1) j1 = nby - 1;
            for (int i = i0; i <= i1; ++i)
                for (int j = j0; j <= j1; ++j) {
                    const int b = j * nbx + i;
                    if (pass == 0) c->box_off[b + 1]++;
                    else c->box_tri[c->box_off[b] + fill[b]++] = t;
                }
        }
        if (pass == 0) {
            for (int b = 0; b < nb; ++b) c->box_off[b + 1] += c->box_off[b];
            c->box_tri = (int *)malloc(sizeof(int) * (size_t)(c->box_off[nb] > 0 ? c->box_off[nb] : 1));
        } else free(fill);
    }
    return c;
}
/* the rule over an index list (all triangles when list == NULL) */
static int locate_list(const orc_ctx *c, const int *list, int n, double R, double Z, double *xi_out, double *eta_out)
{
    double xi, eta, l0, bm = -INFINITY, bxi = 0.0, bet = 0.0;
    int best = -1;
    for (int q = 0; q < n; ++q) {
        const int t = list ? list[q] : q;
        if (inside(c, t, R, Z, &xi, &eta, &l0)) { if (xi_out) { *xi_out = xi; *eta_out = eta; } return t; }
        const double m = min3(xi, eta, l0);
        if (m > bm) { bm = m; best = t; bxi = xi; bet = eta; }       /* first (lowest t) of equal margins */
    }
    if (best >= 0 && bm >= -ORC_GAP_TOL) { if (xi_out) { *xi_out = bxi; *eta_out = bet; } return best; }
    return -1;
}
static int locate_box(const orc_ctx *c, double R, double Z, double *xi_out, double *eta_out)
{
    const double fx = floor((R - c->bx0) / c->bdx), fz = floor((Z - c->bz0) / c->bdz);
    if (!(fx >= -1.0 && fx <= (double)c->nbx && fz >= -1.0 && fz <= (double)c->nby)) return -1;       /* also NaN */
    int i = (int)fx, j = (int)fz;
    if (i < 0) i = 0;                                   /* points on (or a rounding beyond) the outer frame */
    if (i > c->nbx - 1) i = c->nbx - 1;
    if (j < 0) j = 0;
    if (j > c->nby - 1) j = c->nby - 1;
    const int b = j * c->nbx + i;
    return locate_list(c, c->box_tri + c->box_off[b], c->box_off[b + 1] - c->box_off[b], R, Z, xi_out, eta_out);
}
int orc_box_count(const orc_ctx *c) { return c->box_off ? c->box_off[c->nbx * c->nby] : 0; }

void orc_destroy(orc_ctx *c)
{
    if (!c) return;
    free(c->box_off); free(c->box_tri);
    orc_set_equilibrium_table(c, 0, 0, 0, 0, 0, 0, NULL, 0, 0, 0, NULL);
    free(c->r_nodes); free(c->Rv); free(c->Zv); free(c->tri); free(c->geom);
    if (c->basis) { for (int t = 0; t < c->n_tri; ++t) free(c->basis[t]); free(c->basis); }
    free(c->coef_aux[0]); free(c->coef_aux[1]); free(c->coef_spl);
    free(c->mode_n); free(c->coef); free(c);
}

int orc_n_tri(const orc_ctx *c) { return c->n_tri; }
int orc_n_vert(const orc_ctx *c) { return c->n_vert; }
void orc_get_tri(const orc_ctx *c, int *out) { memcpy(out, c->tri, sizeof(int) * 3 * c->n_tri); }
void orc_get_geom(const orc_ctx *c, double *out) { memcpy(out, c->geom, sizeof(double) * 6 * c->n_tri); }
double orc_get_rin2(const orc_ctx *c) { return c->rin2; }
void orc_set_params(orc_ctx *c, const orc_params *p) { c->p = *p; }

void orc_set_modes(orc_ctx *c, int n_modes, const int *mode_n)
{
    free(c->mode_n); free(c->coef);
    free(c->coef_aux[0]); free(c->coef_aux[1]); c->coef_aux[0] = c->coef_aux[1] = NULL;
    c->n_modes = n_modes;
    c->mode_n = (int *)malloc(sizeof(int) * (n_modes > 0 ? n_modes : 1));
    if (n_modes > 0) memcpy(c->mode_n, mode_n, sizeof(int) * n_modes);
    c->coef = (double *)calloc((size_t)c->n_tri * (n_modes > 0 ? n_modes : 1) * ORC_NCOEF * 2, sizeof(double));
}
void orc_set_coef(orc_ctx *c, const double *coef)
{ memcpy(c->coef, coef, sizeof(double) * (size_t)c->n_tri * c->n_modes * ORC_NCOEF * 2); }
void orc_get_coef(const orc_ctx *c, double *coef)
{ memcpy(coef, c->coef, sizeof(double) * (size_t)c->n_tri * c->n_modes * ORC_NCOEF * 2); }

/* ------------------------------------------------- O2 Bell reduced quintic */
/* monomial order, degree-major: k = 0..20 <-> (i,j): for d = 0..5, for j = 0..d: (d-j, j) */
static void mono_ij(int k, int *i, int *j)
{
    int d = 0, kk = k;
    while (kk > d) { kk -= d + 1; ++d; }
    *j = kk; *i = d - kk;
}
static long double ipowl(long double x, int n) { long double r = 1.0L; while (n-- > 0) r *= x; return r; }
static double ipow(double x, int n) { double r = 1.0; while (n-- > 0) r *= x; return r; }
static int falling(int i, int a) { int r = 1; for (int q = 0; q < a; ++q) r *= (i - q); return r; }
/* d^a/dxi^a d^b/deta^b of xi^i eta^j at (xi,eta); 0^0 = 1 */
static long double mono_derivl(int i, int j, int a, int b, long double xi, long double eta)
{
    if (a > i || b > j) return 0.0L;
    return (long double)falling(i, a) * ipowl(xi, i - a) * (long double)falling(j, b) * ipowl(eta, j - b);
}

/* Build the 21x21 matrix of one triangle (rows 1-18: six DOFs of PAPER.md:350-353 at the
 * three vertices; rows 19-21: the quartic term of the normal derivative vanishes on each
 * edge -- the textbook Bell reduction 21 -> 18, reading O2), row-equilibrate, LU-factor with
 * partial pivoting in long double. */
static int bell_factor(const orc_ctx *c, int t, long double A[21][21], long double rowscale[21], int piv[21])
{
    const double *g = c->geom + 6 * t;
    const int *v = c->tri + 3 * t;
    long double xR = g[2], xZ = g[3], eR = g[4], eZ = g[5];
    static const long double vx[3] = {0.0L, 1.0L, 0.0L}, ve[3] = {0.0L, 0.0L, 1.0L};
    for (int pnt = 0; pnt < 3; ++pnt)
        for (int k = 0; k < 21; ++k) {
            int i, j; mono_ij(k, &i, &j);
            long double P   = mono_derivl(i, j, 0, 0, vx[pnt], ve[pnt]);
            long double Px  = mono_derivl(i, j, 1, 0, vx[pnt], ve[pnt]);
            long double Pe  = mono_derivl(i, j, 0, 1, vx[pnt], ve[pnt]);
            long double Pxx = mono_derivl(i, j, 2, 0, vx[pnt], ve[pnt]);
            long double Pxe = mono_derivl(i, j, 1, 1, vx[pnt], ve[pnt]);
            long double Pee = mono_derivl(i, j, 0, 2, vx[pnt], ve[pnt]);
            A[6 * pnt + 0][k] = P;                                              /* f    */
            A[6 * pnt + 1][k] = xR * Px + eR * Pe;                              /* f_R  */
            A[6 * pnt + 2][k] = xZ * Px + eZ * Pe;                              /* f_Z  */
            A[6 * pnt + 3][k] = xR * xR * Pxx + 2.0L * xR * eR * Pxe + eR * eR * Pee;            /* f_RR */
            A[6 * pnt + 4][k] = xR * xZ * Pxx + (xR * eZ + xZ * eR) * Pxe + eR * eZ * Pee;       /* f_RZ */
            A[6 * pnt + 5][k] = xZ * xZ * Pxx + 2.0L * xZ * eZ * Pxe + eZ * eZ * Pee;            /* f_ZZ */
        }
    /* edges a->b with reference direction (dxi, deta) */
    static const int ea[3] = {0, 0, 1}, eb[3] = {1, 2, 2};
    static const long double dxi[3] = {1.0L, 0.0L, -1.0L}, det[3] = {0.0L, 1.0L, 1.0L};
    for (int e = 0; e < 3; ++e) {
        long double tR = (long double)c->Rv[v[eb[e]]] - (long double)c->Rv[v[ea[e]]];
        long double tZ = (long double)c->Zv[v[eb[e]]] - (long double)c->Zv[v[ea[e]]];
        long double nR = tZ, nZ = -tR;                    /* unnormalised normal */
        long double alpha = nR * xR + nZ * xZ, beta = nR * eR + nZ * eZ;
        for (int k = 0; k < 21; ++k) {
            int i, j; mono_ij(k, &i, &j);
            long double val = 0.0L;
            if (i + j == 5) {
                if (i >= 1) val += alpha * i * ipowl(dxi[e], i - 1) * ipowl(det[e], j);
                if (j >= 1) val += beta * j * ipowl(dxi[e], i) * ipowl(det[e], j - 1);
            }
            A[18 + e][k] = val;
        }
    }
    for (int r = 0; r < 21; ++r) {
        long double m = 0.0L;
        for (int k = 0; k < 21; ++k) { long double a = fabsl(A[r][k]); if (a > m) m = a; }
        if (m == 0.0L) return -1;
        rowscale[r] = 1.0L / m;
        for (int k = 0; k < 21; ++k) A[r][k] *= rowscale[r];
    }
    for (int k = 0; k < 21; ++k) {
        int pr = k; long double best = fabsl(A[k][k]);
        for (int r = k + 1; r < 21; ++r) if (fabsl(A[r][k]) > best) { best = fabsl(A[r][k]); pr = r; }
        if (best == 0.0L) return -1;
        piv[k] = pr;
        if (pr != k) for (int q = 0; q < 21; ++q) { long double tmp = A[k][q]; A[k][q] = A[pr][q]; A[pr][q] = tmp; }
        for (int r = k + 1; r < 21; ++r) {
            long double f = A[r][k] / A[k][k];
            A[r][k] = f;
            for (int q = k + 1; q < 21; ++q) A[r][q] -= f * A[k][q];
        }
    }
    return 0;
}
static void bell_solve(long double A[21][21], const long double rowscale[21], const int piv[21], long double b[21])
{
    for (int r = 0; r < 21; ++r) b[r] *= rowscale[r];
    /* whole rows (multipliers included) were swapped while factoring: permute b first */
    for (int k = 0; k < 21; ++k)
        if (piv[k] != k) { long double tmp = b[k]; b[k] = b[piv[k]]; b[piv[k]] = tmp; }
    for (int k = 0; k < 21; ++k)
        for (int r = k + 1; r < 21; ++r) b[r] -= A[r][k] * b[k];
    for (int k = 20; k >= 0; --k) {
        for (int q = k + 1; q < 21; ++q) b[k] -= A[k][q] * b[q];
        b[k] /= A[k][k];
    }
}

/* dofs: [n_modes][n_vert][6][2] (re,im) in the order f, f_R, f_Z, f_RR, f_RZ, f_ZZ */
int orc_bell_from_dofs(orc_ctx *c, const double *dofs)
{
    int bad = 0;
#pragma omp parallel for schedule(static) reduction(+ : bad)
    for (int t = 0; t < c->n_tri; ++t) {
        long double A[21][21], rs[21]; int piv[21];
        if (bell_factor(c, t, A, rs, piv)) { bad += 1; continue; }
        const int *v = c->tri + 3 * t;
        for (int m = 0; m < c->n_modes; ++m)
            for (int part = 0; part < 2; ++part) {
                long double b[21];
                for (int pnt = 0; pnt < 3; ++pnt)
                    for (int d = 0; d < 6; ++d)
                        b[6 * pnt + d] = dofs[(((size_t)m * c->n_vert + v[pnt]) * 6 + d) * 2 + part];
                b[18] = b[19] = b[20] = 0.0L;
                bell_solve(A, rs, piv, b);
                double *out = c->coef + (((size_t)t * c->n_modes + m) * ORC_NCOEF) * 2;
                for (int k = 0; k < 21; ++k) out[2 * k + part] = (double)b[k];
            }
    }
    return bad ? -1 : 0;
}

/* --------------------------------------------------------------- O3 locator */
/* contains(): barycentric test, every operation individually rounded (rule L2). */
static int inside(const orc_ctx *c, int t, double R, double Z, double *xi, double *eta, double *lam0)
{
    const double *g = c->geom + 6 * t;
    double dx = R - g[0], dz = Z - g[1];
    double a = g[2] * dx, b = g[3] * dz;
    *xi = a + b;
    double cc = g[4] * dx, d = g[5] * dz;
    *eta = cc + d;
    double one_m_xi = 1.0 - *xi;
    *lam0 = one_m_xi - *eta;
    return (*xi >= 0.0) && (*eta >= 0.0) && (*lam0 >= 0.0);
}
static double min3(double a, double b, double c) { double m = a < b ? a : b; return m < c ? m : c; }

/* plain definition: lowest t with inside(t); gap fallback as in SURVEY.md §8(c) O3 */
static int locate_brute_one(const orc_ctx *c, double R, double Z)
{
    double xi, eta, l0;
    if (c->n_r == 0) return locate_list(c, NULL, c->n_tri, R, Z, NULL, NULL);      /* O13: the rule over all triangles */
    for (int t = 0; t < c->n_tri; ++t)
        if (inside(c, t, R, Z, &xi, &eta, &l0)) return t;
    double x = R - c->Rv[0], z = Z - c->Zv[0];
    double s = x * x + z * z;
    if (s < c->rin2) {
        int best = -1; double bm = -INFINITY;
        for (int t = 0; t < c->n_tri; ++t) {
            inside(c, t, R, Z, &xi, &eta, &l0);
            double m = min3(xi, eta, l0);
            if (m > bm) { bm = m; best = t; }
        }
        return best;
    }
    return -1;
}

/* O(1) version: (r, theta) ring/sector guess, 3x3 neighbourhood of cells (<= 18 triangles),
 * same inside() and same lowest-t rule (rules L1-L4).  r and theta only choose candidates. */
static int candidates(const orc_ctx *c, double R, double Z, int *cand)
{
    double x = R - c->Rv[0], z = Z - c->Zv[0];
    double r = sqrt(x * x + z * z);
    double th = atan2(z, x);
    if (th < 0.0) th += ORC_TWO_PI;
    int lo = 0, hi = c->n_r;               /* largest i with r_nodes[i] <= r */
    while (hi - lo > 1) { int mid = (lo + hi) / 2; if (c->r_nodes[mid] <= r) lo = mid; else hi = mid; }
    int i0 = lo; if (i0 > c->n_r - 1) i0 = c->n_r - 1;
    double jf = floor(th * c->n_theta / ORC_TWO_PI);
    if (!(jf >= 0.0 && jf < (double)c->n_theta)) jf = 0.0;   /* also catches NaN */
    int j0 = (int)jf;
    int n = 0;
    for (int ii = i0 - 1; ii <= i0 + 1; ++ii) {
        if (ii < 0 || ii > c->n_r - 1) continue;
        for (int dj = -1; dj <= 1; ++dj) {
            int jj = ((j0 + dj) % c->n_theta + c->n_theta) % c->n_theta;
            if (ii == 0) cand[n++] = jj;
            else { int base = c->n_theta + 2 * ((ii - 1) * c->n_theta + jj); cand[n++] = base; cand[n++] = base + 1; }
        }
    }
    /* sort ascending (insertion sort) so that "lowest t" is the first hit */
    for (int a = 1; a < n; ++a) { int v = cand[a], b = a - 1; while (b >= 0 && cand[b] > v) { cand[b + 1] = cand[b]; --b; } cand[b + 1] = v; }
    return n;
}
static int locate_one(const orc_ctx *c, double R, double Z, double *xi_out, double *eta_out)
{
    if (c->n_r == 0) return locate_box(c, R, Z, xi_out, eta_out);                  /* O13 */
    int cand[18];
    int n = candidates(c, R, Z, cand);
    double xi, eta, l0;
    for (int q = 0; q < n; ++q) {
        if (q > 0 && cand[q] == cand[q - 1]) continue;
        if (inside(c, cand[q], R, Z, &xi, &eta, &l0)) { if (xi_out) { *xi_out = xi; *eta_out = eta; } return cand[q]; }
    }
    double x = R - c->Rv[0], z = Z - c->Zv[0];
    double s = x * x + z * z;
    if (s < c->rin2) {
        int best = -1; double bm = -INFINITY, bxi = 0, beta_ = 0;
        for (int q = 0; q < n; ++q) {
            inside(c, cand[q], R, Z, &xi, &eta, &l0);
            double m = min3(xi, eta, l0);
            if (m > bm) { bm = m; best = cand[q]; bxi = xi; beta_ = eta; }
        }
        if (xi_out) { *xi_out = bxi; *eta_out = beta_; }
        return best;
    }
    return -1;
}

void orc_locate_brute(const orc_ctx *c, size_t n, const double *R, const double *Z, int32_t *cell)
{
#pragma omp parallel for schedule(static)
    for (size_t p = 0; p < n; ++p) cell[p] = locate_brute_one(c, R[p], Z[p]);
}
void orc_locate(const orc_ctx *c, size_t n, const double *R, const double *Z, int32_t *cell)
{
#pragma omp parallel for schedule(static)
    for (size_t p = 0; p < n; ++p) cell[p] = locate_one(c, R[p], Z[p], NULL, NULL);
}
/* (xi, eta, lambda0) of point p in triangle t -- test hook */
void orc_bary(const orc_ctx *c, size_t n, const int32_t *t, const double *R, const double *Z, double *out)
{
    for (size_t p = 0; p < n; ++p) inside(c, t[p], R[p], Z[p], out + 3 * p, out + 3 * p + 1, out + 3 * p + 2);
}

/* ---------------------------------------------------------------- O4 gather */
/* Naive monomial sums; E_n = cos(n phi) + i sin(n phi);
 *   dphi        = sum_n Re(P_n E_n)
 *   d/dR, d/dZ  = sum_n Re((xi_X dP/dxi + eta_X dP/deta) E_n)
 *   d/dphi      = sum_n Re(i n P_n E_n)
 * No factor 2 for n > 0; Im of the n = 0 mode is ignored (reading G15). */
static void gather_one_spline(const orc_ctx *c, int t, double xi, double eta, double phi, double out[4]);
static void gather_one(const orc_ctx *c, int t, double xi, double eta, double phi, double out[4])
{
    if (c->n_phi > 0) { gather_one_spline(c, t, xi, eta, phi, out); return; }
    const double *g = c->geom + 6 * t;
    double f = 0.0, fR = 0.0, fZ = 0.0, fp = 0.0;
    for (int m = 0; m < c->n_modes; ++m) {
        const double *cf = c->coef + (((size_t)t * c->n_modes + m) * ORC_NCOEF) * 2;
        double Pr = 0, Pi = 0, Pxr = 0, Pxi_ = 0, Per = 0, Pei = 0;
        for (int k = 0; k < 21; ++k) {
            int i, j; mono_ij(k, &i, &j);
            double mono = ipow(xi, i) * ipow(eta, j);
            double mx = (i >= 1) ? i * ipow(xi, i - 1) * ipow(eta, j) : 0.0;
            double me = (j >= 1) ? j * ipow(xi, i) * ipow(eta, j - 1) : 0.0;
            Pr += cf[2 * k] * mono;  Pi += cf[2 * k + 1] * mono;
            Pxr += cf[2 * k] * mx;   Pxi_ += cf[2 * k + 1] * mx;
            Per += cf[2 * k] * me;   Pei += cf[2 * k + 1] * me;
        }
        double nn = (double)c->mode_n[m];
        double Er = cos(nn * phi), Ei = sin(nn * phi);
        double PRr = g[2] * Pxr + g[4] * Per, PRi = g[2] * Pxi_ + g[4] * Pei;   /* dP/dR */
        double PZr = g[3] * Pxr + g[5] * Per, PZi = g[3] * Pxi_ + g[5] * Pei;   /* dP/dZ */
        f  += Pr * Er - Pi * Ei;
        fR += PRr * Er - PRi * Ei;
        fZ += PZr * Er - PZi * Ei;
        fp += nn * (-Pi * Er - Pr * Ei);      /* Re(i n P E) */
    }
    out[0] = f; out[1] = fR; out[2] = fZ; out[3] = fp;
}

/* cell_out[p] = located triangle (or -1, outputs then 0) */
void orc_gather(const orc_ctx *c, size_t n, const double *R, const double *Z, const double *phi,
                int32_t *cell_out, double *f, double *fR, double *fZ, double *fphi)
{
#pragma omp parallel for schedule(static)
    for (size_t p = 0; p < n; ++p) {
        double xi, eta, o[4] = {0, 0, 0, 0};
        int t = locate_one(c, R[p], Z[p], &xi, &eta);
        if (t >= 0) gather_one(c, t, xi, eta, phi[p], o);
        if (cell_out) cell_out[p] = t;
        f[p] = o[0]; fR[p] = o[1]; fZ[p] = o[2]; if (fphi) fphi[p] = o[3];
    }
}

/* ----------------------------------------------------------- O5 equilibrium */
typedef struct {
    double B, BR, BZ, Bphi, bR, bZ, bphi, dBdR, dBdZ;
    double dbR_dZ, dbZ_dR, dbphi_dR, dbphi_dZ, psi;
    double psiR, psiZ;             /* O14: grad psi (tabulated equilibrium only; the analytic one uses rhat) */
} orc_eq;

/* B = grad psi x grad phi + F grad phi; B_R = -psi_Z/R, B_Z = psi_R/R,
 * B_phi = F/R with psi'(r) = B0 r/q(r) (reading G11), F = B0 R0. */
static void equilibrium_analytic(const orc_params *p, double R, double Z, orc_eq *e)
{
    double x = R - p->R0;
    double s = x * x + Z * Z;
    double a2 = p->a * p->a;
    double qs = p->q2 / a2;                         /* d qbar / d s */
    double qb = p->q0 + qs * s;
    double g = p->R0 * p->R0 + s / (qb * qb);
    double gs = 1.0 / (qb * qb) - 2.0 * s * qs / (qb * qb * qb);
    double sg = sqrt(g);
    double h = 1.0 / (qb * sg);
    double hs = -qs / (qb * qb * sg) - gs / (2.0 * qb * g * sg);
    e->B = p->B0 * sg / R;
    e->BR = -p->B0 * Z / (R * qb);
    e->BZ = p->B0 * x / (R * qb);
    e->Bphi = p->B0 * p->R0 / R;
    e->bR = -Z * h; e->bZ = x * h; e->bphi = p->R0 / sg;
    e->dBdR = p->B0 * (gs * x / (sg * R) - sg / (R * R));
    e->dBdZ = p->B0 * gs * Z / (sg * R);
    e->dbR_dZ = -h - 2.0 * Z * Z * hs;
    e->dbZ_dR = h + 2.0 * x * x * hs;
    e->dbphi_dR = -p->R0 * gs * x / (g * sg);
    e->dbphi_dZ = -p->R0 * gs * Z / (g * sg);
    e->psi = (p->q2 != 0.0) ? p->B0 * a2 / (2.0 * p->q2) * log(1.0 + p->q2 * s / (p->q0 * a2))
                            : p->B0 * s / (2.0 * p->q0);
}
/* ----------------------------------------------------------- O14 tabulated equilibrium */
/* "The equilibrium configuration is computed as functions of (R, Z) ... starting from the magnetic equilibrium constructed from
 * the EQDSK output file ... B_phi = F/R by means of b-spline interpolation of the poloidal current function F";
 * B_R = -psi_Z/R, B_Z = psi_R/R, B_phi = F/R.  Reading G32 (the thesis names the interpolation, not its form):
 *   psi(R, Z) = sum_ij C[i][j] beta((R - Ra)/hR - i) beta((Z - Za)/hZ - j),   F(psi) = sum_k D[k] beta((psi - pa)/hp - k),
 * beta the uniform cubic B-spline of O11, the caller hands in COEFFICIENTS (a prefiltered EQDSK grid).  All sixteen (four)
 * non-zero terms are summed; the F index is clamped to the table (the end pieces extend as cubics).  First and second
 * derivatives of psi and F' give B, grad B, b and the derivatives of b that curl b needs, by the quotient rule.
 * The profile gradients of the weight equation point along grad psi/|grad psi| (= rhat in the circular case). */
typedef struct orc_eqtab {
    int nR, nZ, nF;
    double Ra, Za, hR, hZ, pa, hp;
    double *C, *D;
} orc_eqtab;
static double bspl(double x);
static double bspl_d(double x);
static double bspl_dd(double x) { double a = fabs(x); if (a < 1.0) return -2.0 + 3.0 * a; if (a < 2.0) return 2.0 - a; return 0.0; }
static void equilibrium_table(const orc_eqtab *q, double R, double Z, orc_eq *e)
{
    const double xr = (R - q->Ra) / q->hR, xz = (Z - q->Za) / q->hZ;
    int i0 = (int)floor(xr), j0 = (int)floor(xz);
    double psi = 0, pR = 0, pZ = 0, pRR = 0, pRZ = 0, pZZ = 0;
    for (int i = i0 - 1; i <= i0 + 2; ++i)
        for (int j = j0 - 1; j <= j0 + 2; ++j) {
            if (i < 0 || i >= q->nR || j < 0 || j >= q->nZ) continue;         /* outside the table: no contribution */
            const double c = q->C[(size_t)i * q->nZ + j], a = xr - i, b = xz - j;
            psi += c * bspl(a) * bspl(b);
            pR += c * bspl_d(a) * bspl(b) / q->hR;       pZ += c * bspl(a) * bspl_d(b) / q->hZ;
            pRR += c * bspl_dd(a) * bspl(b) / (q->hR * q->hR);
            pRZ += c * bspl_d(a) * bspl_d(b) / (q->hR * q->hZ);
            pZZ += c * bspl(a) * bspl_dd(b) / (q->hZ * q->hZ);
        }
    const double xp = (psi - q->pa) / q->hp;
    int k0 = (int)floor(xp);
    if (k0 < 1) k0 = 1;
    if (k0 > q->nF - 3) k0 = q->nF - 3;
    double F = 0, Fp = 0;
    {   /* the cubic piece of interval k0, written with the piece's own four polynomials so that it extends beyond the table */
        const double t = xp - k0, u = 1.0 - t;
        const double N[4] = {u * u * u / 6.0, 2.0 / 3.0 - t * t + 0.5 * t * t * t, 2.0 / 3.0 - u * u + 0.5 * u * u * u, t * t * t / 6.0};
        const double M[4] = {-0.5 * u * u, -2.0 * t + 1.5 * t * t, 2.0 * u - 1.5 * u * u, 0.5 * t * t};
        for (int k = 0; k < 4; ++k) { F += q->D[k0 - 1 + k] * N[k]; Fp += q->D[k0 - 1 + k] * M[k] / q->hp; }
    }
    const double BR = -pZ / R, BZ = pR / R, BP = F / R;
    const double BR_R = -pRZ / R + pZ / (R * R), BR_Z = -pZZ / R;
    const double BZ_R = pRR / R - pR / (R * R), BZ_Z = pRZ / R;
    const double BP_R = Fp * pR / R - F / (R * R), BP_Z = Fp * pZ / R;
    const double B = sqrt(BR * BR + BZ * BZ + BP * BP);
    const double B_R = (BR * BR_R + BZ * BZ_R + BP * BP_R) / B, B_Z = (BR * BR_Z + BZ * BZ_Z + BP * BP_Z) / B;
    e->B = B; e->BR = BR; e->BZ = BZ; e->Bphi = BP;
    e->bR = BR / B; e->bZ = BZ / B; e->bphi = BP / B;
    e->dBdR = B_R; e->dBdZ = B_Z;
    e->dbR_dZ = (BR_Z - e->bR * B_Z) / B;
    e->dbZ_dR = (BZ_R - e->bZ * B_R) / B;
    e->dbphi_dR = (BP_R - e->bphi * B_R) / B;
    e->dbphi_dZ = (BP_Z - e->bphi * B_Z) / B;
    e->psi = psi; e->psiR = pR; e->psiZ = pZ;
}
static void equilibrium(const orc_ctx *c, double R, double Z, orc_eq *e)
{
    if (c->eq) equilibrium_table(c->eq, R, Z, e);
    else { equilibrium_analytic(&c->p, R, Z, e); e->psiR = e->psiZ = 0.0; }
}
/* rate of change of the radial label along a velocity: along rhat (analytic equilibrium), along grad psi/|grad psi| (table) */
static double radial_rate(const orc_ctx *c, const orc_eq *e, double R, double Z, double dRdot, double dZdot)
{
    if (c->eq) {
        const double g = sqrt(e->psiR * e->psiR + e->psiZ * e->psiZ);
        return (g > 0.0) ? (dRdot * e->psiR + dZdot * e->psiZ) / g : 0.0;
    }
    const double x = R - c->p.R0, r = sqrt(x * x + Z * Z);
    return (r > 0.0) ? (dRdot * x + dZdot * Z) / r : 0.0;
}
/* C: [nR][nZ] coefficients of psi; D: [nF] coefficients of F; NULL C returns to the analytic equilibrium */
void orc_set_equilibrium_table(orc_ctx *c, int nR, int nZ, double Ra, double Za, double hR, double hZ, const double *C,
                               int nF, double pa, double hp, const double *D)
{
    if (c->eq) { free(c->eq->C); free(c->eq->D); free(c->eq); c->eq = NULL; }
    if (!C) return;
    orc_eqtab *q = (orc_eqtab *)calloc(1, sizeof(orc_eqtab));
    q->nR = nR; q->nZ = nZ; q->nF = nF; q->Ra = Ra; q->Za = Za; q->hR = hR; q->hZ = hZ; q->pa = pa; q->hp = hp;
    q->C = (double *)malloc(sizeof(double) * (size_t)nR * nZ); memcpy(q->C, C, sizeof(double) * (size_t)nR * nZ);
    q->D = (double *)malloc(sizeof(double) * (size_t)nF); memcpy(q->D, D, sizeof(double) * (size_t)nF);
    c->eq = q;
}
void orc_equilibrium(const orc_ctx *c, size_t n, const double *R, const double *Z, double *out /* [n][14] */)
{
    for (size_t p = 0; p < n; ++p) {
        orc_eq e; equilibrium(c, R[p], Z[p], &e);
        memcpy(out + 14 * p, &e, sizeof(double) * 14);
    }
}

/* ------------------------------------------------------------------- O6 RHS */
/* Electrostatic subset (dA^s = dA^h = 0  =>  u_par = v_par, b* = b0*, dG = dPhi).
 * eps = (m_s/q_s) rho_0 B_0 (reading G23). */
static void rhs_point_em_reduced(const orc_ctx *c, double R, double Z, double upar, double mu, double w,
                                 const double fld[3][4], int ohm, double out[5]);
static void rhs_point(const orc_ctx *c, double R, double Z, double vpar, double mu, double w,
                      const double fld[4] /* dphi, d/dR, d/dZ, d/dphi */, double out[5])
{
    const orc_params *p = &c->p;
    if (p->eom_variant == 2) {                        /* O12: the reduced model with dA^s = dA^h = 0 and NO Ohm's-law substitution */
        double f3[3][4];
        memset(f3, 0, sizeof(f3));
        memcpy(f3[0], fld, sizeof(double) * 4);
        rhs_point_em_reduced(c, R, Z, vpar, mu, w, f3, 0, out);
        return;
    }
    orc_eq e; equilibrium(c, R, Z, &e);
    double eps = p->rho0 * p->B0 / p->qs_over_ms;
    double cR = -e.dbphi_dZ;                          /* (curl b)_R   , bracket of A.4 */
    double cZ = e.dbphi_dR + e.bphi / R;              /* (curl b)_Z   , bracket of A.5 */
    double cP = e.dbR_dZ - e.dbZ_dR;                  /* (curl b)_phi , bracket of A.6 */
    double bcurlb = e.bR * cR + e.bZ * cZ + e.bphi * cP;
    double Bsp = e.B + eps * vpar * bcurlb;           /* B*_par */
    double lead = (p->eom_variant == 1) ? e.B / Bsp : 1.0;
    double k = eps * vpar / Bsp;
    double b0R = lead * e.bR + k * cR;                /* A.4 */
    double b0Z = lead * e.bZ + k * cZ;                /* A.5 */
    double b0P = lead * e.bphi + k * cP;              /* A.6 */
    double Cd = eps * mu / (e.B * Bsp);
    double CE = p->rho0 * p->B0 / Bsp;
    double R0dot = b0R * vpar + Cd * e.Bphi * e.dBdZ;                            /* A.10 */
    double Z0dot = b0Z * vpar - Cd * e.Bphi * e.dBdR;                            /* A.11, sign: G1 */
    double P0dot = b0P * vpar / R + (Cd / R) * (e.BZ * e.dBdR - e.BR * e.dBdZ);  /* A.12 */
    double v0dot = -mu * (b0R * e.dBdR + b0Z * e.dBdZ);                          /* A.13 */
    double fR = fld[1], fZ = fld[2], fP = fld[3];
    double dRdot = CE * (e.bphi * fZ - (e.bZ / R) * fP);                         /* A.14 */
    double dZdot = CE * (-e.bphi * fR + (e.bR / R) * fP);                        /* A.15 */
    double dPdot = (CE / R) * (e.bZ * fR - e.bR * fZ);                           /* A.16 */
    double dvdot = -p->qs_over_ms * (b0R * fR + b0Z * fZ + (b0P / R) * fP);      /* A.17, dA = 0 (G3) */
    /* d ln f_M / dt, mbar = 1, kappa_X = -kappa_X rhat (G6, G10) */
    double drdot = radial_rate(c, &e, R, Z, dRdot, dZdot);            /* dRvec . rhat */
    double en = vpar * vpar / p->T + 2.0 * mu * e.B / p->T - 1.5;
    double L = drdot * (-p->kappa_n - en * p->kappa_T)
             - (2.0 * mu / p->T) * (dRdot * e.dBdR + dZdot * e.dBdZ)
             - (2.0 * vpar / p->T) * dvdot;
    out[0] = R0dot + dRdot;
    out[1] = Z0dot + dZdot;
    out[2] = P0dot + dPdot;
    out[3] = v0dot + dvdot;
    out[4] = (p->weight_mode == 0) ? -(1.0 - w) * L : -L;
}

/* full RHS at a phase-space point: locate -> gather -> equilibrium -> equations.
 * returns the triangle, or -1 (out[] untouched) if the point is outside the mesh */
static int rhs_full(const orc_ctx *c, double R, double Z, double phi, double vpar, double mu, double w, double out[5])
{
    double xi, eta, fld[4] = {0, 0, 0, 0};
    int t = locate_one(c, R, Z, &xi, &eta);
    if (t < 0) return -1;
    if (c->n_modes > 0 || c->n_phi > 0) gather_one(c, t, xi, eta, phi, fld);
    rhs_point(c, R, Z, vpar, mu, w, fld, out);
    return t;
}

void orc_rhs(const orc_ctx *c, size_t n, const double *R, const double *Z, const double *phi,
             const double *vpar, const double *mu, const double *w, int32_t *cell_out,
             double *dRdt, double *dZdt, double *dphidt, double *dvpardt, double *dwdt)
{
#pragma omp parallel for schedule(static)
    for (size_t p = 0; p < n; ++p) {
        double o[5] = {0, 0, 0, 0, 0};
        int t = rhs_full(c, R[p], Z[p], phi[p], vpar[p], mu[p], w[p], o);
        if (cell_out) cell_out[p] = t;
        dRdt[p] = o[0]; dZdt[p] = o[1]; dphidt[p] = o[2]; dvpardt[p] = o[3]; dwdt[p] = o[4];
    }
}
/* RHS with the field values handed in (no mesh): test hook for the pointwise identities */
void orc_rhs_point(const orc_ctx *c, size_t n, const double *R, const double *Z, const double *vpar,
                   const double *mu, const double *w, const double *fld /* [n][4] */, double *out /* [n][5] */)
{
    for (size_t p = 0; p < n; ++p) rhs_point(c, R[p], Z[p], vpar[p], mu[p], w[p], fld + 4 * p, out + 5 * p);
}

/* ------------------------------------------------------------------- O7 RK4 */
/* y = (R, Z, phi, v_par, w), mu constant.  phi wrapped to [0, 2 pi) once per step.  A marker
 * whose any stage position, or final position, is outside the mesh is restored to its
 * start-of-step state, flagged cell = -1 and skipped from then on.  Field frozen. */
void orc_push(const orc_ctx *c, size_t n, double *R, double *Z, double *phi, double *vpar,
              const double *mu, double *w, int32_t *cell, double dt, int nsteps, int nthreads)
{
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#else
    (void)nthreads;
#endif
#pragma omp parallel for schedule(static)
    for (size_t p = 0; p < n; ++p) {
        if (cell[p] < 0) continue;          /* already lost */
        double y[5] = {R[p], Z[p], phi[p], vpar[p], w[p]};
        int cl = cell[p];
        for (int s = 0; s < nsteps; ++s) {
            double k1[5], k2[5], k3[5], k4[5], ys[5];
            int lost = 0;
            if (rhs_full(c, y[0], y[1], y[2], y[3], mu[p], y[4], k1) < 0) lost = 1;
            if (!lost) {
                for (int q = 0; q < 5; ++q) ys[q] = y[q] + 0.5 * dt * k1[q];
                if (rhs_full(c, ys[0], ys[1], ys[2], ys[3], mu[p], ys[4], k2) < 0) lost = 1;
            }
            if (!lost) {
                for (int q = 0; q < 5; ++q) ys[q] = y[q] + 0.5 * dt * k2[q];
                if (rhs_full(c, ys[0], ys[1], ys[2], ys[3], mu[p], ys[4], k3) < 0) lost = 1;
            }
            if (!lost) {
                for (int q = 0; q < 5; ++q) ys[q] = y[q] + dt * k3[q];
                if (rhs_full(c, ys[0], ys[1], ys[2], ys[3], mu[p], ys[4], k4) < 0) lost = 1;
            }
            int newcell = -1;
            if (!lost) {
                for (int q = 0; q < 5; ++q) ys[q] = y[q] + (dt / 6.0) * (k1[q] + 2.0 * k2[q] + 2.0 * k3[q] + k4[q]);
                ys[2] = ys[2] - ORC_TWO_PI * floor(ys[2] / ORC_TWO_PI);
                newcell = locate_one(c, ys[0], ys[1], NULL, NULL);
                if (newcell < 0) lost = 1;
            }
            if (lost) { cl = -1; break; }       /* y keeps the start-of-step state */
            for (int q = 0; q < 5; ++q) y[q] = ys[q];
            cl = newcell;
        }
        R[p] = y[0]; Z[p] = y[1]; phi[p] = y[2]; vpar[p] = y[3]; w[p] = y[4]; cell[p] = cl;
    }
}


/* ------------------------------------------------------------ O8 scatter (p2g) */
/* "The charge of each particle is projected onto the basis functions"; the P2G projection is the
 * counterpart of the G2P interpolation.  With the field written as
 *     dphi(R, phi, Z) = sum_n Re( sum_{v,d} Y_{n,v,d} Lambda_{v,d}(R, Z) e^{i n phi} )
 * (Lambda_{v,d}: the C1 basis function of degree of freedom d = f, f_R, f_Z, f_RR, f_RZ, f_ZZ at vertex v),
 * the projection of the marker weights onto the test functions Lambda_{v,d} e^{i n phi} is
 *     rhs[n][v][d] = sum_p w_p Lambda_{v,d}(R_p, Z_p) e^{-i n phi_p}
 * (the conjugate toroidal factor, as in any Galerkin projection onto e^{i n phi}), so that for real weights
 *     sum_p w_p dphi(x_p) = Re sum_{n,v,d} Y_{n,v,d} conj(rhs[n][v][d]):   scatter is the adjoint of gather (O4).
 * Plain definition, marker by marker: locate -> the 18 basis functions of the triangle at (xi, eta) -> add.
 * Lambda_j restricted to a triangle is the quintic whose nodal values are the unit vector e_j: its 21 monomial
 * coefficients are the solution of the same 21 x 21 system as in O2 (bell_factor / bell_solve) with right-hand side e_j. */
static const double *bell_basis(orc_ctx *c, int t)
{
    if (c->basis[t]) return c->basis[t];
    long double A[21][21], rs[21]; int piv[21];
    if (bell_factor(c, t, A, rs, piv)) return NULL;
    double *B = (double *)malloc(sizeof(double) * 21 * 18);
    for (int j = 0; j < 18; ++j) {
        long double b[21];
        for (int r = 0; r < 21; ++r) b[r] = (r == j) ? 1.0L : 0.0L;
        bell_solve(A, rs, piv, b);
        for (int k = 0; k < 21; ++k) B[k * 18 + j] = (double)b[k];
    }
    c->basis[t] = B;
    return B;
}

/* rhs: [n_modes][n_vert][6][2] (re, im), overwritten.  cell_flag may be NULL; markers with cell_flag[p] < 0, and markers
 * outside the mesh, contribute nothing.  Returns the number of markers that contributed, or -1 (singular element). */
long orc_scatter(orc_ctx *c, size_t n, const double *R, const double *Z, const double *phi, const double *w,
                 const int32_t *cell_flag, double *rhs)
{
    const size_t per_mode = (size_t)c->n_vert * 6 * 2;
    memset(rhs, 0, sizeof(double) * per_mode * (c->n_modes > 0 ? c->n_modes : 0));
    if (!c->basis) c->basis = (double **)calloc((size_t)c->n_tri, sizeof(double *));
    /* pass 1 (serial): triangles and local coordinates, basis tables of the triangles that hold markers */
    int32_t *tp = (int32_t *)malloc(sizeof(int32_t) * (n ? n : 1));
    double *xe = (double *)malloc(sizeof(double) * 2 * (n ? n : 1));
    long used = 0;
    for (size_t p = 0; p < n; ++p) {
        tp[p] = -1;
        if (cell_flag && cell_flag[p] < 0) continue;
        double xi, eta;
        int t = locate_one(c, R[p], Z[p], &xi, &eta);
        if (t < 0) continue;
        if (!bell_basis(c, t)) { free(tp); free(xe); return -1; }
        tp[p] = t; xe[2 * p] = xi; xe[2 * p + 1] = eta;
        ++used;
    }
    /* pass 2: one toroidal mode per thread; inside a mode the markers are added in their order */
#pragma omp parallel for schedule(dynamic, 1)
    for (int m = 0; m < c->n_modes; ++m) {
        double *out = rhs + per_mode * m;
        const double nn = (double)c->mode_n[m];
        for (size_t p = 0; p < n; ++p) {
            const int t = tp[p];
            if (t < 0) continue;
            const double *B = c->basis[t];
            const int *v = c->tri + 3 * t;
            const double xi = xe[2 * p], eta = xe[2 * p + 1];
            double mono[21];
            for (int k = 0; k < 21; ++k) { int i, j; mono_ij(k, &i, &j); mono[k] = ipow(xi, i) * ipow(eta, j); }
            const double Er = cos(nn * phi[p]), Ei = -sin(nn * phi[p]);        /* e^{-i n phi} */
            for (int j = 0; j < 18; ++j) {
                double lam = 0.0;
                for (int k = 0; k < 21; ++k) lam += B[k * 18 + j] * mono[k];
                double *o = out + ((size_t)v[j / 6] * 6 + (j % 6)) * 2;
                o[0] += w[p] * lam * Er;
                o[1] += w[p] * lam * Ei;
            }
        }
    }
    free(tp); free(xe);
    return used;
}

/* ------------------------------------------------- O9 electromagnetic right-hand side (mixed variables) */
/* Fields: dPhi (coef), dA^s (coef_aux[0]), dA^h (coef_aux[1]), dA_par = dA^s + dA^h (A.1), all on the same
 * basis.  The marker's velocity coordinate is u_par = v_par + (q_s/m_s) <dA^h>; the gyro-average <.> is the
 * identity (off, as in the thesis's own runs).  Vector form, eps = (m_s/q_s) rho_0 B_0:
 *   B*_par = B + eps u_par b.curl b;  b0* = b + (eps u_par/B*_par) curl b  [variant 1: (B/B*_par) b + ...]   (A.4-A.6 with u_par)
 *   b* = b0* + C_E grad(dA^s) x b,  C_E = rho_0 B_0/B*_par                                                (A.7-A.9)
 *   R0dot, u0dot: A.10-A.13 with u_par (sign of A.11 as reading G1)
 *   dRdot = C_E b x grad(dG) - (q_s/m_s) dA^h b*,   grad(dG) = grad(dPhi) - u_par grad(dA^s + dA^h)       (A.14-A.16)
 *   dudot = -(q_s/m_s) [ (b* - b).grad(dPhi) - u_par b*.grad(dA^h) ] - (Rdot_mu d_R + Zdot_mu d_Z + phidot_mu d_phi) dA^s
 *     = A.17 with the ideal Ohm's law d_t dA^s = -b.grad(dPhi) substituted exactly (reading G26: A.18 as
 *     printed has b instead of b* in the dA^h term, a second-order difference; the phi term of A.18 lacks its 1/R).
 *   weight: d ln f_M/dt of PAPER.md:1208 with v_par = u_par - (q_s/m_s) dA^h and d(u_par)/dt perturbed part.
 * fld[3][4]: (value, d/dR, d/dZ, d/dphi) of dPhi, dA^s, dA^h. */
static void rhs_point_em(const orc_ctx *c, double R, double Z, double upar, double mu, double w,
                         const double fld[3][4], double out[5])
{
    const orc_params *p = &c->p;
    if (p->eom_variant == 2) { rhs_point_em_reduced(c, R, Z, upar, mu, w, fld, 1, out); return; }   /* O12, A.29 */
    orc_eq e; equilibrium(c, R, Z, &e);
    const double eps = p->rho0 * p->B0 / p->qs_over_ms, qom = p->qs_over_ms;
    const double *Phi = fld[0], *As = fld[1], *Ah = fld[2];
    double cR = -e.dbphi_dZ, cZ = e.dbphi_dR + e.bphi / R, cP = e.dbR_dZ - e.dbZ_dR;      /* curl b */
    double Bsp = e.B + eps * upar * (e.bR * cR + e.bZ * cZ + e.bphi * cP);
    double lead = (p->eom_variant == 1) ? e.B / Bsp : 1.0;
    double k = eps * upar / Bsp;
    double b0R = lead * e.bR + k * cR, b0Z = lead * e.bZ + k * cZ, b0P = lead * e.bphi + k * cP;        /* A.4-A.6 */
    double CE = p->rho0 * p->B0 / Bsp, Cd = eps * mu / (e.B * Bsp);
    /* b* (A.7-A.9): b0* + C_E grad(dA^s) x b, with (grad f)_phi = (1/R) d f/d phi */
    double bsR = b0R + CE * ((e.bZ / R) * As[3] - e.bphi * As[2]);
    double bsZ = b0Z + CE * (e.bphi * As[1] - (e.bR / R) * As[3]);
    double bsP = b0P + CE * (e.bR * As[2] - e.bZ * As[1]);
    /* equilibrium part, A.10-A.13 */
    double Rmu = Cd * e.Bphi * e.dBdZ, Zmu = -Cd * e.Bphi * e.dBdR, Pmu = (Cd / R) * (e.BZ * e.dBdR - e.BR * e.dBdZ);
    double R0dot = b0R * upar + Rmu, Z0dot = b0Z * upar + Zmu, P0dot = b0P * upar / R + Pmu;
    double u0dot = -mu * (b0R * e.dBdR + b0Z * e.dBdZ);
    /* perturbed part */
    double GR = Phi[1] - upar * (As[1] + Ah[1]), GZ = Phi[2] - upar * (As[2] + Ah[2]), GP = Phi[3] - upar * (As[3] + Ah[3]);
    double dRdot = CE * (e.bphi * GZ - (e.bZ / R) * GP) - qom * Ah[0] * bsR;                           /* A.14 */
    double dZdot = CE * (-e.bphi * GR + (e.bR / R) * GP) - qom * Ah[0] * bsZ;                          /* A.15 */
    double dPdot = (CE / R) * (e.bZ * GR - e.bR * GZ) - (1.0 / R) * qom * Ah[0] * bsP;                 /* A.16 */
    double dudot = -qom * ((bsR - e.bR) * Phi[1] + (bsZ - e.bZ) * Phi[2] + ((bsP - e.bphi) / R) * Phi[3]
                           - upar * (bsR * Ah[1] + bsZ * Ah[2] + (bsP / R) * Ah[3]))
                   - (Rmu * As[1] + Zmu * As[2] + Pmu * As[3]);                                        /* A.17 + Ohm */
    /* weight */
    double vpar = upar - qom * Ah[0];
    double drdot = radial_rate(c, &e, R, Z, dRdot, dZdot);
    double en = vpar * vpar / p->T + 2.0 * mu * e.B / p->T - 1.5;
    double L = drdot * (-p->kappa_n - en * p->kappa_T) - (2.0 * mu / p->T) * (dRdot * e.dBdR + dZdot * e.dBdZ)
             - (2.0 * vpar / p->T) * dudot;
    out[0] = R0dot + dRdot; out[1] = Z0dot + dZdot; out[2] = P0dot + dPdot; out[3] = u0dot + dudot;
    out[4] = (p->weight_mode == 0) ? -(1.0 - w) * L : -L;
}
/* ------------------------------------------------- O12 reduced equations of motion (eom_variant 2) */
/* "Only the dominant terms ... obtained by replacing b* with b" (A.19-A.29):
 *   R0dot = u_par b + C_d B x grad B,        C_d = (m_s/q_s) rho_0 (u_par^2 + mu B) B_0/B^3                 (A.19-A.21)
 *   u0dot = -mu b.grad B                      (A.22; reading G29: b, as the sentence above says -- A.22 prints b0*, a copy of A.13;
 *                                              with b the unperturbed motion conserves u^2/2 + mu B exactly, and for F = const, as
 *                                              here, (b0* - b).grad B = 0 anyway: R b_phi = F/B, curl b's poloidal part is perpendicular to grad B)
 *   dRdot = C_E b x grad(dG) - (q_s/m_s) dA^h b,   C_E = rho_0 B_0/B,  dG = dPhi - u_par (dA^s + dA^h)    (A.24-A.26)
 *   dudot = -(q_s/m_s) [ b.grad(dPhi) - u_par b.grad(dA^h) ] - v_mu.grad(dA^s),   v_mu = C_mu B x grad B,
 *           C_mu = (m_s/q_s) rho_0 mu B B_0/B^3                                                              (A.28 without d_t dA^s)
 *   reading G30: the velocity in C_d and in the dA^h term of A.28 / A.29 is printed v_par; the coordinate u_par is taken, as in
 *   A.17 from which A.28 follows by b* -> b (the difference is second order in the fields).
 *   weight: d ln f_M/dt of PAPER.md:1208 along the perturbed velocity, v_par = u_par - (q_s/m_s) dA^h in the Maxwellian.
 * ohm = 0: the electrostatic push (orc_rhs / orc_push with eom_variant 2, dA = 0, d_t dA^s = 0); ohm = 1: orc_rhs_em, A.29. */
static void rhs_point_em_reduced(const orc_ctx *c, double R, double Z, double upar, double mu, double w,
                                 const double fld[3][4], int ohm, double out[5])
{
    const orc_params *p = &c->p;
    orc_eq e; equilibrium(c, R, Z, &e);
    const double eps = p->rho0 * p->B0 / p->qs_over_ms, qom = p->qs_over_ms;
    const double *Phi = fld[0], *As = fld[1], *Ah = fld[2];
    const double B3 = e.B * e.B * e.B;
    const double Cd = eps * (upar * upar + mu * e.B) / B3;
    const double Cmu = eps * mu * e.B / B3;
    const double CE = p->rho0 * p->B0 / e.B;
    /* (B x grad B) in (R, phi, Z): (B_phi d_Z B, B_Z d_R B - B_R d_Z B, -B_phi d_R B) */
    const double xR = e.Bphi * e.dBdZ, xZ = -e.Bphi * e.dBdR, xP = e.BZ * e.dBdR - e.BR * e.dBdZ;
    const double R0dot = e.bR * upar + Cd * xR;                                                   /* A.19 */
    const double Z0dot = e.bZ * upar + Cd * xZ;                                                   /* A.20 */
    const double P0dot = e.bphi * upar / R + Cd * xP / R;                                         /* A.21 */
    const double u0dot = -mu * (e.bR * e.dBdR + e.bZ * e.dBdZ);                                   /* A.22 (G29) */
    const double GR = Phi[1] - upar * (As[1] + Ah[1]), GZ = Phi[2] - upar * (As[2] + Ah[2]), GP = Phi[3] - upar * (As[3] + Ah[3]);
    const double dRdot = CE * (e.bphi * GZ - (e.bZ / R) * GP) - qom * Ah[0] * e.bR;               /* A.24 */
    const double dZdot = CE * (-e.bphi * GR + (e.bR / R) * GP) - qom * Ah[0] * e.bZ;              /* A.25 */
    const double dPdot = (CE / R) * (e.bZ * GR - e.bR * GZ) - (1.0 / R) * qom * Ah[0] * e.bphi;   /* A.26 */
    /* A.28; ohm: d_t dA^s = -b.grad(dPhi) cancels the parallel electric field, which leaves A.29 */
    const double keepE = ohm ? 0.0 : 1.0;
    const double dudot = -qom * (e.bR * (keepE * Phi[1] - upar * Ah[1]) + e.bZ * (keepE * Phi[2] - upar * Ah[2])
                                 + (e.bphi / R) * (keepE * Phi[3] - upar * Ah[3]))
                         - Cmu * (xR * As[1] + xZ * As[2] + (xP / R) * As[3]);
    const double vpar = upar - qom * Ah[0];
    const double drdot = radial_rate(c, &e, R, Z, dRdot, dZdot);
    const double en = vpar * vpar / p->T + 2.0 * mu * e.B / p->T - 1.5;
    const double L = drdot * (-p->kappa_n - en * p->kappa_T) - (2.0 * mu / p->T) * (dRdot * e.dBdR + dZdot * e.dBdZ)
                   - (2.0 * vpar / p->T) * dudot;
    out[0] = R0dot + dRdot; out[1] = Z0dot + dZdot; out[2] = P0dot + dPdot; out[3] = u0dot + dudot;
    out[4] = (p->weight_mode == 0) ? -(1.0 - w) * L : -L;
}
void orc_rhs_point_em(const orc_ctx *c, size_t n, const double *R, const double *Z, const double *upar, const double *mu,
                      const double *w, const double *fld /* [n][3][4] */, double *out /* [n][5] */)
{
    for (size_t p = 0; p < n; ++p) {
        double f3[3][4];
        memcpy(f3, fld + 12 * p, sizeof(f3));
        rhs_point_em(c, R[p], Z[p], upar[p], mu[p], w[p], f3, out + 5 * p);
    }
}
void orc_set_aux_coef(orc_ctx *c, int which, const double *coef)
{
    const size_t nn = (size_t)c->n_tri * c->n_modes * ORC_NCOEF * 2;
    free(c->coef_aux[which]); c->coef_aux[which] = NULL;
    if (coef && nn) { c->coef_aux[which] = (double *)malloc(sizeof(double) * nn); memcpy(c->coef_aux[which], coef, sizeof(double) * nn); }
}
/* gather of the three fields at a located point: the same gather_one on each table */
static void gather_three(const orc_ctx *c, int t, double xi, double eta, double phi, double fld[3][4])
{
    memset(fld, 0, sizeof(double) * 12);
    if (c->n_modes == 0) return;
    orc_ctx tmp = *c;
    gather_one(c, t, xi, eta, phi, fld[0]);
    for (int a = 0; a < 2; ++a)
        if (c->coef_aux[a]) { tmp.coef = c->coef_aux[a]; gather_one(&tmp, t, xi, eta, phi, fld[1 + a]); }
}
/* K1 of the thesis: locate -> gather dPhi, dA^s, dA^h -> equilibrium -> equations; five outputs */
void orc_rhs_em(const orc_ctx *c, size_t n, const double *R, const double *Z, const double *phi, const double *upar,
                const double *mu, const double *w, int32_t *cell_out, double *dRdt, double *dZdt, double *dphidt,
                double *dudt, double *dwdt)
{
#pragma omp parallel for schedule(static)
    for (size_t p = 0; p < n; ++p) {
        double o[5] = {0, 0, 0, 0, 0}, xi, eta, fld[3][4];
        int t = locate_one(c, R[p], Z[p], &xi, &eta);
        if (t >= 0) { gather_three(c, t, xi, eta, phi[p], fld); rhs_point_em(c, R[p], Z[p], upar[p], mu[p], w[p], fld, o); }
        if (cell_out) cell_out[p] = t;
        dRdt[p] = o[0]; dZdt[p] = o[1]; dphidt[p] = o[2]; dudt[p] = o[3]; dwdt[p] = o[4];
    }
}

/* ------------------------------------------------------------------- O10 pullback (K2 of the thesis) */
/* PAPER.md:1112-1128 (normalised form): u_new = u_old - (q_s/m_s) <dA^h_old>;
 * delta f_new = delta f_old - (2 q_s/T) v_par <dA^h_old> f_0  (linearised, Maxwellian f_0; the factor 2 from T_N = m_N v_N^2/2).
 * In marker weights (w = delta f/f, 1 - w = f_0/f, reading G7): w_new = w_old - (2 q_s/T) v_par dA^h (1 - w_old)
 * [weight_mode 1: ... x 1]; v_par: the velocity coordinate after the transformation, = u_new (reading G27).
 * Markers outside the mesh (or flagged cell < 0) are left untouched.  The field side (dA^s += dA^h) is not a marker operation. */
void orc_pullback(const orc_ctx *c, size_t n, const double *R, const double *Z, const double *phi, double *upar, double *w,
                  const int32_t *cell_flag)
{
#pragma omp parallel for schedule(static)
    for (size_t p = 0; p < n; ++p) {
        if (cell_flag && cell_flag[p] < 0) continue;
        double xi, eta, fld[3][4];
        int t = locate_one(c, R[p], Z[p], &xi, &eta);
        if (t < 0) continue;
        gather_three(c, t, xi, eta, phi[p], fld);
        const double Ah = fld[2][0];
        const double unew = upar[p] - c->p.qs_over_ms * Ah;
        const double fac = (c->p.weight_mode == 0) ? (1.0 - w[p]) : 1.0;
        w[p] = w[p] - (2.0 * c->p.qs_over_ms / c->p.T) * unew * Ah * fac;
        upar[p] = unew;
    }
}

/* ------------------------------------------------- O11 cubic B-spline toroidal basis (the thesis's own) */
/* Y(R, Phi, Z) = sum_i sum_j Lambda_i(xi, eta) N_j(Phi) Y_ij: C1 triangles in (R, Z), cubic splines in
 * Phi on a uniform periodic grid.  Reading G28: N_j(phi) = beta((phi - phi_j)/h), phi_j = j h,
 * h = 2 pi/N_phi, wrapped periodically, beta the uniform cubic B-spline
 *     beta(x) = 2/3 - x^2 + |x|^3/2  (|x| < 1),  (2 - |x|)^3/6  (1 <= |x| < 2),  0 else.
 * Per triangle and plane j the (R, Z) part is the quintic P_j of the plane's nodal DOFs (O2).  Plain definition: the sum
 * runs over ALL planes.  Outputs as O4: value, d/dR, d/dZ, d/dphi. */
static double bspl(double x) { double a = fabs(x); if (a < 1.0) return 2.0 / 3.0 - a * a + 0.5 * a * a * a; if (a < 2.0) { double u = 2.0 - a; return u * u * u / 6.0; } return 0.0; }
static double bspl_d(double x)
{
    double a = fabs(x), sgn = (x < 0.0) ? -1.0 : 1.0, d;
    if (a < 1.0) d = -2.0 * a + 1.5 * a * a;
    else if (a < 2.0) { double u = 2.0 - a; d = -0.5 * u * u; }
    else d = 0.0;
    return sgn * d;
}
static void gather_one_spline(const orc_ctx *c, int t, double xi, double eta, double phi, double out[4])
{
    const double *g = c->geom + 6 * t;
    const int np = c->n_phi;
    const double h = ORC_TWO_PI / np;
    double f = 0.0, fR = 0.0, fZ = 0.0, fp = 0.0;
    double mono[21], mx[21], me[21];
    for (int k = 0; k < 21; ++k) {
        int i, j; mono_ij(k, &i, &j);
        mono[k] = ipow(xi, i) * ipow(eta, j);
        mx[k] = (i >= 1) ? i * ipow(xi, i - 1) * ipow(eta, j) : 0.0;
        me[k] = (j >= 1) ? j * ipow(xi, i) * ipow(eta, j - 1) : 0.0;
    }
    for (int j = 0; j < np; ++j) {
        double x = (phi - j * h) / h;
        x -= np * floor(x / np + 0.5);                   /* nearest periodic image: x in [-np/2, np/2) */
        const double N = bspl(x), Nd = bspl_d(x) / h;
        if (N == 0.0 && Nd == 0.0) continue;
        const double *cf = c->coef_spl + ((size_t)t * np + j) * ORC_NCOEF;
        double P = 0.0, Px = 0.0, Pe = 0.0;
        for (int k = 0; k < 21; ++k) { P += cf[k] * mono[k]; Px += cf[k] * mx[k]; Pe += cf[k] * me[k]; }
        f += N * P;
        fR += N * (g[2] * Px + g[4] * Pe);
        fZ += N * (g[3] * Px + g[5] * Pe);
        fp += Nd * P;
    }
    out[0] = f; out[1] = fR; out[2] = fZ; out[3] = fp;
}
/* n_phi = 0 returns to the harmonic field of orc_set_modes / orc_set_coef.  coef: [n_tri][n_phi][21] real, or NULL (zeros). */
void orc_set_spline(orc_ctx *c, int n_phi, const double *coef)
{
    free(c->coef_spl); c->coef_spl = NULL; c->n_phi = n_phi > 0 ? n_phi : 0;
    if (c->n_phi == 0) return;
    const size_t nn = (size_t)c->n_tri * c->n_phi * ORC_NCOEF;
    c->coef_spl = (double *)calloc(nn, sizeof(double));
    if (coef) memcpy(c->coef_spl, coef, sizeof(double) * nn);
}
void orc_get_spline(const orc_ctx *c, double *coef) { memcpy(coef, c->coef_spl, sizeof(double) * (size_t)c->n_tri * c->n_phi * ORC_NCOEF); }
/* dofs: [n_phi][n_vert][6] real nodal values per plane; the Bell expansion of O2 plane by plane */
int orc_bell_spline_from_dofs(orc_ctx *c, int n_phi, const double *dofs)
{
    orc_set_spline(c, n_phi, NULL);
    int bad = 0;
#pragma omp parallel for schedule(static) reduction(+ : bad)
    for (int t = 0; t < c->n_tri; ++t) {
        long double A[21][21], rs[21]; int piv[21];
        if (bell_factor(c, t, A, rs, piv)) { bad += 1; continue; }
        const int *v = c->tri + 3 * t;
        for (int j = 0; j < n_phi; ++j) {
            long double b[21];
            for (int pnt = 0; pnt < 3; ++pnt)
                for (int d = 0; d < 6; ++d) b[6 * pnt + d] = dofs[((size_t)j * c->n_vert + v[pnt]) * 6 + d];
            b[18] = b[19] = b[20] = 0.0L;
            bell_solve(A, rs, piv, b);
            double *o = c->coef_spl + ((size_t)t * n_phi + j) * ORC_NCOEF;
            for (int k = 0; k < 21; ++k) o[k] = (double)b[k];
        }
    }
    return bad ? -1 : 0;
}

int orc_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
