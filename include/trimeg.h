/*
 * trimeg.h -- C ABI of libtrimeg: the B200-native (sm_100a) marker-push hot path of the
 * TRIMEG gyrokinetic particle-in-cell method (arxiv/paper_2601_14301).
 *
 * Citations are /root/reference/PAPER.md:<line> (section / equation); readings of passages
 * the paper leaves open are numbered G1..G23, L1..L5, O1..O7 in DESIGN.md §3.
 *
 * The path, per marker ("particle push kernel"):
 *   locate the triangle (contains()) ->
 *   grid-to-particle gather of the perturbed potential dphi and its gradient from C1
 *   quintic triangle elements x toroidal harmonics e^{i n phi}
 *   (Def. 19) ->
 *   analytic equilibrium B = grad psi x grad phi + F grad phi ->
 *   gyro-centre equations of motion A.4-A.6, A.10-A.17 with dA_par = 0
 *   and the delta-f weight rate from d ln f_M / dt ->
 *   classic RK4.
 *
 * Conventions common to every call
 *   - Returns TRIMEG_OK (0) or a negative TRIMEG_ERR_* code; nothing throws or aborts
 *     across this boundary.  trimeg_strerror() names a code.
 *   - "_host" pointers are host memory, read during the call and not retained.
 *     All other data pointers are DEVICE pointers owned by the caller (e.g. PyTorch
 *     tensors); the library never frees or reallocates them.  fp64 everywhere.
 *   - `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).  Work is
 *     enqueued on it and the call returns without synchronising, except where stated.
 *   - Tables (mesh geometry, coefficient table) are owned by the context, uploaded once
 *     ("allocate once, upload static data once").
 *   - One context per GPU (cudaSetDevice before trimeg_mesh_create); every later call runs on
 *     the context's device whatever device is current, and restores the caller's device.  Several
 *     contexts (on one or several GPUs) may live in one process; a context is not thread-safe.  There is no CPU fallback: without a CUDA device calls return
 *     TRIMEG_ERR_CUDA.
 */
#ifndef TRIMEG_H
#define TRIMEG_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define TRIMEG_OK               0
#define TRIMEG_ERR_INVALID_ARG (-1)  /* NULL pointer, negative size, bad enum                   */
#define TRIMEG_ERR_MESH        (-2)  /* nodes not strictly increasing / r_0 != 0 / sagitta rule  */
#define TRIMEG_ERR_NO_FIELD    (-3)  /* a gather/rhs/push was asked before trimeg_field_upload   */
#define TRIMEG_ERR_CUDA        (-4)  /* a CUDA runtime call or kernel launch failed              */
#define TRIMEG_ERR_ALLOC       (-5)  /* device or host allocation failed                         */
#define TRIMEG_ERR_UNSUPPORTED (-6)  /* the call is not defined for the loaded field's toroidal basis */
#define TRIMEG_ERR_CAPACITY    (-7)  /* trimeg_scatter_static: the problem needs more than the fixed static scratch */

#define TRIMEG_NCOEF 21              /* monomials xi^i eta^j, 0 <= i+j <= 5        */

typedef struct trimeg_ctx trimeg_ctx;   /* opaque; owns all device tables */
typedef void *trimeg_stream;            /* cudaStream_t */

/* Physical parameters (plain data, copied by trimeg_mesh_create / trimeg_set_params).
 * Normalised units of PAPER.md:1198: length 1 m, ion mass = charge = 1 in the workloads. */
typedef struct {
    double R0, a, B0;        /* major radius, minor radius, on-axis field                         */
    double q0, q2;           /* cylindrical safety factor q(r) = q0 + q2 (r/a)^2; psi' = B0 r/q   */
    double rho0;             /* rho_0 of A.4-A.6                                  */
    double qs_over_ms;       /* q_s / m_s                                                         */
    double T;                /* Tbar of the Maxwellian; sigma_vpar = sqrt(T/2)    */
    double kappa_n, kappa_T; /* -d ln n0/dr, -d ln T/dr (inverse length)           */
    int eom_variant;         /* 0: b0* as printed in A.4-A.6; 1: (B/B*par) b + ... (reading G2);
                              * 2: the reduced model A.19-A.29, b* -> b, C_d = (m/q) rho_0 (u^2 + mu B) B_0/B^3
                              *    (row f4): in trimeg_rhs / trimeg_push A.28 with dA = 0, in
                              *    trimeg_rhs_em A.24-A.26 and A.29 (ideal Ohm's law); the pullback is unchanged */
    int weight_mode;         /* 0: dw/dt = -(1-w) d ln f_M/dt; 1: dw/dt = -d ln f_M/dt (G7)       */
} trimeg_params;

/* Marker arrays, structure of arrays, each of length n.
 * cell[p] = triangle index of marker p, used as a HINT by the locator (a stale hint costs
 * time, never correctness); cell[p] < 0 marks a marker outside the mesh: it is skipped. */
typedef struct {
    double *R, *Z, *phi;     /* cylindrical position                              */
    double *vpar;            /* parallel velocity v_par = u_par (electrostatic)                   */
    double *mu;              /* magnetic moment v_perp^2 / 2B; never written       */
    double *w;               /* delta-f weight                                 */
    int32_t *cell;
} trimeg_markers;

/* ---- mesh (rows a0, a2 of DESIGN.md §1) --------------------------------------------------
 * Structured ring x sector triangulation of the poloidal plane around the axis (R0, 0):
 * n_vert = 1 + n_r n_theta vertices, n_tri = (2 n_r - 1) n_theta triangles, numbered as in
 * DESIGN.md §3 O1 (axis fan first, then two triangles per ring-sector quad), all
 * counter-clockwise, local coordinates (xi, eta) with the vertices at (0,0),(1,0),(0,1)
 * (PAPER.md:328).
 *   r_nodes_host  n_r + 1 radii, r[0] = 0 < r[1] < ... < r[n_r] = a
 *   vert_R_host, vert_Z_host   n_vert vertex coordinates, or both NULL: the library then
 *                 places v(i,j) at (R0 + r_i cos(2 pi j/n_theta), r_i sin(2 pi j/n_theta))
 *                 with the host libm.  Pass them to get bit-identical geometry to another
 *                 implementation.
 * Errors: INVALID_ARG (NULL, n_r < 2, n_theta < 3), MESH (nodes not increasing, or the chord
 * sagitta r_{k+1}(1 - cos(pi/n_theta)) >= r_{k+2} - r_{k+1}: the locator's 3x3 candidate
 * neighbourhood would not be sufficient, rule L4), CUDA, ALLOC. */
int trimeg_mesh_create(trimeg_ctx **out, int n_r, int n_theta, const double *r_nodes_host,
                       const double *vert_R_host, const double *vert_Z_host,
                       const trimeg_params *params);
/* Row f4, general geometry: any conforming triangulation of the poloidal cross-section with the thesis's own locator
 * (section 3.3: an intermediate grid of boxes, each with the list of the triangles that
 * overlap it; the marker's box is found in O(1), its triangles are tested one by one with the inside-triangle test).
 *   vert_R_host, vert_Z_host: n_vert vertex coordinates; tri_host: int32 [n_tri][3] vertex numbers (a clockwise triple is
 *   turned by swapping its second and third vertex); nbx x nby boxes over the bounding rectangle of the vertices (0: about
 *   one triangle's area per box).  The library builds the geometry table, the neighbour table across the three edges, the
 *   box lists (ascending triangle numbers, bounding boxes inflated by 1e-6 of a box) and the vertex adjacency.
 * Locating rule: the lowest-numbered triangle of the box whose test passes (= of all triangles); if none passes, the one
 * with the largest smallest barycentric coordinate when that is >= -1e-12, else outside (reading G31 of DESIGN.md).
 * Every other call works as on the ring x sector mesh (the equilibrium stays the analytic one of trimeg_params; markers
 * outside the triangulation are lost).  Errors: INVALID_ARG, MESH (vertex number out of range, degenerate triangle, an
 * edge with three owners, non-finite coordinates), CUDA, ALLOC. */
int trimeg_mesh_create_unstructured(trimeg_ctx **out, int n_vert, const double *vert_R_host, const double *vert_Z_host,
                                    int n_tri, const int32_t *tri_host, int nbx, int nby, const trimeg_params *params);
/* Host utility for unstructured meshes (no device work): order_host[q] = the triangle that should get number q so that
 * triangles close in space are close in number -- Hilbert curve over the bounding rectangle, by centroid.  The push keeps the
 * coefficient records of the triangles a CTA's cell-sorted markers sit in in shared memory; when the neighbours of consecutive
 * triangles are unrelated (a shuffled or advancing-front numbering) the CTA meets far more records than it can hold.  Apply
 * the order to the triangle list (tri_new[q] = tri[order[q]]) BEFORE trimeg_mesh_create_unstructured and use the new numbers
 * everywhere; the library never renumbers behind the caller's back (cell numbers are the caller's).
 * Errors: INVALID_ARG, MESH (vertex number out of range, degenerate bounding rectangle), ALLOC. */
int trimeg_mesh_locality_order(int n_vert, const double *vert_R_host, const double *vert_Z_host, int n_tri,
                               const int32_t *tri_host, int32_t *order_host);
int trimeg_mesh_destroy(trimeg_ctx *ctx);
int trimeg_mesh_info(const trimeg_ctx *ctx, int *n_vert, int *n_tri);
int trimeg_set_params(trimeg_ctx *ctx, const trimeg_params *params);
/* Row f4, equilibrium from tables ("the magnetic equilibrium constructed from the EQDSK output file ... B_phi = F/R by means
 * of b-spline interpolation of the poloidal current function F"; B = grad psi x grad phi + F grad phi,
 * B_R = -psi_Z/R, B_Z = psi_R/R).  Reading G32 of DESIGN.md:
 *   psi(R, Z) = sum_ij C[i][j] beta((R - Ra)/hR - i) beta((Z - Za)/hZ - j),   F(psi) = sum_k D[k] beta((psi - pa)/hp - k),
 * beta the uniform cubic B-spline; C_host [nR][nZ] and D_host [nF] are COEFFICIENTS (a prefiltered EQDSK grid), host memory,
 * copied.  |B|, grad B, b, curl b follow from the first and second derivatives of psi and from F'.  The F index is clamped to
 * the table (the end pieces extend as cubics).  While a table is loaded every right-hand side (trimeg_rhs, trimeg_push,
 * trimeg_push_host, trimeg_rhs_em; all eom_variants) uses it in place of the analytic circular equilibrium of trimeg_params
 * (whose R0, a, q0, q2, B0 are then unused), and the profile gradients kappa_n, kappa_T act along grad psi/|grad psi|.
 * C_host = NULL returns to the analytic equilibrium.  Synchronises the device.
 * Errors: INVALID_ARG (sizes < 4, spacings <= 0, or a mesh vertex whose 4 x 4 stencil is not inside the table:
 * every vertex needs Ra + hR <= R <= Ra + (nR - 2) hR and the same in Z), ALLOC, CUDA. */
int trimeg_equilibrium_upload(trimeg_ctx *ctx, int nR, int nZ, double Ra, double Za, double hR, double hZ,
                              const double *C_host, int nF, double pa, double hp, const double *D_host);
/* test hook: geometry table [n_tri][6] = (R_v0, Z_v0, xi_R, xi_Z, eta_R, eta_Z) to device memory */
int trimeg_mesh_download_geom(trimeg_ctx *ctx, double *geom_dev, trimeg_stream stream);

/* ---- field (row a0) -----------------------------------------------------------------------
 * dphi(R, phi, Z) = sum_n Re( P_n(xi, eta) e^{i n phi} ), P_n the C1 quintic of the triangle
 * (PAPER.md:338-363, 365-368 with the toroidal basis replaced by harmonics).
 *   kind 0: data_dev = nodal DOFs [n_modes][n_vert][6] complex128 in the order
 *           (f, f_R, f_Z, f_RR, f_RZ, f_ZZ) of PAPER.md:350-353; the library expands them on
 *           the device to the 21 monomial coefficients per triangle and mode with Bell's
 *           reduction (normal derivative cubic on every edge, reading O2).
 *   kind 1: data_dev = coefficients [n_tri][n_modes][21] complex128, degree-major monomial
 *           order k <-> (i, j): for d = 0..5, for j = 0..d: xi^(d-j) eta^j.
 * mode_n_host: n_modes toroidal mode numbers.  n_modes = 0 is legal (dphi == 0).
 * Ordering: the table is (re)written on `stream`.  A gather / rhs / push that the caller enqueued
 * earlier on ANOTHER stream may still be reading it: order uploads and pushes on one stream (or
 * with events).  trimeg_push_host waits for the upload by itself.  A change of n_modes
 * re-allocates the table and synchronises the device.
 * Errors: INVALID_ARG, ALLOC, CUDA. */
int trimeg_field_upload(trimeg_ctx *ctx, int n_modes, const int *mode_n_host,
                        const void *data_dev, int kind, trimeg_stream stream);
/* test hook: coefficient table in the kind-1 layout to device memory */
int trimeg_field_download_coeffs(trimeg_ctx *ctx, void *coeffs_dev, trimeg_stream stream);

/* ---- field on the cubic B-spline toroidal basis (row f3) ---------------------------------------
 * The thesis's own toroidal discretisation ("the cubic B-spline in the toroidal direction";
 * PAPER.md:365-368 Y = sum_i sum_j Lambda_i(xi, eta) N_j(Phi) Y_ij; PAPER.md:320-326 uniform periodic grid in phi):
 *   dphi(R, phi, Z) = sum_{j=0}^{n_phi-1} N_j(phi) P_j(xi, eta),   N_j(phi) = beta(phi/h - j),  h = 2 pi/n_phi,
 * periodic in j, beta the uniform cubic B-spline (reading G28 of DESIGN.md), P_j the real C1 quintic of plane j.
 * Four planes are non-zero at any phi.
 *   kind 0: data_dev = nodal DOFs [n_phi][n_vert][6] float64, the six per vertex as in trimeg_field_upload;
 *   kind 1: data_dev = coefficients [n_tri][n_phi][21] float64, monomial order as in trimeg_field_upload.
 * n_phi >= 4.  Replaces whatever field was loaded (harmonic table, mode list and the dA^s / dA^h tables are dropped);
 * a later trimeg_field_upload returns to harmonics.  trimeg_locate / gather / rhs / push / push_host / sort / compact
 * work on either basis; trimeg_scatter, trimeg_field_upload_aux, trimeg_rhs_em and trimeg_pullback return
 * UNSUPPORTED while a B-spline field is loaded.  trimeg_field_download_coeffs writes [n_tri][n_phi][21] float64.
 * Ordering as trimeg_field_upload.  Errors: INVALID_ARG (n_phi < 4, NULL), ALLOC, CUDA. */
int trimeg_field_upload_spline(trimeg_ctx *ctx, int n_phi, const double *data_dev, int kind,
                               trimeg_stream stream);

/* ---- locator (row a2) ----------------------------------------------
 * cell[p] = lowest triangle index t whose contains() test passes for (R[p], Z[p]), the test
 * being xi >= 0, eta >= 0, 1 - xi - eta >= 0 with every operation individually rounded in
 * the order of DESIGN.md §3 O3 (no fused multiply-add); -1 outside the outer polygon.
 * The result is bit-identical to the brute-force search over all triangles. */
int trimeg_locate(trimeg_ctx *ctx, size_t n, const double *R, const double *Z, int32_t *cell,
                  trimeg_stream stream);

/* ---- gather only (row a3; BASELINE.json configs[3]) ----------------------------------------
 * The grid-to-particle interpolation on its own ("field gathering/interpolation";
 * PAPER.md:608 section 5.1: "the electrostatic scalar potential needs to always be computed"; the
 * g2p subroutine of the pullback / density / g2p2g kernels):
 * dphi, d dphi/dR, d dphi/dZ (and d dphi/dphi if dphi_dphi != NULL) at the markers.
 * cell_hint may be NULL.  Markers outside the mesh get 0.  NO_FIELD if no field is loaded.
 * Any marker order is correct.  Batches of 2^18 markers and more that come with hints and a field of up
 * to 7 modes: cell-sorted markers (hinted cells that never decrease, markers flagged < 0 aside; up to
 * n / 16 exceptions are tolerated) take a kernel that keeps the coefficient records of its triangles in
 * shared memory and fetches the next markers while it evaluates the current ones; the device decides
 * (both kernels are enqueued, the one not chosen returns at once). */
int trimeg_gather(trimeg_ctx *ctx, size_t n, const double *R, const double *Z, const double *phi,
                  const int32_t *cell_hint, double *dphi, double *dphi_dR, double *dphi_dZ,
                  double *dphi_dphi, trimeg_stream stream);

/* ---- one right-hand-side evaluation (rows a2-a5) -------------------------------------------
 * The paper's push kernel: five time derivatives per marker
 * (dRdt, dZdt, dphidt, dvpardt, dwdt), each n doubles.  Markers are not modified; markers
 * outside the mesh get 0. */
int trimeg_rhs(trimeg_ctx *ctx, const trimeg_markers *m, size_t n, double *dRdt, double *dZdt,
               double *dphidt, double *dvpardt, double *dwdt, trimeg_stream stream);

/* ---- electromagnetic terms (row f2) ------------------------------------------------------------
 * The mixed-variable scheme of the thesis: dA_par = dA^s + dA^h (A.1), the marker's
 * velocity coordinate is u_par = v_par + (q_s/m_s) <dA^h> (stored in markers.vpar), the gyro-average is the
 * identity.  dA^s and dA^h live on the basis and mode list of the uploaded field (dPhi):
 * trimeg_field_upload_aux(which = TRIMEG_FIELD_AS / _AH, data_dev, kind) takes nodal DOFs (kind 0) or
 * coefficients (kind 1) in the layouts of trimeg_field_upload; data_dev = NULL drops the table (the field is
 * zero).  A trimeg_field_upload that changes the number of modes drops both.  Ordering as trimeg_field_upload.
 * Errors: INVALID_ARG, NO_FIELD (upload dPhi first), ALLOC, CUDA. */
#define TRIMEG_FIELD_AS 1
#define TRIMEG_FIELD_AH 2
int trimeg_field_upload_aux(trimeg_ctx *ctx, int which, const void *data_dev, int kind,
                            trimeg_stream stream);
/* K1, the thesis's push kernel with the electromagnetic model on: one right-hand side
 * per marker -- locate, gather dPhi, dA^s, dA^h, analytic equilibrium, b* = b0* + grad(dA^s) x b / B*_par
 * (A.7-A.9), equilibrium motion A.10-A.13 with u_par, perturbed motion A.14-A.16 with
 * dG = dPhi - u_par dA_par, parallel acceleration A.17 with the ideal Ohm's law d_t dA^s = -b.grad dPhi
 * substituted (reading G26 of DESIGN.md), weight rate of PAPER.md:1208 at
 * v_par = u_par - (q_s/m_s) dA^h.  Five outputs (dRdt, dZdt, dphidt, dudt, dwdt), n doubles each; markers are
 * not modified; markers outside the mesh get 0. */
int trimeg_rhs_em(trimeg_ctx *ctx, const trimeg_markers *m, size_t n, double *dRdt, double *dZdt,
                  double *dphidt, double *dudt, double *dwdt, trimeg_stream stream);
/* K2, the pullback kernel (section 5.2.1; normalised equations): per marker
 * u_new = u_old - (q_s/m_s) dA^h, w_new = w_old - (2 q_s/T) u_new dA^h (1 - w_old) (weight_mode 1: x 1), in
 * place on markers.vpar and markers.w; markers with cell < 0 or outside the mesh are left untouched.  Without
 * a dA^h table the call does nothing.  (The field side, dA^s += dA^h, is a table operation of the caller.) */
int trimeg_pullback(trimeg_ctx *ctx, trimeg_markers *m, size_t n, trimeg_stream stream);

/* ---- particle-to-grid projection / scatter (row f1) -----------------------------------------
 * "The charge of each particle is projected onto the basis functions" (section 3.1; the P2G
 * functions of PAPER.md:249; section 6.3: the phase the thesis left on the CPU as "not suitable
 * for GPU offloading").  The adjoint of trimeg_gather: with Lambda_{v,d} the C1 basis function of degree of
 * freedom d = (f, f_R, f_Z, f_RR, f_RZ, f_ZZ) at vertex v,
 *     rhs[n][v][d] = sum_p w_p Lambda_{v,d}(R_p, Z_p) e^{-i n phi_p}
 * for the toroidal modes n of the uploaded field (trimeg_field_upload supplies the mode list; the field values
 * are not used), so that for real weights  sum_p w_p dphi(x_p) = Re sum Y_{n,v,d} conj(rhs[n][v][d])  for any
 * nodal values Y.  rhs_dev: [n_modes][n_vert][6] complex128, device memory, overwritten.
 * m: the marker arrays (R, Z, phi, w and cell are read; cell is a HINT, cell < 0 = marker skipped; markers
 * outside the mesh contribute nothing).  Any marker order is correct and costs the same: the markers are
 * brought into triangle order by an index sort inside (8 B of context scratch per marker, plus 288 B per
 * triangle and mode for the per-triangle results).  The summation order inside a triangle is unspecified
 * (results reproduce to rounding).  Multi-GPU: each GPU scatters its markers; one all-reduce (sum) of rhs
 * is the only collective.  Errors: INVALID_ARG, NO_FIELD (no mode list uploaded), ALLOC, CUDA. */
int trimeg_scatter(trimeg_ctx *ctx, const trimeg_markers *m, size_t n, void *rhs_dev,
                   trimeg_stream stream);

/* The same projection for callers that cannot allocate device memory (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc): trimeg_scatter_static calls no cudaMalloc, cudaFree or any allocating routine.
 * All its scratch -- histogram bins, the two int32 index arrays of the sort, the per-triangle results -- lives in ONE
 * array of TRIMEG_SCATTER_STATIC_BYTES (16 MiB) in the library's device image, which every GPU that loads the library
 * holds until the process exits.  Same arguments, same kernels, same result (to the rounding of the unspecified summation
 * order inside a triangle) as trimeg_scatter.  Capacity: with the scratch laid out as
 *     256-aligned 4 (n_tri + 8)  +  2 x 256-aligned 4 n  +  288 n_tri n_modes   bytes  <=  TRIMEG_SCATTER_STATIC_BYTES
 * (e.g. 480 triangles x 2 modes with up to 2.0e6 markers; 32 512 triangles x 3 modes does not fit), else the call
 * returns TRIMEG_ERR_CAPACITY and does nothing: use trimeg_scatter.  The array is shared by every context of a device and
 * keeps the last call's contents (the call clears what must start at zero): two calls that overlap on the GPU -- on two
 * streams, or from two contexts of one device -- race; calls on one stream are ordered and safe.  The array's device
 * address is looked up once per device (cudaGetSymbolAddress) on the first call.
 * Errors: INVALID_ARG, NO_FIELD, UNSUPPORTED (B-spline field), CAPACITY, CUDA. */
#define TRIMEG_SCATTER_STATIC_BYTES (16 * 1024 * 1024)
int trimeg_scatter_static(trimeg_ctx *ctx, const trimeg_markers *m, size_t n, void *rhs_dev, trimeg_stream stream);

/* ---- cell sort (row a1) ---------------------------------------------------------------------
 * Why: the thesis's kernel reads the field tables with 18 % of its accesses coalesced and leaves the
 * on-chip shared memory unused (section 6.4); with the markers ordered by triangle the
 * lanes of a warp read the same coefficient record and the record can be staged on chip.
 * Counting sort of the markers by cell (markers with cell < 0 go last).  Permutes all seven
 * arrays in place.  perm_dev (int64[n], may be NULL) receives, for every new position, the
 * old index.  The order inside one cell is unspecified.  Uses context-owned scratch of
 * ~60 B/marker, grown on demand (ALLOC if that fails). */
int trimeg_sort(trimeg_ctx *ctx, trimeg_markers *m, size_t n, int64_t *perm_dev,
                trimeg_stream stream);

/* ---- compaction of the active list (row a6) -------------------------------------------------
 * Markers evolve independently of each other (section 5.1), so a marker that has left
 * the mesh (lost-marker rule of trimeg_push, reading G18) can be dropped from the active range
 * without touching the others.  Stable partition: markers with cell >= 0 first (original order
 * kept), lost markers after them.  *n_active_host receives the number of active markers (the call
 * synchronises the stream to return it).  perm_dev as in trimeg_sort. */
int trimeg_compact(trimeg_ctx *ctx, trimeg_markers *m, size_t n, int64_t *perm_dev,
                   size_t *n_active_host, trimeg_stream stream);

/* ---- the push (rows a2-a6) ------------------------------------------------------------------
 * nsteps classic RK4 steps of size dt on y = (R, Z, phi, vpar, w), mu constant, with
 * the field frozen; four locate + gather + equilibrium + RHS evaluations per step (the thesis's push
 * kernel), all in one kernel.  After each step phi is wrapped to [0, 2 pi) and
 * cell is set to the triangle of the new position.  A marker whose any stage position, or new
 * position, is outside the mesh is restored to its start-of-step state, flagged cell = -1 and skipped
 * from then on (reading G18); it keeps its index (use trimeg_compact to drop it).  Markers are not
 * reordered.  INVALID_ARG for a NaN dt or nsteps < 0. */
int trimeg_push(trimeg_ctx *ctx, trimeg_markers *m, size_t n, double dt, int nsteps,
                trimeg_stream stream);
/* Schedule used by trimeg_push / trimeg_push_host (same results, different kernels):
 *  TRIMEG_PUSH_KERNEL_AUTO (the default)  LANE for a field of up to 6 toroidal modes, WCACHE above;
 *  TRIMEG_PUSH_KERNEL_THREAD   one thread per marker, state in registers, coefficients through L1 (the plain schedule);
 *  TRIMEG_PUSH_KERNEL_LANE     lane-owned markers: every warp owns 64 markers, lane l the markers l and l + 32, for the
 *         whole call (state in shared memory; no grouping, no evaluation slots); one marker per evaluation in two phases
 *         (all Horner steps in xi, then those in eta) so that runs of DFMAs share their multiplier (the FP64 pipe reads one
 *         register operand per cycle); the coefficient records of the CTA's triangles sit in a shared,
 *         insert-only hash table in shared memory; 16 warps per CTA, one CTA per SM; no block barrier inside a 10-step call;
 *  TRIMEG_PUSH_KERNEL_WCACHE   every warp owns 59 markers, groups them by triangle with ballots (anew only at a stage where
 *         one of them has changed its triangle) into 64 evaluation slots, every group starting at an even slot, and evaluates
 *         32 slots per pass, one marker per lane in the same two phases: the lanes 2j, 2j+1 read one record, and a warp-wide
 *         16-byte shared-memory load whose addresses agree in such pairs costs 2 wavefronts instead of 4 -- from about seven
 *         modes on the shared-memory pipe cannot deliver a coefficient per marker at 4; same record table; 16 warps per CTA up to
 *         14 modes (128 registers), 12 above (the larger records need the room).
 * Fastest when the markers are cell-sorted (trimeg_sort); any order is correct.
 * INVALID_ARG for a variant outside -1..TRIMEG_PUSH_KERNEL_MAX.  (Schedules of earlier rounds that lost everywhere were
 * removed: lock-step CTA tiles -- commit 3003ca4 --, warp kernels reading the records through L1 -- commit a10a1dc.) */
#define TRIMEG_PUSH_KERNEL_AUTO (-1)
#define TRIMEG_PUSH_KERNEL_THREAD 0
#define TRIMEG_PUSH_KERNEL_LANE 1
#define TRIMEG_PUSH_KERNEL_WCACHE 2
#define TRIMEG_PUSH_KERNEL_MAX 2
int trimeg_set_push_kernel(trimeg_ctx *ctx, int variant);
/* The variant trimeg_push will launch (AUTO resolved for the uploaded field; otherwise the TRIMEG_PUSH_KERNEL
 * environment override at context creation -- ignored unless it parses as an integer in range -- or the last
 * trimeg_set_push_kernel); -2 for a NULL context. */
int trimeg_get_push_kernel(const trimeg_ctx *ctx);

/* ---- end-to-end push from HOST buffers -------------------------------------------------------
 * The thesis's offloading strategy (section 5.5): device memory is allocated once and
 * kept, static tables are uploaded once, only the marker arrays travel.  Same result as: copy the seven
 * arrays to the device, trimeg_locate if locate_first != 0, trimeg_sort, trimeg_push, undo the sort, copy
 * R, Z, phi, vpar, w, cell back.  `m` holds HOST pointers (pinned memory makes the copies asynchronous).
 * The batch is cut into up to 8 chunks of consecutive markers (at least ~100 markers per triangle each);
 * every chunk is copied in, located, cell-sorted, pushed with a re-sort every 10 steps, unsorted and copied
 * out on three streams of the context, so that the copies of one chunk run under the push of another.
 * Results are returned in the caller's order and do not depend on the chunking.  The device buffers
 * (2 marker sets + 3 permutations, 128 B per marker) stay allocated in the context until
 * trimeg_release_host_buffers or trimeg_mesh_destroy.  Waits for the last trimeg_field_upload of the
 * context; synchronises before returning.  INVALID_ARG for a NaN dt. */
int trimeg_push_host(trimeg_ctx *ctx, trimeg_markers *m_host, size_t n, double dt, int nsteps,
                     int locate_first);
/* Frees the device buffers kept by trimeg_push_host / trimeg_sort / trimeg_compact (they are
 * re-allocated on demand).  Synchronises the device. */
int trimeg_release_host_buffers(trimeg_ctx *ctx);

/* ---- statistics ------------------------------------------------------------------------------
 * Totals since context creation (or the last reset): markers flagged lost by trimeg_push,
 * locator calls that left the hinted triangle, kernels launched by the library.
 * Synchronises the device.  Any pointer may be NULL. */
int trimeg_get_stats(trimeg_ctx *ctx, int64_t *n_lost, int64_t *n_relocated, int64_t *n_launches);
int trimeg_reset_stats(trimeg_ctx *ctx);
/* Schedule diagnostics of the warp kernels since the last reset, out8[0..7] (host), summed over warps:
 * [1] stages at which a warp had to group its markers by triangle anew; [5] markers evaluated by the
 * one-marker path; [6] coefficient records copied to shared memory (WCACHE) or triangle groups formed (WARP);
 * [7] RK4 stages run.  [0], [3], [4]: SM cycles of lane 0 spent grouping (+ record lookups), evaluating +
 * finishing, and on markers without a slot -- only in a library built with -DTRIMEG_PROFILE
 * (python -m paper_2601_14301_b200.build --profile), else 0.  Synchronises the device. */
int trimeg_get_tile_counters(trimeg_ctx *ctx, int64_t *out8_host);

/* ---- diagnostics ------------------------------------------------------------------------------
 * Measured FP64 vector (DFMA) throughput of the current device in TFLOP/s (2 flops per DFMA),
 * best of 5 launches of a dependency-free DFMA loop: the denominator of the FP64 roofline in
 * DESIGN.md §6.  Not part of the path.  Synchronises. */
int trimeg_measure_fp64_peak(trimeg_ctx *ctx, double *tflops_out);
/* The same loop with `n_reg_operands` (1, 2 or 3) of the three DFMA source operands coming fresh from
 * the register file in every instruction (the others are constants or sit in the operand reuse
 * cache).  On sm_100 the FP64 pipe reads one 64-bit register operand per cycle, so a DFMA stream whose
 * three operands all change from one instruction to the next -- a Horner step a <- a x + c over several
 * markers -- runs at 2/3 of trimeg_measure_fp64_peak.  INVALID_ARG outside 1..3. */
int trimeg_measure_fp64_peak_operands(trimeg_ctx *ctx, int n_reg_operands, double *tflops_out);

/* Denominator for the gather of markers in random order (configs[3] "as drawn"): GB/s of record bytes when every
 * thread reads a whole record of `record_bytes` (a multiple of 16; e.g. 1008 = 3 modes x 21 complex coefficients), 16
 * bytes at a time, from a record chosen at random in a zero-filled table of `table_bytes` (33 MB: resident in the 126 MB
 * L2; 1.4 GB: from HBM), and nothing else -- the access pattern of gather_kernel without its arithmetic.  Best of 4
 * launches.  Not part of the path.  Allocates and frees the table; synchronises.  Errors: INVALID_ARG, ALLOC, CUDA. */
int trimeg_measure_gather_peak(trimeg_ctx *ctx, size_t table_bytes, int record_bytes, double *gbs_out);

const char *trimeg_strerror(int code);
const char *trimeg_version(void);

#ifdef __cplusplus
}
#endif
#endif /* TRIMEG_H */
