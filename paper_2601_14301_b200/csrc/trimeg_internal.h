// trimeg_internal.h -- host-side context and launch wrappers shared by the library's
// translation units (not part of the public ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/trimeg.h"
#include "trimeg_device.cuh"

#ifndef TRIMEG_AUTO_SMALL_MAX_MODES
#define TRIMEG_AUTO_SMALL_MAX_MODES 6
#endif
#define TRIMEG_WCACHE_16_MAX_MODES 14      /* many-mode kernel: 16 warps per CTA up to here, 12 above (trimeg_push_wcache.cu) */
#define TRIMEG_GATHER_LANE_MAX_MODES 7     /* the gather alone: lane kernel for cell-sorted markers up to here */

namespace trimeg {

struct Stats {                      // device-resident counters
    unsigned long long n_lost;
    unsigned long long n_moved;
    // schedule diagnostics of the warp kernels (trimeg_get_tile_counters)
    unsigned long long tile[8];
};

}  // namespace trimeg

struct trimeg_ctx {
    int device;
    int n_sm;
    int n_r, n_theta, n_vert, n_tri;
    trimeg_params params;
    trimeg::MeshDev mesh;
    trimeg::FieldDev field;
    trimeg::PhysDev phys;
    // device tables
    double *d_geom, *d_r_nodes, *d_vR, *d_vZ;
    double *d_eqC, *d_eqD;          // row f4: tabulated equilibrium (NULL: analytic)
    trimeg::EqTabDev *d_eqdesc;     // its descriptor in device memory
    double bbox[4];                 // R min, R max, Z min, Z max of the vertices
    int *d_tri, *d_nbr, *d_box_off, *d_box_tri;   // row f4, unstructured mesh: vertex triples, neighbours, box grid (NULL on the ring x sector mesh)
    double2 *d_coef;
    double2 *d_coef_aux[2];         // row f2: dA^s, dA^h on the main field's basis and mode list; NULL = identically zero
    double *d_coef_spl;             // row f3: [n_tri][n_phi][21] real, the field on the cubic B-spline toroidal basis (then d_coef == NULL)
    int *d_mode_n;
    int has_field;
    int push_kernel;                // trimeg_set_push_kernel variant
    trimeg::Stats *d_stats;
    int64_t n_launches;
    // scratch for sort / compact / host path (grown on demand)
    void *d_scratch;
    size_t scratch_bytes;
    int *d_bins;                    // n_tri + 2 counters
    // row f1 (scatter): vertex -> (triangle, local vertex) adjacency in CSR form, per-triangle results (grown on demand)
    int *d_adj_off, *d_adj;
    void *d_trirhs;
    size_t trirhs_bytes;
    // host path: two marker sets + permutation of the last trimeg_push_host batch (grown on demand)
    void *d_hbuf;
    size_t hbuf_bytes;
    cudaStream_t hstream[3];        // compute, H2D, D2H
    cudaEvent_t hevent[16];         // per chunk: inputs landed (0..7), results ready (8..15)
    int hstreams_ready;
    cudaEvent_t ev_upload;          // recorded after the last trimeg_field_upload on its stream
};

namespace trimeg {

// TRIMEG_PUSH_KERNEL_AUTO (measurements: DESIGN.md section 5).  Few toroidal modes: the per-stage work around the mode
// loop (equations, locate, bookkeeping) weighs as much as the loop, and the kernel with lane-owned markers -- no grouping by
// triangle, no evaluation slots, 16 warps per SM -- wins although its loads cost twice the shared-memory wavefronts (markers
// that have left their triangle sit at arbitrary lanes).  From seven modes on the shared-memory pipe cannot deliver a
// coefficient per marker at that price, and the kernel that groups its markers by triangle (lane pairs on one record, the
// CTA-shared record table) wins: with 16 warps while its records are small, with 12 from 15 modes on (also beyond 26 modes,
// where only a dozen records fit).
inline int auto_push_kernel(int n_modes)
{
    return (n_modes <= TRIMEG_AUTO_SMALL_MAX_MODES) ? TRIMEG_PUSH_KERNEL_LANE : TRIMEG_PUSH_KERNEL_WCACHE;
}

// The schedule a push call runs.  Row f3 (field on cubic B-spline planes): the lane kernel holds plane records as it holds
// mode records (two planes take the place of a complex mode) when the record is a whole number of 16-byte units (n_phi even)
// and a useful number of records fits into shared memory; else, or when the thread schedule is asked for, thread per marker.
constexpr int TRIMEG_SPLINE_LANE_MAX_PLANES = 48;
inline int effective_push_kernel(const trimeg_ctx *c)
{
    if (c->field.n_phi > 0) {
        const bool lane_ok = (c->field.n_phi % 2 == 0) && c->field.n_phi <= TRIMEG_SPLINE_LANE_MAX_PLANES;
        return (c->push_kernel == TRIMEG_PUSH_KERNEL_THREAD || !lane_ok) ? TRIMEG_PUSH_KERNEL_THREAD : TRIMEG_PUSH_KERNEL_LANE;
    }
    return (c->push_kernel == TRIMEG_PUSH_KERNEL_AUTO) ? auto_push_kernel(c->field.n_modes) : c->push_kernel;
}

// launch wrappers implemented in trimeg_push.cu; each returns the cudaError of the launch
cudaError_t launch_locate(trimeg_ctx *c, size_t n, const double *R, const double *Z, int32_t *cell, cudaStream_t s);
cudaError_t launch_gather(trimeg_ctx *c, size_t n, const double *R, const double *Z, const double *phi,
                          const int32_t *hint, double *f, double *fR, double *fZ, double *fP, cudaStream_t s);
cudaError_t launch_rhs(trimeg_ctx *c, const trimeg_markers &m, size_t n, double *dR, double *dZ, double *dP,
                       double *dV, double *dW, cudaStream_t s);
cudaError_t launch_push(trimeg_ctx *c, const trimeg_markers &m, size_t n, double dt, int nsteps, cudaStream_t s);
// trimeg_lib.cu: exclusive scan of nb ints in place, bins[nb] = total
void launch_scan(int *bins, int nb, cudaStream_t s);
// trimeg_scatter.cu: row f1, rhs [n_modes][n_vert][6] complex; cell, perm: int32[n] scratch; tri_rhs [n_tri][n_modes][18] complex
cudaError_t launch_scatter(trimeg_ctx *c, const trimeg_markers &m, size_t n, double2 *rhs, int32_t *cell, int32_t *perm,
                           double2 *tri_rhs, cudaStream_t s);

// trimeg_push_wcache.cu: warp-autonomous with a CTA-shared record table in shared memory (TRIMEG_PUSH_KERNEL_WCACHE)
cudaError_t launch_push_wcache(trimeg_ctx *c, const trimeg_markers &m, size_t n, double dt, int nsteps, cudaStream_t s);

// trimeg_push_lane.cu: lane-owned markers, one marker per evaluation in two phases, CTA-shared record table
// (TRIMEG_PUSH_KERNEL_LANE)
cudaError_t launch_push_lane(trimeg_ctx *c, const trimeg_markers &m, size_t n, double dt, int nsteps, cudaStream_t s);

// trimeg_push_*_core.cu: the same two kernels compiled without the branches of rows f3 / f4
cudaError_t launch_push_wcache_core(trimeg_ctx *c, const trimeg_markers &m, size_t n, double dt, int nsteps, cudaStream_t s);
cudaError_t launch_push_lane_core(trimeg_ctx *c, const trimeg_markers &m, size_t n, double dt, int nsteps, cudaStream_t s);
// trimeg_push_lane_spline.cu: the lane kernel for a B-spline field on the ring x sector mesh, rigorous equations, analytic equilibrium
cudaError_t launch_push_lane_spline(trimeg_ctx *c, const trimeg_markers &m, size_t n, double dt, int nsteps, cudaStream_t s);
inline bool core_case(const trimeg_ctx *c)
{
    return c->field.n_phi == 0 && c->params.eom_variant != 2 && c->mesh.n_r > 0 && c->phys.eq == nullptr;
}
inline bool spline_core_case(const trimeg_ctx *c)
{
    return c->field.n_phi > 0 && c->params.eom_variant != 2 && c->mesh.n_r > 0 && c->phys.eq == nullptr;
}

// trimeg_push_lane.cu: the gather alone for cell-sorted markers; gate / want: runs iff (*gate * 16 <= n) == want
cudaError_t launch_gather_lane(trimeg_ctx *c, size_t n, const double *R, const double *Z, const double *phi, const int32_t *hint,
                               double *f, double *fR, double *fZ, double *fP, const int *gate, int want, cudaStream_t s);
constexpr size_t GATHER_LANE_MIN = 1 << 18;     // below, two more kernel launches cost more than the lane kernel saves

// trimeg_em.cu: row f2, one EM right-hand side (K1) and the pullback of u_par, w (K2)
cudaError_t launch_rhs_em(trimeg_ctx *c, const trimeg_markers &m, size_t n, double *dR, double *dZ, double *dP, double *dU, double *dW,
                          cudaStream_t s);
cudaError_t launch_pullback(trimeg_ctx *c, const trimeg_markers &m, size_t n, cudaStream_t s);
cudaError_t launch_rhs_em_core(trimeg_ctx *c, const trimeg_markers &m, size_t n, double *dR, double *dZ, double *dP, double *dU, double *dW,
                               cudaStream_t s);

}  // namespace trimeg
