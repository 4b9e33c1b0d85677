// trimeg_scatter.cu -- row f1 of DESIGN.md section 1: particle-to-grid projection of the marker weights onto the C1 basis
// x toroidal harmonics ("the charge of each particle is projected onto the basis functions"; PAPER.md:249
// P2G; PAPER.md:936 the phase the thesis left on the CPU), the adjoint of the gather (row a3):
//     rhs[n][v][d] = sum_p w_p Lambda_{v,d}(R_p, Z_p) e^{-i n phi_p}.
//
// The basis functions of a triangle are quintics: Lambda_j = sum_k B_t[k][j] xi^i eta^j with B_t the triangle's Bell
// matrix (21 x 18).  So the sum over the markers of a triangle factors into
//   (1) the monomial moments  M_t[n][k] = sum_{p in t} w_p xi_p^i eta_p^j e^{-i n phi_p}      (21 per mode, complex),
//   (2) the transposed Bell expansion  r_t[n][j] = sum_k B_t[k][j] M_t[n][k]                  (18 per mode),
//   (3) the assembly over the triangles around a vertex  rhs[n][v][d] = sum_{t ni v} r_t[n][6 loc + d].
// (1) is the hot part: a rank-one update of a 21 x 2M matrix per marker.  Markers are brought into triangle order by an
// index sort (histogram, scan, index scatter -- a few bytes per marker, no marker data is moved), one CTA takes one
// triangle: it stages the monomials and the weighted toroidal factors of a batch of markers in shared memory and every
// thread accumulates a 7 x 2 tile of complex moments in registers (7 monomials x 2 modes), the markers of the batch
// divided among the lanes that share the modes.  (2) uses the same fixed right inverse and edge bubbles as the library's Bell
// expansion (bell_kernel), transposed -- no linear solve.  (3) runs by vertex over a precomputed vertex -> triangle
// adjacency: no atomics, and the result does not depend on the order of the triangles.
#include <mutex>

#include "trimeg_internal.h"
#include "trimeg_mesh.cuh"
#include "bell_tables.inc"

namespace trimeg {

namespace {

constexpr int SC_THREADS = 96;      // 3 warps: warp w accumulates monomials 7 w .. 7 w + 6
constexpr int SC_BATCH = 64;        // markers staged per round
constexpr int SC_MBLK = 16;         // toroidal modes per pass over the markers of a triangle
constexpr int SC_MT = 2;            // toroidal modes per thread

// cell of every marker (hint < 0: lost, skipped), for the index sort
__global__ void __launch_bounds__(256) scatter_locate_kernel(MeshDev M, size_t n, const double *__restrict__ R,
                                                             const double *__restrict__ Z, const int32_t *__restrict__ hint,
                                                             int32_t *__restrict__ cell)
{
    const size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n) return;
    int c = hint[p];
    if (c >= 0) { Bary b; int moved = 0; c = locate(M, R[p], Z[p], c, b, moved); }
    cell[p] = c;
}

__global__ void __launch_bounds__(256) scatter_hist_kernel(size_t n, const int32_t *__restrict__ cell, int n_tri, int *__restrict__ bins)
{
    const size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31;
    int c = -1 - lane;                                   // past the end or lost: a key of its own, nothing counted
    if (p < n) { const int cc = cell[p]; if (cc >= 0 && cc < n_tri) c = cc; }
    const unsigned grp = __match_any_sync(0xffffffffu, c);
    if (c >= 0 && lane == __ffs(grp) - 1) atomicAdd(bins + c, __popc(grp));
}

// perm[position in triangle order] = marker index; afterwards cursor[t] = end of triangle t's segment
__global__ void __launch_bounds__(256) scatter_index_kernel(size_t n, const int32_t *__restrict__ cell, int n_tri, int *__restrict__ cursor,
                                                            int32_t *__restrict__ perm)
{
    const size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31;
    int c = -1 - lane;
    if (p < n) { const int cc = cell[p]; if (cc >= 0 && cc < n_tri) c = cc; }
    const unsigned grp = __match_any_sync(0xffffffffu, c);
    const int leader = __ffs(grp) - 1;
    int first = 0;
    if (c >= 0 && lane == leader) first = atomicAdd(cursor + c, __popc(grp));
    first = __shfl_sync(0xffffffffu, first, leader);
    if (c >= 0) perm[(size_t)first + __popc(grp & ((1u << lane) - 1u))] = (int32_t)p;
}

// (1) + (2): one CTA per triangle.  tri_rhs [n_tri][n_modes][18] complex.
__global__ void __launch_bounds__(SC_THREADS) scatter_moments_kernel(MeshDev M, FieldDev F, int n_theta, const int *__restrict__ tri, const double *__restrict__ vR,
                                                                     const double *__restrict__ vZ, const double *__restrict__ R,
                                                                     const double *__restrict__ Z, const double *__restrict__ phi,
                                                                     const double *__restrict__ w, const int32_t *__restrict__ perm,
                                                                     const int *__restrict__ seg_end, double2 *__restrict__ tri_rhs)
{
    __shared__ double mono[NCOEF][SC_BATCH];             // monomials of the batch, [k][p]
    __shared__ double2 wE[SC_BATCH][SC_MBLK + 1];        // w_p e^{-i n phi_p} of the batch, [p][mode of the block] (+1: bank spread)
    __shared__ double2 mom[SC_MBLK][NCOEF + 1];          // moments of the mode block, then M' of the transposed expansion
    const int t = blockIdx.x, tid = threadIdx.x, lane = tid & 31, wrp = tid >> 5;
    const int s0 = (t == 0) ? 0 : seg_end[t - 1], s1 = seg_end[t];
    const int n_modes = F.n_modes;
    double2 *out = tri_rhs + (size_t)t * n_modes * 18;
    if (s1 <= s0) {                                      // no marker in this triangle
        for (int k = tid; k < n_modes * 18; k += SC_THREADS) out[k] = make_double2(0.0, 0.0);
        return;
    }
    const double2 *g = reinterpret_cast<const double2 *>(M.geom + 6 * (size_t)t);
    const double2 v0 = __ldg(g), gx = __ldg(g + 1), ge = __ldg(g + 2);
    // edge vectors of the triangle (for the transposed map from reference derivatives to (R, Z) derivatives)
    int vtx[3];
    tri_vertices(n_theta, tri, t, vtx);
    const double e1R = vR[vtx[1]] - vR[vtx[0]], e1Z = vZ[vtx[1]] - vZ[vtx[0]];
    const double e2R = vR[vtx[2]] - vR[vtx[0]], e2Z = vZ[vtx[2]] - vZ[vtx[0]];

    for (int m0 = 0; m0 < n_modes; m0 += SC_MBLK) {
        const int mb = min(SC_MBLK, n_modes - m0);       // modes of this block
        int ng = 1;
        while (SC_MT * ng < mb) ng <<= 1;                // lanes of a warp = ng groups of SC_MT modes x (32 / ng) marker slices
        const int n_sl = 32 / ng, my_grp = lane & (ng - 1), my_sl = lane / ng, mfill = SC_MT * ng;
        double ar[7][SC_MT], ai[7][SC_MT];               // 7 monomials x SC_MT modes of complex moments per thread
#pragma unroll
        for (int i = 0; i < 7; ++i)
#pragma unroll
            for (int k = 0; k < SC_MT; ++k) ar[i][k] = ai[i][k] = 0.0;
        // the marker a thread stages in the next batch is fetched (perm -> R, Z, phi, w: two dependent trips to HBM) while
        // the current batch is being accumulated
        double nxR = 0.0, nxZ = 0.0, nxP = 0.0, nxW = 0.0;
        if (tid < SC_BATCH && s0 + tid < s1) { const int p = perm[s0 + tid]; nxR = R[p]; nxZ = Z[p]; nxP = phi[p]; nxW = w[p]; }
        for (int b0 = s0; b0 < s1; b0 += SC_BATCH) {
            const int nb = min(SC_BATCH, s1 - b0);
            __syncthreads();                             // the previous batch has been consumed
            const double cR = nxR, cZ = nxZ, cP = nxP, cW = nxW;
            if (tid < SC_BATCH && b0 + SC_BATCH + tid < s1) {
                const int p = perm[b0 + SC_BATCH + tid];
                nxR = R[p]; nxZ = Z[p]; nxP = phi[p]; nxW = w[p];
            }
            if (tid < nb) {                              // ---- stage: monomials, weighted toroidal factors
                const double dx = __dsub_rn(cR, v0.x), dz = __dsub_rn(cZ, v0.y);   // local coordinates as the locator's (rule L2)
                const double xi = __dadd_rn(__dmul_rn(gx.x, dx), __dmul_rn(gx.y, dz));
                const double eta = __dadd_rn(__dmul_rn(ge.x, dx), __dmul_rn(ge.y, dz));
                double xp[6], ep[6];
                xp[0] = ep[0] = 1.0;
#pragma unroll
                for (int i = 1; i < 6; ++i) { xp[i] = xp[i - 1] * xi; ep[i] = ep[i - 1] * eta; }
#pragma unroll
                for (int d = 0; d < 6; ++d)
#pragma unroll
                    for (int j = 0; j <= d; ++j) mono[d * (d + 1) / 2 + j][tid] = xp[d - j] * ep[j];
                const double ph = cP, wp = cW;
                if (F.is_ap) {                           // e^{-i n phi}: rotation from mode to mode
                    double sr, cr, sd, cd;
                    sincos((double)(F.n_first + m0 * F.n_step) * ph, &sr, &cr);
                    sincos((double)F.n_step * ph, &sd, &cd);
                    double er = wp * cr, ei = -wp * sr;
                    for (int k = 0; k < mb; ++k) {
                        wE[tid][k] = make_double2(er, ei);
                        const double tr = fma(er, cd, ei * sd);          // times e^{-i dn phi}
                        ei = fma(ei, cd, -er * sd);
                        er = tr;
                    }
                } else {
                    for (int k = 0; k < mb; ++k) {
                        double sr, cr;
                        sincos((double)__ldg(F.mode_n + m0 + k) * ph, &sr, &cr);
                        wE[tid][k] = make_double2(wp * cr, -wp * sr);
                    }
                }
                for (int k = mb; k < mfill; ++k) wE[tid][k] = make_double2(0.0, 0.0);     // modes past the end of the list
            }
            __syncthreads();
            // ---- accumulate: a 7 x SC_MT tile of complex moments per thread (15 loaded doubles per 56 multiply-adds: the
            // shared-memory pipe delivers 16 doubles per cycle and SM, the FP64 pipe takes 64 multiply-adds)
            for (int p = my_sl; p < nb; p += n_sl) {
                double2 e[SC_MT];
#pragma unroll
                for (int k = 0; k < SC_MT; ++k) e[k] = wE[p][SC_MT * my_grp + k];
#pragma unroll
                for (int i = 0; i < 7; ++i) {
                    const double mk = mono[7 * wrp + i][p];
#pragma unroll
                    for (int k = 0; k < SC_MT; ++k) { ar[i][k] = fma(mk, e[k].x, ar[i][k]); ai[i][k] = fma(mk, e[k].y, ai[i][k]); }
                }
            }
        }
        // ---- sum over the marker slices, moments to shared memory
#pragma unroll
        for (int i = 0; i < 7; ++i)
#pragma unroll
            for (int k = 0; k < SC_MT; ++k)
                for (int off = ng; off < 32; off <<= 1) {
                    ar[i][k] += __shfl_xor_sync(0xffffffffu, ar[i][k], off);
                    ai[i][k] += __shfl_xor_sync(0xffffffffu, ai[i][k], off);
                }
        __syncthreads();
        if (my_sl == 0)
#pragma unroll
            for (int k = 0; k < SC_MT; ++k)
                if (SC_MT * my_grp + k < mb)
#pragma unroll
                    for (int i = 0; i < 7; ++i) mom[SC_MT * my_grp + k][7 * wrp + i] = make_double2(ar[i][k], ai[i][k]);
        __syncthreads();
        // ---- (2) transposed Bell expansion, one thread per (mode, real / imaginary part)
        for (int q = tid; q < 2 * mb; q += SC_THREADS) {
            const int md = q >> 1, part = q & 1;
            double Mk[NCOEF];
#pragma unroll
            for (int k = 0; k < NCOEF; ++k) Mk[k] = part ? mom[md][k].y : mom[md][k].x;
            // c = c_pre + sum_e z_e N_e with z_e linear in c_pre (bell_kernel): transposed, M' = M + sum_e (N_e . M) dz_e/dc_pre
            const double e11 = e1R * e1R + e1Z * e1Z, e22 = e2R * e2R + e2Z * e2Z, e12 = e1R * e2R + e1Z * e2Z;
            const double ett = e11 - 2.0 * e12 + e22;
            double sb[3] = {0.0, 0.0, 0.0};
#pragma unroll
            for (int k = 0; k < NCOEF; ++k) {
                sb[0] = fma(c_bubble[0][k], Mk[k], sb[0]); sb[1] = fma(c_bubble[1][k], Mk[k], sb[1]); sb[2] = fma(c_bubble[2][k], Mk[k], sb[2]);
            }
            // z_0 = (5 e12 c15 - e11 c16) / e11;  z_1 = -(e22 c19 - 5 e12 c20) / e22;  z_2 = sum_j c_{15+j} (a2 sa_j + b2 sb_j) / ett
            Mk[15] += sb[0] * (5.0 * e12 / e11); Mk[16] -= sb[0];
            Mk[19] -= sb[1]; Mk[20] += sb[1] * (5.0 * e12 / e22);
            const double a2 = e22 - e12, b2 = e11 - e12;
#pragma unroll
            for (int j = 0; j <= 5; ++j) {
                const int i = 5 - j;
                const double sa = (i >= 1) ? (((i - 1) & 1) ? -(double)i : (double)i) : 0.0;     // i (-1)^(i-1)
                const double sbj = (j >= 1) ? ((i & 1) ? -(double)j : (double)j) : 0.0;          // j (-1)^i
                Mk[15 + j] += sb[2] * (a2 * sa + b2 * sbj) / ett;
            }
            // y = P18^T M' (reference-triangle degrees of freedom), then the transposed edge-vector map to (R, Z) derivatives
#pragma unroll
            for (int pv = 0; pv < 3; ++pv) {
                double y[6];
#pragma unroll
                for (int d = 0; d < 6; ++d) {
                    double acc = 0.0;
#pragma unroll
                    for (int k = 0; k < NCOEF; ++k) acc = fma(c_P18[k][6 * pv + d], Mk[k], acc);
                    y[d] = acc;
                }
                double r6[6];
                r6[0] = y[0];
                r6[1] = e1R * y[1] + e2R * y[2];
                r6[2] = e1Z * y[1] + e2Z * y[2];
                r6[3] = e1R * e1R * y[3] + e1R * e2R * y[4] + e2R * e2R * y[5];
                r6[4] = 2.0 * e1R * e1Z * y[3] + (e1R * e2Z + e1Z * e2R) * y[4] + 2.0 * e2R * e2Z * y[5];
                r6[5] = e1Z * e1Z * y[3] + e1Z * e2Z * y[4] + e2Z * e2Z * y[5];
                double *o = reinterpret_cast<double *>(out + (size_t)(m0 + md) * 18 + 6 * pv) + part;
#pragma unroll
                for (int d = 0; d < 6; ++d) o[2 * d] = r6[d];
            }
        }
    }
}

// (3): rhs[n][v][d] = sum over the triangles around v; adjacency entries are 3 t + local vertex
__global__ void __launch_bounds__(256) scatter_assemble_kernel(int n_vert, int n_modes, const int *__restrict__ adj_off,
                                                               const int *__restrict__ adj, const double2 *__restrict__ tri_rhs,
                                                               double2 *__restrict__ rhs)
{
    const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;        // (mode, vertex, d)
    if (idx >= (size_t)n_modes * n_vert * 6) return;
    const int d = (int)(idx % 6), v = (int)((idx / 6) % n_vert), md = (int)(idx / (6 * (size_t)n_vert));
    double sr = 0.0, si = 0.0;
    for (int a = adj_off[v]; a < adj_off[v + 1]; ++a) {
        const int e = adj[a], t = e / 3, loc = e - 3 * t;
        const double2 x = tri_rhs[((size_t)t * n_modes + md) * 18 + 6 * loc + d];
        sr += x.x; si += x.y;
    }
    rhs[idx] = make_double2(sr, si);
}

}  // namespace

// scratch: int32 cell[n], int32 perm[n] (context scratch), bins (context), tri_rhs (context, grown on demand)
cudaError_t launch_scatter(trimeg_ctx *c, const trimeg_markers &m, size_t n, double2 *rhs, int32_t *cell, int32_t *perm,
                           double2 *tri_rhs, cudaStream_t s)
{
    const int n_modes = c->field.n_modes;
    if (n_modes == 0) return cudaSuccess;
    cudaError_t e = cudaMemsetAsync(c->d_bins, 0, sizeof(int) * ((size_t)c->n_tri + 2), s);
    if (e != cudaSuccess) return e;
    if (n > 0) {
        const unsigned grid = (unsigned)((n + 255) / 256);
        scatter_locate_kernel<<<grid, 256, 0, s>>>(c->mesh, n, m.R, m.Z, m.cell, cell);
        scatter_hist_kernel<<<grid, 256, 0, s>>>(n, cell, c->n_tri, c->d_bins);
        launch_scan(c->d_bins, c->n_tri + 1, s);
        scatter_index_kernel<<<grid, 256, 0, s>>>(n, cell, c->n_tri, c->d_bins, perm);
        c->n_launches += 4;
    }
    scatter_moments_kernel<<<c->n_tri, SC_THREADS, 0, s>>>(c->mesh, c->field, c->n_theta, c->d_tri, c->d_vR, c->d_vZ, m.R, m.Z, m.phi, m.w,
                                                          perm, c->d_bins, tri_rhs);
    const size_t work = (size_t)n_modes * c->n_vert * 6;
    scatter_assemble_kernel<<<(unsigned)((work + 255) / 256), 256, 0, s>>>(c->n_vert, n_modes, c->d_adj_off, c->d_adj, tri_rhs, rhs);
    c->n_launches += 2;
    return cudaGetLastError();
}

}  // namespace trimeg

// ------------------------------------------------------------------------------------ scatter without any allocation
// trimeg_scatter_static (include/trimeg.h): the same kernels in the same order as launch_scatter, with ALL scratch -- the
// histogram bins / cursors, the two int32 index arrays and the per-triangle results -- in one file-scope device array of
// TRIMEG_SCATTER_STATIC_BYTES.  Every GPU that loads the library holds the array until the process exits.  In host code the
// array's name is a host-side stand-in, not a device address: its address is fetched with cudaGetSymbolAddress once per
// device, with that device current, and handed to the kernels as an ordinary pointer.
namespace {

static __device__ __align__(256) unsigned char g_scatter_static[TRIMEG_SCATTER_STATIC_BYTES];

constexpr int SCS_MAX_DEVICES = 64;
std::mutex g_scs_mutex;
unsigned char *g_scs_addr[SCS_MAX_DEVICES];              // device address of g_scatter_static on device k, nullptr = not looked up yet

inline size_t scs_align(size_t x) { return (x + 255) / 256 * 256; }

}  // namespace

extern "C" int trimeg_scatter_static(trimeg_ctx *c, const trimeg_markers *m, size_t n, void *rhs_dev, trimeg_stream stream)
{
    using namespace trimeg;
    if (!c || n > 0x7fffffffULL) return TRIMEG_ERR_INVALID_ARG;
    if (n > 0 && (!m || !m->R || !m->Z || !m->phi || !m->w || !m->cell)) return TRIMEG_ERR_INVALID_ARG;
    if (!c->has_field) return TRIMEG_ERR_NO_FIELD;
    if (c->field.n_phi > 0) return TRIMEG_ERR_UNSUPPORTED;
    const int n_modes = c->field.n_modes;
    if (n_modes == 0) return TRIMEG_OK;
    if (!rhs_dev) return TRIMEG_ERR_INVALID_ARG;
    // layout of the static array: bins | cell | perm | per-triangle results
    const size_t off_cell = scs_align(sizeof(int) * ((size_t)c->n_tri + 8));
    const size_t off_perm = off_cell + scs_align(sizeof(int32_t) * (n ? n : 1));
    const size_t off_tri = off_perm + scs_align(sizeof(int32_t) * (n ? n : 1));
    const size_t need = off_tri + sizeof(double2) * 18 * (size_t)c->n_tri * n_modes;
    if (need > (size_t)TRIMEG_SCATTER_STATIC_BYTES) return TRIMEG_ERR_CAPACITY;
    if (c->device < 0 || c->device >= SCS_MAX_DEVICES) return TRIMEG_ERR_CAPACITY;
    int cur = -1;
    if (cudaGetDevice(&cur) != cudaSuccess) { cudaGetLastError(); return TRIMEG_ERR_CUDA; }
    if (cur != c->device && cudaSetDevice(c->device) != cudaSuccess) { cudaGetLastError(); return TRIMEG_ERR_CUDA; }
    int rc = TRIMEG_OK;
    unsigned char *base = nullptr;
    {
        std::lock_guard<std::mutex> lock(g_scs_mutex);
        if (!g_scs_addr[c->device]) {                    // set-up, once per device, with that device current
            void *p = nullptr;
            if (cudaGetSymbolAddress(&p, g_scatter_static) != cudaSuccess || !p) { cudaGetLastError(); rc = TRIMEG_ERR_CUDA; }
            else g_scs_addr[c->device] = (unsigned char *)p;
        }
        base = g_scs_addr[c->device];
    }
    if (rc == TRIMEG_OK) {
        cudaStream_t s = (cudaStream_t)stream;
        int *bins = (int *)base;
        int32_t *cell = (int32_t *)(base + off_cell), *perm = (int32_t *)(base + off_perm);
        double2 *tri_rhs = (double2 *)(base + off_tri);
        // the array keeps the last call's contents: the bins must start at zero; cell, perm and the per-triangle results are
        // written in full before they are read (scatter_moments_kernel writes every triangle's block, zeros for an empty one)
        cudaError_t e = cudaMemsetAsync(bins, 0, sizeof(int) * ((size_t)c->n_tri + 2), s);
        if (e == cudaSuccess) {
            if (n > 0) {
                const unsigned grid = (unsigned)((n + 255) / 256);
                scatter_locate_kernel<<<grid, 256, 0, s>>>(c->mesh, n, m->R, m->Z, m->cell, cell);
                scatter_hist_kernel<<<grid, 256, 0, s>>>(n, cell, c->n_tri, bins);
                launch_scan(bins, c->n_tri + 1, s);
                scatter_index_kernel<<<grid, 256, 0, s>>>(n, cell, c->n_tri, bins, perm);
                c->n_launches += 4;
            }
            const double *nul = nullptr;
            scatter_moments_kernel<<<c->n_tri, SC_THREADS, 0, s>>>(c->mesh, c->field, c->n_theta, c->d_tri, c->d_vR, c->d_vZ, n ? m->R : nul,
                                                                  n ? m->Z : nul, n ? m->phi : nul, n ? m->w : nul, perm, bins, tri_rhs);
            const size_t work = (size_t)n_modes * c->n_vert * 6;
            scatter_assemble_kernel<<<(unsigned)((work + 255) / 256), 256, 0, s>>>(c->n_vert, n_modes, c->d_adj_off, c->d_adj, tri_rhs,
                                                                                   (double2 *)rhs_dev);
            c->n_launches += 2;
            e = cudaGetLastError();
        }
        if (e != cudaSuccess) { cudaGetLastError(); rc = TRIMEG_ERR_CUDA; }
    }
    if (cur != c->device) cudaSetDevice(cur);
    return rc;
}
