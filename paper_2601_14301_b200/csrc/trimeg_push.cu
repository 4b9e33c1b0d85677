// trimeg_push.cu -- hot-path kernels: locate, gather, one RHS evaluation, fused RK4 push.
//
// One thread per marker, marker streams are SoA and coalesced; the RK4 state lives in
// registers for all `nsteps` (the field is frozen, reading O7), so a marker is read once and
// written once per call.  Coefficient records are fetched through the read-only path; when
// the markers are cell-sorted (trimeg_sort) the lanes of a warp read the same record and
// the loads coalesce to one L1 line each.
#include "trimeg_internal.h"

namespace trimeg {

constexpr int PUSH_BLOCK = 128;
static inline unsigned grid_for(size_t n, int block) { return (unsigned)((n + block - 1) / block); }
constexpr double TWO_PI = 6.283185307179586476925286766559;

__device__ __forceinline__ void add_stats(Stats *st, int lost, int moved)
{
    const unsigned mask = __activemask();
    const int l = __reduce_add_sync(mask, lost);
    const int m = __reduce_add_sync(mask, moved);
    if ((threadIdx.x & 31) == (__ffs(mask) - 1)) {
        if (l) atomicAdd(&st->n_lost, (unsigned long long)l);
        if (m) atomicAdd(&st->n_moved, (unsigned long long)m);
    }
}

__global__ void __launch_bounds__(256) locate_kernel(MeshDev M, size_t n, const double *__restrict__ R,
                                                     const double *__restrict__ Z, int32_t *__restrict__ cell)
{
    const size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n) return;
    Bary b;
    int moved = 0;
    cell[p] = locate(M, R[p], Z[p], -1, b, moved);
}

// GATED: device-side choice between this kernel and gather_lane_kernel (runs iff (*gate * 16 <= n) == want), grid-stride loop
// over the markers so that the launch that is not chosen costs nothing; else one thread per marker.
template <bool GATED>
__global__ void __launch_bounds__(256) gather_kernel(MeshDev M, FieldDev F, size_t n, const double *__restrict__ R,
                                                     const double *__restrict__ Z, const double *__restrict__ phi,
                                                     const int32_t *__restrict__ hint, double *__restrict__ f,
                                                     double *__restrict__ fR, double *__restrict__ fZ,
                                                     double *__restrict__ fP, const int *gate, int want)
{
    if (GATED && (((size_t)*gate * 16 <= n) ? 1 : 0) != want) return;
    size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (!GATED && p >= n) return;
    do {
        if (GATED && p >= n) break;
        Bary b;
        int moved = 0;
        const double r = R[p], z = Z[p];
        const int t = locate(M, r, z, hint ? hint[p] : -1, b, moved);
        FieldVal v;
        v.f = v.fR = v.fZ = v.fphi = 0.0;
        if (t >= 0) v = gather(F, t, b, phi[p]);
        f[p] = v.f; fR[p] = v.fR; fZ[p] = v.fZ;
        if (fP) fP[p] = v.fphi;
        p += (size_t)gridDim.x * blockDim.x;
    } while (GATED);
}

// estimate of the number of places where the hinted cells decrease (markers flagged < 0 aside): 0 for cell-sorted markers.
// Only a heuristic hangs on it (which of two correct kernels runs), so it looks at every HINT_SAMPLE-th run of 32 consecutive
// hints (one 128-byte line each, the pairs inside the run) and scales the count: 1/16 of the hint bytes.
constexpr int HINT_SAMPLE = 16;
__global__ void __launch_bounds__(256) hint_order_kernel(size_t n, const int32_t *__restrict__ hint, int *__restrict__ count)
{
    int bad = 0;
    const int lane = threadIdx.x & 31;
    const size_t n_runs = (n + 31) / 32, n_samp = (n_runs + HINT_SAMPLE - 1) / HINT_SAMPLE;
    const size_t warp = ((size_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5, n_warps = ((size_t)gridDim.x * blockDim.x) >> 5;
    for (size_t k = warp; k < n_samp; k += n_warps) {
        const size_t p = (k * HINT_SAMPLE) * 32 + lane;
        if (lane > 0 && p < n) { const int a = hint[p - 1], c = hint[p]; bad += (a >= 0 && c >= 0 && c < a) ? 1 : 0; }
    }
    bad = __reduce_add_sync(0xffffffffu, bad);
    if (lane == 0 && bad) atomicAdd(count, bad * HINT_SAMPLE);
}

// locate -> gather -> equilibrium -> equations at one phase-space point (rows a2-a5)
__device__ __forceinline__ bool rhs_full(const MeshDev &M, const FieldDev &F, const PhysDev &P, double R, double Z,
                                         double phi, double v, double mu, double w, int &cell, Rates &k, int &moved)
{
    Bary b;
    const int t = locate(M, R, Z, cell, b, moved);
    if (t < 0) return false;
    cell = t;
    const FieldVal fv = gather(F, t, b, phi);
    k = rhs_point(P, R, Z, v, mu, w, fv);
    return true;
}

__global__ void __launch_bounds__(256) rhs_kernel(MeshDev M, FieldDev F, PhysDev P, trimeg_markers m, size_t n,
                                                  double *__restrict__ dR, double *__restrict__ dZ,
                                                  double *__restrict__ dP, double *__restrict__ dV,
                                                  double *__restrict__ dW)
{
    const size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n) return;
    Rates k;
    k.R = k.Z = k.phi = k.vpar = k.w = 0.0;
    int cell = m.cell ? m.cell[p] : -1, moved = 0;
    rhs_full(M, F, P, m.R[p], m.Z[p], m.phi[p], m.vpar[p], m.mu[p], m.w[p], cell, k, moved);
    dR[p] = k.R; dZ[p] = k.Z; dP[p] = k.phi; dV[p] = k.vpar; dW[p] = k.w;
}

// Fused RK4 (row a6): y <- y + dt/6 (k1 + 2 k2 + 2 k3 + k4), four full RHS evaluations per
// step at the stage positions, phi wrapped once per step, lost markers restored and flagged.
__global__ void __launch_bounds__(PUSH_BLOCK) push_kernel(MeshDev M, FieldDev F, PhysDev P, trimeg_markers m, size_t n,
                                                          double dt, int nsteps, Stats *st)
{
    const size_t p = (size_t)blockIdx.x * PUSH_BLOCK + threadIdx.x;
    int lost = 0, moved = 0;
    if (p < n) {
        int cell = m.cell[p];
        if (cell >= 0) {
            double R = m.R[p], Z = m.Z[p], phi = m.phi[p], v = m.vpar[p], w = m.w[p];
            const double mu = m.mu[p];
            const double hdt = 0.5 * dt, dt6 = dt / 6.0;
#pragma unroll 1
            for (int s = 0; s < nsteps; ++s) {
                Rates k, a;
                int c = cell;
                bool ok = rhs_full(M, F, P, R, Z, phi, v, mu, w, c, k, moved);
                a = k;
                if (ok) ok = rhs_full(M, F, P, fma(hdt, k.R, R), fma(hdt, k.Z, Z), fma(hdt, k.phi, phi),
                                      fma(hdt, k.vpar, v), mu, fma(hdt, k.w, w), c, k, moved);
                if (ok) {
                    a.R = fma(2.0, k.R, a.R); a.Z = fma(2.0, k.Z, a.Z); a.phi = fma(2.0, k.phi, a.phi);
                    a.vpar = fma(2.0, k.vpar, a.vpar); a.w = fma(2.0, k.w, a.w);
                    ok = rhs_full(M, F, P, fma(hdt, k.R, R), fma(hdt, k.Z, Z), fma(hdt, k.phi, phi),
                                  fma(hdt, k.vpar, v), mu, fma(hdt, k.w, w), c, k, moved);
                }
                if (ok) {
                    a.R = fma(2.0, k.R, a.R); a.Z = fma(2.0, k.Z, a.Z); a.phi = fma(2.0, k.phi, a.phi);
                    a.vpar = fma(2.0, k.vpar, a.vpar); a.w = fma(2.0, k.w, a.w);
                    ok = rhs_full(M, F, P, fma(dt, k.R, R), fma(dt, k.Z, Z), fma(dt, k.phi, phi),
                                  fma(dt, k.vpar, v), mu, fma(dt, k.w, w), c, k, moved);
                }
                double Rn = 0.0, Zn = 0.0, pn = 0.0, vn = 0.0, wn = 0.0;
                if (ok) {
                    Rn = fma(dt6, a.R + k.R, R); Zn = fma(dt6, a.Z + k.Z, Z);
                    pn = fma(dt6, a.phi + k.phi, phi);
                    vn = fma(dt6, a.vpar + k.vpar, v); wn = fma(dt6, a.w + k.w, w);
                    pn = fma(-TWO_PI, floor(pn * (1.0 / TWO_PI)), pn);
                    Bary b;
                    c = locate(M, Rn, Zn, c, b, moved);
                    ok = (c >= 0);
                }
                if (!ok) { cell = -1; lost = 1; break; }        // keep the start-of-step state
                R = Rn; Z = Zn; phi = pn; v = vn; w = wn; cell = c;
            }
            m.R[p] = R; m.Z[p] = Z; m.phi[p] = phi; m.vpar[p] = v; m.w[p] = w; m.cell[p] = cell;
        }
    }
    add_stats(st, lost, moved);
}

// ------------------------------------------------------------------------------- wrappers

cudaError_t launch_locate(trimeg_ctx *c, size_t n, const double *R, const double *Z, int32_t *cell, cudaStream_t s)
{
    if (n == 0) return cudaSuccess;
    locate_kernel<<<grid_for(n, 256), 256, 0, s>>>(c->mesh, n, R, Z, cell);
    c->n_launches++;
    return cudaGetLastError();
}

cudaError_t launch_gather(trimeg_ctx *c, size_t n, const double *R, const double *Z, const double *phi,
                          const int32_t *hint, double *f, double *fR, double *fZ, double *fP, cudaStream_t s)
{
    if (n == 0) return cudaSuccess;
    int *gate = nullptr;
    const bool two = hint && n >= GATHER_LANE_MIN && c->field.n_modes > 0 && c->field.n_modes <= TRIMEG_GATHER_LANE_MAX_MODES;
    if (two) {
        // Large batches with hints: cell-sorted markers (hinted cells that never decrease; up to n / 16 exceptions are
        // tolerated) take the lane kernel (records in shared memory, inputs prefetched), anything else the thread-per-marker
        // kernel.  The device decides: both are enqueued, the one not chosen returns at once.
        gate = c->d_bins + c->n_tri + 4;
        cudaError_t e = cudaMemsetAsync(gate, 0, sizeof(int), s);
        if (e != cudaSuccess) return e;
        hint_order_kernel<<<(unsigned)min((size_t)grid_for(n, 256), (size_t)c->n_sm * 8), 256, 0, s>>>(n, hint, gate);
        c->n_launches++;
    }
    // the thread-per-marker kernel lives on L1 (every lane fetches its own record): keep the SM's carve-out at maximum L1
    // whatever kernel ran before
    if (!two) {
        gather_kernel<false><<<grid_for(n, 256), 256, 0, s>>>(c->mesh, c->field, n, R, Z, phi, hint, f, fR, fZ, fP, nullptr, 0);
        c->n_launches++;
        return cudaGetLastError();
    }
    cudaFuncSetAttribute(gather_kernel<true>, cudaFuncAttributePreferredSharedMemoryCarveout, (int)cudaSharedmemCarveoutMaxL1);
    // a fixed grid (grid-stride loop): when the lane kernel is chosen, this launch costs its CTAs' start-up alone
    // (65 536 CTAs that return at once: 0.23 ms, a tenth of the lane kernel's time on 2^26 markers; 9472: 0.03 ms)
    gather_kernel<true><<<(unsigned)min((size_t)grid_for(n, 256), (size_t)c->n_sm * 64), 256, 0, s>>>(c->mesh, c->field, n, R, Z, phi, hint,
                                                                                                    f, fR, fZ, fP, gate, 0);
    c->n_launches++;
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    return launch_gather_lane(c, n, R, Z, phi, hint, f, fR, fZ, fP, gate, 1, s);
}

cudaError_t launch_rhs(trimeg_ctx *c, const trimeg_markers &m, size_t n, double *dR, double *dZ, double *dP,
                       double *dV, double *dW, cudaStream_t s)
{
    if (n == 0) return cudaSuccess;
    rhs_kernel<<<grid_for(n, 256), 256, 0, s>>>(c->mesh, c->field, c->phys, m, n, dR, dZ, dP, dV, dW);
    c->n_launches++;
    return cudaGetLastError();
}

cudaError_t launch_push(trimeg_ctx *c, const trimeg_markers &m, size_t n, double dt, int nsteps, cudaStream_t s)
{
    if (n == 0 || nsteps <= 0) return cudaSuccess;
    const int variant = effective_push_kernel(c);
    if (variant == TRIMEG_PUSH_KERNEL_LANE)
        return core_case(c) ? launch_push_lane_core(c, m, n, dt, nsteps, s)
                            : spline_core_case(c) ? launch_push_lane_spline(c, m, n, dt, nsteps, s) : launch_push_lane(c, m, n, dt, nsteps, s);
    if (variant == TRIMEG_PUSH_KERNEL_WCACHE) return core_case(c) ? launch_push_wcache_core(c, m, n, dt, nsteps, s) : launch_push_wcache(c, m, n, dt, nsteps, s);
    push_kernel<<<grid_for(n, PUSH_BLOCK), PUSH_BLOCK, 0, s>>>(c->mesh, c->field, c->phys, m, n, dt, nsteps, c->d_stats);
    c->n_launches++;
    return cudaGetLastError();
}

}  // namespace trimeg
