// trimeg_push_warp.cu -- warp-autonomous, triangle-batched fused RK4 push (rows a2-a6 of DESIGN.md §1).
//
// Why: with one thread per marker every lane fetches every coefficient itself (21 x 16-byte loads per
// mode and stage) and the SM's load/store data pipe, not the FP64 pipe, bounds the kernel
// (profiles/r01_baseline_push_kernel.md).  A coefficient held in a register must serve several markers,
// which therefore have to sit in the same triangle at the moment of the evaluation.
//
// How: every WARP owns NW = 32 P - slack consecutive markers for the whole call (their RK4 state
// sits in a warp-private slice of shared memory) and runs the stage loop on its own, with
// __syncwarp() only.  Warps of an SM drift apart, so the latency-bound work of one warp hides
// under the FP64 work of the others.  Per RK4 stage:
//   1  grouping (home role: lane l looks after markers l, l + 32, ...): the warp's markers are
//      partitioned by triangle with ballots; every triangle gets a run of evaluation slots padded
//      to a multiple of P.  The slots of the last stage stand if no marker has changed its triangle;
//   2  evaluation (slot role): lane l takes slots [P l, P l + P) -- by construction one triangle --
//      and runs the bivariate Horner scheme for the P markers off ONE load of each coefficient;
//      lanes of a warp mostly share the triangle, so the loads are warp-uniform L1 hits;
//   3  still in the slot role, the same lane finishes each of its P markers: chain rule,
//      equilibrium + equations of motion (a4, a5), RK4 bookkeeping (a6), next stage position,
//      and the locate (a2) of that position -- which is what the next stage's grouping needs.
// Markers beyond the NB_MAX-th distinct triangle of a warp (unsorted input) are evaluated by
// their home lane with the one-marker gather of trimeg_device.cuh: slower, same arithmetic.
// The arithmetic per marker (order of operations, fused multiply-adds) is that of push_kernel.
#include "trimeg_internal.h"
#include "trimeg_multi.cuh"
#include "trimeg_rk4.cuh"

namespace trimeg {

namespace {

constexpr int NB_MAX = 12;          // distinct triangles per warp and stage that get evaluation slots

template <int P, int SLACK>
struct WarpCfg {
    static constexpr int NW = 32 * P - SLACK;                       // markers per warp (SLACK slots left for bin padding)
    static constexpr int NE = 32 * P;                               // evaluation slots: exactly one pass of the warp
    static constexpr size_t WARP_BYTES =
        (sizeof(double) * (size_t)N_STATE * NW + sizeof(int) * ((size_t)NW + 2 * (size_t)NE) + NW + 15) / 16 * 16;
};

// MINB: CTAs per SM the kernel is compiled for (3 -> 168 registers, 4 -> 128; without it ptxas takes 214 for P = 2)
template <int P, int WARPS, int SLACK, int MINB>
__global__ void __launch_bounds__(32 * WARPS, MINB) push_warp_kernel(MeshDev M, FieldDev F, PhysDev Ph, trimeg_markers m, size_t n,
                                                               double dt, int nsteps, Stats *st)
{
    using Cfg = WarpCfg<P, SLACK>;
    constexpr int NW = Cfg::NW, NE = Cfg::NE;
    constexpr unsigned FULL = 0xffffffffu;
    extern __shared__ __align__(16) unsigned char smem_w[];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    unsigned char *wbase = smem_w + (size_t)wib * Cfg::WARP_BYTES;
    double *S = reinterpret_cast<double *>(wbase);                 // [N_STATE][NW]
    int *cell = reinterpret_cast<int *>(S + (size_t)N_STATE * NW);  // [NW] current triangle
    int *ev_own = cell + NW;                                        // [NE] marker of an evaluation slot, -1 = padding
    int *ev_tri = ev_own + NE;                                      // [NE] triangle of an evaluation slot
    unsigned char *flags = reinterpret_cast<unsigned char *>(ev_tri + NE);   // [NW]

    const size_t base = ((size_t)blockIdx.x * WARPS + wib) * NW;
    if (base >= n) return;                                          // warps never synchronise with each other
    const int nt = (int)((n - base < (size_t)NW) ? (n - base) : (size_t)NW);
    const bool has_field = F.n_modes > 0;
    const double hdt = 0.5 * dt, dt6 = dt / 6.0;
    const unsigned lt_mask = (1u << lane) - 1u;
    TRIMEG_PHASE_CLOCK_INIT                                         // lane 0: grouping, evaluation + equations, fallback
    unsigned n_fallback = 0, n_bins = 0, n_stages = 0, n_regroup = 0;
    int t_last[P], slot[P], n_ev = 0;                               // triangle and evaluation slot of the lane's markers at the last grouping
#pragma unroll
    for (int p = 0; p < P; ++p) { t_last[p] = -2; slot[p] = -1; }

    // ---- load the warp's markers (home role), locate the start positions
#pragma unroll
    for (int p = 0; p < P; ++p) {
        const int q = lane + 32 * p;
        if (q >= NW) continue;
        unsigned char fl = 0;
        int c = -1;
        if (q < nt) {
            const size_t g = base + q;
            c = m.cell[g];
            if (c >= 0) {
                const double R = m.R[g], Z = m.Z[g];
                S[Y_R * NW + q] = R; S[Y_Z * NW + q] = Z; S[Y_P * NW + q] = m.phi[g];
                S[Y_V * NW + q] = m.vpar[g]; S[Y_W * NW + q] = m.w[g]; S[S_MU * NW + q] = m.mu[g];
                fl = FL_ACTIVE | FL_WASACTIVE;
                Bary b;
                int moved = 0;
                const int t = locate(M, R, Z, c, b, moved);
                if (moved) fl |= FL_MOVED;
                if (t < 0) fl = (fl | FL_LOST) & ~FL_ACTIVE;
                else c = t;
            }
        }
        cell[q] = c; flags[q] = fl;
    }
    __syncwarp();

#pragma unroll 1
    for (int step = 0; step < nsteps; ++step) {
#pragma unroll 1
        for (int stage = 0; stage < 4; ++stage) {
            // ------------------------------------------------------------ 1: grouping by triangle (home role)
            int t[P];
            unsigned rem[P];
            bool same = true;
#pragma unroll
            for (int p = 0; p < P; ++p) {
                const int q = lane + 32 * p;
                const bool act = (q < NW) && (flags[q] & FL_ACTIVE);
                t[p] = act ? cell[q] : -1;
                same = same && (t[p] == t_last[p]);
                if (act && stage == 0) {
#pragma unroll
                    for (int k = 0; k < 5; ++k) S[(S_R + k) * NW + q] = S[(Y_R + k) * NW + q];
                }
            }
            int nb = 0;
            // no marker of the warp has changed its triangle since the last stage: the slots of that stage stand
            if (has_field && !__all_sync(FULL, same)) {
                n_ev = 0;
                ++n_regroup;
#pragma unroll
                for (int p = 0; p < P; ++p) { slot[p] = -1; rem[p] = __ballot_sync(FULL, t[p] >= 0); t_last[p] = t[p]; }
#pragma unroll 1
                while (nb < NB_MAX && n_ev < NE) {
                    int pl = -1;
#pragma unroll
                    for (int p = P - 1; p >= 0; --p) if (rem[p]) pl = p;
                    if (pl < 0) break;
                    int cand = 0;
                    unsigned rl = 0;
#pragma unroll
                    for (int p = 0; p < P; ++p) if (p == pl) { cand = t[p]; rl = rem[p]; }
                    const int tl = __shfl_sync(FULL, cand, __ffs(rl) - 1);
                    const int room = NE - n_ev;                    // a multiple of P; markers beyond it keep slot -1
                    int count = 0;
#pragma unroll
                    for (int p = 0; p < P; ++p) {
                        const bool mine = (t[p] == tl);
                        const unsigned mm = __ballot_sync(FULL, mine);
                        const int rank = count + __popc(mm & lt_mask);
                        if (mine && rank < room) slot[p] = n_ev + rank;
                        count += __popc(mm);
                        rem[p] &= ~mm;
                    }
                    count = min(count, room);
                    const int padded = (count + P - 1) / P * P;
                    if (lane < padded - count) ev_own[n_ev + count + lane] = -1;
                    n_ev += padded;
                    ++nb;
                }
#pragma unroll
                for (int p = 0; p < P; ++p)
                    if (slot[p] >= 0) { ev_own[slot[p]] = lane + 32 * p; ev_tri[slot[p]] = t[p]; }
            }
            __syncwarp();
            if (lane == 0) { TRIMEG_PHASE_CLOCK(0) n_bins += nb; ++n_stages; }

            // ------------------------------------------------------------ 2 + 3: batched evaluation, equations (slot role)
            if (lane * P < n_ev) {
                const int e0 = lane * P;
                const int tri = ev_tri[e0];                                          // first slot of a group is real
                const double2 *g = reinterpret_cast<const double2 *>(M.geom + 6 * (size_t)tri);
                const double2 v0 = __ldg(g), gx = __ldg(g + 1), ge = __ldg(g + 2);
                TriGeom tg;
                tg.t = tri; tg.v0 = v0; tg.gx = gx; tg.ge = ge;
                int own[P];
                double xi[P], eta[P], phi[P], f[P], fx[P], fe[P], fp[P];
#pragma unroll
                for (int p = 0; p < P; ++p) {
                    own[p] = ev_own[e0 + p];
                    xi[p] = eta[p] = phi[p] = 0.0;
                    if (own[p] >= 0) {                 // local coordinates exactly as bary_rn() (rule L2)
                        const double dx = __dsub_rn(S[S_R * NW + own[p]], v0.x), dz = __dsub_rn(S[S_Z * NW + own[p]], v0.y);
                        xi[p] = __dadd_rn(__dmul_rn(gx.x, dx), __dmul_rn(gx.y, dz));
                        eta[p] = __dadd_rn(__dmul_rn(ge.x, dx), __dmul_rn(ge.y, dz));
                        phi[p] = S[S_P * NW + own[p]];
                    }
                }
                gather_multi<P, true>(F, F.coef + (size_t)tri * F.n_modes * NCOEF, xi, eta, phi, f, fx, fe, fp);
#pragma unroll 1
                for (int p = 0; p < P; ++p) {
                    // select without dynamic register indexing
                    int q = -1;
                    FieldVal fv;
                    fv.f = fv.fR = fv.fZ = fv.fphi = 0.0;
#pragma unroll
                    for (int pp = 0; pp < P; ++pp)
                        if (pp == p) {
                            q = own[pp]; fv.f = f[pp]; fv.fphi = fp[pp];
                            fv.fR = fma(gx.x, fx[pp], ge.x * fe[pp]);                // d/dR
                            fv.fZ = fma(gx.y, fx[pp], ge.y * fe[pp]);                // d/dZ
                        }
                    if (q >= 0) advance(M, Ph, S, NW, cell, flags, q, stage, fv, dt, hdt, dt6, &tg);
                }
            }
            __syncwarp();
            if (lane == 0) { TRIMEG_PHASE_CLOCK(1) }

            // ------------------------------------------------------------ markers without a slot (home role)
#pragma unroll 1
            for (int p = 0; p < P; ++p) {
                int tt = -1, sl = -1;
#pragma unroll
                for (int pp = 0; pp < P; ++pp) if (pp == p) { tt = t[pp]; sl = slot[pp]; }
                if (tt < 0 || sl >= 0) continue;
                const int q = lane + 32 * p;
                FieldVal fv;
                fv.f = fv.fR = fv.fZ = fv.fphi = 0.0;
                if (has_field) {
                    const Bary b = bary_rn(M, tt, S[S_R * NW + q], S[S_Z * NW + q]);
                    fv = gather(F, tt, b, S[S_P * NW + q]);
                    ++n_fallback;
                }
                advance(M, Ph, S, NW, cell, flags, q, stage, fv, dt, hdt, dt6);
            }
            __syncwarp();
            if (lane == 0) { TRIMEG_PHASE_CLOCK(2) }
        }
    }

    // ---- write back (home role), statistics
    int lost = 0, moved = 0;
#pragma unroll
    for (int p = 0; p < P; ++p) {
        const int q = lane + 32 * p;
        if (q >= nt) continue;
        const unsigned char fl = flags[q];
        if (!(fl & FL_WASACTIVE)) continue;
        const size_t g = base + q;
        m.R[g] = S[Y_R * NW + q]; m.Z[g] = S[Y_Z * NW + q]; m.phi[g] = S[Y_P * NW + q];
        m.vpar[g] = S[Y_V * NW + q]; m.w[g] = S[Y_W * NW + q];
        m.cell[g] = (fl & FL_LOST) ? -1 : cell[q];
        lost += (fl & FL_LOST) ? 1 : 0;
        moved += (fl & FL_MOVED) ? 1 : 0;
    }
    lost = __reduce_add_sync(FULL, lost);
    moved = __reduce_add_sync(FULL, moved);
    n_fallback = __reduce_add_sync(FULL, n_fallback);
    if (lane == 0) {
        if (lost) atomicAdd(&st->n_lost, (unsigned long long)lost);
        if (moved) atomicAdd(&st->n_moved, (unsigned long long)moved);
        atomicAdd(&st->tile[1], (unsigned long long)n_regroup);
        TRIMEG_PHASE_CLOCK_FLUSH(st)
        if (n_fallback) atomicAdd(&st->tile[5], (unsigned long long)n_fallback);
        atomicAdd(&st->tile[6], (unsigned long long)n_bins);
        atomicAdd(&st->tile[7], (unsigned long long)n_stages);
    }
}

template <int P, int WARPS, int SLACK, int MINB>
cudaError_t launch_warp(trimeg_ctx *c, const trimeg_markers &m, size_t n, double dt, int nsteps, cudaStream_t s)
{
    using Cfg = WarpCfg<P, SLACK>;
    const size_t shm = Cfg::WARP_BYTES * WARPS;
    // function attributes are per device: set on every launch (cheap), not once per process
    cudaError_t e = cudaFuncSetAttribute(push_warp_kernel<P, WARPS, SLACK, MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)shm);
    if (e != cudaSuccess) return e;
    const size_t per_cta = (size_t)Cfg::NW * WARPS;
    const size_t ctas = (n + per_cta - 1) / per_cta;
    push_warp_kernel<P, WARPS, SLACK, MINB><<<(unsigned)ctas, 32 * WARPS, shm, s>>>(c->mesh, c->field, c->phys, m, n, dt, nsteps, c->d_stats);
    c->n_launches++;
    return cudaGetLastError();
}

}  // namespace

cudaError_t launch_push_warp(trimeg_ctx *c, const trimeg_markers &m, size_t n, double dt, int nsteps, int variant,
                             cudaStream_t s)
{
    if (n == 0 || nsteps <= 0) return cudaSuccess;
    switch (variant) {
    case TRIMEG_PUSH_KERNEL_WARP: return launch_warp<2, 4, 6, 3>(c, m, n, dt, nsteps, s);
    case TRIMEG_PUSH_KERNEL_WARP128: return launch_warp<2, 4, 6, 4>(c, m, n, dt, nsteps, s);
    default: return cudaErrorInvalidValue;
    }
}

}  // namespace trimeg
