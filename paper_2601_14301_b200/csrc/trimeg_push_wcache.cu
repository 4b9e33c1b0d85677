// trimeg_push_wcache.cu -- warp-autonomous fused RK4 push with a CTA-shared cache of coefficient records in
// shared memory (rows a2-a6 of DESIGN.md §1).
//
// Why (profiles/r01_fused_push_kernel.md): the CTA-tile kernel has the coefficient records in shared memory but runs its 12
// warps in lock-step (two block barriers per RK4 stage), so its latency-bound phases -- binning, scan, equations -- never
// hide under the Horner loop of another warp: 30 % of its time.  The warp-autonomous kernel has no barrier but reads the
// records through L1, which neither holds them all nor delivers them cheaply.  This kernel takes the warp-autonomous
// schedule (every warp owns 32 P - SLACK markers for the whole call, groups them by triangle with ballots into evaluation
// slots -- anew only at a stage where one of them has changed its triangle, else the slots of the last stage stand --,
// evaluates the slots 32 at a time, one marker per lane, finishes and re-locates them) and gives the CTA's warps ONE shared,
// insert-only hash table of records in shared memory:
//   * the first warp that meets a triangle claims a bin (atomicCAS on the tag), copies the record (coefficients + geometry
//     row) global -> shared with all its lanes, fences, and publishes it (state READY);
//   * a warp that finds the bin claimed but not yet READY polls it (bounded; the copying warp never waits for anybody), and
//     gives the triangle's markers to the one-marker path if the record does not show up or there is no slot left;
//   * every tenth RK4 step of a call all warps of the CTA meet at a barrier, and the table is emptied if it is nearly full
//     (the bench fuses 10 steps per call: no barrier at all; meeting every step costs 4 %, every third step 2 %).
// Everything else -- the arithmetic per marker, the locator rule, lost-marker handling -- is that of the other push kernels.
#include "trimeg_internal.h"
#include "trimeg_lane.cuh"
#include "trimeg_rk4.cuh"

namespace trimeg {

namespace {

constexpr int WC_NBIN = 64;         // hash bins of the CTA's record table
constexpr int WC_NPROBE = 8;
constexpr int WC_NB_MAX = 12;       // distinct triangles per warp and stage that get evaluation slots
constexpr int WC_EMPTY = -1;
constexpr int WC_SYNC_EVERY = 10;   // RK4 steps between two meetings of the CTA's warps (table check)
constexpr int WC_MAXSPIN = 400;     // polls of a record another warp is copying (64 ns apart) before giving up
enum { WC_LOADING = 1, WC_READY = 2 };

template <int P, int SLACK>
struct WCacheCfg {
    static constexpr int NW = 32 * P - SLACK;                       // markers per warp
    static constexpr int NE = 32 * P;                               // evaluation slots: one pass of the warp
    static constexpr size_t WARP_BYTES =
        (sizeof(double) * (size_t)N_STATE * NW + sizeof(int) * ((size_t)NW + 2 * (size_t)NE) + NW + 15) / 16 * 16;
    static constexpr size_t TABLE_BYTES = sizeof(int) * (3 * WC_NBIN + 4);     // tag, state, rec_of, counters
};

__device__ __forceinline__ unsigned wc_hash(int t) { return ((unsigned)t * 0x9E3779B1u) >> 26; }   // 6 bits

// Record slot of triangle tl in the CTA's table, copying the record in if this warp is the first to ask; -1 = none (no slot
// left, probe sequence exhausted, or a record in the making that did not become READY in time).  All 32 lanes call it with
// the same tl.
__device__ __forceinline__ int wc_lookup(int tl, int lane, int *tag, volatile int *state, int *rec_of, int *counters, int nslot,
                                         const MeshDev &M, const FieldDev &F, double2 *REC, int rec_len, int rec_stride,
                                         unsigned &n_copied)
{
    constexpr unsigned FULL = 0xffffffffu;
    int code = -1;                                       // -1 none, (h << 2) | 1 found, (h << 2) | 2 claimed with slot
    if (lane == 0) {
        unsigned h = wc_hash(tl);
        volatile int *vtag = tag;
#pragma unroll 1
        for (int pr = 0; pr < WC_NPROBE; ++pr) {
            int prev = vtag[h];                          // plain look first: the triangle is usually there already
            if (prev == WC_EMPTY) prev = atomicCAS(&tag[h], WC_EMPTY, tl);
            if (prev == WC_EMPTY) {
                const int r = atomicAdd(&counters[0], 1);
                if (r < nslot) { rec_of[h] = r; state[h] = WC_LOADING; code = (int)(h << 2) | 2; }
                else { rec_of[h] = -1; __threadfence_block(); state[h] = WC_READY; }
                break;
            }
            if (prev == tl) { code = (int)(h << 2) | 1; break; }
            h = (h + 1) & (WC_NBIN - 1);
        }
    }
    code = __shfl_sync(FULL, code, 0);
    if (code < 0) return -1;
    const int h = code >> 2;
    int rec = -1;
    if ((code & 3) == 2) {                               // this warp copies the record: coefficients, then the geometry row
        rec = rec_of[h];
        rec = __shfl_sync(FULL, rec, 0);
        const double2 *src = F.coef + (size_t)tl * rec_len;
        const double2 *geo = reinterpret_cast<const double2 *>(M.geom + 6 * (size_t)tl);
        double2 *dst = REC + (size_t)rec * rec_stride;
#pragma unroll 4
        for (int k = lane; k < rec_len; k += 32) dst[k] = __ldg(src + k);
        if (lane < 3) dst[rec_len + lane] = __ldg(geo + lane);
        __threadfence_block();
        __syncwarp();
        if (lane == 0) state[h] = WC_READY;
        ++n_copied;
    } else {
        if (lane == 0) {
            int s = state[h];
#pragma unroll 1
            for (int it = 0; it < WC_MAXSPIN && s != WC_READY; ++it) { __nanosleep(64); s = state[h]; }
            if (s == WC_READY) { __threadfence_block(); rec = rec_of[h]; }
        }
        rec = __shfl_sync(FULL, rec, 0);
    }
    return rec;
}

// Evaluation: P passes; in pass k lane l evaluates slot 32 k + l, one marker, in the two-phase form of trimeg_lane.cuh (2.21
// cycles per FP64 instruction; two markers of one triangle per lane off one load per coefficient, the form of round 1 and
// of trimeg_multi.cuh, cost 2.65).  Every group of slots (one triangle) starts at an even slot, so the lanes 2j, 2j+1 of a
// pass read the same record: a warp-wide 16-byte shared-memory load whose addresses agree in such lane pairs costs 2
// wavefronts of the data pipe instead of 4 (profiles/r02_mode_loop.md) -- per marker as much as one load for two markers.
// zero: a run-time 0 the compiler cannot see through (trimeg_lane.cuh).
template <int P, int WARPS, int SLACK>
__global__ void __launch_bounds__(32 * WARPS, 1) push_wcache_kernel(MeshDev M, FieldDev F, PhysDev Ph, trimeg_markers m, size_t n,
                                                                    double dt, int nsteps, Stats *st, int nslot, int zero)
{
    using Cfg = WCacheCfg<P, SLACK>;
    constexpr int NW = Cfg::NW, NE = Cfg::NE;
    constexpr unsigned FULL = 0xffffffffu;
    extern __shared__ __align__(16) unsigned char smem_c[];
    const int tid = threadIdx.x, lane = tid & 31, wib = tid >> 5;
    unsigned char *wbase = smem_c + (size_t)wib * Cfg::WARP_BYTES;
    double *S = reinterpret_cast<double *>(wbase);                 // [N_STATE][NW]
    int *cell = reinterpret_cast<int *>(S + (size_t)N_STATE * NW);  // [NW] current triangle
    int *ev_own = cell + NW;                                        // [NE] marker of an evaluation slot, -1 = padding
    int *ev_rec = ev_own + NE;                                      // [NE] record slot of an evaluation slot
    unsigned char *flags = reinterpret_cast<unsigned char *>(ev_rec + NE);   // [NW]
    int *tag = reinterpret_cast<int *>(smem_c + (size_t)WARPS * Cfg::WARP_BYTES);   // [WC_NBIN] triangle of a bin
    volatile int *state = tag + WC_NBIN;                            // [WC_NBIN] 0 / WC_LOADING / WC_READY
    int *rec_of = tag + 2 * WC_NBIN;                                // [WC_NBIN] record slot, -1 = none
    int *counters = tag + 3 * WC_NBIN;                              // [0] bins claimed since the table was emptied
    const int rec_len = F.n_modes * NCOEF;
    const int rec_stride = (rec_len + 3) | 1;                       // odd number of 16-byte units (banks), as the CTA-tile kernel
    double2 *REC = reinterpret_cast<double2 *>(smem_c + ((size_t)WARPS * Cfg::WARP_BYTES + Cfg::TABLE_BYTES + 15) / 16 * 16);

    const size_t base = ((size_t)blockIdx.x * WARPS + wib) * NW;
    const int nt = (base >= n) ? 0 : (int)((n - base < (size_t)NW) ? (n - base) : (size_t)NW);   // empty warps stay for the barriers
    const bool has_field = F.n_modes > 0;
    const double hdt = 0.5 * dt, dt6 = dt / 6.0;
    const unsigned lt_mask = (1u << lane) - 1u;
    TRIMEG_PHASE_CLOCK_INIT                                         // lane 0: grouping (+ lookups), evaluation + finish, one-marker path
    unsigned n_fallback = 0, n_copied = 0, n_stages = 0;
    int t_last[P], r_last[P];                                       // triangle and record slot of the lane's markers at the last stage
    int slot[P], recp[P], n_ev = 0;                                 // evaluation slot and record of the lane's markers; slots in use
    unsigned n_regroup = 0;
#pragma unroll
    for (int p = 0; p < P; ++p) { t_last[p] = -2; r_last[p] = -1; slot[p] = -1; recp[p] = -1; }

    if (tid < WC_NBIN) { tag[tid] = WC_EMPTY; state[tid] = 0; rec_of[tid] = -1; }
    if (tid < 4) counters[tid] = 0;
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
    __syncthreads();

#pragma unroll 1
    for (int step = 0; step < nsteps; ++step) {
#pragma unroll 1
        for (int stage = 0; stage < 4; ++stage) {
            // ------------------------------------------------------------ 1: grouping by triangle (home role) + record lookup
            const int ps = (stage == 0) ? Y_R : S_R;   // stage 0 is evaluated at the start-of-step state itself (no copy Y -> S)
            int t[P];
            unsigned rem[P];
            bool same = true;
#pragma unroll
            for (int p = 0; p < P; ++p) {
                const int q = lane + 32 * p;
                const bool act = (q < NW) && (flags[q] & FL_ACTIVE);
                t[p] = act ? cell[q] : -1;
                same = same && (t[p] == t_last[p]);
            }
            // no marker of the warp has changed its triangle since the last stage: the slots of that stage stand
            if (has_field && !__all_sync(FULL, same)) {
                int nb = 0;
                n_ev = 0;
                ++n_regroup;
#pragma unroll
                for (int p = 0; p < P; ++p) { slot[p] = -1; recp[p] = -1; rem[p] = __ballot_sync(FULL, t[p] >= 0); }
                // every lane first looks the triangles of its own markers up (plain loads, all lanes at once): the triangle is
                // usually in the table already.  kr: record slot, -2 = in the table without a slot, -1 = not (yet) there
                int kr[P];
#pragma unroll
                for (int p = 0; p < P; ++p) {
                    kr[p] = (t[p] >= 0 && t[p] == t_last[p] && r_last[p] >= 0) ? r_last[p] : -1;
                    if (t[p] >= 0 && kr[p] < 0) {
                        unsigned h = wc_hash(t[p]);
                        const volatile int *vtag = tag;
#pragma unroll 1
                        for (int pr = 0; pr < WC_NPROBE; ++pr) {
                            const int th = vtag[h];
                            if (th == t[p]) {
                                if (state[h] == WC_READY) { __threadfence_block(); const int r = rec_of[h]; kr[p] = (r >= 0) ? r : -2; }
                                break;
                            }
                            if (th == WC_EMPTY) break;
                            h = (h + 1) & (WC_NBIN - 1);
                        }
                    }
                }
#pragma unroll 1
                while (nb < WC_NB_MAX && n_ev < NE) {
                    int pl = -1;
#pragma unroll
                    for (int p = P - 1; p >= 0; --p) if (rem[p]) pl = p;
                    if (pl < 0) break;
                    int cand = 0, known = -1;
                    unsigned rl = 0;
#pragma unroll
                    for (int p = 0; p < P; ++p)
                        if (p == pl) { cand = t[p]; known = kr[p]; rl = rem[p]; }
                    const int tl = __shfl_sync(FULL, cand, __ffs(rl) - 1);
                    int rec = __shfl_sync(FULL, known, __ffs(rl) - 1);
                    if (rec == -1) rec = wc_lookup(tl, lane, tag, state, rec_of, counters, nslot, M, F, REC, rec_len, rec_stride, n_copied);
                    else if (rec == -2) rec = -1;
                    const int start = (n_ev + 1) & ~1;            // a group starts at an even slot (lane pairs read one record)
                    const int room = (rec >= 0) ? NE - start : 0;  // no record: the triangle's markers keep slot -1
                    int count = 0;
#pragma unroll
                    for (int p = 0; p < P; ++p) {
                        const bool mine = (t[p] == tl);
                        const unsigned mm = __ballot_sync(FULL, mine);
                        const int rank = count + __popc(mm & lt_mask);
                        if (mine && rank < room) { slot[p] = start + rank; recp[p] = rec; }
                        count += __popc(mm);
                        rem[p] &= ~mm;
                    }
                    count = min(count, room);
                    if (count > 0) {
                        if (lane == 0 && start > n_ev) ev_own[n_ev] = -1;          // the padding slot in front of the group
                        n_ev = start + count;
                    }
                    ++nb;
                }
#pragma unroll
                for (int p = 0; p < P; ++p) {
                    if (slot[p] >= 0) { ev_own[slot[p]] = lane + 32 * p; ev_rec[slot[p]] = recp[p]; }
                    t_last[p] = t[p]; r_last[p] = recp[p];
                }
            }
            __syncwarp();
            if (lane == 0) { TRIMEG_PHASE_CLOCK(0) ++n_stages; }

            // ------------------------------------------------------------ 2 + 3: batched evaluation, equations (slot role)
#pragma unroll 1
            for (int pass = 0; pass < P; ++pass) {
                const int e = 32 * pass + lane;
                const int own1 = (e < n_ev) ? ev_own[e] : -1;
                if (own1 >= 0) {
                    const double2 *recp1 = REC + (size_t)ev_rec[e] * rec_stride;
                    TriGeom tg;
                    tg.t = cell[own1];
                    tg.v0 = recp1[rec_len]; tg.gx = recp1[rec_len + 1]; tg.ge = recp1[rec_len + 2];
                    // local coordinates exactly as bary_rn() (rule L2)
                    const double dx = __dsub_rn(S[(ps + 0) * NW + own1], tg.v0.x), dz = __dsub_rn(S[(ps + 1) * NW + own1], tg.v0.y);
                    const double xi1 = __dadd_rn(__dmul_rn(tg.gx.x, dx), __dmul_rn(tg.gx.y, dz));
                    const double eta1 = __dadd_rn(__dmul_rn(tg.ge.x, dx), __dmul_rn(tg.ge.y, dz));
                    double f1, fx1, fe1, fp1;
                    gather_lane_harmonic(F, recp1, xi1, eta1, S[(ps + 2) * NW + own1], zero, f1, fx1, fe1, fp1);
                    FieldVal fv;
                    fv.f = f1; fv.fphi = fp1;
                    fv.fR = fma(tg.gx.x, fx1, tg.ge.x * fe1);                    // d/dR
                    fv.fZ = fma(tg.gx.y, fx1, tg.ge.y * fe1);                    // d/dZ
                    advance(M, Ph, S, NW, cell, flags, own1, stage, fv, dt, hdt, dt6, &tg);
                }
                __syncwarp();
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
                    const Bary b = bary_rn(M, tt, S[(ps + 0) * NW + q], S[(ps + 1) * NW + q]);
                    fv = gather(F, tt, b, S[(ps + 2) * NW + q]);
                    ++n_fallback;
                }
                advance(M, Ph, S, NW, cell, flags, q, stage, fv, dt, hdt, dt6);
            }
            __syncwarp();
            if (lane == 0) { TRIMEG_PHASE_CLOCK(2) }
        }
        // ---- every WC_SYNC_EVERY steps all warps meet; the table is emptied when it is nearly full of triangles the markers
        // have left (a full table is not an error: triangles without a record go down the one-marker path)
        if (has_field && step % WC_SYNC_EVERY == WC_SYNC_EVERY - 1 && step + 1 < nsteps) {
            __syncthreads();
            const int claimed = counters[0];
            __syncthreads();                                        // everybody has read the counter before anybody claims again
            if (claimed > min(nslot, WC_NBIN) - 8) {                // uniform
                if (tid < WC_NBIN) { tag[tid] = WC_EMPTY; state[tid] = 0; rec_of[tid] = -1; }
                if (tid == 0) counters[0] = 0;
#pragma unroll
                for (int p = 0; p < P; ++p) { t_last[p] = -2; r_last[p] = -1; }
                __syncthreads();
            }
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
        if (n_copied) atomicAdd(&st->tile[6], (unsigned long long)n_copied);
        atomicAdd(&st->tile[7], (unsigned long long)n_stages);
    }
}

template <int P, int WARPS, int SLACK>
cudaError_t launch_wcache(trimeg_ctx *c, const trimeg_markers &m, size_t n, double dt, int nsteps, cudaStream_t s)
{
    using Cfg = WCacheCfg<P, SLACK>;
    constexpr size_t SMEM_MAX = 227 * 1024;
    // function attributes are per device: set on every launch (cheap), not once per process
    cudaError_t e = cudaFuncSetAttribute(push_wcache_kernel<P, WARPS, SLACK>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_MAX);
    if (e != cudaSuccess) return e;
    const size_t fixed = ((size_t)WARPS * Cfg::WARP_BYTES + Cfg::TABLE_BYTES + 15) / 16 * 16;
    const size_t rec_bytes = sizeof(double2) * ((NCOEF * (size_t)c->field.n_modes + 3) | 1);    // as rec_stride in the kernel
    int nslot = c->field.n_modes ? (int)((SMEM_MAX - fixed) / rec_bytes) : 0;
    if (nslot > WC_NBIN) nslot = WC_NBIN;
    const size_t shm = fixed + (size_t)nslot * rec_bytes;
    const size_t per_cta = (size_t)Cfg::NW * WARPS;
    const size_t ctas = (n + per_cta - 1) / per_cta;
    push_wcache_kernel<P, WARPS, SLACK><<<(unsigned)ctas, 32 * WARPS, shm, s>>>(c->mesh, c->field, c->phys, m, n, dt, nsteps, c->d_stats, nslot, 0);
    c->n_launches++;
    return cudaGetLastError();
}

}  // namespace

#ifdef TRIMEG_CORE_ONLY
cudaError_t launch_push_wcache_core(trimeg_ctx *c, const trimeg_markers &m, size_t n, double dt, int nsteps, cudaStream_t s)
#else
cudaError_t launch_push_wcache(trimeg_ctx *c, const trimeg_markers &m, size_t n, double dt, int nsteps, cudaStream_t s)
#endif
{
    if (n == 0 || nsteps <= 0) return cudaSuccess;
    // 16 warps at 128 registers while enough of the smaller records fit beside their state (cfg5 mesh, 2^24 markers, 12 / 16
    // warps: 7 modes 3.29e9 / 3.43e9, 10 modes 2.62e9 / 2.70e9, 14 modes 2.05e9 / 2.07e9, 16 modes 1.843e9 / 1.839e9 -- 17
    // record slots for 944 markers there, 2.6 times the markers without a slot)
    // (the core build only: with the branches of rows f3 / f4 the kernel does not fit 128 registers without spilling)
#ifdef TRIMEG_CORE_ONLY
    if (c->field.n_modes <= TRIMEG_WCACHE_16_MAX_MODES) return launch_wcache<2, 16, 5>(c, m, n, dt, nsteps, s);
#endif
    return launch_wcache<2, 12, 5>(c, m, n, dt, nsteps, s);
}

}  // namespace trimeg
