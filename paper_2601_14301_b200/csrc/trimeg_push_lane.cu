// trimeg_push_lane.cu -- fused RK4 push (rows a2-a6 of DESIGN.md section 1) with lane-owned markers: the schedule of
// TRIMEG_PUSH_KERNEL_LANE.
//
// Every warp owns 64 consecutive markers for the whole call, lane l the markers l and l + 32; their RK4 state sits in a
// warp-private slice of shared memory (conflict-free: lane = column).  Per RK4 stage a lane takes its two markers one
// after the other: local coordinates, toroidal factors, the mode loop of trimeg_lane.cuh (one marker per evaluation, two
// phases, so that runs of DFMAs share their multiplier: the FP64 pipe reads one register operand per cycle), chain rule,
// equilibrium + equations of motion, RK4 bookkeeping, next stage position, locate.  No marker ever changes its lane: no
// grouping by triangle, no evaluation slots, no padding (all 64 lanes-slots of a warp carry a marker).
//
// The coefficient records (and geometry rows) of the triangles the CTA's markers sit in live in ONE insert-only hash table
// in shared memory, shared by the CTA's warps, as in the round-1 kernel: the first warp that meets a triangle claims a bin
// (atomicCAS on the tag), copies the record global -> shared with all its lanes, fences and publishes it; the others find
// it there.  A lane remembers the record of each of its markers and asks again only when the marker has changed its
// triangle.  Cell-sorted markers (trimeg_sort) put the 32 markers of a pass into one or two triangles, whose records are
// read by broadcast (records of different triangles start in different banks).  A triangle that finds no record slot sends
// its markers down the one-marker path (coefficients from global memory, same arithmetic).  The warps never meet inside a
// 10-step call; every tenth step of a longer call they do, and the table is emptied if it is nearly full.
#include "trimeg_internal.h"
#include "trimeg_lane.cuh"
#include "trimeg_rk4.cuh"

namespace trimeg {

namespace {

constexpr int LN_NW = 64;           // markers per warp (two per lane)
constexpr int LN_NBIN = 128;        // hash bins of the CTA's record table
constexpr int LN_NPROBE = 8;
constexpr int LN_EMPTY = -1;
constexpr int LN_SYNC_EVERY = 10;   // RK4 steps between two meetings of the CTA's warps (table check)
constexpr int LN_MAXSPIN = 400;     // polls of a record another warp is copying (64 ns apart) before giving up
enum { LN_LOADING = 1, LN_READY = 2 };

constexpr size_t LN_WARP_BYTES = (sizeof(double) * (size_t)N_STATE * LN_NW + sizeof(int) * (size_t)LN_NW + 2 * LN_NW + 15) / 16 * 16;
constexpr size_t LN_TABLE_BYTES = sizeof(int) * (3 * LN_NBIN + 4);     // tag, state, rec_of, counters

__device__ __forceinline__ unsigned ln_hash(int t) { return ((unsigned)t * 0x9E3779B1u) >> 25; }   // 7 bits

// Record slot of triangle tl in the CTA's table, copying the record in if this warp is the first to ask; -1 = none (no slot
// left, probe sequence exhausted, or a record in the making that did not become READY in time).  All 32 lanes call it with
// the same tl.
__device__ __forceinline__ int ln_lookup(int tl, int lane, int *tag, volatile int *state, int *rec_of, int *counters, int nslot,
                                         const MeshDev &M, const FieldDev &F, double2 *REC, int rec_len, int rec_stride,
                                         unsigned &n_copied)
{
    constexpr unsigned FULL = 0xffffffffu;
    int code = -1;                                       // -1 none, (h << 2) | 1 found, (h << 2) | 2 claimed with slot
    if (lane == 0) {
        unsigned h = ln_hash(tl);
        volatile int *vtag = tag;
#pragma unroll 1
        for (int pr = 0; pr < LN_NPROBE; ++pr) {
            int prev = vtag[h];                          // plain look first: the triangle is usually there already
            if (prev == LN_EMPTY) prev = atomicCAS(&tag[h], LN_EMPTY, tl);
            if (prev == LN_EMPTY) {
                const int r = atomicAdd(&counters[0], 1);
                if (r < nslot) { rec_of[h] = r; state[h] = LN_LOADING; code = (int)(h << 2) | 2; }
                else { rec_of[h] = -1; __threadfence_block(); state[h] = LN_READY; }
                break;
            }
            if (prev == tl) { code = (int)(h << 2) | 1; break; }
            h = (h + 1) & (LN_NBIN - 1);
        }
    }
    code = __shfl_sync(FULL, code, 0);
    if (code < 0) return -1;
    const int h = code >> 2;
    int rec = -1;
    if ((code & 3) == 2) {                               // this warp copies the record: coefficients, then the geometry row
        rec = rec_of[h];
        rec = __shfl_sync(FULL, rec, 0);
        const double2 *src = lane_rec_src(F, tl);
        const double2 *geo = reinterpret_cast<const double2 *>(M.geom + 6 * (size_t)tl);
        double2 *dst = REC + (size_t)rec * rec_stride;
#pragma unroll 4
        for (int k = lane; k < rec_len; k += 32) dst[k] = __ldg(src + k);
        if (lane < 3) dst[rec_len + lane] = __ldg(geo + lane);
        __threadfence_block();
        __syncwarp();
        if (lane == 0) state[h] = LN_READY;
        ++n_copied;
    } else {
        if (lane == 0) {
            int s = state[h];
#pragma unroll 1
            for (int it = 0; it < LN_MAXSPIN && s != LN_READY; ++it) { __nanosleep(64); s = state[h]; }
            if (s == LN_READY) { __threadfence_block(); rec = rec_of[h]; }
        }
        rec = __shfl_sync(FULL, rec, 0);
    }
    return rec;
}

// zero: a run-time 0 the compiler cannot see through (trimeg_lane.cuh)
template <int WARPS>
__global__ void __launch_bounds__(32 * WARPS, 1) push_lane_kernel(MeshDev M, FieldDev F, PhysDev Ph, trimeg_markers m, size_t n,
                                                                  double dt, int nsteps, Stats *st, int nslot, int zero)
{
    constexpr int NW = LN_NW;
    constexpr unsigned FULL = 0xffffffffu;
    extern __shared__ __align__(16) unsigned char smem_l[];
    const int tid = threadIdx.x, lane = tid & 31, wib = tid >> 5;
    unsigned char *wbase = smem_l + (size_t)wib * LN_WARP_BYTES;
    double *S = reinterpret_cast<double *>(wbase);                  // [N_STATE][NW]
    int *cell = reinterpret_cast<int *>(S + (size_t)N_STATE * NW);   // [NW] current triangle
    unsigned char *flags = reinterpret_cast<unsigned char *>(cell + NW);     // [NW]
    unsigned char *orig = flags + NW;                                // [NW] marker (offset in the warp's 64) that sits in a slot
    int *tag = reinterpret_cast<int *>(smem_l + (size_t)WARPS * LN_WARP_BYTES);      // [LN_NBIN] triangle of a bin
    volatile int *state = tag + LN_NBIN;                             // [LN_NBIN] 0 / LN_LOADING / LN_READY
    int *rec_of = tag + 2 * LN_NBIN;                                 // [LN_NBIN] record slot, -1 = none
    int *counters = tag + 3 * LN_NBIN;                               // [0] bins claimed since the table was emptied
    const int rec_len = lane_rec_len(F);
    const int rec_stride = (rec_len + 3) | 1;                        // odd number of 16-byte units: records start in different banks
    double2 *REC = reinterpret_cast<double2 *>(smem_l + ((size_t)WARPS * LN_WARP_BYTES + LN_TABLE_BYTES + 15) / 16 * 16);

    const size_t base = ((size_t)blockIdx.x * WARPS + wib) * NW;
    const int nt = (base >= n) ? 0 : (int)((n - base < (size_t)NW) ? (n - base) : (size_t)NW);   // empty warps stay for the barriers
    const bool has_field = F.n_modes > 0 || TRIMEG_HAS_SPL(F);
    const double hdt = 0.5 * dt, dt6 = dt / 6.0;
    TRIMEG_PHASE_CLOCK_INIT                                          // lane 0: record lookups, evaluation + finish, (unused)
    unsigned n_fallback = 0, n_copied = 0, n_stages = 0, n_regroup = 0;
    int t_last0 = -2, t_last1 = -2, r_last0 = -1, r_last1 = -1;      // triangle and record slot of the lane's markers at the last stage

    for (int k = tid; k < LN_NBIN; k += 32 * WARPS) { tag[k] = LN_EMPTY; state[k] = 0; rec_of[k] = -1; }
    if (tid < 4) counters[tid] = 0;
    // ---- load the warp's markers, locate the start positions.  B-spline field: the warp's markers take their slots in the
    // order of (triangle, toroidal plane), so that the lanes of a pass read neighbouring planes of a record -- different
    // shared-memory banks (planes are 21 doubles apart) -- instead of planes at random (bank conflicts); the order holds for
    // the call (a marker crosses a small fraction of a plane spacing per step).  orig[] takes every marker home at the end.
    unsigned *skey = reinterpret_cast<unsigned *>(S + (size_t)A_R * NW);      // scratch: the accumulators are written at stage 0
    double ldR[2], ldZ[2], ldP[2], ldV[2], ldW[2], ldM[2];
    int ldc[2];
    unsigned char ldf[2];
#pragma unroll
    for (int p = 0; p < 2; ++p) {
        const int q = lane + 32 * p;
        unsigned char fl = 0;
        int c = -1;
        ldR[p] = ldZ[p] = ldP[p] = ldV[p] = ldW[p] = ldM[p] = 0.0;
        if (q < nt) {
            const size_t g = base + q;
            c = m.cell[g];
            if (c >= 0) {
                ldR[p] = m.R[g]; ldZ[p] = m.Z[g]; ldP[p] = m.phi[g]; ldV[p] = m.vpar[g]; ldW[p] = m.w[g]; ldM[p] = m.mu[g];
                fl = FL_ACTIVE | FL_WASACTIVE;
                Bary b;
                int moved = 0;
                const int t = locate(M, ldR[p], ldZ[p], c, b, moved);
                if (moved) fl |= FL_MOVED;
                if (t < 0) fl = (fl | FL_LOST) & ~FL_ACTIVE;
                else c = t;
            }
        }
        ldc[p] = c; ldf[p] = fl;
        if (TRIMEG_HAS_SPL(F)) {
            unsigned key = 0xffffffffu;
            if (fl & FL_ACTIVE) key = (((unsigned)c << 6) | (unsigned)spline_weights(F.n_phi, F.inv_h, ldP[p]).j0) & 0x7fffffffu;
            skey[q] = key;
        }
    }
    int slot[2] = {lane, lane + 32};
    if (TRIMEG_HAS_SPL(F)) {
        __syncwarp();
#pragma unroll
        for (int p = 0; p < 2; ++p) {
            const int q = lane + 32 * p;
            const unsigned key = skey[q];
            int r = 0;
#pragma unroll 8
            for (int o = 0; o < NW; ++o) {
                const unsigned ko = skey[o];
                r += (ko < key || (ko == key && o < q)) ? 1 : 0;
            }
            slot[p] = r;
        }
        __syncwarp();
    }
#pragma unroll
    for (int p = 0; p < 2; ++p) {
        const int q = slot[p];
        if (ldf[p] & FL_WASACTIVE) {
            S[Y_R * NW + q] = ldR[p]; S[Y_Z * NW + q] = ldZ[p]; S[Y_P * NW + q] = ldP[p];
            S[Y_V * NW + q] = ldV[p]; S[Y_W * NW + q] = ldW[p]; S[S_MU * NW + q] = ldM[p];
        }
        cell[q] = ldc[p]; flags[q] = ldf[p]; orig[q] = (unsigned char)(lane + 32 * p);
    }
    __syncthreads();

#pragma unroll 1
    for (int step = 0; step < nsteps; ++step) {
#pragma unroll 1
        for (int stage = 0; stage < 4; ++stage) {
            const int ps = (stage == 0) ? Y_R : S_R;                 // stage 0 is evaluated at the start-of-step state itself
#pragma unroll 1
            for (int p = 0; p < 2; ++p) {
                const int q = lane + 32 * p;
                const bool act = (flags[q] & FL_ACTIVE) != 0;
                const int t = act ? cell[q] : -1;
                // ------------------------------------------------ the record of the marker's triangle
                const int tl_prev = p ? t_last1 : t_last0;
                int rec = (t == tl_prev) ? (p ? r_last1 : r_last0) : -1;      // still in the triangle of the last stage: same record
                bool ask = has_field && t >= 0 && t != tl_prev;
                if (ask) {                                           // every lane looks its new triangle up by itself: it is usually there
                    unsigned h = ln_hash(t);
                    const volatile int *vtag = tag;
#pragma unroll 1
                    for (int pr = 0; pr < LN_NPROBE; ++pr) {
                        const int tg_h = vtag[h];
                        if (tg_h == t) {
                            if (state[h] == LN_READY) { __threadfence_block(); rec = rec_of[h]; ask = false; }
                            break;
                        }
                        if (tg_h == LN_EMPTY) break;
                        h = (h + 1) & (LN_NBIN - 1);
                    }
                }
                unsigned need = __ballot_sync(FULL, ask);            // triangles not in the table yet: the warp brings them in, one by one
                if (need) ++n_regroup;
#pragma unroll 1
                while (need) {
                    const int tl = __shfl_sync(FULL, t, __ffs(need) - 1);
                    const int r = ln_lookup(tl, lane, tag, state, rec_of, counters, nslot, M, F, REC, rec_len, rec_stride, n_copied);
                    const bool mine = ask && (t == tl);
                    if (mine) rec = r;
                    need &= ~__ballot_sync(FULL, mine);
                }
                if (p) { t_last1 = t; r_last1 = rec; } else { t_last0 = t; r_last0 = rec; }
                if (lane == 0) { TRIMEG_PHASE_CLOCK(0) }
                // ------------------------------------------------ field at the stage position, equations, RK4, locate
                if (act) {
                    FieldVal fv;
                    fv.f = fv.fR = fv.fZ = fv.fphi = 0.0;
                    TriGeom tg;
                    tg.t = -1;
                    if (has_field) {
                        if (rec >= 0) {
                            const double2 *recp = REC + (size_t)rec * rec_stride;
                            tg.t = t; tg.v0 = recp[rec_len]; tg.gx = recp[rec_len + 1]; tg.ge = recp[rec_len + 2];
                            // local coordinates exactly as bary_rn() (rule L2)
                            const double dx = __dsub_rn(S[(ps + 0) * NW + q], tg.v0.x), dz = __dsub_rn(S[(ps + 1) * NW + q], tg.v0.y);
                            const double xi = __dadd_rn(__dmul_rn(tg.gx.x, dx), __dmul_rn(tg.gx.y, dz));
                            const double eta = __dadd_rn(__dmul_rn(tg.ge.x, dx), __dmul_rn(tg.ge.y, dz));
                            double f, fx, fe, fp;
                            gather_lane(F, recp, xi, eta, S[(ps + 2) * NW + q], zero, f, fx, fe, fp);
                            fv.f = f; fv.fphi = fp;
                            fv.fR = fma(tg.gx.x, fx, tg.ge.x * fe);             // d/dR
                            fv.fZ = fma(tg.gx.y, fx, tg.ge.y * fe);             // d/dZ
                        } else {                                                 // no record slot: coefficients from global memory
                            const Bary b = bary_rn(M, t, S[(ps + 0) * NW + q], S[(ps + 1) * NW + q]);
                            fv = gather(F, t, b, S[(ps + 2) * NW + q]);
                            ++n_fallback;
                        }
                    }
                    if (lane == 0) { TRIMEG_PHASE_CLOCK(1) }
                    advance(M, Ph, S, NW, cell, flags, q, stage, fv, dt, hdt, dt6, (tg.t >= 0) ? &tg : nullptr);
                }
                __syncwarp();
                if (lane == 0) { TRIMEG_PHASE_CLOCK(2) }
            }
            if (lane == 0) ++n_stages;
        }
        // ---- every LN_SYNC_EVERY steps all warps meet; the table is emptied when it is nearly full of triangles the markers
        // have left (a full table is not an error: triangles without a record go down the one-marker path)
        if (has_field && step % LN_SYNC_EVERY == LN_SYNC_EVERY - 1 && step + 1 < nsteps) {
            __syncthreads();
            const int claimed = counters[0];
            __syncthreads();                                        // everybody has read the counter before anybody claims again
            if (claimed > min(nslot, LN_NBIN * 3 / 4) - 8) {         // uniform
                for (int k = tid; k < LN_NBIN; k += 32 * WARPS) { tag[k] = LN_EMPTY; state[k] = 0; rec_of[k] = -1; }
                if (tid == 0) counters[0] = 0;
                t_last0 = t_last1 = -2; r_last0 = r_last1 = -1;
                __syncthreads();
            }
        }
    }

    // ---- write back, statistics
    int lost = 0, moved = 0;
#pragma unroll
    for (int p = 0; p < 2; ++p) {
        const int q = lane + 32 * p;
        const unsigned char fl = flags[q];
        if (!(fl & FL_WASACTIVE)) continue;              // empty slots of a ragged last warp, markers flagged on entry
        const size_t g = base + orig[q];
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


// ---------------------------------------------------------------------------------------------- gather alone (configs[3])
// The gather for cell-sorted markers, with the machinery above and no RK4 state: a CTA of GL_WARPS warps walks over chunks of
// n_pass x 32 consecutive markers per warp (n_pass <= GL_PASSES_MAX, fewer for small batches so that every SM gets chunks); a lane takes one marker per pass: the inputs of the next pass are fetched
// while the current one is evaluated (the thread-per-marker kernel waits for its loads at 12-24 warps per SM), the record of
// the marker's triangle (coefficients + geometry row) comes from the CTA's table in shared memory, the evaluation is the
// two-phase mode loop.  The warps meet once per chunk; the table is emptied there when it is nearly full.  gate / want:
// device-side choice between this kernel and gather_kernel (*gate = number of places where the hinted cells decrease).
constexpr int GL_WARPS = 16;
constexpr int GL_PASSES_MAX = 16;

__global__ void __launch_bounds__(32 * GL_WARPS, 1) gather_lane_kernel(MeshDev M, FieldDev F, size_t n, const double *__restrict__ R,
                                                                       const double *__restrict__ Z, const double *__restrict__ phi,
                                                                       const int32_t *__restrict__ hint, double *__restrict__ f,
                                                                       double *__restrict__ fR, double *__restrict__ fZ,
                                                                       double *__restrict__ fP, int nslot, int zero, const int *gate, int want,
                                                                       int n_pass)
{
    if ((((size_t)*gate * 16 <= n) ? 1 : 0) != want) return;
    constexpr unsigned FULL = 0xffffffffu;
    extern __shared__ __align__(16) unsigned char smem_g[];
    const int tid = threadIdx.x, lane = tid & 31, wib = tid >> 5;
    int *tag = reinterpret_cast<int *>(smem_g);
    volatile int *state = tag + LN_NBIN;
    int *rec_of = tag + 2 * LN_NBIN;
    int *counters = tag + 3 * LN_NBIN;
    const int rec_len = lane_rec_len(F);
    const int rec_stride = (rec_len + 3) | 1;
    double2 *REC = reinterpret_cast<double2 *>(smem_g + (LN_TABLE_BYTES + 15) / 16 * 16);
    for (int k = tid; k < LN_NBIN; k += 32 * GL_WARPS) { tag[k] = LN_EMPTY; state[k] = 0; rec_of[k] = -1; }
    if (tid < 4) counters[tid] = 0;
    __syncthreads();
    const size_t PER_WARP = 32 * (size_t)n_pass, PER_CTA = PER_WARP * GL_WARPS;
    const size_t n_chunks = (n + PER_CTA - 1) / PER_CTA;
    unsigned n_copied = 0;
    for (size_t chunk = blockIdx.x; chunk < n_chunks; chunk += gridDim.x) {
        const size_t w0 = chunk * PER_CTA + (size_t)wib * PER_WARP;
        size_t p = w0 + lane;
        double nR = 0.0, nZ = 0.0, nP = 0.0;
        int nH = -1;
        if (p < n) { nR = R[p]; nZ = Z[p]; nP = phi[p]; nH = hint[p]; }
#pragma unroll 1
        for (int pass = 0; pass < n_pass; ++pass, p += 32) {
            const double r = nR, z = nZ, ph = nP;
            const int h = nH;
            const bool in = p < n;
            if (pass + 1 < n_pass && p + 32 < n) { nR = R[p + 32]; nZ = Z[p + 32]; nP = phi[p + 32]; nH = hint[p + 32]; }
            // the hinted triangle first, with the geometry row of its record in shared memory (no trip to global memory on the
            // way): inside by the margin (rule L3) -> done; else the complete locator and a second look-up
            int t = (in && h >= 0 && h < M.n_tri) ? h : -1;
            int rec = -1;
            Bary b;
            b.xi = b.eta = b.l0 = b.xR = b.xZ = b.eR = b.eZ = 0.0;
            bool redo = in;
#pragma unroll 1
            for (int round = 0; round < 2; ++round) {
                bool ask = redo && t >= 0;
                if (ask) {                                   // own probe
                    unsigned hh = ln_hash(t);
                    const volatile int *vtag = tag;
#pragma unroll 1
                    for (int pr = 0; pr < LN_NPROBE; ++pr) {
                        const int th = vtag[hh];
                        if (th == t) {
                            if (state[hh] == LN_READY) { __threadfence_block(); rec = rec_of[hh]; ask = false; }
                            break;
                        }
                        if (th == LN_EMPTY) break;
                        hh = (hh + 1) & (LN_NBIN - 1);
                    }
                }
                unsigned need = __ballot_sync(FULL, ask);    // triangles not in the table yet: the warp brings them in
#pragma unroll 1
                while (need) {
                    const int tl = __shfl_sync(FULL, t, __ffs(need) - 1);
                    const int rr = ln_lookup(tl, lane, tag, state, rec_of, counters, nslot, M, F, REC, rec_len, rec_stride, n_copied);
                    const bool mine = ask && (t == tl);
                    if (mine) rec = rr;
                    need &= ~__ballot_sync(FULL, mine);
                }
                if (round == 1) break;
                if (redo && t >= 0 && rec >= 0) {            // barycentric test exactly as bary_rn() (rule L2)
                    const double2 *gq = REC + (size_t)rec * rec_stride + rec_len;
                    const double2 v0 = gq[0], gx = gq[1], ge = gq[2];
                    const double dx = __dsub_rn(r, v0.x), dz = __dsub_rn(z, v0.y);
                    b.xi = __dadd_rn(__dmul_rn(gx.x, dx), __dmul_rn(gx.y, dz));
                    b.eta = __dadd_rn(__dmul_rn(ge.x, dx), __dmul_rn(ge.y, dz));
                    b.l0 = __dsub_rn(__dsub_rn(1.0, b.xi), b.eta);
                    b.xR = gx.x; b.xZ = gx.y; b.eR = ge.x; b.eZ = ge.y;
                    if (fmin(fmin(b.xi, b.eta), b.l0) > LOC_TAU) redo = false;
                }
                if (!__any_sync(FULL, redo)) break;
                if (redo) { int moved = 0; t = locate(M, r, z, h, b, moved); rec = -1; }
            }
            if (in) {
                double v = 0.0, vR = 0.0, vZ = 0.0, vP = 0.0;
                if (t >= 0) {
                    if (rec >= 0) {
                        double fx, fe;
                        gather_lane_harmonic(F, REC + (size_t)rec * rec_stride, b.xi, b.eta, ph, zero, v, fx, fe, vP);
                        vR = fma(b.xR, fx, b.eR * fe);
                        vZ = fma(b.xZ, fx, b.eZ * fe);
                    } else {
                        const FieldVal fv = gather(F, t, b, ph);
                        v = fv.f; vR = fv.fR; vZ = fv.fZ; vP = fv.fphi;
                    }
                }
                f[p] = v; fR[p] = vR; fZ[p] = vZ;
                if (fP) fP[p] = vP;
            }
        }
        // ---- all warps meet; the table is emptied when it is nearly full
        __syncthreads();
        const int claimed = counters[0];
        __syncthreads();
        if (claimed > min(nslot, LN_NBIN * 3 / 4) - 16) {
            for (int k = tid; k < LN_NBIN; k += 32 * GL_WARPS) { tag[k] = LN_EMPTY; state[k] = 0; rec_of[k] = -1; }
            if (tid == 0) counters[0] = 0;
            __syncthreads();
        }
    }
}

template <int WARPS>
cudaError_t launch_lane(trimeg_ctx *c, const trimeg_markers &m, size_t n, double dt, int nsteps, cudaStream_t s)
{
    constexpr size_t SMEM_MAX = 227 * 1024;
    // function attributes are per device: set on every launch (cheap), not once per process
    cudaError_t e = cudaFuncSetAttribute(push_lane_kernel<WARPS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_MAX);
    if (e != cudaSuccess) return e;
    const size_t fixed = ((size_t)WARPS * LN_WARP_BYTES + LN_TABLE_BYTES + 15) / 16 * 16;
    const size_t rec_bytes = sizeof(double2) * (((size_t)lane_rec_len(c->field) + 3) | 1);    // as rec_stride in the kernel
    int nslot = lane_rec_len(c->field) ? (int)((SMEM_MAX - fixed) / rec_bytes) : 0;
    if (nslot > LN_NBIN * 3 / 4) nslot = LN_NBIN * 3 / 4;
    const size_t shm = fixed + (size_t)nslot * rec_bytes;
    const size_t per_cta = (size_t)LN_NW * WARPS;
    const size_t ctas = (n + per_cta - 1) / per_cta;
    push_lane_kernel<WARPS><<<(unsigned)ctas, 32 * WARPS, shm, s>>>(c->mesh, c->field, c->phys, m, n, dt, nsteps, c->d_stats, nslot, 0);
    c->n_launches++;
    return cudaGetLastError();
}

}  // namespace

#if !defined(TRIMEG_CORE_ONLY) && !defined(TRIMEG_SPLINE_ONLY)
cudaError_t launch_gather_lane(trimeg_ctx *c, size_t n, const double *R, const double *Z, const double *phi, const int32_t *hint,
                               double *f, double *fR, double *fZ, double *fP, const int *gate, int want, cudaStream_t s)
{
    constexpr size_t SMEM = 160 * 1024;
    cudaError_t e = cudaFuncSetAttribute(gather_lane_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM);
    if (e != cudaSuccess) return e;
    const size_t fixed = (LN_TABLE_BYTES + 15) / 16 * 16;
    const size_t rec_bytes = sizeof(double2) * (((size_t)lane_rec_len(c->field) + 3) | 1);
    int nslot = (int)((SMEM - fixed) / rec_bytes);
    if (nslot > LN_NBIN * 3 / 4) nslot = LN_NBIN * 3 / 4;
    size_t n_pass = n / ((size_t)c->n_sm * 4 * 32 * GL_WARPS);                 // at least ~4 chunks per SM
    n_pass = n_pass < 1 ? 1 : (n_pass > GL_PASSES_MAX ? GL_PASSES_MAX : n_pass);
    const size_t per_cta = (size_t)32 * n_pass * GL_WARPS;
    size_t ctas = (n + per_cta - 1) / per_cta;
    if (ctas > (size_t)c->n_sm * 4) ctas = (size_t)c->n_sm * 4;
    gather_lane_kernel<<<(unsigned)ctas, 32 * GL_WARPS, fixed + (size_t)nslot * rec_bytes, s>>>(c->mesh, c->field, n, R, Z, phi, hint, f, fR, fZ, fP,
                                                                                                 nslot, 0, gate, want, (int)n_pass);
    c->n_launches++;
    return cudaGetLastError();
}

#endif

#if defined(TRIMEG_CORE_ONLY)
cudaError_t launch_push_lane_core(trimeg_ctx *c, const trimeg_markers &m, size_t n, double dt, int nsteps, cudaStream_t s)
#elif defined(TRIMEG_SPLINE_ONLY)
cudaError_t launch_push_lane_spline(trimeg_ctx *c, const trimeg_markers &m, size_t n, double dt, int nsteps, cudaStream_t s)
#else
cudaError_t launch_push_lane(trimeg_ctx *c, const trimeg_markers &m, size_t n, double dt, int nsteps, cudaStream_t s)
#endif
{
    if (n == 0 || nsteps <= 0) return cudaSuccess;
#ifndef TRIMEG_SPLINE_LANE_WARPS
#define TRIMEG_SPLINE_LANE_WARPS 16
#endif
#ifndef TRIMEG_CORE_ONLY
    if (c->field.n_phi > 0) return launch_lane<TRIMEG_SPLINE_LANE_WARPS>(c, m, n, dt, nsteps, s);
#endif
    return launch_lane<16>(c, m, n, dt, nsteps, s);      // 16 warps at 128 registers (12 at 168 lose 8 % with 3 modes, 1 % with 16)
}

}  // namespace trimeg
