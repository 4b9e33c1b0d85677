// trimeg_push_fused.cu -- CTA-tile fused RK4 push with resident coefficient records (rows a2-a6 of
// DESIGN.md §1).
//
// Why (profiles/r01_fused_push_kernel.md): the batched Horner evaluation is 88 % of the FP64 work.  Fed
// through L1 (warp kernel) it is held back by the load path: a warp-wide LDG.128 costs 4.6 cycles of the
// SM's data pipe -- more when the lanes sit in several triangles --, and the records of all resident warps
// do not fit in what is left of L1 next to their shared-memory state.  From shared memory a warp-wide
// LDS.128 costs 3.15 cycles whatever the mix of triangles (records padded by 16 B), with a fixed latency.
//
// This kernel: one CTA owns a tile of NT consecutive markers for the whole call (RK4 state in shared
// memory) and keeps the coefficient records of the tile's triangles in shared memory BETWEEN stages and
// steps -- only a triangle that no marker of the tile was in before costs a copy.  Per RK4 stage (two
// block barriers)
//   B  the records of new triangles (coefficients + geometry row) are copied global -> shared (cp.async,
//      16 B per lane); every warp scans the bin sizes, each padded to a multiple of P, into evaluation
//      slots sorted by triangle, and every marker writes its index into its slot;
//   D  one pass, no barrier inside: each thread takes P consecutive slots -- one triangle --, runs the
//      bivariate Horner scheme for the P markers off ONE shared-memory load of each coefficient, then
//      finishes the same P markers: chain rule, equilibrium + equations (a4, a5), RK4 bookkeeping (a6),
//      next stage position and the locate (a2) of that position, and bins them by their new triangle
//      for the next stage (small hash table, warp-aggregated: one probe sequence and one atomicAdd per
//      distinct triangle of a warp).
// Markers without a record (more distinct triangles than record slots: unsorted input) or without a
// slot are evaluated one per thread with the one-marker gather of trimeg_device.cuh: same arithmetic.
#include "trimeg_internal.h"
#include "trimeg_multi.cuh"
#include "trimeg_rk4.cuh"

namespace trimeg {

namespace {

constexpr int NBIN = 64;            // hash bins (distinct triangles the tile can track)
constexpr int NPROBE = 8;
constexpr int BIN_EMPTY = -1;

// misc[] slots
enum { MI_NEV, MI_NREC, MI_NLOAD0, MI_NLOAD1, MI_NFB0, MI_NFB1, MI_COUNT = 8 };   // NLOAD / NFB: one per stage parity

template <int P, int T>
struct FusedCfg {
    static constexpr int NE = P * T;                              // evaluation slots: one pass of the CTA
    static constexpr int NT = NE - 12 * P;                        // markers per tile (slack for bin padding)
    static constexpr size_t BASE_BYTES =
        (sizeof(double) * (size_t)N_STATE * NT +
         sizeof(int) * (3 * (size_t)NT + (size_t)NE + 6 * NBIN + MI_COUNT) + NT + 15) / 16 * 16;
};

__device__ __forceinline__ unsigned hash_tri(int t) { return ((unsigned)t * 0x9E3779B1u) >> 26; }   // 6 bits

// One marker evaluated on its own (coefficients from global memory) and finished.  Rare on cell-sorted input, so it is kept
// out of line: the kernel's hot path stays small for the instruction caches (L0 6 KB, L1.5 32 KB).
static __device__ __noinline__ void finish_single(const MeshDev &M, const FieldDev &F, const PhysDev &Ph, double *S, int NT,
                                                  int *cell, unsigned char *flags, int q, int stage, double dt, double hdt,
                                                  double dt6)
{
    const int tt = cell[q];
    const Bary b = bary_rn(M, tt, S[S_R * NT + q], S[S_Z * NT + q]);
    const FieldVal fv = gather(F, tt, b, S[S_P * NT + q]);
    advance(M, Ph, S, NT, cell, flags, q, stage, fv, dt, hdt, dt6);
}

template <int P, int T, int CTAS>
__global__ void __launch_bounds__(T, CTAS) push_fused_kernel(MeshDev M, FieldDev F, PhysDev Ph, trimeg_markers m, size_t n,
                                                          double dt, int nsteps, Stats *st, int nslot)
{
    using Cfg = FusedCfg<P, T>;
    constexpr int NT = Cfg::NT, NE = Cfg::NE;
    constexpr unsigned FULL = 0xffffffffu;
    extern __shared__ __align__(16) double smem_f[];
    double *S = smem_f;                                   // [N_STATE][NT]
    int *cell = reinterpret_cast<int *>(S + (size_t)N_STATE * NT);   // [NT] current triangle
    int *binrank = cell + NT;                             // [NT] bin << 16 | rank, -1 = not binned
    int *fb_list = binrank + NT;                          // [NT] markers evaluated one per thread
    int *ev = fb_list + NT;                               // [NE] owner | record slot << 16, -1 = padding
    int *tag = ev + NE;                                   // [NBIN] triangle of a bin (kept between stages)
    int *cnt = tag + NBIN;                                // [2][NBIN] markers in the bin, by parity of the stage that evaluates them
    int *rec_of = cnt + 2 * NBIN;                         // [NBIN] record slot of the bin, -1 = none
    int *load_list = rec_of + NBIN;                       // [2][NBIN] bins whose record must be copied, same parity rule
    int *misc = load_list + 2 * NBIN;                     // [MI_COUNT]
    unsigned char *flags = reinterpret_cast<unsigned char *>(misc + MI_COUNT);   // [NT]
    const int rec_len = F.n_modes * NCOEF;                // double2 elements per record
    const int rec_copy = rec_len + 3;                     // + the triangle's geometry row (3 double2)
    const int rec_stride = rec_copy | 1;                  // odd number of 16-byte units: records of different triangles start in different banks
    double2 *REC = reinterpret_cast<double2 *>(reinterpret_cast<unsigned char *>(smem_f) + Cfg::BASE_BYTES);

    const int tid = threadIdx.x, lane = tid & 31;
    const size_t base = (size_t)blockIdx.x * NT;
    const int nt = (int)((n - base < (size_t)NT) ? (n - base) : (size_t)NT);
    const bool has_field = F.n_modes > 0;
    const double hdt = 0.5 * dt, dt6 = dt / 6.0;
    unsigned n_fallback = 0;

    // ---- load the tile, locate the start positions
    for (int q = tid; q < NT; q += T) {
        unsigned char fl = 0;
        int c = -1;
        if (q < nt) {
            const size_t g = base + q;
            c = m.cell[g];
            if (c >= 0) {
                const double R = m.R[g], Z = m.Z[g];
                S[Y_R * NT + q] = R; S[Y_Z * NT + q] = Z; S[Y_P * NT + q] = m.phi[g];
                S[Y_V * NT + q] = m.vpar[g]; S[Y_W * NT + q] = m.w[g]; S[S_MU * NT + q] = m.mu[g];
#pragma unroll
                for (int k = 0; k < 5; ++k) S[(S_R + k) * NT + q] = S[(Y_R + k) * NT + q];
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
    if (tid < NBIN) { tag[tid] = BIN_EMPTY; cnt[tid] = 0; cnt[NBIN + tid] = 0; rec_of[tid] = -1; }
    if (tid < MI_COUNT) misc[tid] = 0;
    __syncthreads();

    unsigned n_copied = 0, n_stages = 0;
    long long tph[6] = {0, 0, 0, 0, 0, 0}, tlast = clock64();       // thread 0: cycles per phase
#define FUSED_TICK(k) do { if (tid == 0) { const long long now_ = clock64(); tph[k] += now_ - tlast; tlast = now_; } } while (0)

    // Bin marker q (triangle t) for the NEXT evaluation: warp-aggregated -- one probe sequence and one
    // atomicAdd per distinct triangle of the warp.  Must be called by all 32 lanes (act = false: no marker).
    auto bin_marker = [&](bool act, int q, int t, int set) {
        const int key = act ? t : -1 - lane;
        const unsigned grp = __match_any_sync(FULL, key);
        const int leader = __ffs(grp) - 1;
        int bin = -1, rank0 = 0;
        if (act && lane == leader) {
            unsigned h = hash_tri(t);
#pragma unroll 1
            for (int pr = 0; pr < NPROBE; ++pr) {
                const int prev = atomicCAS(&tag[h], BIN_EMPTY, t);
                if (prev == BIN_EMPTY) {                   // first marker of the tile in this triangle: record slot + copy
                    const int r = atomicAdd(&misc[MI_NREC], 1);
                    if (r < nslot) { rec_of[h] = r; load_list[set * NBIN + atomicAdd(&misc[MI_NLOAD0 + set], 1)] = (int)h; }
                    else rec_of[h] = -1;
                }
                if (prev == BIN_EMPTY || prev == t) { bin = (int)h; break; }
                h = (h + 1) & (NBIN - 1);
            }
            if (bin >= 0) rank0 = atomicAdd(&cnt[set * NBIN + bin], __popc(grp));
        }
        bin = __shfl_sync(FULL, bin, leader);
        rank0 = __shfl_sync(FULL, rank0, leader);
        if (act) binrank[q] = (bin >= 0) ? ((bin << 16) | (rank0 + __popc(grp & ((1u << lane) - 1u)))) : -1;
    };

    if (has_field) {                                       // bins of the first stage
#pragma unroll 1
        for (int q0 = 0; q0 < NT; q0 += T) {
            const int q = q0 + tid;
            const bool act = (q < NT) && (flags[q] & FL_ACTIVE);
            bin_marker(act, q, act ? cell[q] : -1, 0);
        }
        __syncthreads();
    }

#pragma unroll 1
    for (int step = 0; step < nsteps; ++step) {
#pragma unroll 1
        for (int stage = 0; stage < 4; ++stage) {
            if (!has_field) {                              // no field: equations only, one marker per thread and turn
#pragma unroll 1
                for (int q = tid; q < NT; q += T) {
                    if (!(flags[q] & FL_ACTIVE)) continue;
                    FieldVal fv;
                    fv.f = fv.fR = fv.fZ = fv.fphi = 0.0;
                    advance(M, Ph, S, NT, cell, flags, q, stage, fv, dt, hdt, dt6);
                    if (stage == 3) {
#pragma unroll
                        for (int k = 0; k < 5; ++k) S[(S_R + k) * NT + q] = S[(Y_R + k) * NT + q];
                    }
                }
                continue;                                  // a thread only ever touches its own markers here
            }
            // ------------------------------------------------- B: copy new records; bins -> slots; markers -> slots
            const int cur = stage & 1, nxt = cur ^ 1;                          // 4 stages per step: parity of the global stage count
            {
                const int n_load = misc[MI_NLOAD0 + cur];
                const int total = n_load * rec_copy;
#pragma unroll 1
                for (int idx = tid; idx < total; idx += T) {
                    const int i = idx / rec_copy, k = idx - i * rec_copy;
                    const int b = load_list[cur * NBIN + i];
                    const double2 *src = (k < rec_len) ? F.coef + (size_t)tag[b] * rec_len + k
                                                       : reinterpret_cast<const double2 *>(M.geom + 6 * (size_t)tag[b]) + (k - rec_len);
                    const unsigned dst = (unsigned)__cvta_generic_to_shared(REC + (size_t)rec_of[b] * rec_stride + k);
                    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
                }
                asm volatile("cp.async.commit_group;" ::: "memory");
                if (tid == 0) n_copied += (unsigned)n_load;
            }
            // every warp scans the 64 bin sizes itself (lane l: bins l and l + 32), each padded to a multiple of P
            int off0, off1;
            {
                const int c0 = (rec_of[lane] >= 0) ? cnt[cur * NBIN + lane] : 0;             // no record: one marker per thread
                const int c1 = (rec_of[32 + lane] >= 0) ? cnt[cur * NBIN + 32 + lane] : 0;
                const int pad0 = (c0 + P - 1) / P * P, pad1 = (c1 + P - 1) / P * P;
                int in0 = pad0, in1 = pad1;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const int v0 = __shfl_up_sync(FULL, in0, o), v1 = __shfl_up_sync(FULL, in1, o);
                    if (lane >= o) { in0 += v0; in1 += v1; }
                }
                const int o0 = in0 - pad0, o1 = __shfl_sync(FULL, in0, 31) + in1 - pad1;
                const bool fit0 = (c0 > 0) && (o0 + pad0 <= NE), fit1 = (c1 > 0) && (o1 + pad1 <= NE);   // else: one marker per thread
                off0 = fit0 ? o0 : -1; off1 = fit1 ? o1 : -1;
                if (tid < 32) {
                    if (fit0) for (int e = o0 + c0; e < o0 + pad0; ++e) ev[e] = -1;            // padding slots
                    if (fit1) for (int e = o1 + c1; e < o1 + pad1; ++e) ev[e] = -1;
                    const int n_ev = __reduce_max_sync(FULL, max(fit0 ? o0 + pad0 : 0, fit1 ? o1 + pad1 : 0));
                    if (lane == 0) { misc[MI_NEV] = n_ev; misc[MI_NFB0 + nxt] = 0; }
                }
            }
#pragma unroll
            for (int q0 = 0; q0 < NT; q0 += T) {
                const int q = q0 + tid;
                const bool act = (q < NT) && (flags[q] & FL_ACTIVE);
                const int br = act ? binrank[q] : -1;
                const int b = (br >= 0) ? (br >> 16) : 0;
                const int oa = __shfl_sync(FULL, off0, b & 31), ob = __shfl_sync(FULL, off1, b & 31);
                const int o = (b < 32) ? oa : ob;
                if (act) {
                    if (br >= 0 && o >= 0) ev[o + (br & 0xffff)] = q | (rec_of[b] << 16);
                    else fb_list[atomicAdd(&misc[MI_NFB0 + cur], 1)] = q;
                }
            }
            // the table is nearly full of triangles the markers have left: start it afresh with the bins of the next step
            const bool clear = (stage == 3) && (misc[MI_NREC] > min(nslot, NBIN) - 8);   // MI_NREC only changes in phase D
            asm volatile("cp.async.wait_group 0;" ::: "memory");
            __syncthreads();
            FUSED_TICK(1);
            if (clear) {                                                      // uniform; rec_of / tag were read above
                if (tid < NBIN) { tag[tid] = BIN_EMPTY; rec_of[tid] = -1; }
                if (tid == 0) misc[MI_NREC] = 0;
                __syncthreads();
            }
            // counters of this parity were read above; phase D of the NEXT stage is the first to add to them again
            if (tid < NBIN) cnt[cur * NBIN + tid] = 0;
            if (tid == 0) misc[MI_NLOAD0 + cur] = 0;
            FUSED_TICK(2);
            // ---------------------------------------------------------------- D: evaluate + finish, P slots per thread
            const int n_ev = misc[MI_NEV];
            int own[P];
#pragma unroll
            for (int p = 0; p < P; ++p) own[p] = -1;
            if (tid * P < n_ev) {
                const int e0 = tid * P;
#pragma unroll
                for (int p = 0; p < P; ++p) { const int v = ev[e0 + p]; own[p] = (v >= 0) ? (v & 0xffff) : -1; }
                const int rec = ev[e0] >> 16;                                // first slot of a group is real
                const double2 *recp = REC + (size_t)rec * rec_stride;          // coefficients, then the geometry row
                TriGeom tg;
                tg.t = cell[own[0]];
                tg.v0 = recp[rec_len]; tg.gx = recp[rec_len + 1]; tg.ge = recp[rec_len + 2];
                const double2 v0 = tg.v0, gx = tg.gx, ge = tg.ge;
                double xi[P], eta[P], phi[P], f[P], fx[P], fe[P], fp[P];
#pragma unroll
                for (int p = 0; p < P; ++p) {
                    xi[p] = eta[p] = phi[p] = 0.0;
                    if (own[p] >= 0) {                 // local coordinates exactly as bary_rn() (rule L2)
                        const double dx = __dsub_rn(S[S_R * NT + own[p]], v0.x), dz = __dsub_rn(S[S_Z * NT + own[p]], v0.y);
                        xi[p] = __dadd_rn(__dmul_rn(gx.x, dx), __dmul_rn(gx.y, dz));
                        eta[p] = __dadd_rn(__dmul_rn(ge.x, dx), __dmul_rn(ge.y, dz));
                        phi[p] = S[S_P * NT + own[p]];
                    }
                }
                double Er[P], Ei[P], Dr[P], Di[P];
                gather_phases<P>(F, phi, Er, Ei, Dr, Di);
                FUSED_TICK(0);
                gather_modes<P, false>(F, recp, xi, eta, phi, Er, Ei, Dr, Di, f, fx, fe, fp);
                FUSED_TICK(3);
#pragma unroll 1
                for (int p = 0; p < P; ++p) {
                    int q = -1;                                              // select without dynamic register indexing
                    FieldVal fv;
                    fv.f = fv.fR = fv.fZ = fv.fphi = 0.0;
#pragma unroll
                    for (int pp = 0; pp < P; ++pp)
                        if (pp == p) {
                            q = own[pp]; fv.f = f[pp]; fv.fphi = fp[pp];
                            fv.fR = fma(gx.x, fx[pp], ge.x * fe[pp]);            // d/dR
                            fv.fZ = fma(gx.y, fx[pp], ge.y * fe[pp]);            // d/dZ
                        }
                    if (q >= 0) advance(M, Ph, S, NT, cell, flags, q, stage, fv, dt, hdt, dt6, &tg);
                }
            }
            // the markers this thread finished: start-of-step copy, bin for the next stage (all lanes take part)
#pragma unroll
            for (int p = 0; p < P; ++p) {
                const int q = own[p];
                const bool act = (q >= 0) && (flags[q] & FL_ACTIVE);
                if (act && stage == 3) {
#pragma unroll
                    for (int k = 0; k < 5; ++k) S[(S_R + k) * NT + q] = S[(Y_R + k) * NT + q];
                }
                bin_marker(act, q, act ? cell[q] : -1, nxt);
            }
            // markers without a slot: one per thread, coefficients from global memory
            {
                const int n_fb = misc[MI_NFB0 + cur];
#pragma unroll 1
                for (int i0 = 0; i0 < n_fb; i0 += T) {
                    const int i = i0 + tid;
                    int q = -1;
                    if (i < n_fb) {
                        q = fb_list[i];
                        ++n_fallback;
                        finish_single(M, F, Ph, S, NT, cell, flags, q, stage, dt, hdt, dt6);
                    }
                    const bool act = (q >= 0) && (flags[q] & FL_ACTIVE);
                    if (act && stage == 3) {
#pragma unroll
                        for (int k = 0; k < 5; ++k) S[(S_R + k) * NT + q] = S[(Y_R + k) * NT + q];
                    }
                    bin_marker(act, q, act ? cell[q] : -1, nxt);
                }
            }
            FUSED_TICK(4);
            __syncthreads();
            FUSED_TICK(5);
            if (tid == 0) ++n_stages;
        }
    }
#undef FUSED_TICK
    // ---- write back, statistics
    int lost = 0, moved = 0;
    for (int q = tid; q < nt; q += T) {
        const unsigned char fl = flags[q];
        if (!(fl & FL_WASACTIVE)) continue;
        const size_t g = base + q;
        m.R[g] = S[Y_R * NT + q]; m.Z[g] = S[Y_Z * NT + q]; m.phi[g] = S[Y_P * NT + q];
        m.vpar[g] = S[Y_V * NT + q]; m.w[g] = S[Y_W * NT + q];
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
        if (n_fallback) atomicAdd(&st->tile[5], (unsigned long long)n_fallback);
    }
    if (tid == 0) {
        atomicAdd(&st->tile[6], (unsigned long long)n_copied);
#pragma unroll
        for (int k = 0; k < 5; ++k) atomicAdd(&st->tile[k], (unsigned long long)(k == 4 ? tph[4] + tph[5] : tph[k]));
        atomicAdd(&st->tile[7], (unsigned long long)n_stages);
    }
}

template <int P, int T, int CTAS = 1>
cudaError_t launch_fused(trimeg_ctx *c, const trimeg_markers &m, size_t n, double dt, int nsteps, cudaStream_t s)
{
    using Cfg = FusedCfg<P, T>;
    static bool configured = false;
    constexpr size_t SMEM_MAX = (228 * 1024) / CTAS - 1024;  // 228 KB per SM, 1 KB per CTA reserved by the system
    if (!configured) {
        cudaError_t e = cudaFuncSetAttribute(push_fused_kernel<P, T, CTAS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_MAX);
        if (e != cudaSuccess) return e;
        configured = true;
    }
    // record slots: what is left of the CTA's shared memory
    const size_t rec_bytes = sizeof(double2) * ((NCOEF * (size_t)c->field.n_modes + 3) | 1);   // as rec_stride in the kernel
    int nslot = c->field.n_modes ? (int)((SMEM_MAX - Cfg::BASE_BYTES) / rec_bytes) : 0;
    if (nslot > NBIN) nslot = NBIN;
    const size_t shm = Cfg::BASE_BYTES + (size_t)nslot * rec_bytes;
    const size_t tiles = (n + Cfg::NT - 1) / Cfg::NT;
    push_fused_kernel<P, T, CTAS><<<(unsigned)tiles, T, shm, s>>>(c->mesh, c->field, c->phys, m, n, dt, nsteps, c->d_stats, nslot);
    c->n_launches++;
    return cudaGetLastError();
}

}  // namespace

cudaError_t launch_push_fused(trimeg_ctx *c, const trimeg_markers &m, size_t n, double dt, int nsteps, int variant,
                              cudaStream_t s)
{
    if (n == 0 || nsteps <= 0) return cudaSuccess;
    switch (variant) {
    case 3: return launch_fused<2, 384>(c, m, n, dt, nsteps, s);
    case 4: return launch_fused<3, 256>(c, m, n, dt, nsteps, s);
    case 5: return launch_fused<4, 256>(c, m, n, dt, nsteps, s);
    case 6: return launch_fused<2, 192, 2>(c, m, n, dt, nsteps, s);
    default: return cudaErrorInvalidValue;
    }
}

}  // namespace trimeg
