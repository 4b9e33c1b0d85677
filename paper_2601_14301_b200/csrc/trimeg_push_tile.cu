// trimeg_push_tile.cu -- triangle-batched fused RK4 push (rows a2-a6 of DESIGN.md §1).
//
// Why: with one thread per marker every lane fetches every coefficient of its triangle
// itself (21 x 16-byte loads per mode and stage); on B200 a warp-wide load costs 2-4 cycles
// of the SM's load/store data pipe even when all lanes read the same address, so the load
// path, not the FP64 pipe, bounds the kernel (profiles/r01_baseline_push_kernel.md).  The
// only way to lower load-pipe cycles per FP64 operation is to let one loaded coefficient
// feed several markers from a REGISTER.  That needs the markers evaluated together to sit
// in the same triangle, which a cell sort alone cannot keep true for long: markers drift
// across edges between sorts.
//
// How: one CTA owns a tile of NT consecutive markers for the whole call; their RK4 state
// lives in shared memory.  Every RK4 stage is five block-synchronous phases:
//   A  locate the stage position of every marker (hinted walk, bit-exact rule O3) and bin
//      it by triangle in a small open-addressing hash table (warp-aggregated atomics);
//   B  the coefficient records of the stage's triangles (n_modes x 21 complex each) are
//      copied HBM/L2 -> shared memory with cp.async (no register staging; the copy runs
//      under phases B and C); exclusive scan of the bin counts, each bin padded to a
//      multiple of P slots;
//   C  scatter (xi, eta, phi, owner) of every marker to its evaluation slot;
//   D  evaluation: each thread takes P consecutive slots -- by construction the same
//      triangle -- and runs the bivariate Horner scheme for all P markers off ONE
//      shared-memory load of each coefficient (warp-uniform address = broadcast, fixed
//      ~30-cycle latency instead of an L1/L2 round trip that 12 warps per SM cannot hide);
//   E  each marker reads back its field values, evaluates equilibrium + equations of motion
//      (a4, a5) and does its RK4 bookkeeping (a6).
// Markers whose triangle finds no bin or no shared-memory record (more distinct triangles
// in the tile than record slots: unsorted input) are evaluated by their owner with the
// one-marker gather of trimeg_device.cuh -- slower, same arithmetic.  The arithmetic of
// every marker (order of operations, fused multiply-adds) is the same as in push_kernel.
#include "trimeg_internal.h"
#include "trimeg_multi.cuh"

namespace trimeg {

namespace {

constexpr double TWO_PI = 6.283185307179586476925286766559;
constexpr int NBIN = 64;            // hash bins per stage (distinct triangles of a tile)
constexpr int NPROBE = 8;
constexpr int BIN_EMPTY = -1;

enum : unsigned char { FL_ACTIVE = 1, FL_LOST = 2, FL_MOVED = 4, FL_WASACTIVE = 8 };

// indices of the per-marker fp64 state arrays in shared memory
enum { S_R, S_Z, S_P, S_V, S_W, S_MU, A_R, A_Z, A_P, A_V, A_W, Y_R, Y_Z, Y_P, Y_V, Y_W, N_STATE };
// S_* = stage position, A_* = RK4 accumulator k1 + 2 k2 + 2 k3, Y_* = start-of-step state

template <int P, int T>
struct TileCfg {
    static constexpr int NT = P * T - 12 * P;                 // markers per tile (slack for bin padding)
    static constexpr int NE = NT + (P - 1) * NBIN;            // evaluation slots, worst case
    // without the coefficient records, rounded up to 16 bytes
    static constexpr size_t BASE_BYTES =
        (sizeof(double) * ((size_t)N_STATE * NT + 4 * (size_t)NE) +
         sizeof(int) * (3 * (size_t)NT + 2 * (size_t)NE + 5 * NBIN + 8) + NT + 15) / 16 * 16;
};

__device__ __forceinline__ unsigned hash_tri(int t) { return ((unsigned)t * 0x9E3779B1u) >> 26; }   // 6 bits

template <int P, int T>
__global__ void __launch_bounds__(T) push_tile_kernel(MeshDev M, FieldDev F, PhysDev Ph, trimeg_markers m, size_t n,
                                                      double dt, int nsteps, Stats *st, int nslot)
{
    using Cfg = TileCfg<P, T>;
    constexpr int NT = Cfg::NT, NE = Cfg::NE;
    extern __shared__ __align__(16) double smem_d[];
    double *S = smem_d;                                   // [N_STATE][NT]
    double *EV = S + (size_t)N_STATE * NT;                // [4][NE]: in (xi, eta, phi, -) / out (f, fR, fZ, fphi)
    int *cell = reinterpret_cast<int *>(EV + 4 * (size_t)NE);   // [NT] current triangle (hint)
    int *binrank = cell + NT;                             // [NT] bin << 16 | rank, -1 = not binned
    int *slot = binrank + NT;                             // [NT] evaluation slot of the marker
    int *ev_own = slot + NT;                              // [NE] owner marker of a slot, -1 = padding
    int *ev_rec = ev_own + NE;                            // [NE] coefficient-record slot of an evaluation slot
    int *tag = ev_rec + NE;                               // [NBIN] triangle of a bin
    int *cnt = tag + NBIN;                                // [NBIN]
    int *off = cnt + NBIN;                                // [NBIN]
    int *rec_of = off + NBIN;                             // [NBIN] record slot of a bin (order of first claim)
    int *bin_of = rec_of + NBIN;                          // [NBIN] bin of a record slot
    int *misc = bin_of + NBIN;                            // [0] = number of evaluation slots, [3] = bins claimed this stage
    unsigned char *flags = reinterpret_cast<unsigned char *>(misc + 8);   // [NT]
    // coefficient records of the stage's triangles: [nslot][n_modes][21] complex
    double2 *REC = reinterpret_cast<double2 *>(reinterpret_cast<unsigned char *>(smem_d) + Cfg::BASE_BYTES);
    const int rec_len = F.n_modes * NCOEF;               // double2 elements per record

    const int tid = threadIdx.x, lane = tid & 31;
    const size_t base = (size_t)blockIdx.x * NT;
    const int nt = (int)((n - base < (size_t)NT) ? (n - base) : (size_t)NT);
    const bool has_field = F.n_modes > 0;
    const double hdt = 0.5 * dt, dt6 = dt / 6.0;
    long long tph[5] = {0, 0, 0, 0, 0}, tlast = 0;      // phase timers (thread 0 only)
    unsigned n_fallback = 0, n_bins = 0, n_stages = 0;
#define TILE_TICK(k) do { if (tid == 0) { const long long now_ = clock64(); tph[k] += now_ - tlast; tlast = now_; } } while (0)
    if (tid == 0) tlast = clock64();

    // ---- load the tile
    for (int q = tid; q < NT; q += T) {
        unsigned char fl = 0;
        int c = -1;
        if (q < nt) {
            const size_t g = base + q;
            c = m.cell[g];
            if (c >= 0) {
                fl = FL_ACTIVE | FL_WASACTIVE;
                S[Y_R * NT + q] = m.R[g]; S[Y_Z * NT + q] = m.Z[g]; S[Y_P * NT + q] = m.phi[g];
                S[Y_V * NT + q] = m.vpar[g]; S[Y_W * NT + q] = m.w[g]; S[S_MU * NT + q] = m.mu[g];
            }
        }
        cell[q] = c; flags[q] = fl;
    }
    if (tid < NBIN) { tag[tid] = BIN_EMPTY; cnt[tid] = 0; }
    if (tid < 8) misc[tid] = 0;
    __syncthreads();

#pragma unroll 1
    for (int step = 0; step < nsteps; ++step) {
#pragma unroll 1
        for (int stage = 0; stage < 4; ++stage) {
            // ---------------------------------------------------------------- A: locate + bin
#pragma unroll 1
            for (int q0 = 0; q0 < NT; q0 += T) {
                const int q = q0 + tid;
                const bool act = (q < NT) && (flags[q] & FL_ACTIVE);
                int t = -1;
                if (act) {
                    if (stage == 0) {
#pragma unroll
                        for (int k = 0; k < 5; ++k) S[(S_R + k) * NT + q] = S[(Y_R + k) * NT + q];
                    }
                    Bary b;
                    int moved = 0;
                    t = locate(M, S[S_R * NT + q], S[S_Z * NT + q], cell[q], b, moved);
                    unsigned char fl = flags[q];
                    if (moved) fl |= FL_MOVED;
                    if (t < 0) fl = (fl | FL_LOST) & ~FL_ACTIVE;     // dropped for the rest of the call
                    else cell[q] = t;
                    flags[q] = fl;
                }
                if (has_field) {
                    // warp-aggregated insertion: one probe sequence and one atomicAdd per distinct triangle
                    const bool ok = act && t >= 0;
                    const int key = ok ? t : -1 - lane;
                    const unsigned grp = __match_any_sync(0xffffffffu, key);
                    const int leader = __ffs(grp) - 1;
                    int bin = -1, rank0 = 0;
                    if (ok && lane == leader) {
                        unsigned h = hash_tri(t);
#pragma unroll 1
                        for (int pr = 0; pr < NPROBE; ++pr) {
                            const int prev = atomicCAS(&tag[h], BIN_EMPTY, t);
                            if (prev == BIN_EMPTY) {                   // first claim: take the next record slot
                                const int r = atomicAdd(&misc[3], 1);
                                rec_of[h] = r;
                                if (r < NBIN) bin_of[r] = (int)h;
                            }
                            if (prev == BIN_EMPTY || prev == t) { bin = (int)h; break; }
                            h = (h + 1) & (NBIN - 1);
                        }
                        if (bin >= 0) rank0 = atomicAdd(&cnt[bin], __popc(grp));
                    }
                    bin = __shfl_sync(0xffffffffu, bin, leader);
                    rank0 = __shfl_sync(0xffffffffu, rank0, leader);
                    if (q < NT) binrank[q] = (ok && bin >= 0) ? ((bin << 16) | (rank0 + __popc(grp & ((1u << lane) - 1u)))) : -1;
                }
            }
            if (has_field) {
                __syncthreads();
                TILE_TICK(0);
                // ------------------------------------------------------------ B: records -> shared memory (async)
                {
                    const int n_rec = min(misc[3], nslot);
                    const int total = n_rec * rec_len;
#pragma unroll 1
                    for (int idx = tid; idx < total; idx += T) {
                        const int r = idx / rec_len, k = idx - r * rec_len;
                        const double2 *src = F.coef + (size_t)tag[bin_of[r]] * rec_len + k;
                        const unsigned dst = (unsigned)__cvta_generic_to_shared(REC + idx);
                        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
                    }
                    asm volatile("cp.async.commit_group;" ::: "memory");
                }
                // ------------------------------------------------------------ B: scan of padded bin sizes
                if (tid < 32) {
                    int run = 0;
#pragma unroll
                    for (int k = 0; k < NBIN / 32; ++k) {
                        const int b = k * 32 + lane;
                        const int c = (rec_of[b] < nslot) ? cnt[b] : 0;      // no record slot: owner evaluates
                        const int padded = (c + P - 1) / P * P;
                        int incl = padded;
#pragma unroll
                        for (int o = 1; o < 32; o <<= 1) {
                            const int v = __shfl_up_sync(0xffffffffu, incl, o);
                            if (lane >= o) incl += v;
                        }
                        const int o0 = run + incl - padded;
                        off[b] = o0;
                        for (int e = o0 + c; e < o0 + padded; ++e) ev_own[e] = -1;      // padding slots
                        run += __shfl_sync(0xffffffffu, incl, 31);
                    }
                    if (lane == 0) misc[0] = run;
                }
                __syncthreads();
                TILE_TICK(1);
                if (tid == 0) { n_bins += (unsigned)misc[3]; ++n_stages; }
                // ------------------------------------------------------------ C: scatter to evaluation slots
#pragma unroll 1
                for (int q = tid; q < NT; q += T) {
                    const int br = binrank[q];
                    if (br >= 0) {
                        const int r = rec_of[br >> 16];
                        if (r >= nslot) { binrank[q] = -1; continue; }
                        const int e = off[br >> 16] + (br & 0xffff);
                        const int t = cell[q];
                        const Bary b = bary_rn(M, t, S[S_R * NT + q], S[S_Z * NT + q]);
                        EV[e] = b.xi; EV[NE + e] = b.eta; EV[2 * NE + e] = S[S_P * NT + q];
                        ev_own[e] = q; ev_rec[e] = r;
                        slot[q] = e;
                    }
                }
                asm volatile("cp.async.wait_group 0;" ::: "memory");
                __syncthreads();
                TILE_TICK(2);
                // ------------------------------------------------------------ D: batched evaluation
                const int n_ev = misc[0];
#pragma unroll 1
                for (int e0 = tid * P; e0 < n_ev; e0 += T * P) {
                    const double2 *rec = REC + (size_t)ev_rec[e0] * rec_len;         // first slot of a group is real
                    double xi[P], eta[P], phi[P], f[P], fx[P], fe[P], fp[P];
                    bool real[P];
#pragma unroll
                    for (int p = 0; p < P; ++p) {
                        real[p] = ev_own[e0 + p] >= 0;
                        xi[p] = real[p] ? EV[e0 + p] : 0.0;
                        eta[p] = real[p] ? EV[NE + e0 + p] : 0.0;
                        phi[p] = real[p] ? EV[2 * NE + e0 + p] : 0.0;
                    }
                    gather_multi<P, false>(F, rec, xi, eta, phi, f, fx, fe, fp);
#pragma unroll
                    for (int p = 0; p < P; ++p) {
                        if (real[p]) {                                               // d/dxi, d/deta: chain rule in E
                            EV[e0 + p] = f[p]; EV[NE + e0 + p] = fx[p]; EV[2 * NE + e0 + p] = fe[p];
                            EV[3 * NE + e0 + p] = fp[p];
                        }
                    }
                }
                __syncthreads();
                TILE_TICK(3);
                if (tid < NBIN) { tag[tid] = BIN_EMPTY; cnt[tid] = 0; }             // for the next stage
                if (tid == 0) misc[3] = 0;
            }
            // ---------------------------------------------------------------- E: equations + RK4
#pragma unroll 1
            for (int q = tid; q < NT; q += T) {
                if (!(flags[q] & FL_ACTIVE)) continue;
                const double R = S[S_R * NT + q], Z = S[S_Z * NT + q], ph = S[S_P * NT + q];
                const double v = S[S_V * NT + q], w = S[S_W * NT + q], mu = S[S_MU * NT + q];
                FieldVal fv;
                fv.f = fv.fR = fv.fZ = fv.fphi = 0.0;
                if (has_field) {
                    if (binrank[q] >= 0) {
                        const int e = slot[q];
                        const double2 *g = reinterpret_cast<const double2 *>(M.geom + 6 * (size_t)cell[q]);
                        const double2 gx = __ldg(g + 1), ge = __ldg(g + 2);
                        const double fx = EV[NE + e], fe = EV[2 * NE + e];
                        fv.f = EV[e]; fv.fphi = EV[3 * NE + e];
                        fv.fR = fma(gx.x, fx, ge.x * fe);                            // d/dR
                        fv.fZ = fma(gx.y, fx, ge.y * fe);                            // d/dZ
                    } else {                               // no bin: one-marker gather, same arithmetic
                        const int t = cell[q];
                        const Bary b = bary_rn(M, t, R, Z);
                        fv = gather(F, t, b, ph);
                        ++n_fallback;
                    }
                }
                const Rates k = rhs_point(Ph, R, Z, v, mu, w, fv);
                const double yR = S[Y_R * NT + q], yZ = S[Y_Z * NT + q], yP = S[Y_P * NT + q];
                const double yV = S[Y_V * NT + q], yW = S[Y_W * NT + q];
                if (stage < 3) {
                    if (stage == 0) {
                        S[A_R * NT + q] = k.R; S[A_Z * NT + q] = k.Z; S[A_P * NT + q] = k.phi;
                        S[A_V * NT + q] = k.vpar; S[A_W * NT + q] = k.w;
                    } else {
                        S[A_R * NT + q] = fma(2.0, k.R, S[A_R * NT + q]); S[A_Z * NT + q] = fma(2.0, k.Z, S[A_Z * NT + q]);
                        S[A_P * NT + q] = fma(2.0, k.phi, S[A_P * NT + q]); S[A_V * NT + q] = fma(2.0, k.vpar, S[A_V * NT + q]);
                        S[A_W * NT + q] = fma(2.0, k.w, S[A_W * NT + q]);
                    }
                    const double c = (stage == 2) ? dt : hdt;
                    S[S_R * NT + q] = fma(c, k.R, yR); S[S_Z * NT + q] = fma(c, k.Z, yZ); S[S_P * NT + q] = fma(c, k.phi, yP);
                    S[S_V * NT + q] = fma(c, k.vpar, yV); S[S_W * NT + q] = fma(c, k.w, yW);
                } else {
                    const double Rn = fma(dt6, S[A_R * NT + q] + k.R, yR), Zn = fma(dt6, S[A_Z * NT + q] + k.Z, yZ);
                    double pn = fma(dt6, S[A_P * NT + q] + k.phi, yP);
                    const double vn = fma(dt6, S[A_V * NT + q] + k.vpar, yV), wn = fma(dt6, S[A_W * NT + q] + k.w, yW);
                    pn = fma(-TWO_PI, floor(pn * (1.0 / TWO_PI)), pn);
                    Bary b;
                    int moved = 0;
                    const int c = locate(M, Rn, Zn, cell[q], b, moved);
                    unsigned char fl = flags[q];
                    if (moved) fl |= FL_MOVED;
                    if (c < 0) fl = (fl | FL_LOST) & ~FL_ACTIVE;            // start-of-step state is kept
                    else {
                        cell[q] = c;
                        S[Y_R * NT + q] = Rn; S[Y_Z * NT + q] = Zn; S[Y_P * NT + q] = pn;
                        S[Y_V * NT + q] = vn; S[Y_W * NT + q] = wn;
                    }
                    flags[q] = fl;
                }
            }
            __syncthreads();
            TILE_TICK(4);
        }
    }
#undef TILE_TICK

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
    lost = __reduce_add_sync(0xffffffffu, lost);
    moved = __reduce_add_sync(0xffffffffu, moved);
    n_fallback = __reduce_add_sync(0xffffffffu, n_fallback);
    if (lane == 0 && n_fallback) atomicAdd(&st->tile[5], (unsigned long long)n_fallback);
    if (tid == 0) {
#pragma unroll
        for (int k = 0; k < 5; ++k) atomicAdd(&st->tile[k], (unsigned long long)tph[k]);
        atomicAdd(&st->tile[6], (unsigned long long)n_bins);
        atomicAdd(&st->tile[7], (unsigned long long)n_stages);
    }
    if (lane == 0) {
        if (lost) atomicAdd(&st->n_lost, (unsigned long long)lost);
        if (moved) atomicAdd(&st->n_moved, (unsigned long long)moved);
    }
}

template <int P, int T>
cudaError_t launch_tile(trimeg_ctx *c, const trimeg_markers &m, size_t n, double dt, int nsteps, cudaStream_t s)
{
    using Cfg = TileCfg<P, T>;
    static bool configured = false;
    constexpr size_t SMEM_MAX = 227 * 1024;                 // per-CTA limit on sm_100
    constexpr int CTAS = (2 * Cfg::BASE_BYTES + 32 * 1024 <= SMEM_MAX && 2 * T <= 1024) ? 2 : 1;   // CTAs per SM aimed at
    if (!configured) {
        cudaError_t e = cudaFuncSetAttribute(push_tile_kernel<P, T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_MAX);
        if (e != cudaSuccess) return e;
        configured = true;
    }
    // record slots: what is left of the SM's shared memory (1 KB per CTA is reserved by the system)
    const size_t rec_bytes = sizeof(double2) * NCOEF * (size_t)c->field.n_modes;
    const size_t avail = (SMEM_MAX + 1024) / CTAS - 1024 - Cfg::BASE_BYTES;
    int nslot = rec_bytes ? (int)(avail / rec_bytes) : 0;
    if (nslot > NBIN) nslot = NBIN;
    const size_t shm = Cfg::BASE_BYTES + (size_t)nslot * rec_bytes;
    const size_t tiles = (n + Cfg::NT - 1) / Cfg::NT;
    push_tile_kernel<P, T><<<(unsigned)tiles, T, shm, s>>>(c->mesh, c->field, c->phys, m, n, dt, nsteps, c->d_stats, nslot);
    c->n_launches++;
    return cudaGetLastError();
}

}  // namespace

cudaError_t launch_push_tile(trimeg_ctx *c, const trimeg_markers &m, size_t n, double dt, int nsteps, int variant,
                             cudaStream_t s)
{
    if (n == 0 || nsteps <= 0) return cudaSuccess;
    switch (variant) {
    case 1: return launch_tile<2, 192>(c, m, n, dt, nsteps, s);
    case 2: return launch_tile<2, 384>(c, m, n, dt, nsteps, s);
    case 3: return launch_tile<4, 128>(c, m, n, dt, nsteps, s);
    case 4: return launch_tile<4, 256>(c, m, n, dt, nsteps, s);
    case 5: return launch_tile<3, 256>(c, m, n, dt, nsteps, s);
    case 6: return launch_tile<3, 320>(c, m, n, dt, nsteps, s);
    default: return cudaErrorInvalidValue;
    }
}

}  // namespace trimeg
