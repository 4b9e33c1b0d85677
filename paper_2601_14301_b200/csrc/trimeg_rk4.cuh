// trimeg_rk4.cuh -- row a6 building blocks shared by the shared-memory push kernels: per-marker RK4
// state layout, marker flags, and "finish a marker at one stage" (equations a4/a5, RK4 bookkeeping,
// next stage position, locate of that position).  The arithmetic per marker is that of push_kernel.
#pragma once
#include "trimeg_device.cuh"

// In-kernel phase timers of the warp kernels (lane 0, clock64): compiled in only with -DTRIMEG_PROFILE
// (python -m paper_2601_14301_b200.build --profile); the default build carries the cheap event counters alone.
#ifdef TRIMEG_PROFILE
#define TRIMEG_PHASE_CLOCK_INIT long long tph[3] = {0, 0, 0}, tlast = clock64();
#define TRIMEG_PHASE_CLOCK(k) { const long long now__ = clock64(); tph[k] += now__ - tlast; tlast = now__; }
#define TRIMEG_PHASE_CLOCK_FLUSH(st)                              \
    atomicAdd(&(st)->tile[0], (unsigned long long)tph[0]);        \
    atomicAdd(&(st)->tile[3], (unsigned long long)tph[1]);        \
    atomicAdd(&(st)->tile[4], (unsigned long long)tph[2]);
#else
#define TRIMEG_PHASE_CLOCK_INIT
#define TRIMEG_PHASE_CLOCK(k)
#define TRIMEG_PHASE_CLOCK_FLUSH(st)
#endif

namespace trimeg {

constexpr double TWO_PI = 6.283185307179586476925286766559;

enum : unsigned char { FL_ACTIVE = 1, FL_LOST = 2, FL_MOVED = 4, FL_WASACTIVE = 8 };
// per-marker fp64 state: Y = start-of-step state, A = k1 + 2 k2 + 2 k3, S = stage position
enum { Y_R, Y_Z, Y_P, Y_V, Y_W, S_MU, A_R, A_Z, A_P, A_V, A_W, S_R, S_Z, S_P, S_V, S_W, N_STATE };

// Geometry row of a triangle held in registers by the caller (R_v0, Z_v0 | xi_R, xi_Z | eta_R, eta_Z).
struct TriGeom { int t; double2 v0, gx, ge; };

// Finish one marker at one stage (slot or home role): equations, RK4 bookkeeping, next position,
// locate of the next position.  q = index of the marker in the warp's slice.  tg: geometry of the
// triangle the marker is in, if the caller holds it (saves the locator's loads when the marker stays).
__device__ __forceinline__ void advance(const MeshDev &M, const PhysDev &Ph, double *S, int NW, int *cell,
                                        unsigned char *flags, int q, int stage, const FieldVal &fv, double dt,
                                        double hdt, double dt6, const TriGeom *tg = nullptr)
{
    const int ps = (stage == 0) ? Y_R : S_R;               // stage 0 is evaluated at the start-of-step state itself (no copy Y -> S)
    const double R = S[(ps + 0) * NW + q], Z = S[(ps + 1) * NW + q];
    const double v = S[(ps + 3) * NW + q], w = S[(ps + 4) * NW + q], mu = S[S_MU * NW + q];
    const Rates k = rhs_point(Ph, R, Z, v, mu, w, fv);
    const double yR = S[Y_R * NW + q], yZ = S[Y_Z * NW + q], yP = S[Y_P * NW + q];
    const double yV = S[Y_V * NW + q], yW = S[Y_W * NW + q];
    double nR, nZ, nP, nV, nW_;
    if (stage < 3) {
        if (stage == 0) {
            S[A_R * NW + q] = k.R; S[A_Z * NW + q] = k.Z; S[A_P * NW + q] = k.phi;
            S[A_V * NW + q] = k.vpar; S[A_W * NW + q] = k.w;
        } else {
            S[A_R * NW + q] = fma(2.0, k.R, S[A_R * NW + q]); S[A_Z * NW + q] = fma(2.0, k.Z, S[A_Z * NW + q]);
            S[A_P * NW + q] = fma(2.0, k.phi, S[A_P * NW + q]); S[A_V * NW + q] = fma(2.0, k.vpar, S[A_V * NW + q]);
            S[A_W * NW + q] = fma(2.0, k.w, S[A_W * NW + q]);
        }
        const double c = (stage == 2) ? dt : hdt;
        nR = fma(c, k.R, yR); nZ = fma(c, k.Z, yZ); nP = fma(c, k.phi, yP);
        nV = fma(c, k.vpar, yV); nW_ = fma(c, k.w, yW);
    } else {
        nR = fma(dt6, S[A_R * NW + q] + k.R, yR); nZ = fma(dt6, S[A_Z * NW + q] + k.Z, yZ);
        nP = fma(dt6, S[A_P * NW + q] + k.phi, yP);
        nV = fma(dt6, S[A_V * NW + q] + k.vpar, yV); nW_ = fma(dt6, S[A_W * NW + q] + k.w, yW);
        nP = fma(-TWO_PI, floor(nP * (1.0 / TWO_PI)), nP);
    }
    Bary b;
    int moved = 0, tn = -2;
    if (tg != nullptr) {                                   // rule L3 on the current triangle, arithmetic of bary_rn() (rule L2)
        const double dx = __dsub_rn(nR, tg->v0.x), dz = __dsub_rn(nZ, tg->v0.y);
        const double xi = __dadd_rn(__dmul_rn(tg->gx.x, dx), __dmul_rn(tg->gx.y, dz));
        const double eta = __dadd_rn(__dmul_rn(tg->ge.x, dx), __dmul_rn(tg->ge.y, dz));
        const double l0 = __dsub_rn(__dsub_rn(1.0, xi), eta);
        if (fmin(fmin(xi, eta), l0) > LOC_TAU) tn = tg->t;
    }
    if (tn == -2) tn = locate(M, nR, nZ, cell[q], b, moved);
    unsigned char fl = flags[q];
    if (moved) fl |= FL_MOVED;
    if (tn < 0) fl = (fl | FL_LOST) & ~FL_ACTIVE;        // start-of-step state Y is kept; dropped for the rest of the call
    else {
        cell[q] = tn;
        const int o = (stage < 3) ? S_R : Y_R;             // S_* and Y_* are both (R, Z, phi, vpar, w) in this order
        S[(o + 0) * NW + q] = nR; S[(o + 1) * NW + q] = nZ; S[(o + 2) * NW + q] = nP;
        S[(o + 3) * NW + q] = nV; S[(o + 4) * NW + q] = nW_;
    }
    flags[q] = fl;
}

}  // namespace trimeg
