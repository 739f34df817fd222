// Lennard-Jones pair term on the device.  PAPER.md:56-62 (Eq. 2-3), readings R1/R2.
//   f_LJ(r)/r = 24 eps (2 s6^2 - s6) / r^2,  U_LJ = 4 eps (s6^2 - s6),  s6 = (sigma^2/r^2)^3
// An in-range pair is evaluated in FP64 when r2 < precise_r2 (default: always), because the
// per-component force tolerance sits at the FP32 rounding floor; the
// FP32 variant is the "fast" branch for pairs whose |f| is small enough not to need it.
#pragma once
#include "common.cuh"

// 1/x for a normal positive double: hardware seed (MUFU.RCP64H, ~20 good bits) and two
// Newton steps -> relative error ~1e-16.  No slow path: r2 is never 0, inf or denormal here.
__device__ __forceinline__ double rcp_f64(double x)
{
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    double e = fma(-x, y, 1.0);
    y = fma(y, e, y);
    e = fma(-x, y, 1.0);
    y = fma(y, e, y);
    return y;
}

// Second pair potential ("trivial to replace this potential by other
// pair-potentials, including the coulombic interaction"): screened Coulomb (Yukawa) between equal charges,
//   U_Y = A exp(-kappa r) / r,   f_Y = -dU_Y/dr = U_Y (1/r + kappa),
// the bare Coulomb pair for kappa = 0; same cutoff and shift modes (ushift = U_Y(rc), f_rc = f_Y(rc)).
// Evaluated in FP64 on every path (md_set_potential makes the FP32 window of the cell and list kernels empty).
// U and f/r of a pair inside rc:
__device__ __forceinline__ void yukawa_fu64(const PairParams &P, double r2, double &fr, double &u)
{
    const double r = sqrt(r2), ir = 1.0 / r;
    const double e = P.yA * exp(-P.ykappa * r) * ir;
    double f = e * (ir + P.ykappa);
    u = e - P.ushift;
    if (P.mode == 2) {
        u += (r - P.rc) * P.f_rc;
        f -= P.f_rc;
    }
    fr = f * ir;
}

// FP64 pair term.  d = r_j - r_i (minimum image applied).  Returns true when r2 < rc^2
// (strict) and then adds this pair's contribution:  F_i -= (f/r) d  (Eq. 1),
// pe += U, w += r f.  Callers halve pe and w when they visit each pair twice.
__device__ __forceinline__ bool pair_f64(const PairParams &P, double dx, double dy, double dz,
                                         double &fx, double &fy, double &fz, double &pe, double &w)
{
    double r2 = fma(dx, dx, fma(dy, dy, dz * dz));
    if (!(r2 < P.rc2)) return false;
    if (P.kind == 1) {
        double fr, u;
        yukawa_fu64(P, r2, fr, u);
        fx = fma(-fr, dx, fx);
        fy = fma(-fr, dy, fy);
        fz = fma(-fr, dz, fz);
        pe += u;
        w = fma(fr, r2, w);
        return true;
    }
    double inv = rcp_f64(r2);
    double s2 = P.sig2 * inv;
    double s6 = s2 * s2 * s2;
    double fr = P.eps24 * inv * s6 * (2.0 * s6 - 1.0);
    double u = P.eps4 * s6 * (s6 - 1.0) - P.ushift;
    if (P.mode == 2) {                       // PAPER.md:61 (Eq. 3): f = f_LJ(r) - f_LJ(rc)
        double r = sqrt(r2);
        u += (r - P.rc) * P.f_rc;
        fr -= P.f_rc * inv * r;              // f_rc / r
    }
    fx = fma(-fr, dx, fx);
    fy = fma(-fr, dy, fy);
    fz = fma(-fr, dz, fz);
    pe += u;
    w = fma(fr, r2, w);
    return true;
}

// FP32 pair term for pairs already known to satisfy precise_r2 <= r2 < rc^2 (classification
// was done in FP64 by the caller); d in FP32.
__device__ __forceinline__ void pair_f32(const PairParams &P, float dx, float dy, float dz, float r2,
                                         float &fx, float &fy, float &fz, float &pe, float &w)
{
    float inv = __frcp_rn(r2);
    float s2 = P.sig2f * inv;
    float s6 = s2 * s2 * s2;
    float fr = P.eps24f * inv * s6 * (2.0f * s6 - 1.0f);
    float u = P.eps4f * s6 * (s6 - 1.0f) - P.ushiftf;
    if (P.mode == 2) {
        float r = sqrtf(r2);
        u += (r - P.rcf) * P.f_rcf;
        fr -= P.f_rcf * inv * r;
    }
    fx = fmaf(-fr, dx, fx);
    fy = fmaf(-fr, dy, fy);
    fz = fmaf(-fr, dz, fz);
    pe += u;
    w = fmaf(fr, r2, w);
}
