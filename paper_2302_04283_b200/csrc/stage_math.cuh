// stage_math.cuh -- device helpers shared by the kernels: the pinned four-term chain, warp reductions, the tetrad-frame
// fluid velocity and the quartic solve of Eq.49.
#pragma once
#include <math.h>

#include "async_copy.cuh"
#include "rad_internal.h"

namespace rad {

constexpr double kFourPi = 12.566370614359172954;
constexpr double kInvFourPi = 0.079577471545947667884;

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// pinned order (decides upwind signs, compared bit for bit with the oracle): fma(r3,n3, fma(r2,n2, fma(r1,n1, r0)))
__device__ __forceinline__ double chain4(double r0, double r1, double r2, double r3, double n1, double n2, double n3) {
    return fma(r3, n3, fma(r2, n2, fma(r1, n1, r0)));
}

// tetrad-frame four-velocity from the normal-frame spatial velocity u^a':
// u^ahat = theta^ahat_j u^j' (the co-triad is the spatial inverse tetrad), u^0hat = sqrt(1 + |u^ahat|^2).
// th = cell record [44..49] = theta (1x,1y,1z,2y,2z,3z)
__device__ __forceinline__ void tetrad_velocity(const double th[6], double u1, double u2, double u3, double uh[4]) {
    uh[1] = th[0] * u1 + th[1] * u2 + th[2] * u3;
    uh[2] = th[3] * u2 + th[4] * u3;
    uh[3] = th[5] * u3;
    uh[0] = sqrt(1.0 + (uh[1] * uh[1] + uh[2] * uh[2] + uh[3] * uh[3]));
}

// Quartic Eq.49 solved for the temperature change d = T_+ - T_- (R13): g(d) = B4 (T_- + d)^4 + B1 d + Bp,
// Bp = A_1 - (1 - A_2 alpha_s) Ebar_-.  Eq.48 needs exactly this difference; solving for it directly keeps
// Ebar_+ accurate in gas-dominated cells where C_v T >> Ebar.  g is convex and increasing on T > 0, so Newton converges
// monotonically from the right of the root and from the left lands right of it after one step.  Start: the Newton step
// from T_- (d = 0), which is close for cells near equilibrium; where it lands far away (more than T_- beyond T_-) the
// upper bound min(-B0/B1, (-B0/B4)^(1/4)) caps it (fourth root from the hardware rsqrt seeds: the start only has to be
// near the bound).  Reciprocals by rcp3.  Stop when the step is at rounding level, or when the error it leaves behind,
// <= 1.5 dd^2 / T (quadratic convergence: g''/2g' <= 1.5/T), is below 1e-16 |d|: a bound RELATIVE TO d, so that Eq.48's
// C_v d keeps full accuracy however large C_v T / Ebar is.
// Returns false when there is no positive root (B0 = Bp - B1 T_- >= 0) or a coefficient is not finite.
__device__ __forceinline__ bool quartic_delta(double B4, double B1, double Bp, double Tm, double &d) {
    const double B0 = Bp - B1 * Tm;
    if (!(B0 < 0.0) || !(B1 > 0.0) || !(B4 >= 0.0) || !isfinite(B0) || !isfinite(B1) || !isfinite(B4)) return false;
    if (B4 == 0.0) { d = -Bp * rcp3(B1); return true; }
    const double B44 = 4.0 * B4, aBp = fabs(Bp);
    {
        const double T2 = Tm * Tm, q = B4 * (T2 * T2);
        d = -(q + Bp) * rcp3(fma(B44, T2 * Tm, B1));
    }
    if (d > Tm) {
        const double y = -B0 * rcp3(B4);
        double r1, r2;
        asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(r1) : "d"(y));
        const double sy = y * r1;
        asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(r2) : "d"(sy));
        double T0 = sy * r2;                         // ~ y^(1/4)
        if (!(T0 > 0.0)) T0 = __longlong_as_double(0x7ff0000000000000ll);  // y outside the range of the approximation: the other bound alone
        d = fmin(d, fmin(-B0 * rcp3(B1), T0) - Tm);
    }
    for (int it = 0; it < 60; it++) {
        const double T = Tm + d, T2 = T * T, T3 = T2 * T, q = B4 * (T2 * T2);
        const double g = q + fma(B1, d, Bp), gp = fma(B44, T3, B1);
        const double rgp = rcp3(gp);  // gp >= B1 > 0, finite
        const double dd = g * rgp;
        d -= dd;
        const double add = fabs(dd);
        if (add <= 1e-15 * (fabs(d) + (aBp + q) * rgp) || 1.5 * add * add <= 1e-16 * fabs(d) * T) break;
    }
    return true;
}

}  // namespace rad
