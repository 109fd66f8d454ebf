// stage_math.cuh -- device helpers shared by the stage kernels (stage.cu, coupling.cu): fast FP64 reciprocal,
// warp reductions, the tetrad-frame fluid velocity and the quartic solve of Eq.49.
#pragma once
#include <math.h>

#include "rad_internal.h"

namespace rad {

constexpr double kFourPi = 12.566370614359172954;
constexpr double kInvFourPi = 0.079577471545947667884;

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// 1/d for normal, finite d: hardware seed (MUFU.RCP64H, ~20 bits) + two Newton steps = 4 DFMA, last-bit accurate
// (measured on B200 against IEEE division over 40 decades: identical).  No special-case path: callers never
// use the result when d is 0, subnormal or not finite.
__device__ __forceinline__ double fast_rcp(double d) {
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(d));
    double e = fma(-d, r, 1.0);
    r = fma(r, e, r);
    e = fma(-d, r, 1.0);
    return fma(r, e, r);
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
// Ebar_+ accurate in gas-dominated cells where C_v T >> Ebar.  Newton from an upper bound (g convex, increasing).
// Returns false when there is no positive root (B0 = Bp - B1 T_- >= 0) or a coefficient is not finite.
__device__ __forceinline__ bool quartic_delta(double B4, double B1, double Bp, double Tm, double &d) {
    const double B0 = Bp - B1 * Tm;
    if (!(B0 < 0.0) || !(B1 > 0.0) || !(B4 >= 0.0) || !isfinite(B0) || !isfinite(B1) || !isfinite(B4)) return false;
    const double rB1 = 1.0 / B1;
    if (B4 == 0.0) { d = -Bp * rB1; return true; }
    d = fmin(-B0 * rB1, sqrt(sqrt(-B0 / B4))) - Tm;
    for (int it = 0; it < 60; it++) {
        const double T = Tm + d, T3 = T * T * T, q = B4 * T3 * T;
        const double g = q + fma(B1, d, Bp), gp = fma(4.0 * B4, T3, B1);
        const double rgp = fast_rcp(gp);  // gp >= B1 > 0, finite
        const double dd = g * rgp;
        d -= dd;
        if (fabs(dd) <= 1e-15 * (fabs(d) + (fabs(Bp) + q) * rgp)) break;
    }
    return true;
}

// What a warp needs about its cell for the coupling (all warp-uniform)
struct CoupleCell {
    double nup0;        // n^0 = 1/alpha
    double E[4];        // E_alphahat: n_0 = E_0 + E_a n^a
    double th[6];       // co-triad
    double rho, Tm, u1, u2, u3, aP, aEa, aS;
};

// Locally implicit coupling of one cell by one warp (paper section 2.5, Eq.31-50), the ergosphere mask
// and the fluid increment.  Each lane holds NITER angles n = it*32 + lane (n < N): direction
// (n1,n2,n3), dOmega in dom[], and the post-transport intensity in Is[], which is replaced by the post-coupling
// intensity.  Returns T_+ and dR[4] = change of R^0_alpha (all lanes), and whether the quartic had a root.
template <int NITER>
__device__ __forceinline__ void couple_cell(const Params &p, const CoupleCell &cc, double dt, int lane, int N,
                                            const double (&n1)[NITER], const double (&n2)[NITER], const double (&n3)[NITER],
                                            const double (&dom)[NITER], double (&Is)[NITER], double &Tp, double (&dR)[4],
                                            bool &noroot, bool enable = true) {
    // `enable` (warp-uniform) = this cell takes part (false for excised cells: nothing changes).  All shuffles below run in warp-uniform control flow: cells that are not coupled (params.couple == 0) still
    // take the same path with src = 0, g1 = 1 so that Is is unchanged.
    double uh[4] = {1.0, 0.0, 0.0, 0.0};
    if (p.couple && enable) tetrad_velocity(cc.th, cc.u1, cc.u2, cc.u3, uh);
    const double aE = cc.aEa + cc.aS;  // Eq.33b
    // sweep 1: fluid-frame quantities and the four reductions.  With g1 = n^0/(n^0 + n^0bar alpha_E dt) and
    // g2 = n^0bar/(n^0 + n^0bar alpha_E dt):  A_1 = sum g1 Ibar dOmega_bar, A_2 = dt/4pi sum g2 dOmega_bar (Eq.42),
    // and Eq.40 back in the tetrad frame is  Ihat_+ = g1 Ihat_- + g2 (n^0bar)^-4 dt/4pi (alpha_P a T^4 + alpha_s Ebar_+).
    double g1[NITER], g2r4[NITER];
    double W = 0.0, A1 = 0.0, A2 = 0.0, Em = 0.0;
#pragma unroll
    for (int it = 0; it < NITER; it++) {
        const double nb = uh[0] - (uh[1] * n1[it] + uh[2] * n2[it] + uh[3] * n3[it]);  // n^0bar = -u_alpha n^alpha
        const double nb2 = nb * nb;
        const double r2 = fast_rcp(nb2);
        const double dOm = (it * 32 + lane < N) ? dom[it] * r2 : 0.0;                  // dOmega_bar (R11); 0 for idle lanes
        const double Ib = nb2 * nb2 * Is[it];                                          // Ibar_- = (n^0bar)^4 Ihat (R11)
        const double rd = fast_rcp(fma(nb * aE, dt, cc.nup0));                         // 1/(n^0 + n^0bar alpha_E dt)
        g1[it] = cc.nup0 * rd;
        const double g2 = nb * rd;
        g2r4[it] = g2 * (r2 * r2);
        W += dOm;
        A1 = fma(g1[it] * Ib, dOm, A1);                                                // Eq.42a
        A2 = fma(g2, dOm, A2);                                                         // Eq.42b
        Em = fma(Ib, dOm, Em);                                                         // Eq.38
    }
    W = warp_sum(W); A1 = warp_sum(A1); A2 = warp_sum(A2); Em = warp_sum(Em);
    Tp = cc.Tm;
    noroot = false;
    bool coupled = false;
    double src = 0.0;
    if (p.couple && enable) {
        const double scale = p.renorm ? kFourPi / W : 1.0;                             // R12
        A1 *= scale; Em *= scale; A2 *= scale * dt / kFourPi;
        const double Cv = cc.rho / (p.gamma_gas - 1.0);
        const double B4 = A2 * cc.aP * p.a_rad, om = 1.0 - A2 * cc.aS;                 // Eq.50
        const double B1 = Cv * om, Bp = A1 - om * Em;
        double dTemp = 0.0;
        if (!quartic_delta(B4, B1, Bp, cc.Tm, dTemp)) {
            noroot = true;
        } else {
            coupled = true;
            Tp = cc.Tm + dTemp;
            const double Ep = Em - Cv * dTemp;                                         // Eq.48
            const double T2 = Tp * Tp;
            src = (cc.aP * p.a_rad * T2 * T2 + cc.aS * Ep) * dt / kFourPi;
        }
    }
    // sweep 2: Eq.40, fluid increment through the tetrad-frame first moments of the change, mask
    double M0 = 0.0, M1 = 0.0, M2 = 0.0, M3 = 0.0;
#pragma unroll
    for (int it = 0; it < NITER; it++) {
        const double Iold = Is[it];
        double Inew = coupled ? fma(src, g2r4[it], g1[it] * Iold) : Iold;
        const double wI = (it * 32 + lane < N) ? dom[it] * (Inew - Iold) : 0.0;
        M0 += wI; M1 = fma(wI, n1[it], M1); M2 = fma(wI, n2[it], M2); M3 = fma(wI, n3[it], M3);
        if (p.n0_crit > 0.0 && enable) {
            const double n0 = chain4(cc.E[0], cc.E[1], cc.E[2], cc.E[3], n1[it], n2[it], n3[it]);  // cell-centre n_0
            if (fabs(n0) < p.n0_crit) Inew = 0.0;
        }
        Is[it] = Inew;
    }
    M0 = warp_sum(M0); M1 = warp_sum(M1); M2 = warp_sum(M2); M3 = warp_sum(M3);
    // R^0_alpha = sum n^0 n_alpha I dOmega; n_0 = E_ahat n^ahat, n_i = theta^a_i n^a
    dR[0] = cc.nup0 * (cc.E[0] * M0 + cc.E[1] * M1 + cc.E[2] * M2 + cc.E[3] * M3);
    dR[1] = cc.nup0 * (cc.th[0] * M1);
    dR[2] = cc.nup0 * (cc.th[1] * M1 + cc.th[3] * M2);
    dR[3] = cc.nup0 * (cc.th[2] * M1 + cc.th[4] * M2 + cc.th[5] * M3);
}

}  // namespace rad
