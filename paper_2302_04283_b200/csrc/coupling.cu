// coupling.cu -- subsystem 3: locally implicit matter-radiation coupling (paper section 2.5),
// the ergosphere mask and the angular moments (Eq.45, Eq.38).
//
// One warp per cell.  Lanes stride over the angles; the angle reductions that form A_1, A_2 (Eq.42),
// Ebar_- (Eq.38) and the fluid-frame weight normalisation W (R12) are warp-shuffle trees; the quartic
// Eq.49 for T_+ is solved redundantly by every lane in registers; a second sweep applies Eq.40, transforms
// back to the tetrad frame, masks |n_0| < n_0^crit and accumulates the fluid increment
// dT^0_alpha = -sum_n n^0 n_alpha (I_+ - I*) dOmega_n with a second shuffle tree.
#include "stage_math.cuh"

#ifndef RAD_MOM_CTAS
#define RAD_MOM_CTAS 6
#endif

namespace rad {
namespace {

constexpr int kWarpsPerCta = 12;

// legacy signature of tetrad_velocity on a cell record
__device__ __forceinline__ void tetrad_velocity_rec(const double *cg, double u1, double u2, double u3, double uh[4]) {
    const double th[6] = {cg[44], cg[45], cg[46], cg[47], cg[48], cg[49]};
    rad::tetrad_velocity(th, u1, u2, u3, uh);
}

// ------------------------------------------------------------------------------------------------
// coupling, one warp per cell, angles in registers (the same couple_cell the fused stage kernel uses)
// ------------------------------------------------------------------------------------------------
template <int NITER>
__global__ void __launch_bounds__(32 * kWarpsPerCta) k_coupling_w(DeviceTables t, Params p, double *__restrict__ I,
                                                                  const double *__restrict__ fluid, const double *__restrict__ aP_,
                                                                  const double *__restrict__ aE_, const double *__restrict__ aS_,
                                                                  double dt, double *__restrict__ T_out, double *__restrict__ dT0,
                                                                  unsigned long long *__restrict__ noroot_count) {
    const int lane = threadIdx.x & 31;
    const long long wid = (long long)blockIdx.x * kWarpsPerCta + (threadIdx.x >> 5);
    const long long nint = (long long)t.n[0] * t.n[1] * t.n[2];
    if (wid >= nint) return;
    const int i = (int)(wid % t.n[0]) + t.ng, j = (int)((wid / t.n[0]) % t.n[1]) + t.ng, k = (int)(wid / ((long long)t.n[0] * t.n[1])) + t.ng;
    const long long c = ((long long)k * t.NJ + j) * t.NI + i;
    const int N = t.N;
    const double *cg = t.cell + c * RAD_NCELL;
    double *Ic = I + c * N;
    const double Tm = fluid[1 * t.ncell + c];
    if (cg[50] != 0.0) {  // excised
        if (lane == 0) {
            if (T_out) T_out[c] = Tm;
            if (dT0) for (int m = 0; m < 4; m++) dT0[m * t.ncell + c] = 0.0;
        }
        return;
    }
    double n1[NITER], n2[NITER], n3[NITER], dom[NITER], Is[NITER], Iold[NITER];
#pragma unroll
    for (int it = 0; it < NITER; it++) {
        const int n = min(it * 32 + lane, N - 1);  // lanes past the last angle redo angle N-1 and do not store
        n1[it] = __ldg(t.nhat + 3 * n); n2[it] = __ldg(t.nhat + 3 * n + 1); n3[it] = __ldg(t.nhat + 3 * n + 2); dom[it] = __ldg(t.domega + n); Is[it] = Ic[n];
        Iold[it] = Is[it];
    }
    CoupleCell cc;
    cc.nup0 = cg[0];
    for (int q = 0; q < 4; q++) cc.E[q] = cg[1 + q];
    for (int q = 0; q < 6; q++) cc.th[q] = cg[44 + q];
    cc.Tm = Tm;
    cc.rho = cc.u1 = cc.u2 = cc.u3 = cc.aP = cc.aEa = cc.aS = 0.0;
    if (p.couple) {
        cc.rho = fluid[c]; cc.u1 = fluid[2 * t.ncell + c]; cc.u2 = fluid[3 * t.ncell + c]; cc.u3 = fluid[4 * t.ncell + c];
        cc.aP = aP_[c]; cc.aEa = aE_[c]; cc.aS = aS_[c];
    }
    double Tp, dR[4];
    bool noroot;
    couple_cell<NITER>(p, cc, dt, lane, N, n1, n2, n3, dom, Is, Tp, dR, noroot);
    if (noroot && lane == 0 && noroot_count) atomicAdd(noroot_count, 1ull);
#pragma unroll
    for (int it = 0; it < NITER; it++) {
        const int n = it * 32 + lane;
        if (n < N && Is[it] != Iold[it]) Ic[n] = Is[it];
    }
    if (lane == 0) {
        if (T_out) T_out[c] = Tp;
        if (dT0) for (int m = 0; m < 4; m++) dT0[m * t.ncell + c] = -dR[m];
    }
}

// generic fallback for angle grids with more than 192 angles: lanes stride over the angles, two sweeps over memory
__global__ void __launch_bounds__(32 * kWarpsPerCta) k_coupling(DeviceTables t, Params p, double *__restrict__ I,
                                                                const double *__restrict__ fluid, const double *__restrict__ aP_,
                                                                const double *__restrict__ aE_, const double *__restrict__ aS_,
                                                                double dt, double *__restrict__ T_out, double *__restrict__ dT0,
                                                                unsigned long long *__restrict__ noroot) {
    const int lane = threadIdx.x & 31;
    const long long wid = (long long)blockIdx.x * kWarpsPerCta + (threadIdx.x >> 5);
    const long long nint = (long long)t.n[0] * t.n[1] * t.n[2];
    if (wid >= nint) return;
    const int i = (int)(wid % t.n[0]) + t.ng, j = (int)((wid / t.n[0]) % t.n[1]) + t.ng, k = (int)(wid / ((long long)t.n[0] * t.n[1])) + t.ng;
    const long long c = ((long long)k * t.NJ + j) * t.NI + i;
    const int N = t.N;
    const double *cg = t.cell + c * RAD_NCELL;
    double *Ic = I + c * N;
    const double Tm = fluid[1 * t.ncell + c];
    if (cg[50] != 0.0) {  // excised
        if (lane == 0) {
            if (T_out) T_out[c] = Tm;
            if (dT0) for (int m = 0; m < 4; m++) dT0[m * t.ncell + c] = 0.0;
        }
        return;
    }
    const double nup0 = cg[0], E0 = cg[1], E1 = cg[2], E2 = cg[3], E3 = cg[4];
    double Tp = Tm;
    double dR[4] = {0.0, 0.0, 0.0, 0.0};
    bool coupled = false;
    double uh[4] = {1.0, 0.0, 0.0, 0.0}, aE = 0.0, src = 0.0;
    if (p.couple) {
        const double rho = fluid[c];
        tetrad_velocity_rec(cg, fluid[2 * t.ncell + c], fluid[3 * t.ncell + c], fluid[4 * t.ncell + c], uh);
        const double aP = aP_[c], aS = aS_[c];
        aE = aE_[c] + aS;  // Eq.33b
        // sweep 1: fluid-frame quantities and the four reductions
        double W = 0.0, A1 = 0.0, A2 = 0.0, Em = 0.0;
        for (int n = lane; n < N; n += 32) {
            const double n1 = __ldg(t.nhat + 3 * n), n2 = __ldg(t.nhat + 3 * n + 1), n3 = __ldg(t.nhat + 3 * n + 2);
            const double nb = uh[0] - (uh[1] * n1 + uh[2] * n2 + uh[3] * n3);  // n^0bar = -u_alpha n^alpha
            const double nb2 = nb * nb;
            const double dOm = __ldg(t.domega + n) / nb2;                       // dOmega_bar (R11)
            const double Ib = nb2 * nb2 * Ic[n];                                // Ibar_- = (n^0bar)^4 Ihat (R11)
            const double rd = 1.0 / fma(nb * aE, dt, nup0);                     // 1/(n^0 + n^0bar alpha_E dt)
            W += dOm;
            A1 = fma(nup0 * rd * Ib, dOm, A1);                                  // Eq.42a
            A2 = fma(nb * rd, dOm, A2);                                         // Eq.42b
            Em = fma(Ib, dOm, Em);                                              // Eq.38
        }
        W = warp_sum(W); A1 = warp_sum(A1); A2 = warp_sum(A2); Em = warp_sum(Em);
        const double scale = p.renorm ? kFourPi / W : 1.0;                      // R12
        A1 *= scale; Em *= scale; A2 *= scale * dt / kFourPi;
        const double Cv = rho / (p.gamma_gas - 1.0);
        const double B4 = A2 * aP * p.a_rad, om = 1.0 - A2 * aS;                // Eq.50
        const double B1 = Cv * om, Bp = A1 - om * Em;
        double dTemp = 0.0;
        if (!quartic_delta(B4, B1, Bp, Tm, dTemp)) {
            if (lane == 0 && noroot) atomicAdd(noroot, 1ull);
        } else {
            coupled = true;
            Tp = Tm + dTemp;
            const double Ep = Em - Cv * dTemp;                                  // Eq.48
            const double T2 = Tp * Tp;
            src = (aP * p.a_rad * T2 * T2 + aS * Ep) * dt / kFourPi;
        }
    }
    // sweep 2: Eq.40, back to the tetrad frame, mask, fluid increment
    for (int n = lane; n < N; n += 32) {
        const double n1 = __ldg(t.nhat + 3 * n), n2 = __ldg(t.nhat + 3 * n + 1), n3 = __ldg(t.nhat + 3 * n + 2);
        const double Iold = Ic[n];
        double Inew = Iold;
        if (coupled) {
            const double nb = uh[0] - (uh[1] * n1 + uh[2] * n2 + uh[3] * n3);
            const double nb2 = nb * nb, nb4 = nb2 * nb2;
            const double rd = 1.0 / fma(nb * aE, dt, nup0);
            Inew = fma(nup0 * nb4, Iold, nb * src) * rd / nb4;                  // Eq.40 then Ihat = Ibar/(n^0bar)^4
            const double w = nup0 * __ldg(t.domega + n) * (Inew - Iold);
            const double n0 = fma(E3, n3, fma(E2, n2, fma(E1, n1, E0)));
            dR[0] = fma(w, n0, dR[0]);
            dR[1] = fma(w, cg[44] * n1, dR[1]);                                  // n_i = theta^a_i n^a
            dR[2] = fma(w, fma(cg[47], n2, cg[45] * n1), dR[2]);
            dR[3] = fma(w, fma(cg[49], n3, fma(cg[48], n2, cg[46] * n1)), dR[3]);
        }
        if (p.n0_crit > 0.0) {
            const double n0 = fma(E3, n3, fma(E2, n2, fma(E1, n1, E0)));       // pinned chain, cell-centre n_0
            if (fabs(n0) < p.n0_crit) Inew = 0.0;
        }
        if (Inew != Iold) Ic[n] = Inew;
    }
    if (dT0) {
#pragma unroll
        for (int m = 0; m < 4; m++) dR[m] = warp_sum(dR[m]);
        if (lane == 0) for (int m = 0; m < 4; m++) dT0[m * t.ncell + c] = -dR[m];
    }
    if (lane == 0 && T_out) T_out[c] = Tp;
}

// ------------------------------------------------------------------------------------------------
// moments
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(32 * kWarpsPerCta) k_moments(DeviceTables t, const double *__restrict__ I, int frame,
                                                               const double *__restrict__ fluid, double *__restrict__ out) {
    const int lane = threadIdx.x & 31;
    const long long wid = (long long)blockIdx.x * kWarpsPerCta + (threadIdx.x >> 5);
    const long long nint = (long long)t.n[0] * t.n[1] * t.n[2];
    if (wid >= nint) return;
    const int i = (int)(wid % t.n[0]) + t.ng, j = (int)((wid / t.n[0]) % t.n[1]) + t.ng, k = (int)(wid / ((long long)t.n[0] * t.n[1])) + t.ng;
    const long long c = ((long long)k * t.NJ + j) * t.NI + i;
    const int N = t.N;
    const double *cg = t.cell + c * RAD_NCELL;
    double acc[10];
#pragma unroll
    for (int q = 0; q < 10; q++) acc[q] = 0.0;
    double uh[4] = {1.0, 0.0, 0.0, 0.0};
    if (frame == 3) tetrad_velocity_rec(cg, fluid[2 * t.ncell + c], fluid[3 * t.ncell + c], fluid[4 * t.ncell + c], uh);
    const double nup0 = cg[0];
    for (int n = lane; n < N; n += 32) {
        const double n1 = __ldg(t.nhat + 3 * n), n2 = __ldg(t.nhat + 3 * n + 1), n3 = __ldg(t.nhat + 3 * n + 2);
        const double w = I[c * N + n] * __ldg(t.domega + n);
        double v[4];
        if (frame == 0) {  // n^mu = e^mu_0 + e^mu_a n^a, e^i_0 = -beta^i / alpha = -beta^i n^0
            v[0] = nup0;
            v[1] = fma(cg[40], n3, fma(cg[39], n2, fma(cg[38], n1, -cg[35] * nup0)));
            v[2] = fma(cg[42], n3, fma(cg[41], n2, -cg[36] * nup0));
            v[3] = fma(cg[43], n3, -cg[37] * nup0);
        } else if (frame == 2) {
            v[0] = 1.0; v[1] = n1; v[2] = n2; v[3] = n3;
        } else if (frame == 3) {  // boost Eq.13-14 (G2: denominator 1 + u^0hat)
            const double un = uh[1] * n1 + uh[2] * n2 + uh[3] * n3;
            const double f = un / (1.0 + uh[0]) - 1.0;
            v[0] = uh[0] - un;
            v[1] = fma(uh[1], f, n1); v[2] = fma(uh[2], f, n2); v[3] = fma(uh[3], f, n3);
        }
        if (frame == 1) {  // R^0_alpha = sum n^0 n_alpha I dOmega
            const double w0 = w * nup0;
            acc[0] = fma(w0, fma(cg[4], n3, fma(cg[3], n2, fma(cg[2], n1, cg[1]))), acc[0]);
            acc[1] = fma(w0, cg[44] * n1, acc[1]);
            acc[2] = fma(w0, fma(cg[47], n2, cg[45] * n1), acc[2]);
            acc[3] = fma(w0, fma(cg[49], n3, fma(cg[48], n2, cg[46] * n1)), acc[3]);
        } else if (frame == 3) {
#pragma unroll
            for (int q = 0; q < 4; q++) acc[q] = fma(w * v[0], v[q], acc[q]);
        } else {
            int q = 0;
#pragma unroll
            for (int a = 0; a < 4; a++)
#pragma unroll
                for (int b = a; b < 4; b++) { acc[q] = fma(w * v[a], v[b], acc[q]); q++; }
        }
    }
    const int ncomp = (frame == 0 || frame == 2) ? 10 : 4;
    for (int q = 0; q < ncomp; q++) {
        const double s = warp_sum(acc[q]);
        if (lane == 0) out[q * t.ncell + c] = s;
    }
}

// sums of ten values over the warp, delivered to every lane: a transposing butterfly (at distance 16, 8, 4, 2 a lane keeps half of
// the values it carries and hands the other half to its partner), 16 + 10 shuffles instead of 50
__device__ __forceinline__ void warp_sum10(double (&m)[10], int lane) {
    const unsigned full = 0xffffffffu;
    double a[16];
#pragma unroll
    for (int q = 0; q < 16; q++) a[q] = q < 10 ? m[q] : 0.0;
    double b[8], c[4], d[2];
    const bool h16 = (lane & 16) != 0, h8 = (lane & 8) != 0, h4 = (lane & 4) != 0, h2 = (lane & 2) != 0;
#pragma unroll
    for (int q = 0; q < 8; q++) b[q] = (h16 ? a[8 + q] : a[q]) + __shfl_xor_sync(full, h16 ? a[q] : a[8 + q], 16);
#pragma unroll
    for (int q = 0; q < 4; q++) c[q] = (h8 ? b[4 + q] : b[q]) + __shfl_xor_sync(full, h8 ? b[q] : b[4 + q], 8);
#pragma unroll
    for (int q = 0; q < 2; q++) d[q] = (h4 ? c[2 + q] : c[q]) + __shfl_xor_sync(full, h4 ? c[q] : c[2 + q], 4);
    double e = (h2 ? d[1] : d[0]) + __shfl_xor_sync(full, h2 ? d[0] : d[1], 2);
    e += __shfl_xor_sync(full, e, 1);  // lanes 2q, 2q+1 hold the sum of value q
#pragma unroll
    for (int q = 0; q < 10; q++) m[q] = __shfl_sync(full, e, 2 * q);
}

// ------------------------------------------------------------------------------------------------
// moments, leaner version: persistent warps, the angle set in registers, one cell per warp iteration.
// By linearity every frame's moments follow from the ten tetrad-frame sums M^{ab} = sum_n I dOmega ntil^a ntil^b,
// ntil = (1, n^1hat, n^2hat, n^3hat): 13 FP64 operations per angle instead of ~35, all loads of a row issued together;
// the per-cell transform (tetrad e^mu_ahat for frame 0, n_alpha rows for frame 1, boost Eq.13-14 for frame 3) is done
// once per cell after the warp reduction.
// ------------------------------------------------------------------------------------------------
template <int NITER>
__global__ void __launch_bounds__(256, 3) k_moments_t(DeviceTables t, const double *__restrict__ I, int frame, const double *__restrict__ fluid,
                                                   double *__restrict__ out) {
    const int lane = threadIdx.x & 31, N = t.N;
    const long long nwarp = (long long)gridDim.x * (blockDim.x >> 5), nint = (long long)t.n[0] * t.n[1] * t.n[2];
    // per-angle table {dOmega, n^1hat, n^2hat, n^3hat} in shared memory (registers are for warps in flight: the kernel is latency bound)
    __shared__ double4 sAng[NITER * 32];
    for (int q = threadIdx.x; q < NITER * 32; q += blockDim.x)
        sAng[q] = q < N ? make_double4(t.domega[q], t.nhat[3 * q], t.nhat[3 * q + 1], t.nhat[3 * q + 2]) : make_double4(0.0, 0.0, 0.0, 0.0);
    __syncthreads();
    for (long long wid = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); wid < nint; wid += nwarp) {
        const int i = (int)(wid % t.n[0]) + t.ng, j = (int)((wid / t.n[0]) % t.n[1]) + t.ng, k = (int)(wid / ((long long)t.n[0] * t.n[1])) + t.ng;
        const long long c = ((long long)k * t.NJ + j) * t.NI + i;
        const double *row = I + c * N;
        double w[NITER];
#pragma unroll
        for (int it = 0; it < NITER; it++) w[it] = row[min(it * 32 + lane, N - 1)];
        double m[10];
#pragma unroll
        for (int q = 0; q < 10; q++) m[q] = 0.0;
#pragma unroll
        for (int it = 0; it < NITER; it++) {
            const double4 an = sAng[it * 32 + lane];  // dOmega = 0 for the idle slots of the last group
            const double w0 = w[it] * an.x, w1 = w0 * an.y, w2 = w0 * an.z, w3 = w0 * an.w;
            m[0] += w0; m[1] += w1; m[2] += w2; m[3] += w3;
            m[4] = fma(w1, an.y, m[4]); m[5] = fma(w1, an.z, m[5]); m[6] = fma(w1, an.w, m[6]);
            m[7] = fma(w2, an.z, m[7]); m[8] = fma(w2, an.w, m[8]); m[9] = fma(w3, an.w, m[9]);
        }
        warp_sum10(m, lane);
        if (lane != 0) continue;
        const double *cg = t.cell + c * RAD_NCELL;
        // full symmetric M[a][b]
        const double M[4][4] = {{m[0], m[1], m[2], m[3]}, {m[1], m[4], m[5], m[6]}, {m[2], m[5], m[7], m[8]}, {m[3], m[6], m[8], m[9]}};
        if (frame == 2) {
#pragma unroll
            for (int q = 0; q < 10; q++) out[q * t.ncell + c] = m[q];
        } else if (frame == 1) {  // R^0_alpha = n^0 sum n_alpha I dOmega; n_0 = E_ahat ntil^ahat, n_i = theta^a_i n^a
            const double nup0 = cg[0];
            out[c] = nup0 * (cg[1] * m[0] + cg[2] * m[1] + cg[3] * m[2] + cg[4] * m[3]);
            out[t.ncell + c] = nup0 * (cg[44] * m[1]);
            out[2 * t.ncell + c] = nup0 * (cg[45] * m[1] + cg[47] * m[2]);
            out[3 * t.ncell + c] = nup0 * (cg[46] * m[1] + cg[48] * m[2] + cg[49] * m[3]);
        } else if (frame == 0) {  // R^{mu nu} = e^mu_a e^nu_b M^{ab}; e^0_0 = n^0, e^i_0 = -beta^i n^0, e^i_a = triad (upper triangular, R2)
            const double nup0 = cg[0];
            const double E[4][4] = {{nup0, 0.0, 0.0, 0.0}, {-cg[35] * nup0, cg[38], cg[39], cg[40]}, {-cg[36] * nup0, 0.0, cg[41], cg[42]}, {-cg[37] * nup0, 0.0, 0.0, cg[43]}};
            double EM[4][4];
#pragma unroll
            for (int mu = 0; mu < 4; mu++)
#pragma unroll
                for (int b = 0; b < 4; b++) EM[mu][b] = E[mu][0] * M[0][b] + E[mu][1] * M[1][b] + E[mu][2] * M[2][b] + E[mu][3] * M[3][b];
            int q = 0;
#pragma unroll
            for (int mu = 0; mu < 4; mu++)
#pragma unroll
                for (int nu = mu; nu < 4; nu++) {
                    out[q * t.ncell + c] = EM[mu][0] * E[nu][0] + EM[mu][1] * E[nu][1] + EM[mu][2] * E[nu][2] + EM[mu][3] * E[nu][3];
                    q++;
                }
        } else {  // fluid frame (Eq.13-14 with G2): nbar^0 = u^0 - u_a n^a, nbar^a = n^a + u^a (u_b n^b / (1 + u^0) - 1)
            double uh[4];
            tetrad_velocity_rec(cg, fluid[2 * t.ncell + c], fluid[3 * t.ncell + c], fluid[4 * t.ncell + c], uh);
            const double r = 1.0 / (1.0 + uh[0]);
            double L[4][4];
            L[0][0] = uh[0]; L[0][1] = -uh[1]; L[0][2] = -uh[2]; L[0][3] = -uh[3];
#pragma unroll
            for (int a = 1; a < 4; a++) {
                L[a][0] = -uh[a];
#pragma unroll
                for (int b = 1; b < 4; b++) L[a][b] = (a == b ? 1.0 : 0.0) + uh[a] * uh[b] * r;
            }
            double LM[4];  // Lambda^0_a M^{ab}
#pragma unroll
            for (int b = 0; b < 4; b++) LM[b] = L[0][0] * M[0][b] + L[0][1] * M[1][b] + L[0][2] * M[2][b] + L[0][3] * M[3][b];
#pragma unroll
            for (int q = 0; q < 4; q++) out[q * t.ncell + c] = LM[0] * L[q][0] + LM[1] * L[q][1] + LM[2] * L[q][2] + LM[3] * L[q][3];
        }
    }
}

}  // namespace

int launch_coupling(const DeviceTables &t, const Params &p, double *I, const double *fluid, const double *aP, const double *aE,
                    const double *aS, double dt, double *T_out, double *dT0, unsigned long long *noroot, cudaStream_t s) {
    const long long nint = (long long)t.n[0] * t.n[1] * t.n[2];
    const long long blocks = (nint + kWarpsPerCta - 1) / kWarpsPerCta;
#define RAD_CPL(NIT) k_coupling_w<NIT><<<(unsigned)blocks, 32 * kWarpsPerCta, 0, s>>>(t, p, I, fluid, aP, aE, aS, dt, T_out, dT0, noroot)
    switch ((t.N + 31) / 32) {
        case 1: RAD_CPL(1); break;
        case 2: RAD_CPL(2); break;
        case 3: RAD_CPL(3); break;
        case 4: RAD_CPL(4); break;
        case 5: RAD_CPL(5); break;
        case 6: RAD_CPL(6); break;
        default: k_coupling<<<(unsigned)blocks, 32 * kWarpsPerCta, 0, s>>>(t, p, I, fluid, aP, aE, aS, dt, T_out, dT0, noroot);
    }
#undef RAD_CPL
    return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

int launch_moments(const DeviceTables &t, const double *I, int frame, const double *fluid, double *out, cudaStream_t s) {
    const long long nint = (long long)t.n[0] * t.n[1] * t.n[2];
    const long long blocks = (nint + kWarpsPerCta - 1) / kWarpsPerCta;
    const int grid = 148 * RAD_MOM_CTAS;
    switch ((t.N + 31) / 32) {
        case 1: k_moments_t<1><<<grid, 256, 0, s>>>(t, I, frame, fluid, out); break;
        case 2: k_moments_t<2><<<grid, 256, 0, s>>>(t, I, frame, fluid, out); break;
        case 3: k_moments_t<3><<<grid, 256, 0, s>>>(t, I, frame, fluid, out); break;
        case 4: k_moments_t<4><<<grid, 256, 0, s>>>(t, I, frame, fluid, out); break;
        case 5: k_moments_t<5><<<grid, 256, 0, s>>>(t, I, frame, fluid, out); break;
        case 6: k_moments_t<6><<<grid, 256, 0, s>>>(t, I, frame, fluid, out); break;
        case 7: k_moments_t<7><<<grid, 256, 0, s>>>(t, I, frame, fluid, out); break;
        case 8: k_moments_t<8><<<grid, 256, 0, s>>>(t, I, frame, fluid, out); break;
        default: k_moments<<<(unsigned)blocks, 32 * kWarpsPerCta, 0, s>>>(t, I, frame, fluid, out);  // N > 256: per-angle version
    }
    return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

}  // namespace rad
