// coupling.cu -- subsystem 3: locally implicit matter-radiation coupling (paper section 2.5),
// the ergosphere mask and the angular moments (Eq.45, Eq.38).
//
// Generic kernels for any angle grid (odd N, N > 256); stream.cu holds the streaming versions that serve the rest.
// One warp per cell.  Lanes stride over the angles; the angle reductions that form A_1, A_2 (Eq.42),
// Ebar_- (Eq.38) and the fluid-frame weight normalisation W (R12) are warp-shuffle trees; the quartic
// Eq.49 for T_+ is solved redundantly by every lane in registers; a second sweep applies Eq.40, transforms
// back to the tetrad frame, masks |n_0| < n_0^crit and accumulates the fluid increment
// dT^0_alpha = -sum_n n^0 n_alpha (I_+ - I*) dOmega_n with a second shuffle tree.
#include "stage_math.cuh"

namespace rad {
namespace {

constexpr int kWarpsPerCta = 12;

// legacy signature of tetrad_velocity on a cell record
__device__ __forceinline__ void tetrad_velocity_rec(const double *cg, double u1, double u2, double u3, double uh[4]) {
    const double th[6] = {cg[44], cg[45], cg[46], cg[47], cg[48], cg[49]};
    rad::tetrad_velocity(th, u1, u2, u3, uh);
}

// ------------------------------------------------------------------------------------------------
// coupling, generic version for any angle grid (the streaming kernel of stream.cu serves even N that fit shared memory):
// one warp per cell, lanes stride over the angles, two sweeps over memory
// ------------------------------------------------------------------------------------------------
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

}  // namespace

int launch_coupling(const DeviceTables &t, const Params &p, double *I, const double *fluid, const double *aP, const double *aE,
                    const double *aS, double dt, double *T_out, double *dT0, unsigned long long *noroot, cudaStream_t s) {
    const long long nint = (long long)t.n[0] * t.n[1] * t.n[2];
    const long long blocks = (nint + kWarpsPerCta - 1) / kWarpsPerCta;
    k_coupling<<<(unsigned)blocks, 32 * kWarpsPerCta, 0, s>>>(t, p, I, fluid, aP, aE, aS, dt, T_out, dT0, noroot);
    return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

int launch_moments(const DeviceTables &t, const double *I, int frame, const double *fluid, double *out, cudaStream_t s) {
    const long long nint = (long long)t.n[0] * t.n[1] * t.n[2];
    const long long blocks = (nint + kWarpsPerCta - 1) / kWarpsPerCta;
    k_moments<<<(unsigned)blocks, 32 * kWarpsPerCta, 0, s>>>(t, I, frame, fluid, out);
    return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

}  // namespace rad
