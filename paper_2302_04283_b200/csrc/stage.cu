// stage.cu -- the fused stage kernel: spatial + angular flux divergence (Eq.22, 24, 25), cons -> prim
// and, in the same launch, the locally implicit coupling (section 2.5), the ergosphere mask and the
// fluid increment.
//
// Mapping:
//   * one WARP per cell; a lane holds the angles n = it*32 + lane, it < NITER, whose directions stay in
//     registers for the whole kernel.  Intensities are I[cell][angle], angle innermost, so every load and
//     store of a warp is a run of consecutive doubles.
//   * a warp marches along x through a run of KX cells of one pencil; the flux through the upper x face is
//     carried in registers to the next step.  Warps are independent (no block barrier): while one waits for
//     memory the others compute.  The y and z face fluxes are computed by both cells that share the face,
//     with bitwise identical results (same inputs, same non-contracted products), so the scheme stays
//     conservative to rounding.  The warps of a CTA take neighbouring pencils, so the rows one warp loads as
//     its y/z neighbours are the rows its neighbours load as their own: L1 serves the overlap.
//   * geometry per face and per cell (5 x 8 + 5 doubles) is warp-uniform and read once per cell.
//   * angular fluxes: every unique edge is owned by one of its two angles (edges.cpp).  The owner reads the
//     stored edge coefficient q_e = +-dlambda_e c_e n_0e (one coalesced load; its lowest mantissa bit says which
//     end is upwind), multiplies by the upwind intensity taken from the cell's row in shared memory, and
//     publishes the flux for the partner angle (warp-private shared memory, __syncwarp only).
//   * the warp then holds all N post-transport intensities of its cell in registers, so the coupling's angle
//     reductions are warp shuffles and the intermediate I* never goes to memory.
#include "stage_math.cuh"

#ifndef RAD_PREFETCH
#define RAD_PREFETCH 1
#endif
#if RAD_PREFETCH == 2
#define RAD_PF(p) prefetch_l2(p)
#else
#define RAD_PF(p) prefetch_l1(p)
#endif

namespace rad {
namespace {

#ifndef RAD_TY
#define RAD_TY 4
#define RAD_TZ 3
#endif
constexpr int TY = RAD_TY, TZ = RAD_TZ, NW = TY * TZ;

__device__ __forceinline__ double2 ldg2(const double *p) { return __ldg(reinterpret_cast<const double2 *>(p)); }

struct FaceRec {
    double e0, e1, e2, e3, E0, E1, E2, E3;
};
__device__ __forceinline__ FaceRec load_face(const double *f) {
    const double2 a = ldg2(f), b = ldg2(f + 2), c = ldg2(f + 4), d = ldg2(f + 6);
    return {a.x, a.y, b.x, b.y, c.x, c.y, d.x, d.y};
}

__device__ __forceinline__ FaceRec load_face_s(const double *f) {  // shared memory, warp-uniform address
    const double2 a = *reinterpret_cast<const double2 *>(f), b = *reinterpret_cast<const double2 *>(f + 2),
                  c = *reinterpret_cast<const double2 *>(f + 4), d = *reinterpret_cast<const double2 *>(f + 6);
    return {a.x, a.y, b.x, b.y, c.x, c.y, d.x, d.y};
}

// Upwind flux n^a n_0 I (Eq.24) through the face between cells L and R; qLL, qL, qR, qRR are the
// intensities of the four cells around it.  PLM: van Leer limited slope of the upwind cell (R7): with
// (far, mid, oth) = (LL, L, R) for n^a > 0 and (RR, R, L) otherwise, the face value is mid + dl dr / (dl + dr),
// dl = mid - far, dr = oth - mid (the harmonic mean is odd under reversal, so one formula serves both signs).
// Branch free; the two products are never contracted, so the two cells that share a face get the same bits.
// TAU: optical-depth-aware flux (Eq.26-29; readings R15-R18, G1 in DESIGN.md).  With G_c = -(1 + 1/n^0bar_c) per cell and
// angle and f the interpolating factor of the face, g_L/R = f G_L/R, g = (g_L + g_R)/2, and the factor of Eq.28,
// 1 - g_up + g, is 1 + (f/2) (G_R - G_L) for n^a > 0 and 1 + (f/2) (G_L - G_R) otherwise; fh = f/2.
template <bool PLM, bool TAU>
__device__ __forceinline__ double face_flux(const FaceRec &f, double n1, double n2, double n3, double qLL, double qL, double qR,
                                            double qRR, double GL = 0.0, double GR = 0.0, double fh = 0.0) {
    const double na = chain4(f.e0, f.e1, f.e2, f.e3, n1, n2, n3);
    const double n0 = chain4(f.E0, f.E1, f.E2, f.E3, n1, n2, n3);
    const bool pos = na > 0.0;
    double up = pos ? qL : qR;
    if (PLM) {
        const double far = pos ? qLL : qRR, oth = pos ? qR : qL;
        const double dl = up - far, dr = oth - up, pr = dl * dr;
        const double h = pr * fast_rcp(dl + dr);
        up += pr > 0.0 ? h : 0.0;
    }
    if (TAU) up *= fma(fh, pos ? GR - GL : GL - GR, 1.0);
    return __dmul_rn(__dmul_rn(na, n0), up);  // n^a = 0 gives 0 for finite intensities
}

// G = -(1 + 1/n^0bar) of one cell for one angle; v = {u^0hat, u^1hat, u^2hat, u^3hat} of the cell (Eq.29)
__device__ __forceinline__ double tau_G(const double *v, double n1, double n2, double n3) {
    const double nb = v[0] - (v[1] * n1 + v[2] * n2 + v[3] * n3);
    return -(1.0 + fast_rcp(nb));
}
// f/2 of a face between cells L and R (Eq.26-27): vL, vR = {u^alphahat (4), alpha_E}
__device__ __forceinline__ double tau_fh(const double *vL, const double *vR, double tau_dt) {
    const double tau = tau_dt * (0.5 * (vL[4] + vR[4])) / (0.5 * (vL[0] + vR[0]));
    return -0.5 * expm1(-tau * tau);
}

// v[it] = row[angle of (lane, it)]; lanes past the last angle re-read angle N-1 (last_off)
template <int NITER>
__device__ __forceinline__ void load_row(const double *__restrict__ row, int lane, int last_off, double (&v)[NITER]) {
#pragma unroll
    for (int it = 0; it < NITER - 1; it++) v[it] = __ldg(row + lane + it * 32);
    v[NITER - 1] = __ldg(row + last_off);
}

__device__ __forceinline__ void prefetch_l1(const void *p) { asm volatile("prefetch.global.L1 [%0];" ::"l"(p)); }
__device__ __forceinline__ void prefetch_l2(const void *p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

template <int NITER, bool PLM, bool COUPLE, bool TAU>
__global__ void __launch_bounds__(NW * 32, 1) k_stage(const DeviceTables t, const Params p, const StageArgs a, const int KX) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int N = t.N, Np = (N + 2) & ~1;  // even, > N: slot N of a row is scratch
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int wy = w % TY, wz = w / TY;
    double *sm = reinterpret_cast<double *>(smem_raw);
    double *sI = sm + (size_t)w * 4 * Np;                    // [Np]    this warp's cell, all angles
    double *sG = sI + Np;                                    // [3*N+1] fluxes of owned edges, position j*N + n; [3N] = 0
    double *sU = sm + (size_t)NW * 4 * Np + (size_t)w * 128;  // [128] this cell's warp-uniform records (see below)
    double *sWinv = sm + (size_t)NW * (4 * Np + 128);         // [Np] 1/dOmega
    double *sDom = sWinv + Np;                               // [Np] dOmega
    uint4 *sRec = reinterpret_cast<uint4 *>(sDom + Np);      // [N]  {own_partner[3], pull_pos[3]} as uint16
    for (int q = threadIdx.x; q < N; q += blockDim.x) {
        sWinv[q] = t.winv[q];
        sDom[q] = t.domega[q];
        sRec[q] = reinterpret_cast<const uint4 *>(t.ang_rec)[q];
    }
    if (lane == 0) sG[3 * N] = 0.0;
    __syncthreads();

    const int ng = t.ng;
    const int j = blockIdx.y * TY + wy + ng, k = blockIdx.z * TZ + wz + ng;
    if (j >= t.n[1] + ng || k >= t.n[2] + ng) return;  // no block barrier below
    const int i_begin = blockIdx.x * KX + ng, i_end = min(i_begin + KX, t.n[0] + ng);
    const long long sy = (long long)t.NI * N, sz = (long long)t.NI * t.NJ * N;  // strides in doubles
    const double idx0 = t.inv_dx[0], idx1 = t.inv_dx[1], idx2 = t.inv_dx[2];
    const int last_off = min((NITER - 1) * 32 + lane, N - 1);
    const bool last_valid = (NITER - 1) * 32 + lane < N;

    double n1[NITER], n2[NITER], n3[NITER], carry[NITER];
#pragma unroll
    for (int it = 0; it < NITER; it++) {
        const int nc = it < NITER - 1 ? it * 32 + lane : last_off;
        n1[it] = t.nhat[3 * nc]; n2[it] = t.nhat[3 * nc + 1]; n3[it] = t.nhat[3 * nc + 2];
    }
    {   // flux through the lower x face of the first cell of this run
        const long long c = ((long long)k * t.NJ + j) * t.NI + i_begin;
        const FaceRec f = load_face(t.face + (c * 3 + 0) * RAD_NFACE);
        const double *Ic = a.I_in + c * N;
        double qLL[NITER], qL[NITER], qR[NITER], qRR[NITER];
        load_row<NITER>(Ic - N, lane, last_off, qL); load_row<NITER>(Ic, lane, last_off, qR);
        if (PLM) { load_row<NITER>(Ic - 2 * N, lane, last_off, qLL); load_row<NITER>(Ic + N, lane, last_off, qRR); }
        double vL[5] = {1.0, 0.0, 0.0, 0.0, 0.0}, vR[5] = {1.0, 0.0, 0.0, 0.0, 0.0}, fh = 0.0;
        if (TAU) {
#pragma unroll
            for (int r = 0; r < 5; r++) { vL[r] = __ldg(a.vel + 5 * (c - 1) + r); vR[r] = __ldg(a.vel + 5 * c + r); }
            fh = tau_fh(vL, vR, a.tau_dt);
        }
#pragma unroll
        for (int it = 0; it < NITER; it++)
            carry[it] = face_flux<PLM, TAU>(f, n1[it], n2[it], n3[it], PLM ? qLL[it] : 0.0, qL[it], qR[it], PLM ? qRR[it] : 0.0,
                                            TAU ? tau_G(vL, n1[it], n2[it], n3[it]) : 0.0, TAU ? tau_G(vR, n1[it], n2[it], n3[it]) : 0.0, fh);
    }

    // Warp-uniform records of a cell, gathered two per lane in one round trip and broadcast through shared memory:
    //   sU[0..7] x face above, [8..15] y face below, [16..23] y face above, [24..31] z face below, [32..39] z face above,
    //   [40..44] cell n^0, E_0..E_3, [45] excised flag, [46..51] co-triad, [52..56] rho, T, u1', u2', u3', [57..59] alpha_P, alpha_E, alpha_s
    const double *ptrA, *ptrB;
    int strideB = RAD_NCELL;
    {
        const long long c = ((long long)k * t.NJ + j) * t.NI + i_begin, cz = (long long)t.NI * t.NJ;
        const int g = lane >> 3, r = lane & 7;
        ptrA = t.face + ((g == 0 ? c + 1 : (g == 2 ? c + t.NI : c)) * 3 + (g == 0 ? 0 : (g == 3 ? 2 : 1))) * RAD_NFACE + r;
        ptrB = t.cell + c * RAD_NCELL;  // lanes 28..31: unused
        if (lane < 8) { ptrB = t.face + ((c + cz) * 3 + 2) * RAD_NFACE + lane; strideB = 3 * RAD_NFACE; }
        else if (lane < 13) ptrB += lane - 8;
        else if (lane == 13) ptrB += 50;
        else if (lane < 20) ptrB += 44 + (lane - 14);
        else if (COUPLE && p.couple && lane < 28) {
            ptrB = lane < 25 ? a.fluid + (long long)(lane - 20) * t.ncell + c : (lane == 25 ? a.aP : (lane == 26 ? a.aE : a.aS)) + c;
            strideB = 1;
        } else if (COUPLE && lane == 21) { ptrB = a.fluid + t.ncell + c; strideB = 1; }  // T_- is reported even when not coupling
    }

    for (int i = i_begin; i < i_end; i++) {
        const long long c = ((long long)k * t.NJ + j) * t.NI + i;
        const double *Ic = a.I_in + c * N;
        const long long cint = ((long long)(k - ng) * t.n[1] + (j - ng)) * t.n[0] + (i - ng);
        double div[NITER], Iown[NITER];
#if RAD_PREFETCH
        if (i + 1 < i_end) {  // pull the next step's rows towards the SM while this step computes
            const double *In = Ic + N;
            const int lines = (N * 8 + 127) / 128 + 1;
            if (lane < lines) {
                const long long lo = lane * 16;
                RAD_PF(In + 2 * N + lo);
                RAD_PF(In - sy + lo); RAD_PF(In + sy + lo); RAD_PF(In - sz + lo); RAD_PF(In + sz + lo);
                if (PLM) { RAD_PF(In - 2 * sy + lo); RAD_PF(In + 2 * sy + lo); RAD_PF(In - 2 * sz + lo); RAD_PF(In + 2 * sz + lo); }
            }
            const double *kn = t.ke + (cint + 1) * 3 * N;
            if (lane * 16 < 3 * N) RAD_PF(kn + lane * 16);
        }
#endif
        // ---- angular fluxes (Eq.25, donor cell in angle)
        {
            const double *kec = t.ke + cint * 3 * N;
            double q0[NITER], q1[NITER], q2[NITER];
            const double uA = __ldg(ptrA), uB = __ldg(ptrB);
            ptrA += 3 * RAD_NFACE; ptrB += strideB;
            double uV = 0.0;  // TAU: {u^alphahat, alpha_E} of this cell and its +x, -y, +y, -z, +z neighbours, one double per lane
            if (TAU && lane < 30) {
                const int q = lane / 5;
                const long long cq = c + (q == 1 ? 1 : (q == 2 ? -(long long)t.NI : (q == 3 ? (long long)t.NI : (q == 4 ? -(long long)t.NI * t.NJ : (q == 5 ? (long long)t.NI * t.NJ : 0)))));
                uV = __ldg(a.vel + 5 * cq + (lane - 5 * q));
            }
            load_row<NITER>(Ic, lane, last_off, Iown);
            load_row<NITER>(kec, lane, last_off, q0); load_row<NITER>(kec + N, lane, last_off, q1); load_row<NITER>(kec + 2 * N, lane, last_off, q2);
            __syncwarp();  // the previous step's readers of sI / sG / sU are done
            sU[lane] = uA; sU[32 + lane] = uB;
            if (TAU) sU[64 + lane] = uV;
#pragma unroll
            for (int it = 0; it < NITER; it++)
                if (it < NITER - 1 || last_valid) sI[it * 32 + lane] = Iown[it];
            __syncwarp();
            if (TAU) {  // f/2 of the five faces computed below: x above (0,1), y below (2,0), y above (0,3), z below (4,0), z above (0,5)
                if (lane < 5) {
                    const int L = lane == 1 ? 2 : (lane == 3 ? 4 : 0), R = lane == 0 ? 1 : (lane == 2 ? 3 : (lane == 4 ? 5 : 0));
                    sU[96 + lane] = tau_fh(sU + 64 + 5 * L, sU + 64 + 5 * R, a.tau_dt);
                }
                __syncwarp();
            }
#pragma unroll
            for (int it = 0; it < NITER; it++) {
                const int n = it < NITER - 1 ? it * 32 + lane : last_off;
                const uint4 rec = sRec[n];
                const unsigned pj[3] = {rec.x & 0xffffu, rec.x >> 16, rec.y & 0xffffu};
                const double qq[3] = {q0[it], q1[it], q2[it]};
                double asum = 0.0;
#pragma unroll
                for (int jj = 0; jj < 3; jj++) {  // unused slots have q = 0
                    const bool owner_up = (__double2loint(qq[jj]) & 1) != 0;
                    const double G = qq[jj] * sI[owner_up ? (unsigned)n : pj[jj]];
                    asum += G;
                    if (it < NITER - 1 || last_valid) sG[jj * N + n] = G;
                }
                div[it] = asum;
            }
            __syncwarp();
#pragma unroll
            for (int it = 0; it < NITER; it++) {
                const int n = it < NITER - 1 ? it * 32 + lane : last_off;
                const uint4 rec = sRec[n];
                const double asum = div[it] - ((sG[rec.y >> 16] + sG[rec.z & 0xffffu]) + sG[rec.z >> 16]);  // unused -> sG[3N] = 0
                div[it] = asum * sWinv[n];
            }
        }
        double G0[NITER];  // TAU: G of this cell per angle
#pragma unroll
        for (int it = 0; it < NITER; it++) G0[it] = TAU ? tau_G(sU + 64, n1[it], n2[it], n3[it]) : 0.0;
        // ---- x: flux through the upper face (the lower x face of cell i+1); the lower one is carried
        {
            const FaceRec f = load_face_s(sU);
            double qLL[NITER], qR[NITER], qRR[NITER];
            load_row<NITER>(Ic + N, lane, last_off, qR);
            if (PLM) { load_row<NITER>(Ic - N, lane, last_off, qLL); load_row<NITER>(Ic + 2 * N, lane, last_off, qRR); }
#pragma unroll
            for (int it = 0; it < NITER; it++) {
                const double F = face_flux<PLM, TAU>(f, n1[it], n2[it], n3[it], PLM ? qLL[it] : 0.0, Iown[it], qR[it], PLM ? qRR[it] : 0.0, G0[it],
                                                     TAU ? tau_G(sU + 69, n1[it], n2[it], n3[it]) : 0.0, TAU ? sU[96] : 0.0);
                div[it] = fma(F - carry[it], idx0, div[it]);
                carry[it] = F;
            }
        }
        // ---- y and z: both faces (rows -2, -1, +1, +2 serve the two of them)
#pragma unroll
        for (int ax = 1; ax <= 2; ax++) {
            const long long st = ax == 1 ? sy : sz;
            const double idx = ax == 1 ? idx1 : idx2;
            const FaceRec flo = load_face_s(sU + (ax == 1 ? 8 : 24)), fhi = load_face_s(sU + (ax == 1 ? 16 : 32));
            double m2[NITER], m1[NITER], p1[NITER], p2[NITER];
            load_row<NITER>(Ic - st, lane, last_off, m1); load_row<NITER>(Ic + st, lane, last_off, p1);
            if (PLM) { load_row<NITER>(Ic - 2 * st, lane, last_off, m2); load_row<NITER>(Ic + 2 * st, lane, last_off, p2); }
#pragma unroll
            for (int it = 0; it < NITER; it++) {
                const double Glo = TAU ? tau_G(sU + (ax == 1 ? 74 : 84), n1[it], n2[it], n3[it]) : 0.0, Ghi = TAU ? tau_G(sU + (ax == 1 ? 79 : 89), n1[it], n2[it], n3[it]) : 0.0;
                const double Flo = face_flux<PLM, TAU>(flo, n1[it], n2[it], n3[it], PLM ? m2[it] : 0.0, m1[it], Iown[it], p1[it], Glo, G0[it], TAU ? sU[ax == 1 ? 97 : 99] : 0.0);
                const double Fhi = face_flux<PLM, TAU>(fhi, n1[it], n2[it], n3[it], m1[it], Iown[it], p1[it], PLM ? p2[it] : 0.0, G0[it], Ghi, TAU ? sU[ax == 1 ? 98 : 100] : 0.0);
                div[it] = fma(Fhi - Flo, idx, div[it]);
            }
        }
        // ---- flux-divergence update of C = n^0 n_0 I (Eq.22, stage form R8) and cons -> prim
        const double2 c01 = *reinterpret_cast<const double2 *>(sU + 40), c23 = *reinterpret_cast<const double2 *>(sU + 42),
                      c45 = *reinterpret_cast<const double2 *>(sU + 44);
        const double nup0 = c01.x, E0 = c01.y, E1 = c23.x, E2 = c23.y, E3 = c45.x;
        const bool excised = c45.y != 0.0;
        double Is[NITER];
        {
            double I0v[NITER];
            if (a.I0 != nullptr) load_row<NITER>(a.I0 + c * N, lane, last_off, I0v);
#pragma unroll
            for (int it = 0; it < NITER; it++) {
                const double wgt = nup0 * chain4(E0, E1, E2, E3, n1[it], n2[it], n3[it]);  // n^0 n_0
                double v = a.gam1 * Iown[it];
                if (a.I0 != nullptr) v = fma(a.gam0, I0v[it], v);
                v = fma(-a.beta_dt * div[it], fast_rcp(wgt), v);
                Is[it] = excised ? 0.0 : v;
            }
        }
        if (COUPLE) {
            CoupleCell cc;
            cc.nup0 = nup0; cc.E[0] = E0; cc.E[1] = E1; cc.E[2] = E2; cc.E[3] = E3;
            const double2 t0 = *reinterpret_cast<const double2 *>(sU + 46), t1 = *reinterpret_cast<const double2 *>(sU + 48),
                          t2 = *reinterpret_cast<const double2 *>(sU + 50), f0 = *reinterpret_cast<const double2 *>(sU + 52),
                          f1 = *reinterpret_cast<const double2 *>(sU + 54), f2 = *reinterpret_cast<const double2 *>(sU + 56),
                          f3 = *reinterpret_cast<const double2 *>(sU + 58);
            cc.th[0] = t0.x; cc.th[1] = t0.y; cc.th[2] = t1.x; cc.th[3] = t1.y; cc.th[4] = t2.x; cc.th[5] = t2.y;
            cc.rho = f0.x; cc.Tm = f0.y; cc.u1 = f1.x; cc.u2 = f1.y; cc.u3 = f2.x; cc.aP = f2.y; cc.aEa = f3.x; cc.aS = f3.y;
            double dom[NITER];
#pragma unroll
            for (int it = 0; it < NITER; it++) dom[it] = sDom[it < NITER - 1 ? it * 32 + lane : last_off];
            double Tp, dR[4];
            bool noroot;
            couple_cell<NITER>(p, cc, a.beta_dt, lane, N, n1, n2, n3, dom, Is, Tp, dR, noroot, !excised);
            if (lane == 0) {
                if (noroot && a.noroot) atomicAdd(a.noroot, 1ull);
                if (a.T_out) a.T_out[c] = Tp;
                if (a.dT0) {
#pragma unroll
                    for (int m = 0; m < 4; m++) a.dT0[m * t.ncell + c] = -dR[m];
                }
            }
        }
        double *out = a.I_out + c * N;
#pragma unroll
        for (int it = 0; it < NITER; it++)
            if (it < NITER - 1 || last_valid) out[it * 32 + lane] = Is[it];
    }
}

// ------------------------------------------------------------------------------------------------
// stored edge coefficients: q[cell][j][n] = s * dlambda_e * (c_e * n_0e) for the edge e that angle n owns in slot
// j (s = +1 if n is the edge's lower angle, else -1, so that q I_up is the flux LEAVING n), lowest mantissa bit
// = 1 if n is the upwind end.  c_e by the pinned 30-term chain (the one RAD_TAB_EDGE_SIGN reports).
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_build_ke(const DeviceTables t, double *__restrict__ ke) {
    const long long nint = (long long)t.n[0] * t.n[1] * t.n[2];
    const long long total = nint * 3 * t.N;
    for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < total; idx += (long long)gridDim.x * blockDim.x) {
        const int n = (int)(idx % t.N);
        const int jj = (int)((idx / t.N) % 3);
        const long long cint = idx / (3 * t.N);
        const int i = (int)(cint % t.n[0]) + t.ng, j = (int)((cint / t.n[0]) % t.n[1]) + t.ng, k = (int)(cint / ((long long)t.n[0] * t.n[1])) + t.ng;
        const long long c = ((long long)k * t.NJ + j) * t.NI + i;
        const int e = t.own_edge[n * 3 + jj];
        double q = 0.0;
        if (e >= 0) {
            const double *S = t.cell + c * RAD_NCELL + 5, *T = t.edge_T + (long long)e * 30;
            double acc = 0.0;
#pragma unroll
            for (int m = 0; m < 30; m++) acc = fma(S[m], T[m], acc);  // pinned 30-term chain
            const double ce = -acc;
            const double *cg = t.cell + c * RAD_NCELL;
            const double n0e = chain4(cg[1], cg[2], cg[3], cg[4], t.edge_mid[3 * e], t.edge_mid[3 * e + 1], t.edge_mid[3 * e + 2]);
            const bool owner_is_lo = t.edge_lo[e] == n;
            if (ce != 0.0) {
                q = (owner_is_lo ? t.edge_len[e] : -t.edge_len[e]) * (ce * n0e);
                const bool owner_up = (ce > 0.0) == owner_is_lo;
                long long bits = __double_as_longlong(q);
                bits = (bits & ~1ll) | (owner_up ? 1ll : 0ll);
                q = __longlong_as_double(bits);
            }
        }
        ke[idx] = q;
    }
}

size_t stage_smem_bytes(int N) {
    const int Np = (N + 2) & ~1;
    return sizeof(double) * ((size_t)NW * (4 * Np + 128) + 2 * (size_t)Np) + sizeof(uint4) * (size_t)N;
}

template <int NITER>
int launch_niter(const DeviceTables &t, const Params &p, const StageArgs &a, bool couple, dim3 grid, size_t smem, int KX, cudaStream_t s) {
#define RAD_LAUNCH(PLM, CPL)                                                                                         \
    do {                                                                                                             \
        if (a.vel != nullptr) {                                                                                      \
            if (cudaFuncSetAttribute(k_stage<NITER, PLM, CPL, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return -1; \
            k_stage<NITER, PLM, CPL, true><<<grid, NW * 32, smem, s>>>(t, p, a, KX);                                   \
        } else {                                                                                                     \
            if (cudaFuncSetAttribute(k_stage<NITER, PLM, CPL, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return -1; \
            k_stage<NITER, PLM, CPL, false><<<grid, NW * 32, smem, s>>>(t, p, a, KX);                                  \
        }                                                                                                            \
    } while (0)
    if (p.recon_space == 1) { if (couple) RAD_LAUNCH(true, true); else RAD_LAUNCH(true, false); }
    else { if (couple) RAD_LAUNCH(false, true); else RAD_LAUNCH(false, false); }
#undef RAD_LAUNCH
    return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

}  // namespace

int launch_stage_fused(const DeviceTables &t, const Params &p, const StageArgs &a, bool couple, cudaStream_t s) {
    if (!t.fused_ok || t.ke == nullptr) return 0;
    const int niter = (t.N + 31) / 32;
    if (niter > 6) return 0;
    const size_t smem = stage_smem_bytes(t.N);
    if (smem > 227 * 1024) return 0;
    // run length along x: long runs amortise the first face of a run, short runs fill the SMs of small grids
    const long long tiles = (long long)((t.n[1] + TY - 1) / TY) * ((t.n[2] + TZ - 1) / TZ);
    int KX = 64;
    while (KX > 8 && tiles * ((t.n[0] + KX - 1) / KX) < 2 * 148) KX /= 2;
    dim3 grid((t.n[0] + KX - 1) / KX, (t.n[1] + TY - 1) / TY, (t.n[2] + TZ - 1) / TZ);
    if (grid.y > 65535 || grid.z > 65535) return 0;
    switch (niter) {
        case 1: return launch_niter<1>(t, p, a, couple, grid, smem, KX, s);
        case 2: return launch_niter<2>(t, p, a, couple, grid, smem, KX, s);
        case 3: return launch_niter<3>(t, p, a, couple, grid, smem, KX, s);
        case 4: return launch_niter<4>(t, p, a, couple, grid, smem, KX, s);
        case 5: return launch_niter<5>(t, p, a, couple, grid, smem, KX, s);
        default: return launch_niter<6>(t, p, a, couple, grid, smem, KX, s);
    }
}

int launch_build_ke(const DeviceTables &t, double *ke, cudaStream_t s) {
    k_build_ke<<<148 * 8, 256, 0, s>>>(t, ke);
    return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

}  // namespace rad
