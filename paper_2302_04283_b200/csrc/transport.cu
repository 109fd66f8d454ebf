// transport.cu -- subsystems 2 and 4: fused spatial+angular flux-divergence kernel and ghost fill.
//
// Paper: section 2.3-2.4.  Eq.24 spatial upwind flux, Eq.25 angular upwind flux, Eq.22 update
// of C = n^0 n_0 I, then I* = C*/(n^0 n_0).  Intensities are I[cell][angle], angle innermost.
#include <math.h>
#include <stdint.h>

#include "rad_internal.h"

namespace rad {
namespace {

// ------------------------------------------------------------------------------------------------
// ghost fill: one launch per axis, in x, y, z order so that edges and corners are filled
// ------------------------------------------------------------------------------------------------
// bc: 0 caller-filled, 1 periodic, 2 outflow, 3 reflecting wall: mirror cell across the wall, direction with the wall-normal tetrad
// component flipped (R20); mirror[N] = that angle permutation for this axis
__global__ void k_fill_ghosts(double *__restrict__ I, int N, int NI, int NJ, int NK, int ng, int axis, int nint, int bc_lo, int bc_hi, int vec2,
                              const int *__restrict__ mirror) {
    // one CTA per ghost cell of this axis' two slabs; threads over angles
    const int dims[3] = {NI, NJ, NK};
    int d[3];
    // enumerate ghost cells: along `axis` 2*ng layers, full extent in the other two
    int ext[3] = {NI, NJ, NK};
    ext[axis] = 2 * ng;
    long long b = blockIdx.x;
    d[0] = (int)(b % ext[0]); b /= ext[0];
    d[1] = (int)(b % ext[1]); b /= ext[1];
    d[2] = (int)b;
    int q = d[axis];
    const bool low = q < ng;
    if (!low) q = dims[axis] - 2 * ng + q;  // upper slab
    d[axis] = q;
    const int bc = low ? bc_lo : bc_hi;
    if (bc == 0) return;
    int src = q;
    if (bc == 1) src = ng + (((q - ng) % nint) + nint) % nint;
    else if (bc == 3) src = low ? 2 * ng - 1 - q : 2 * (dims[axis] - ng) - 1 - q;
    else src = low ? ng : ng + nint - 1;
    int s[3] = {d[0], d[1], d[2]};
    s[axis] = src;
    const long long cd = ((long long)d[2] * NJ + d[1]) * NI + d[0], cs = ((long long)s[2] * NJ + s[1]) * NI + s[0];
    const double2 *ps = reinterpret_cast<const double2 *>(I + cs * N);
    double2 *pd = reinterpret_cast<double2 *>(I + cd * N);
    if (bc == 3) {
        for (int n = threadIdx.x; n < N; n += blockDim.x) I[cd * N + n] = I[cs * N + mirror[n]];
    } else if (vec2) {  // rows are 16-byte aligned: N even and the array itself aligned
        for (int n = threadIdx.x; n < N / 2; n += blockDim.x) pd[n] = ps[n];
    } else {
        for (int n = threadIdx.x; n < N; n += blockDim.x) I[cd * N + n] = I[cs * N + n];
    }
}

// ------------------------------------------------------------------------------------------------
// halo copy between two blocks that touch along `axis` (the communication task of a stage, on one device): nlayers
// layers of `src` starting at index src_first along the axis go to the layers of `dst` starting at dst_first; the other two
// extents (ghosts included) are the same in both blocks.  One CTA per cell, threads over angles.
// ------------------------------------------------------------------------------------------------
__global__ void k_copy_halo(const double *__restrict__ src, double *__restrict__ dst, int N, int e0, int e1, int e2, int axis, int src_first, int dst_first,
                            int src_ext, int dst_ext, int vec2) {
    int d[3];
    long long b = blockIdx.x;
    d[0] = (int)(b % e0); b /= e0;
    d[1] = (int)(b % e1); b /= e1;
    d[2] = (int)b;
    int sdim[3] = {e0, e1, e2}, ddim[3] = {e0, e1, e2}, sidx[3] = {d[0], d[1], d[2]}, didx[3] = {d[0], d[1], d[2]};
    sdim[axis] = src_ext; ddim[axis] = dst_ext;
    sidx[axis] = src_first + d[axis]; didx[axis] = dst_first + d[axis];
    const long long cs = ((long long)sidx[2] * sdim[1] + sidx[1]) * sdim[0] + sidx[0], cd = ((long long)didx[2] * ddim[1] + didx[1]) * ddim[0] + didx[0];
    if (vec2) {
        const double2 *ps = reinterpret_cast<const double2 *>(src + cs * N);
        double2 *pd = reinterpret_cast<double2 *>(dst + cd * N);
        for (int n = threadIdx.x; n < N / 2; n += blockDim.x) pd[n] = ps[n];
    } else {
        for (int n = threadIdx.x; n < N; n += blockDim.x) dst[cd * N + n] = src[cs * N + n];
    }
}

// ------------------------------------------------------------------------------------------------
// fused flux divergence, version 1: one CTA per run of CX cells along x
// ------------------------------------------------------------------------------------------------
constexpr int CX = 8;

__device__ __forceinline__ double chain4(const double *r, double n1, double n2, double n3) {
    // pinned order (decides upwind signs): fma(r3,n3, fma(r2,n2, fma(r1,n1, r0)))
    return fma(r[3], n3, fma(r[2], n2, fma(r[1], n1, r[0])));
}

__device__ __forceinline__ double vl_slope(double qm, double q0, double qp) {
    // van Leer harmonic-mean limiter (R7)
    const double dl = q0 - qm, dr = qp - q0, pr = dl * dr;
    return pr > 0.0 ? 2.0 * pr / (dl + dr) : 0.0;
}

// PPM (Colella & Woodward 1984) on uniform spacing, no characteristic tracing: the monotonised parabola of the cell with
// values q[-2..2] around it (p points at the cell, stride st); returns its value at the upper (upper = true) or lower face.
// CW84 Eq.1.6-1.8 (interface values from van Leer-limited average slopes), Eq.1.10 (monotonisation).
__device__ __forceinline__ double ppm_dq(double qm, double q0, double qp) {
    const double dl = q0 - qm, dr = qp - q0;
    if (dl * dr <= 0.0) return 0.0;
    const double d = 0.5 * (qp - qm), lim = fmin(2.0 * fabs(dl), 2.0 * fabs(dr));
    return (d > 0.0 ? 1.0 : -1.0) * fmin(fabs(d), lim);
}
__device__ __forceinline__ double ppm_face(const double *__restrict__ p, long long st, bool upper) {
    const double q0 = p[-2 * st], q1 = p[-st], q2 = p[0], q3 = p[st], q4 = p[2 * st];
    const double dqm = ppm_dq(q0, q1, q2), dq0 = ppm_dq(q1, q2, q3), dqp = ppm_dq(q2, q3, q4);
    double qm = q1 + 0.5 * (q2 - q1) - (dq0 - dqm) / 6.0;
    double qp = q2 + 0.5 * (q3 - q2) - (dqp - dq0) / 6.0;
    if ((qp - q2) * (q2 - qm) <= 0.0) { qm = q2; qp = q2; }
    else {
        const double dq = qp - qm, q6 = 6.0 * (q2 - 0.5 * (qm + qp));
        if (dq * q6 > dq * dq) qm = 3.0 * q2 - 2.0 * qp;
        else if (-dq * dq > dq * q6) qp = 3.0 * q2 - 2.0 * qm;
    }
    return upper ? qp : qm;
}

// flux through the face whose record is `f`, between cells L (lower) and R (upper) along a stride `st`.
// RECON: 0 donor cell, 1 PLM (van Leer, R7), 2 PPM.
// TAU: the optical-depth-aware flux of Eq.26-29 (readings R15-R18, G1 in DESIGN.md): vL, vR = {u^alphahat (4),
// alpha_E} of the two cells, tau = tau_dt (alpha_E,L + alpha_E,R)/2 / ((u^0hat_L + u^0hat_R)/2), f = -expm1(-tau^2),
// g_L/R = -f (1 + 1/n^0bar_L/R), g = (g_L + g_R)/2, the upwind intensity is multiplied by 1 - g_up + g.
template <int RECON, bool TAU>
__device__ __forceinline__ double face_flux(const double *f, double n1, double n2, double n3, const double *__restrict__ pR, long long st,
                                            const double *__restrict__ vL, const double *__restrict__ vR, double tau_dt) {
    const double na = chain4(f, n1, n2, n3), n0 = chain4(f + 4, n1, n2, n3);
    double up;
    if (na > 0.0) {
        const double qL = pR[-st];
        up = qL;
        if (RECON == 1) up = qL + 0.5 * vl_slope(pR[-2 * st], qL, pR[0]);
        if (RECON == 2) up = ppm_face(pR - st, st, true);
    } else if (na < 0.0) {
        const double qR = pR[0];
        up = qR;
        if (RECON == 1) up = qR - 0.5 * vl_slope(pR[-st], qR, pR[st]);
        if (RECON == 2) up = ppm_face(pR, st, false);
    } else {
        return 0.0;
    }
    if (TAU) {
        const double aE = 0.5 * (vL[4] + vR[4]), v0 = 0.5 * (vL[0] + vR[0]);
        const double tau = tau_dt * aE / v0;                                         // Eq.26
        const double fint = -expm1(-tau * tau);                                      // Eq.27 (G1)
        const double nbL = vL[0] - (vL[1] * n1 + vL[2] * n2 + vL[3] * n3);           // n^0bar_L
        const double nbR = vR[0] - (vR[1] * n1 + vR[2] * n2 + vR[3] * n3);
        const double gL = -fint * (1.0 + 1.0 / nbL), gR = -fint * (1.0 + 1.0 / nbR);  // Eq.29
        const double g = 0.5 * (gL + gR);
        up *= (na > 0.0) ? (1.0 - gL + g) : (1.0 - gR + g);                          // Eq.28
    }
    return na * n0 * up;
}

// tetrad-frame fluid velocity and alpha_E of EVERY cell (ghosts included), vel[cell][5], for the optical-depth-aware flux:
// u^ahat = theta^ahat_j u^j' (co-triad of the cell record), u^0hat = sqrt(1 + |u^ahat|^2) (R10), alpha_E = alpha^a_E + alpha^s
__global__ void __launch_bounds__(256) k_cell_velocity(DeviceTables t, const double *__restrict__ fluid, const double *__restrict__ aE,
                                                       const double *__restrict__ aS, double *__restrict__ vel) {
    for (long long c = blockIdx.x * (long long)blockDim.x + threadIdx.x; c < t.ncell; c += (long long)gridDim.x * blockDim.x) {
        const double *th = t.cell + c * RAD_NCELL + 44;
        const double u1 = fluid[2 * t.ncell + c], u2 = fluid[3 * t.ncell + c], u3 = fluid[4 * t.ncell + c];
        const double h1 = th[0] * u1 + th[1] * u2 + th[2] * u3, h2 = th[3] * u2 + th[4] * u3, h3 = th[5] * u3;
        vel[5 * c] = sqrt(1.0 + (h1 * h1 + h2 * h2 + h3 * h3));
        vel[5 * c + 1] = h1; vel[5 * c + 2] = h2; vel[5 * c + 3] = h3;
        vel[5 * c + 4] = aE[c] + aS[c];
    }
}

// R21: van Leer PLM in index space on the latitude-longitude grid for the edge value of the upwind angle a_up; beyond a pole
// the row of cell (l, m) continues in cell (l, m + N_psi / 2); periodic in psi.  slot of this edge in the upwind cell: 0 zeta-, 1 zeta+,
// 2 psi-, 3 psi+
__device__ __noinline__ double plm_angle(const int *__restrict__ nbr_edge, int np, int nzeta, const double *__restrict__ row, int a_up, int e, double Iup) {
    int slot = 0;
    while (__ldg(nbr_edge + a_up * RAD_MAXNBR + slot) != e) slot++;
    const int l = a_up / np, m = a_up - l * np;
    int lo, hi;
    if (slot < 2) {
        const int across = l * np + (m + np / 2) % np;
        lo = l > 0 ? a_up - np : across;
        hi = l + 1 < nzeta ? a_up + np : across;
    } else {
        lo = l * np + (m + np - 1) % np;
        hi = l * np + (m + 1) % np;
    }
    const double sl = vl_slope(row[lo], Iup, row[hi]);
    return (slot & 1) ? Iup + 0.5 * sl : Iup - 0.5 * sl;
}

template <int RECON, bool TAU>
__global__ void __launch_bounds__(256, 4) k_fluxdiv(DeviceTables t, const double *__restrict__ I_in, const double *__restrict__ I0,
                                                   double gam0, double gam1, double beta_dt, double *__restrict__ I_out,
                                                   const double *__restrict__ vel, double tau_dt) {
    extern __shared__ double smem[];
    const int N = t.N, E = t.E;
    double *sCell = smem;                 // [CX][36]: n^0, E[4], S[30], excised
    double *sFx = sCell + CX * 36;        // [CX+1][8]  lower x-face of cells i0..i0+CX
    double *sFy = sFx + (CX + 1) * 8;     // [2][CX][8] lower y-face of (j) and (j+1)
    double *sFz = sFy + 2 * CX * 8;       // [2][CX][8]
    double *sFe = sFz + 2 * CX * 8;       // [CX][E]   dlambda_e * c_e * n_0e * I_up

    const int nxb = (t.n[0] + CX - 1) / CX;
    long long b = blockIdx.x;
    const int ib = (int)(b % nxb); b /= nxb;
    const int j = (int)(b % t.n[1]) + t.ng;
    const int k = (int)(b / t.n[1]) + t.ng;
    const int i0 = ib * CX + t.ng;
    const int ncx = min(CX, t.n[0] + t.ng - i0);
    const long long sy = t.NI, sz = (long long)t.NI * t.NJ;
    const long long c0 = ((long long)k * t.NJ + j) * t.NI + i0;

    for (int q = threadIdx.x; q < ncx * 36; q += blockDim.x) {
        const int cl = q / 36, w = q % 36;
        sCell[q] = (w < 35) ? t.cell[(c0 + cl) * RAD_NCELL + w] : t.cell[(c0 + cl) * RAD_NCELL + 50];
    }
    for (int q = threadIdx.x; q < (ncx + 1) * 8; q += blockDim.x) sFx[q] = t.face[((c0 + q / 8) * 3 + 0) * RAD_NFACE + q % 8];
    for (int q = threadIdx.x; q < 2 * ncx * 8; q += blockDim.x) {
        const int up = q / (ncx * 8), r = q % (ncx * 8);
        sFy[up * CX * 8 + r] = t.face[((c0 + r / 8 + up * sy) * 3 + 1) * RAD_NFACE + r % 8];
        sFz[up * CX * 8 + r] = t.face[((c0 + r / 8 + up * sz) * 3 + 2) * RAD_NFACE + r % 8];
    }
    __syncthreads();

    // phase A: angular fluxes, once per unique edge (Eq.25, donor cell in angle).  A thread takes an edge for all cells of the run:
    // the edge's 30 products N^c (n^a n^b), its midpoint direction, length and end angles are loaded once and stay in registers
    // (they were fetched per cell before: 90 loads per intensity update through L1, the kernel's bottleneck); the cell's S comes
    // from shared memory as a broadcast.  The 30-term chain keeps its order, so the results are the same bit for bit.
    for (int e = threadIdx.x; e < E; e += blockDim.x) {
        double acc[CX];  // the chains of the run's cells side by side (each a dependent sequence of 30 FP64 operations)
#pragma unroll
        for (int cl = 0; cl < CX; cl++) acc[cl] = 0.0;
#pragma unroll
        for (int half = 0; half < 2; half++) {  // the edge's products in two halves of 15: fewer registers, the chain order is kept
            double T[15];
#pragma unroll
            for (int w = 0; w < 15; w++) T[w] = __ldg(t.edge_T + (long long)e * 30 + half * 15 + w);
#pragma unroll
            for (int w = 0; w < 15; w++) {
#pragma unroll
                for (int cl = 0; cl < CX; cl++) acc[cl] = fma(sCell[min(cl, ncx - 1) * 36 + 5 + half * 15 + w], T[w], acc[cl]);  // pinned 30-term chain
            }
        }
        const double m1 = __ldg(t.edge_mid + 3 * e), m2 = __ldg(t.edge_mid + 3 * e + 1), m3 = __ldg(t.edge_mid + 3 * e + 2);
        const double len = __ldg(t.edge_len + e);
        const int elo = __ldg(t.edge_lo + e), ehi = __ldg(t.edge_hi + e);
#pragma unroll
        for (int cl = 0; cl < CX; cl++) {
            if (cl >= ncx) break;
            const double ce = -acc[cl];
            const double n0e = chain4(sCell + cl * 36 + 1, m1, m2, m3);
            const int a_up = ce > 0.0 ? elo : ehi;
            const double *row = I_in + (c0 + cl) * N;
            double Iup = row[a_up];
            if (t.recon_angle == 1 && ce != 0.0) Iup = plm_angle(t.nbr_edge, t.npsi, t.nzeta, row, a_up, e, Iup);
            sFe[cl * E + e] = (ce == 0.0) ? 0.0 : len * (ce * n0e * Iup);
        }
    }
    __syncthreads();
    // Delta A_a / Delta V of the cells of this run (Eq.20b,c with sqrt(-g) = 1): 1 / dx, or 1 / (the cell's width) on a stretched axis
    const double idy = t.inv_w[1] ? t.inv_w[1][j] : t.inv_dx[1], idz = t.inv_w[2] ? t.inv_w[2][k] : t.inv_dx[2];

    // phase B: spatial fluxes and the update, per (cell, angle)
    for (int q = threadIdx.x; q < ncx * N; q += blockDim.x) {
        const int cl = q / N, n = q % N;
        const long long c = c0 + cl;
        const double *cg = sCell + cl * 36;
        double *out = I_out + c * N + n;
        if (cg[35] != 0.0) { *out = 0.0; continue; }
        const double n1 = __ldg(t.nhat_t + n), n2 = __ldg(t.nhat_t + N + n), n3 = __ldg(t.nhat_t + 2 * N + n);  // (angle-innermost tables: coalesced)
        const double *p = I_in + c * N + n;
        const long long sx = N;
        double div = 0.0;
        const double *vc = TAU ? vel + 5 * c : nullptr;  // this cell's velocity record; the neighbours' are 5 * stride away
        div += (face_flux<RECON, TAU>(sFx + (cl + 1) * 8, n1, n2, n3, p + sx, sx, vc, vc + 5, tau_dt) -
                face_flux<RECON, TAU>(sFx + cl * 8, n1, n2, n3, p, sx, vc - 5, vc, tau_dt)) * (t.inv_w[0] ? t.inv_w[0][i0 + cl] : t.inv_dx[0]);
        div += (face_flux<RECON, TAU>(sFy + CX * 8 + cl * 8, n1, n2, n3, p + sy * N, sy * N, vc, vc + 5 * sy, tau_dt) -
                face_flux<RECON, TAU>(sFy + cl * 8, n1, n2, n3, p, sy * N, vc - 5 * sy, vc, tau_dt)) * idy;
        div += (face_flux<RECON, TAU>(sFz + CX * 8 + cl * 8, n1, n2, n3, p + sz * N, sz * N, vc, vc + 5 * sz, tau_dt) -
                face_flux<RECON, TAU>(sFz + cl * 8, n1, n2, n3, p, sz * N, vc - 5 * sz, vc, tau_dt)) * idz;
        double adiv = 0.0;
#pragma unroll
        for (int s = 0; s < RAD_MAXNBR; s++) {
            const int e = __ldg(t.nbr_edge_t + s * N + n);
            if (e >= 0) adiv = fma(__ldg(t.nbr_w_t + s * N + n), sFe[cl * E + e], adiv);
        }
        div += adiv;
        const double w = cg[0] * chain4(cg + 1, n1, n2, n3);  // n^0 n_0
        double C = gam1 * (w * p[0]);
        if (I0 != nullptr) C = fma(gam0, w * I0[c * N + n], C);
        *out = (C - beta_dt * div) / w;
    }
}

}  // namespace

int launch_fill_ghosts(const DeviceTables &t, const int bc_lo[3], const int bc_hi[3], double *I, cudaStream_t s) {
    int launches = 0;
    for (int ax = 0; ax < 3; ax++) {
        if (bc_lo[ax] == 0 && bc_hi[ax] == 0) continue;
        long long ext[3] = {t.NI, t.NJ, t.NK};
        ext[ax] = 2 * t.ng;
        const long long blocks = ext[0] * ext[1] * ext[2];
        k_fill_ghosts<<<(unsigned)blocks, 64, 0, s>>>(I, t.N, t.NI, t.NJ, t.NK, t.ng, ax, t.n[ax], bc_lo[ax], bc_hi[ax], (t.N & 1) == 0 && ((uintptr_t)I & 15) == 0,
                                                      t.mirror ? t.mirror + ax * t.N : nullptr);
        if (cudaGetLastError() != cudaSuccess) return -1;
        launches++;
    }
    return launches;
}

// both directions of the exchange between block `lo` and block `hi` = its neighbour above along `axis`: 2 launches, -1 on a CUDA error
int launch_exchange_halo(const DeviceTables &lo, double *I_lo, const DeviceTables &hi, double *I_hi, int axis, cudaStream_t s) {
    const int ng = lo.ng, N = lo.N;
    int e[3] = {lo.NI, lo.NJ, lo.NK};
    const int lo_ext = e[axis], hi_ext = axis == 0 ? hi.NI : (axis == 1 ? hi.NJ : hi.NK);
    e[axis] = ng;
    const long long blocks = (long long)e[0] * e[1] * e[2];
    const int vec2 = (N & 1) == 0 && ((uintptr_t)I_lo & 15) == 0 && ((uintptr_t)I_hi & 15) == 0;
    // the upper ghost layers of lo <- the first interior layers of hi; the lower ghost layers of hi <- the last interior layers of lo
    k_copy_halo<<<(unsigned)blocks, 64, 0, s>>>(I_hi, I_lo, N, e[0], e[1], e[2], axis, ng, lo_ext - ng, hi_ext, lo_ext, vec2);
    k_copy_halo<<<(unsigned)blocks, 64, 0, s>>>(I_lo, I_hi, N, e[0], e[1], e[2], axis, lo_ext - 2 * ng, 0, lo_ext, hi_ext, vec2);
    return cudaGetLastError() == cudaSuccess ? 2 : -1;
}

int launch_cell_velocity(const DeviceTables &t, const double *fluid, const double *aE, const double *aS, double *vel, cudaStream_t s) {
    k_cell_velocity<<<t.sms * 4, 256, 0, s>>>(t, fluid, aE, aS, vel);
    return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

// vel != nullptr: optical-depth-aware flux (Eq.26-29) with tau_dt = tau_factor * beta_dt
int launch_fluxdiv(const DeviceTables &t, const Params &p, const double *I_in, const double *I0, double gam0, double gam1,
                   double beta_dt, double *I_out, cudaStream_t s, const double *vel, double tau_dt) {
    const int nxb = (t.n[0] + CX - 1) / CX;
    const long long blocks = (long long)nxb * t.n[1] * t.n[2];
    const size_t smem = sizeof(double) * (CX * 36 + (CX + 1) * 8 + 4 * CX * 8 + (size_t)CX * t.E);
#define RAD_LAUNCH_FD(RECON, TAU)                                                                                     \
    do {                                                                                                              \
        if (cudaFuncSetAttribute(k_fluxdiv<RECON, TAU>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return -1; \
        k_fluxdiv<RECON, TAU><<<(unsigned)blocks, 256, smem, s>>>(t, I_in, I0, gam0, gam1, beta_dt, I_out, vel, tau_dt); \
    } while (0)
    if (p.recon_space == 2) { if (vel) RAD_LAUNCH_FD(2, true); else RAD_LAUNCH_FD(2, false); }
    else if (p.recon_space == 1) { if (vel) RAD_LAUNCH_FD(1, true); else RAD_LAUNCH_FD(1, false); }
    else { if (vel) RAD_LAUNCH_FD(0, true); else RAD_LAUNCH_FD(0, false); }
#undef RAD_LAUNCH_FD
    return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

}  // namespace rad
