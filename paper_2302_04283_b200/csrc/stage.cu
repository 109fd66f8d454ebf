// stage.cu -- the fused stage kernel: spatial + angular flux divergence (Eq.22, 24, 25), cons -> prim
// and, in the same launch, the locally implicit coupling (section 2.5), the ergosphere mask and the
// fluid increment.
//
// Mapping:
//   * one WARP per cell; a lane holds the angles n = it*32 + lane, it < NITER, whose directions stay in
//     registers for the whole kernel.  Intensities are I[cell][angle], angle innermost, so every load and
//     store of a warp is a run of consecutive doubles.
//   * a CTA is a TY x TZ bundle of such warps (neighbouring pencils in y and z) that marches along x in lock
//     step, one cell per step.  The flux through the upper x face is carried in registers to the next step;
//     the fluxes through the lower y and z faces are published in shared memory for the warps of the
//     neighbouring pencils (one __syncthreads per step, double-buffered), so every face flux is computed once
//     except on the rim of the bundle.
//   * geometry per face and per cell (8 + 8 + 8 + 5 doubles) is warp-uniform and read once per cell.
//   * angular fluxes: every unique edge is owned by one of its two angles (edges.cpp).  The owner reads the
//     stored edge coefficient q_e = +-dlambda_e c_e n_0e (one coalesced load; its lowest mantissa bit says which
//     end is upwind), multiplies by the upwind intensity taken from the cell's row in shared memory, and
//     publishes the flux for the partner angle.
//   * the warp then holds all N post-transport intensities of its cell in registers, so the coupling's angle
//     reductions are warp shuffles and the intermediate I* never goes to memory.
#include "stage_math.cuh"

namespace rad {
namespace {

constexpr int TY = 4, TZ = 3, NW = TY * TZ;

__device__ __forceinline__ double2 ldg2(const double *p) { return __ldg(reinterpret_cast<const double2 *>(p)); }

struct FaceRec {
    double e0, e1, e2, e3, E0, E1, E2, E3;
};
__device__ __forceinline__ FaceRec load_face(const double *f) {
    const double2 a = ldg2(f), b = ldg2(f + 2), c = ldg2(f + 4), d = ldg2(f + 6);
    return {a.x, a.y, b.x, b.y, c.x, c.y, d.x, d.y};
}

// Upwind flux n^a n_0 I (Eq.24) through the face between cells L and R; qLL, qL, qR, qRR are the
// intensities of the four cells around it.  PLM: van Leer limited slope of the upwind cell (R7), written as
// q +- dl dr / (dl + dr).  Branch free; the two products are never contracted, so the two cells that share a
// face get the same bits from every call site.
template <bool PLM>
__device__ __forceinline__ double face_flux(const FaceRec &f, double n1, double n2, double n3, double qLL, double qL, double qR,
                                            double qRR) {
    const double na = chain4(f.e0, f.e1, f.e2, f.e3, n1, n2, n3);
    const double n0 = chain4(f.E0, f.E1, f.E2, f.E3, n1, n2, n3);
    const bool pos = na > 0.0;
    double up;
    if (PLM) {
        const double a = pos ? qLL : qL, b = pos ? qL : qR, c = pos ? qR : qRR;
        const double dl = b - a, dr = c - b, pr = dl * dr;
        double h = pr * fast_rcp(dl + dr);
        h = pr > 0.0 ? h : 0.0;
        up = pos ? b + h : b - h;
    } else {
        up = pos ? qL : qR;
    }
    const double F = __dmul_rn(__dmul_rn(na, n0), up);
    return na == 0.0 ? 0.0 : F;
}

template <int NITER, bool PLM, bool COUPLE>
__global__ void __launch_bounds__(NW * 32, 1) k_stage(const DeviceTables t, const Params p, const StageArgs a, const int KX) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int N = t.N, Np = (N + 1) & ~1;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int wy = w % TY, wz = w / TY;
    double *sm = reinterpret_cast<double *>(smem_raw);
    double *sI = sm + (size_t)w * 4 * Np;             // [Np]    this warp's cell, all angles
    double *sG = sI + Np;                             // [3*Np]  fluxes of owned edges, position j*N + n
    double *sF = sm + (size_t)NW * 4 * Np;            // [2 buf][2 axis][NW][Np] lower y / z face fluxes
    double *sWinv = sF + (size_t)4 * NW * Np;         // [Np] 1/dOmega
    double *sDom = sWinv + Np;                        // [Np] dOmega
    int4 *sRec = reinterpret_cast<int4 *>(sDom + Np); // [N]  {own_partner[3], pull_pos[3]} as int16
    for (int q = threadIdx.x; q < N; q += blockDim.x) {
        sWinv[q] = t.winv[q];
        sDom[q] = t.domega[q];
        sRec[q] = reinterpret_cast<const int4 *>(t.ang_rec)[q];
    }
    __syncthreads();

    const int ng = t.ng;
    const int j = blockIdx.y * TY + wy + ng, k = blockIdx.z * TZ + wz + ng;
    const bool active = (j < t.n[1] + ng) && (k < t.n[2] + ng);
    const int i_begin = blockIdx.x * KX + ng, i_end = min(i_begin + KX, t.n[0] + ng);
    const bool top_y = (wy == TY - 1) || (j == t.n[1] + ng - 1);  // nobody in this CTA publishes my upper y flux
    const bool top_z = (wz == TZ - 1) || (k == t.n[2] + ng - 1);
    const long long sy = (long long)t.NI * N, sz = (long long)t.NI * t.NJ * N;  // strides in doubles
    const double idx0 = t.inv_dx[0], idx1 = t.inv_dx[1], idx2 = t.inv_dx[2];

    double n1[NITER], n2[NITER], n3[NITER], carry[NITER];
#pragma unroll
    for (int it = 0; it < NITER; it++) {
        const int nc = min(it * 32 + lane, N - 1);
        carry[it] = 0.0;
        n1[it] = t.nhat[3 * nc]; n2[it] = t.nhat[3 * nc + 1]; n3[it] = t.nhat[3 * nc + 2];
    }
    if (active && i_begin < i_end) {  // flux through the lower x face of the first cell of this run
        const long long c = ((long long)k * t.NJ + j) * t.NI + i_begin;
        const FaceRec f = load_face(t.face + (c * 3 + 0) * RAD_NFACE);
        const double *Ic = a.I_in + c * N;
#pragma unroll
        for (int it = 0; it < NITER; it++) {
            const int nc = min(it * 32 + lane, N - 1);
            const double qLL = PLM ? __ldg(Ic - 2 * N + nc) : 0.0, qL = __ldg(Ic - N + nc), qR = __ldg(Ic + nc), qRR = PLM ? __ldg(Ic + N + nc) : 0.0;
            carry[it] = face_flux<PLM>(f, n1[it], n2[it], n3[it], qLL, qL, qR, qRR);
        }
    }

    for (int i = i_begin; i < i_end; i++) {
        const int buf = (i - i_begin) & 1;
        double *sFy = sF + (size_t)(buf * 2 + 0) * NW * Np, *sFz = sF + (size_t)(buf * 2 + 1) * NW * Np;
        const long long c = ((long long)k * t.NJ + j) * t.NI + i;
        double div[NITER];
        // Lanes past the last angle (n >= N) redo angle N-1 (index nc) and simply do not store: the code below
        // is straight-line, so the loads of all NITER angles of a phase are in flight together.
        if (active) {
            const double *Ic = a.I_in + c * N;
            const long long cint = ((long long)(k - ng) * t.n[1] + (j - ng)) * t.n[0] + (i - ng);
            // ---- angular fluxes (Eq.25, donor cell in angle)
            double Iown[NITER];
#pragma unroll
            for (int it = 0; it < NITER; it++) Iown[it] = __ldg(Ic + min(it * 32 + lane, N - 1));
#pragma unroll
            for (int it = 0; it < NITER; it++)
                if (it * 32 + lane < N) sI[it * 32 + lane] = Iown[it];
            __syncwarp();
            const double *kec = t.ke + cint * 3 * N;
            double q[NITER][3];
#pragma unroll
            for (int it = 0; it < NITER; it++)
#pragma unroll
                for (int jj = 0; jj < 3; jj++) q[it][jj] = __ldg(kec + jj * N + min(it * 32 + lane, N - 1));
#pragma unroll
            for (int it = 0; it < NITER; it++) {
                const int n = it * 32 + lane, nc = min(n, N - 1);
                const int4 rec = sRec[nc];
                const int pj[3] = {(short)(rec.x & 0xffff), (short)(rec.x >> 16), (short)(rec.y & 0xffff)};
                double asum = 0.0;
#pragma unroll
                for (int jj = 0; jj < 3; jj++) {
                    const bool owner_up = (__double2loint(q[it][jj]) & 1) != 0;
                    const double G = q[it][jj] * (owner_up ? Iown[it] : sI[max(pj[jj], 0)]);  // q = 0 in unused slots
                    asum += G;
                    if (n < N && pj[jj] >= 0) sG[jj * N + n] = G;
                }
                div[it] = asum;
            }
            __syncwarp();
#pragma unroll
            for (int it = 0; it < NITER; it++) {
                const int nc = min(it * 32 + lane, N - 1);
                const int4 rec = sRec[nc];
                const int pp[3] = {(short)(rec.y >> 16), (short)(rec.z & 0xffff), (short)(rec.z >> 16)};
                double asum = div[it];
#pragma unroll
                for (int s = 0; s < 3; s++) {
                    const double G = sG[max(pp[s], 0)];
                    asum -= pp[s] >= 0 ? G : 0.0;
                }
                div[it] = asum * sWinv[nc];
            }
            // ---- x: flux through the upper face (the lower x face of cell i+1); the lower one is carried
            {
                const FaceRec f = load_face(t.face + ((c + 1) * 3 + 0) * RAD_NFACE);
#pragma unroll
                for (int it = 0; it < NITER; it++) {
                    const int nc = min(it * 32 + lane, N - 1);
                    const double qLL = PLM ? __ldg(Ic - N + nc) : 0.0, qL = Iown[it], qR = __ldg(Ic + N + nc), qRR = PLM ? __ldg(Ic + 2 * N + nc) : 0.0;
                    const double F = face_flux<PLM>(f, n1[it], n2[it], n3[it], qLL, qL, qR, qRR);
                    div[it] = fma(F - carry[it], idx0, div[it]);
                    carry[it] = F;
                }
            }
            // ---- y: flux through the lower face, published for the warp below; the rim computes its upper face too
            {
                const FaceRec f = load_face(t.face + (c * 3 + 1) * RAD_NFACE);
#pragma unroll
                for (int it = 0; it < NITER; it++) {
                    const int n = it * 32 + lane, nc = min(n, N - 1);
                    const double qLL = PLM ? __ldg(Ic - 2 * sy + nc) : 0.0, qL = __ldg(Ic - sy + nc), qR = Iown[it], qRR = PLM ? __ldg(Ic + sy + nc) : 0.0;
                    const double F = face_flux<PLM>(f, n1[it], n2[it], n3[it], qLL, qL, qR, qRR);
                    div[it] = fma(-F, idx1, div[it]);
                    if (n < N) sFy[w * Np + n] = F;
                }
                if (top_y) {
                    const FaceRec fu = load_face(t.face + ((c + t.NI) * 3 + 1) * RAD_NFACE);
#pragma unroll
                    for (int it = 0; it < NITER; it++) {
                        const int nc = min(it * 32 + lane, N - 1);
                        const double qLL = PLM ? __ldg(Ic - sy + nc) : 0.0, qL = Iown[it], qR = __ldg(Ic + sy + nc), qRR = PLM ? __ldg(Ic + 2 * sy + nc) : 0.0;
                        div[it] = fma(face_flux<PLM>(fu, n1[it], n2[it], n3[it], qLL, qL, qR, qRR), idx1, div[it]);
                    }
                }
            }
            // ---- z
            {
                const FaceRec f = load_face(t.face + (c * 3 + 2) * RAD_NFACE);
#pragma unroll
                for (int it = 0; it < NITER; it++) {
                    const int n = it * 32 + lane, nc = min(n, N - 1);
                    const double qLL = PLM ? __ldg(Ic - 2 * sz + nc) : 0.0, qL = __ldg(Ic - sz + nc), qR = Iown[it], qRR = PLM ? __ldg(Ic + sz + nc) : 0.0;
                    const double F = face_flux<PLM>(f, n1[it], n2[it], n3[it], qLL, qL, qR, qRR);
                    div[it] = fma(-F, idx2, div[it]);
                    if (n < N) sFz[w * Np + n] = F;
                }
                if (top_z) {
                    const FaceRec fu = load_face(t.face + ((c + (long long)t.NI * t.NJ) * 3 + 2) * RAD_NFACE);
#pragma unroll
                    for (int it = 0; it < NITER; it++) {
                        const int nc = min(it * 32 + lane, N - 1);
                        const double qLL = PLM ? __ldg(Ic - sz + nc) : 0.0, qL = Iown[it], qR = __ldg(Ic + sz + nc), qRR = PLM ? __ldg(Ic + 2 * sz + nc) : 0.0;
                        div[it] = fma(face_flux<PLM>(fu, n1[it], n2[it], n3[it], qLL, qL, qR, qRR), idx2, div[it]);
                    }
                }
            }
        }
        __syncthreads();
        if (active) {
            // ---- flux-divergence update of C = n^0 n_0 I (Eq.22, stage form R8) and cons -> prim
            const double *cg = t.cell + c * RAD_NCELL;
            const double2 c01 = ldg2(cg), c23 = ldg2(cg + 2), c45 = ldg2(cg + 4);
            const double nup0 = c01.x, E0 = c01.y, E1 = c23.x, E2 = c23.y, E3 = c45.x;
            const bool excised = __ldg(cg + 50) != 0.0;
            double Is[NITER];
#pragma unroll
            for (int it = 0; it < NITER; it++) {
                const int nc = min(it * 32 + lane, N - 1);
                double d = div[it];
                if (!top_y) d = fma(sFy[(w + 1) * Np + nc], idx1, d);
                if (!top_z) d = fma(sFz[(w + TY) * Np + nc], idx2, d);
                const double wgt = nup0 * chain4(E0, E1, E2, E3, n1[it], n2[it], n3[it]);  // n^0 n_0
                double v = a.gam1 * sI[nc];
                if (a.I0 != nullptr) v = fma(a.gam0, __ldg(a.I0 + c * N + nc), v);
                v = fma(-a.beta_dt * d, fast_rcp(wgt), v);
                Is[it] = excised ? 0.0 : v;
            }
            if (COUPLE) {
                const double Tm = __ldg(a.fluid + 1 * t.ncell + c);
                double Tp = Tm, dR[4] = {0.0, 0.0, 0.0, 0.0};
                if (!excised) {
                    CoupleCell cc;
                    cc.nup0 = nup0; cc.E[0] = E0; cc.E[1] = E1; cc.E[2] = E2; cc.E[3] = E3;
                    const double2 t0 = ldg2(cg + 44), t1 = ldg2(cg + 46), t2 = ldg2(cg + 48);
                    cc.th[0] = t0.x; cc.th[1] = t0.y; cc.th[2] = t1.x; cc.th[3] = t1.y; cc.th[4] = t2.x; cc.th[5] = t2.y;
                    cc.Tm = Tm;
                    cc.rho = cc.u1 = cc.u2 = cc.u3 = cc.aP = cc.aEa = cc.aS = 0.0;
                    if (p.couple) {
                        cc.rho = __ldg(a.fluid + c);
                        cc.u1 = __ldg(a.fluid + 2 * t.ncell + c); cc.u2 = __ldg(a.fluid + 3 * t.ncell + c); cc.u3 = __ldg(a.fluid + 4 * t.ncell + c);
                        cc.aP = __ldg(a.aP + c); cc.aEa = __ldg(a.aE + c); cc.aS = __ldg(a.aS + c);
                    }
                    double dom[NITER];
#pragma unroll
                    for (int it = 0; it < NITER; it++) dom[it] = sDom[min(it * 32 + lane, N - 1)];
                    bool noroot;
                    couple_cell<NITER>(p, cc, a.beta_dt, lane, N, n1, n2, n3, dom, Is, Tp, dR, noroot);
                    if (noroot && lane == 0 && a.noroot) atomicAdd(a.noroot, 1ull);
                }
                if (lane == 0) {
                    if (a.T_out) a.T_out[c] = Tp;
                    if (a.dT0) {
#pragma unroll
                        for (int m = 0; m < 4; m++) a.dT0[m * t.ncell + c] = -dR[m];
                    }
                }
            }
            double *out = a.I_out + c * N;
#pragma unroll
            for (int it = 0; it < NITER; it++) {
                const int n = it * 32 + lane;
                if (n < N) out[n] = Is[it];
            }
        }
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
    const int Np = (N + 1) & ~1;
    return sizeof(double) * ((size_t)NW * 4 * Np + (size_t)4 * NW * Np + 2 * (size_t)Np) + sizeof(int4) * (size_t)N;
}

template <int NITER>
int launch_niter(const DeviceTables &t, const Params &p, const StageArgs &a, bool couple, dim3 grid, size_t smem, int KX, cudaStream_t s) {
#define RAD_LAUNCH(PLM, CPL)                                                                                         \
    do {                                                                                                             \
        if (cudaFuncSetAttribute(k_stage<NITER, PLM, CPL>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return -1; \
        k_stage<NITER, PLM, CPL><<<grid, NW * 32, smem, s>>>(t, p, a, KX);                                            \
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
