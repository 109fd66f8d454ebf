// stream.cu -- the per-cell angle reductions as streaming kernels: the locally implicit coupling (section 2.5, Eq.31-50, with
// the radiation-dominated velocity estimate of Eq.51-55), the ergosphere mask, the fluid increment, and the
// angular moments (Eq.45, Eq.38).
//
// Both kernels read every intensity once, so they are built around the memory system and around the issue slots (one warp
// instruction per clock and scheduler is the bound that bites first on B200 for FP64 work like this):
//   * a warp owns a ring of shared-memory slots; bulk asynchronous copies (TMA, 1-D cp.async.bulk, mbarrier completion) bring the
//     rows of a GROUP of cells that are neighbours along x into a slot, one group ahead of the one being worked on;
//   * coupling: a group is 4 cells, a warp pass is 4 cells x 8 angles (lane = cell * 8 + angle slot), so every lane works for ONE
//     cell: that cell's scalars stay in its registers, the twelve angle sums are accumulated per lane and reduced over the 8
//     lanes of the cell by three shuffle steps, and the per-cell scalar work (tetrad-frame velocity, velocity estimate, quartic
//     Eq.49) is shared by 4 cells per warp pass.  Rows are padded to Np = 8 (mod 16) doubles: conflict-free;
//   * moments: a group is 8 cells and the sums are a DMMA contraction (below).
// The coupling makes two sweeps over the slot: sweep 1 forms the sums and leaves g1 I (in place) and g2 / n0bar^4 of Eq.40 in
// shared memory, sweep 2 is one fused multiply-add per intensity and the store.  The fluid increment needs no second reduction:
// with I_+ - I* = (g1 - 1) I* + src g2', its moments are P + src Q, and P, Q are sums of sweep 1.
#include <stdint.h>

#include <algorithm>

#include "async_copy.cuh"
#include "stage_math.cuh"

namespace rad {
namespace {

constexpr int kCG = 4;      // cells per group (coupling)
constexpr int kCA = 8;      // angle slots per cell in a warp pass
constexpr int kDepth = 2;   // ring slots per warp
constexpr int kCellF = 20;  // per-cell scalars fetched for the coupling: fluid (5), opacities (3), n^0, E_alphahat (4), co-triad (6), excised


__host__ __device__ inline int couple_row_stride(int N) { return ((N + 7) / 8 * 8 + 7) / 16 * 16 + 8; }  // >= 8 ceil(N/8), = 8 (mod 16)

// position of a group of G cells along x in the block, advanced by integer adds only
struct GroupIt {
    int ig, j, k;  // group number along x, interior row (j, k)
    long long c;   // flat index of the group's first cell
};
__device__ __forceinline__ GroupIt group_at(const DeviceTables &t, long long g, int gpr, int G, int kzb) {
    const long long row = g / gpr;
    GroupIt it;
    it.ig = (int)(g - row * gpr); it.j = (int)(row % t.n[1]); it.k = (int)(row / t.n[1]) + kzb;
    it.c = ((long long)(it.k + t.ng) * t.NJ + (it.j + t.ng)) * t.NI + (G * it.ig + t.ng);
    return it;
}
__device__ __forceinline__ void group_next(const DeviceTables &t, GroupIt &it, int gpr, int G) {
    it.c += G;
    if (++it.ig == gpr) {
        it.ig = 0; it.c += t.NI - (long long)G * gpr;
        if (++it.j == t.n[1]) { it.j = 0; ++it.k; it.c += (long long)t.NI * (t.NJ - t.n[1]); }
    }
}

// sum over the 8 lanes of a cell (lanes that differ in bits 0..2)
__device__ __forceinline__ double cell_sum8(double v) {
    v += __shfl_xor_sync(0xffffffffu, v, 1);
    v += __shfl_xor_sync(0xffffffffu, v, 2);
    v += __shfl_xor_sync(0xffffffffu, v, 4);
    return v;
}

// per-cell scalars of the coupling, in the registers of the cell's lanes
struct CellK {
    double uh0, uh1, uh2, uh3;  // tetrad-frame fluid four-velocity used in the coupling (R10; Eq.55 when the estimate applies)
    double aEdt, nup0;          // alpha_E beta dt (Eq.33b), n^0
    double E0, E1, E2, E3;      // E_alphahat: n_0 = E_0 + E_a n^a (mask)
};

// sweep 1 for one intensity: fluid-frame factors (R11), the twelve summands, and the two numbers sweep 2 needs.
// With dd = n^0 + n^0bar alpha_E dt, rp = 1/(n^0bar dd):  dOmega_bar = dOmega / n^0bar^2, Ibar dOmega_bar = n^0bar^2 Ihat dOmega,
// A_1 = sum (n^0/dd) Ibar dOmega_bar, A_2 = dt/4pi sum dOmega rp (Eq.42), and Eq.40 back in the tetrad frame is
// Ihat_+ = g1 Ihat_- + src g2',  g1 = n^0 / dd,  g2' = 1 / (dd n^0bar^3).
__device__ __forceinline__ void sweep1_item(const CellK &c, const double4 an, double I, double (&acc)[12], double &a_out, double &b_out) {
    const double nbar = c.uh0 - fma(c.uh3, an.w, fma(c.uh2, an.z, c.uh1 * an.y));  // n^0bar = -u_alpha n^alpha
    const double dd = fma(nbar, c.aEdt, c.nup0);
    const double rp = rcp3(nbar * dd);
    const double rd = nbar * rp, rn = dd * rp, rn2 = rn * rn;
    const double Id = I * an.x;
    const double x = (nbar * nbar) * Id;  // Ibar dOmega_bar (Eq.38 summand)
    const double g1 = c.nup0 * rd, g2 = rn2 * rp;
    acc[0] = fma(an.x, rn2, acc[0]);  // W
    acc[1] = fma(g1, x, acc[1]);      // A_1 (Eq.42a)
    acc[2] = fma(an.x, rp, acc[2]);   // A_2 (Eq.42b), x dt / 4 pi later
    acc[3] += x;                      // Ebar_- (Eq.38)
    const double pI = Id * (-(nbar * c.aEdt) * rd);  // dOmega (g1 - 1) I
    acc[4] += pI; acc[5] = fma(pI, an.y, acc[5]); acc[6] = fma(pI, an.z, acc[6]); acc[7] = fma(pI, an.w, acc[7]);
    const double qI = an.x * g2;
    acc[8] += qI; acc[9] = fma(qI, an.y, acc[9]); acc[10] = fma(qI, an.z, acc[10]); acc[11] = fma(qI, an.w, acc[11]);
    a_out = g1 * I;
    b_out = g2;
}

// ---------------------------------------------------------------------------------------------------------------------------------
// coupling.  VEST: the radiation-dominated velocity estimate of Eq.51-55 (NEXT-2; reading G8 in DESIGN.md).
// smem per CTA: the angle table {dOmega, n^1, n^2, n^3}[8 ceil(N/8)] (zero past N); per warp: kDepth slots of 4 rows of Np doubles
// (intensities; sweep 1 leaves g1 I there), one buffer b[4][Np], 4 x kCellF cell scalars, the mbarriers.
// ---------------------------------------------------------------------------------------------------------------------------------
struct CoupleArgs {
    double *I;
    const double *fluid, *aP, *aE, *aS;
    double dt;
    double *T_out, *dT0;
    unsigned long long *noroot;
    int kz0, kz1;  // interior planes kz0 <= k < kz1 (0-based, without ghosts); kz1 <= kz0 = the whole block
};

// NPASS: the number of passes ceil(N / 8) as a compile-time constant (the sweeps are then straight-line code), or 0 = taken from N
template <bool VEST, int NPASS>
__global__ void __launch_bounds__(384) k_couple_stream(const DeviceTables t, const Params p, const CoupleArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int N = t.N, npass = NPASS ? NPASS : (N + kCA - 1) / kCA, Np = couple_row_stride(N);
    double *sm = reinterpret_cast<double *>(smem_raw);
    double2 *sA01 = reinterpret_cast<double2 *>(sm), *sA23 = sA01 + npass * kCA;  // {dOmega, n^1}[npass * 8], {n^2, n^3}[npass * 8]
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
    const int perWarp = (kDepth + 1) * kCG * Np + kCG * kCellF + 2 * kDepth;  // doubles (the last 2 kDepth: mbarriers, 8 B each, 16 B apart)
    double *wbase = sm + 4 * npass * kCA + (size_t)w * perWarp;
    double *slots = wbase, *bbuf = wbase + kDepth * kCG * Np, *scell = bbuf + kCG * Np;
    const uint32_t bar0 = smem_u32(scell + kCG * kCellF);
    for (int q = threadIdx.x; q < npass * kCA; q += blockDim.x) {
        sA01[q] = q < N ? make_double2(t.domega[q], t.nhat[3 * q]) : make_double2(0.0, 0.0);
        sA23[q] = q < N ? make_double2(t.nhat[3 * q + 1], t.nhat[3 * q + 2]) : make_double2(0.0, 0.0);
    }
    for (int q = lane; q < (kDepth + 1) * kCG * Np; q += 32) wbase[q] = 0.0;  // the pad of every row (and rows never loaded) stay finite
    if (lane == 0) {
        for (int d = 0; d < kDepth; d++) mbar_init(bar0 + 16u * d, 1);
        fence_mbar_init();
    }
    fence_proxy_async();
    __syncthreads();

    const int gpr = (t.n[0] + kCG - 1) / kCG;  // groups per row
    const int kzb = a.kz1 > a.kz0 ? a.kz0 : 0, kze = a.kz1 > a.kz0 ? a.kz1 : t.n[2];
    const long long ngroups = (long long)gpr * t.n[1] * (kze - kzb);
    const long long nwarp = (long long)gridDim.x * nwarps, wid = (long long)blockIdx.x * nwarps + w;
    // a warp takes a contiguous chunk of groups (consecutive groups are consecutive in memory)
    const long long chunk = (ngroups + nwarp - 1) / nwarp, gbeg = wid * chunk, gend = min(ngroups, gbeg + chunk);
    if (gbeg >= gend) return;
    GroupIt cur = group_at(t, gbeg, gpr, kCG, kzb), ahead = cur, nxt = cur;  // the group worked on, the next to be copied, the next group's scalars
    long long gahead = gbeg;
    int sl_ahead = 0;
    auto issue = [&]() {  // the rows of group `ahead` into its ring slot, one bulk copy per cell
        const int cnt = min(kCG, t.n[0] - kCG * ahead.ig);
        const uint32_t bar = bar0 + 16u * sl_ahead;
        fence_proxy_async();  // every lane: sweep 1 wrote into this slot through the generic proxy, the copies below go through the asynchronous one
        if (lane == 0) mbar_expect_tx(bar, (uint32_t)(cnt * N * 8));
        __syncwarp();
        if (lane < cnt) bulk_g2s(smem_u32(slots + (sl_ahead * kCG + lane) * Np), a.I + (ahead.c + lane) * N, (uint32_t)(N * 8), bar);
        group_next(t, ahead, gpr, kCG);
        gahead++;
        if (++sl_ahead == kDepth) sl_ahead = 0;
    };
    // the 20 per-cell scalars of a group (80 values), fetched by the lanes one group ahead: item q = lane + 32 m = cell * 20 + field;
    // its address is pfbase + (first cell of the group + cell) * pfstride (a field array: stride 1, the cell table: stride RAD_NCELL)
    const double *pfbase[3];
    int pfcell[3], pfstride[3];
    double pfdefault[3];  // value of a missing item: a missing cell counts as excised (n^0 = 1 keeps its idle lanes finite)
#pragma unroll
    for (int m = 0; m < 3; m++) {
        const int q = lane + 32 * m, cl = q / kCellF, f = q - cl * kCellF;
        pfcell[m] = q < kCG * kCellF ? cl : kCG;  // items past the table are never fetched
        pfstride[m] = f < 8 ? 1 : RAD_NCELL;
        pfdefault[m] = (f == 19 || f == 8) ? 1.0 : 0.0;
        if (f < 5) pfbase[m] = a.fluid + (long long)f * t.ncell;
        else if (f < 8) { pfbase[m] = p.couple ? (f == 5 ? a.aP : (f == 6 ? a.aE : a.aS)) : nullptr; if (!p.couple) pfcell[m] = kCG; pfdefault[m] = 0.0; }
        else if (f < 13) pfbase[m] = t.cell + (f - 8);        // n^0, E_0..3
        else if (f < 19) pfbase[m] = t.cell + 44 + (f - 13);  // co-triad
        else pfbase[m] = t.cell + 50;                         // excised
    }
    auto fetch_cell = [&](double (&v)[3]) {  // of group `nxt`
        const int cnt = min(kCG, t.n[0] - kCG * nxt.ig);
        const long long c0 = nxt.c;
        group_next(t, nxt, gpr, kCG);
#pragma unroll
        for (int m = 0; m < 3; m++) {
            v[m] = pfdefault[m];
            if (pfcell[m] < cnt) v[m] = __ldg(pfbase[m] + (c0 + pfcell[m]) * pfstride[m]);
        }
    };
    for (int d = 0; d < kDepth - 1 && gahead < gend; d++) issue();
    double cellv[3];
    fetch_cell(cellv);
    const int mycell = lane >> 3, kk = lane & 7;
    const uint32_t aA01 = smem_u32(sA01) + 16u * kk, aA23 = smem_u32(sA23) + 16u * kk, aB = smem_u32(bbuf) + 8u * (uint32_t)(mycell * Np + kk);
    const double n0crit = p.n0_crit;
    int sl = 0, par = 0;

    for (long long g = gbeg; g < gend; g++) {
        const int cnt = min(kCG, t.n[0] - kCG * cur.ig);
        const long long c0 = cur.c;
        group_next(t, cur, gpr, kCG);
        // cell scalars of this group to shared memory, next group's on their way
        __syncwarp();
#pragma unroll
        for (int m = 0; m < 3; m++) if (lane + 32 * m < kCG * kCellF) scell[lane + 32 * m] = cellv[m];
        if (g + 1 < gend) fetch_cell(cellv);
        if (gahead < gend) issue();  // its slot was released at the end of the previous iteration
        __syncwarp();
        // ---- per-cell preparation: every lane for its own cell (the 8 lanes of a cell compute the same values)
        const double *sc = scell + mycell * kCellF;
        const double rho = sc[0], Tm = sc[1], aPc = sc[5], aEc = sc[6], aSc = sc[7], nup0 = sc[8];
        const bool excised = sc[19] != 0.0, docouple = p.couple && !excised;
        CellK ck;
        ck.uh0 = 1.0; ck.uh1 = ck.uh2 = ck.uh3 = 0.0;
        ck.aEdt = docouple ? (aEc + aSc) * a.dt : 0.0;  // Eq.33b
        ck.nup0 = nup0; ck.E0 = sc[9]; ck.E1 = sc[10]; ck.E2 = sc[11]; ck.E3 = sc[12];
        if (docouple) {
            const double u1 = sc[2], u2 = sc[3], u3 = sc[4];
            ck.uh1 = sc[13] * u1 + sc[14] * u2 + sc[15] * u3; ck.uh2 = sc[16] * u2 + sc[17] * u3; ck.uh3 = sc[18] * u3;  // u^ahat = theta^ahat_j u^j' (R10)
            ck.uh0 = sqrt_ge1(1.0 + (ck.uh1 * ck.uh1 + ck.uh2 * ck.uh2 + ck.uh3 * ck.uh3));
        }
        // |n_0| = |E_0 + E_a n^a| >= |E_0| - |E|: only cells with |E_0| - |E| < n_0^crit can have a masked angle (1e-9: rounding of the bound)
        // (compared in squares: |E_0| - n_0^crit (1 + 1e-9) < |E|  <=>  that difference is negative or its square is below |E|^2)
        const double mgap = fabs(ck.E0) - n0crit * (1.0 + 1e-9);
        const bool mymask = n0crit > 0.0 && !excised && (mgap < 0.0 || mgap * mgap < ck.E1 * ck.E1 + ck.E2 * ck.E2 + ck.E3 * ck.E3);
        const bool anymask = __any_sync(0xffffffffu, mymask);
        mbar_wait(bar0 + 16u * sl, (uint32_t)par);
        const uint32_t aI = smem_u32(slots + (sl * kCG + mycell) * Np) + 8u * kk;  // this lane's item of pass j: + 64 j

        if (VEST) {
            // ---- Eq.51-55: tetrad-frame moments of I*, radiation velocity, force, clamped fractions, blended velocity
            double M[10];
#pragma unroll
            for (int q = 0; q < 10; q++) M[q] = 0.0;
#pragma unroll(NPASS ? NPASS : 2)
            for (int j = 0; j < npass; j++) {
                const double2 a01 = lds2(aA01 + 128u * j), a23 = lds2(aA23 + 128u * j);
                const double w0 = lds(aI + 64u * j) * a01.x;
                const double w1 = w0 * a01.y, w2 = w0 * a23.x, w3 = w0 * a23.y;
                M[0] += w0; M[1] += w1; M[2] += w2; M[3] += w3;
                M[4] = fma(w1, a01.y, M[4]); M[5] = fma(w1, a23.x, M[5]); M[6] = fma(w1, a23.y, M[6]);
                M[7] = fma(w2, a23.x, M[7]); M[8] = fma(w2, a23.y, M[8]); M[9] = fma(w3, a23.y, M[9]);
            }
#pragma unroll
            for (int q = 0; q < 10; q++) M[q] = cell_sum8(M[q]);
            if (docouple) {
                // R^{ahat bhat} = M: (00,01,02,03,11,12,13,22,23,33).  Ebar = u_a u_b R^{ab} with u_0 = -u^0 (Eq.38 in covariant form)
                const double R[4][4] = {{M[0], M[1], M[2], M[3]}, {M[1], M[4], M[5], M[6]}, {M[2], M[5], M[7], M[8]}, {M[3], M[6], M[8], M[9]}};
                const double ul[4] = {-ck.uh0, ck.uh1, ck.uh2, ck.uh3}, uu[4] = {ck.uh0, ck.uh1, ck.uh2, ck.uh3};
                double uR[4], Ebar = 0.0;  // uR^a = u_b R^{ab}
#pragma unroll
                for (int al = 0; al < 4; al++) {
                    uR[al] = ul[0] * R[al][0] + ul[1] * R[al][1] + ul[2] * R[al][2] + ul[3] * R[al][3];
                }
#pragma unroll
                for (int al = 0; al < 4; al++) Ebar += ul[al] * uR[al];
                const double ugas = rho * Tm * p.rgm1, wgas = rho + ugas + rho * Tm;  // rho + u + p (k_B / mu m_p = 1)
                if (Ebar > rho + ugas && M[0] > 0.0) {  // radiation dominates
                    const double rE = 1.0 / M[0];
                    const double v1 = M[1] * rE, v2 = M[2] * rE, v3 = M[3] * rE;  // Eq.51
                    const double vv = fmin(v1 * v1 + v2 * v2 + v3 * v3, 1.0 - 1e-12);  // R19: keep the Lorentz factor finite
                    const double W0 = 1.0 / sqrt(1.0 - vv);
                    const double ur[4] = {W0, W0 * v1, W0 * v2, W0 * v3};
                    const double T2 = Tm * Tm, emis = aPc * p.a_rad * T2 * T2 + aSc * Ebar, aEt = aEc + aSc;
                    double un[4];
                    un[0] = 0.0;
#pragma unroll
                    for (int q = 1; q < 4; q++) {
                        const double G = -emis * uu[q] - aEt * uR[q];                      // Eq.53
                        const double den = wgas * (ur[0] * ur[q] - uu[0] * uu[q]);         // Eq.52b - Eq.52a
                        double fr = den != 0.0 ? G * a.dt / den : 0.0;                     // Eq.54 (G8)
                        fr = fmin(fmax(fr, 0.0), 1.0);
                        if (!(fr == fr)) fr = 0.0;
                        un[q] = (1.0 - fr) * uu[q] + fr * ur[q];                           // Eq.55
                    }
                    ck.uh1 = un[1]; ck.uh2 = un[2]; ck.uh3 = un[3];
                    ck.uh0 = sqrt(1.0 + (un[1] * un[1] + un[2] * un[2] + un[3] * un[3]));
                }
            }
        }
        // ---- sweep 1: the lane's items of its cell, angle n = 8 j + kk
        double S[12];
#pragma unroll
        for (int q = 0; q < 12; q++) S[q] = 0.0;
#pragma unroll(NPASS ? NPASS : 3)
        for (int j = 0; j < npass; j++) {
            const double2 a01 = lds2(aA01 + 128u * j), a23 = lds2(aA23 + 128u * j);
            const double4 an = make_double4(a01.x, a01.y, a23.x, a23.y);  // zeros past N: such an item adds zeros
            const double I = lds(aI + 64u * j);
            double a_o, b_o;
            sweep1_item(ck, an, I, S, a_o, b_o);
            if (anymask) {  // warp-uniform: some cell of the group lies where |n_0| can drop below n_0^crit
                const bool masked = mymask && fabs(chain4(ck.E0, ck.E1, ck.E2, ck.E3, an.y, an.z, an.w)) < n0crit;  // pinned chain
                a_o = masked ? 0.0 : a_o; b_o = masked ? 0.0 : b_o;
            }
            sts(aI + 64u * j, a_o); sts(aB + 64u * j, b_o);
        }
#pragma unroll
        for (int q = 0; q < 12; q++) S[q] = cell_sum8(S[q]);
        // ---- per cell: quartic Eq.49 (R13), T_+, source, fluid increment
        double Tp = Tm, src = 0.0;
        bool coupled = false, noroot = false;
        if (docouple) {
            const double scale = p.renorm ? kFourPi * rcp3(S[0]) : 1.0;  // R12
            const double A1 = S[1] * scale, Em = S[3] * scale, A2 = S[2] * (scale * (a.dt * kInvFourPi));
            const double Cv = rho * p.rgm1;
            const double B4 = A2 * aPc * p.a_rad, om = 1.0 - A2 * aSc;  // Eq.50
            const double B1 = Cv * om, Bp = A1 - om * Em;
            double dTemp = 0.0;
            if (!quartic_delta(B4, B1, Bp, Tm, dTemp)) noroot = true;
            else {
                coupled = true;
                Tp = Tm + dTemp;
                const double Ep = Em - Cv * dTemp;  // Eq.48
                const double T2 = Tp * Tp;
                src = (aPc * p.a_rad * T2 * T2 + aSc * Ep) * (a.dt * kInvFourPi);
            }
        }
        if (kk == 0 && mycell < cnt) {
            const long long c = c0 + mycell;
            if (noroot && a.noroot) atomicAdd(a.noroot, 1ull);
            if (a.T_out) a.T_out[c] = Tp;
            if (a.dT0) {  // -(change of R^0_alpha) = -n^0 n_alpha-moments of I_+ - I* (P:L472); n_0 = E_ahat ntil^ahat, n_i = theta^a_i n^a
                double M0 = 0.0, M1 = 0.0, M2 = 0.0, M3 = 0.0;
                if (coupled) { M0 = fma(src, S[8], S[4]); M1 = fma(src, S[9], S[5]); M2 = fma(src, S[10], S[6]); M3 = fma(src, S[11], S[7]); }
                a.dT0[c] = -(nup0 * (sc[9] * M0 + sc[10] * M1 + sc[11] * M2 + sc[12] * M3));
                a.dT0[t.ncell + c] = -(nup0 * (sc[13] * M1));
                a.dT0[2 * t.ncell + c] = -(nup0 * (sc[14] * M1 + sc[16] * M2));
                a.dT0[3 * t.ncell + c] = -(nup0 * (sc[15] * M1 + sc[17] * M2 + sc[18] * M3));
            }
        }
        // ---- sweep 2: Eq.40 in the tetrad frame, store.  A cell that is not coupled keeps what the transport wrote, except for
        // its masked intensities (b = 0 marks them: g2' is positive otherwise); excised cells keep their zeros.
        __syncwarp();
        {
            double *out = a.I + (c0 + mycell) * N + kk;
            const int myn = (mycell < cnt && !excised) ? (N - kk + kCA - 1) / kCA : 0;  // this lane's items
            if (__all_sync(0xffffffffu, coupled || myn == 0)) {  // the usual case: every cell of the group has a root
                const int nall = NPASS ? (NPASS - 1) : N / kCA;  // items every lane has; the last pass may be partial
#pragma unroll(NPASS ? NPASS : 4)
                for (int j = 0; j < nall; j++)
                    if (myn) out[kCA * j] = fma(src, lds(aB + 64u * j), lds(aI + 64u * j));
                for (int j = nall; j < myn; j++) out[kCA * j] = fma(src, lds(aB + 64u * j), lds(aI + 64u * j));
            } else {
                for (int j = 0; j < myn; j++) {
                    const double b_ = lds(aB + 64u * j);
                    if (coupled) out[kCA * j] = fma(src, b_, lds(aI + 64u * j));
                    else if (b_ == 0.0) out[kCA * j] = 0.0;
                }
            }
        }
        __syncwarp();  // the slot is free for the copy issued at the top of the next iteration
        if (++sl == kDepth) { sl = 0; par ^= 1; }
    }
}

// ---------------------------------------------------------------------------------------------------------------------------------
// moments: by linearity every frame's moments follow from the ten tetrad-frame sums M^{ab} = sum_n I dOmega ntil^a ntil^b,
// ntil = (1, n^1hat, n^2hat, n^3hat) -- a dense contraction [cells x N] . [N x 10] (Eq.45 in the tetrad frame).  It runs on the
// FP64 matrix instruction DMMA m8n8k4 (same FP64 pipe as DFMA on B200, measured; 256 multiply-adds per issue slot and no
// cross-lane reduction): a warp takes 8 cells that are neighbours along x; per step of 4 angles lane l holds
// A[cell l/4][angle l%4] = I (from the ring slot the bulk copies filled) and B[angle l%4][column l/4] = the table entry for the
// first eight sums; sums 9 and 10 are two ordinary FMAs per step on the same A value, reduced over the four lanes of a cell at
// the end.  The per-cell transform (tetrad e^mu_ahat for frame 0, n_alpha rows for frame 1, boost Eq.13-14 with G2 for frame 3)
// is done once per cell afterwards, one lane per output component.
// Shared memory rows are padded to Np = 4 (mod 16) doubles so that the eight cells' rows fall into different banks.
// ---------------------------------------------------------------------------------------------------------------------------------
constexpr int kMomCells = 8;
constexpr int kMomCellF = 24;  // per-cell scalars of the epilogue: cell record [0..4], [35..49], fluid u^1', u^2', u^3', pad

__device__ __forceinline__ void dmma884(double &d0, double &d1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};" : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}
__host__ __device__ inline int mom_row_stride(int N) { return ((N + 3) / 4 * 4 + 11) / 16 * 16 + 4; }  // >= 4 ceil(N/4), = 4 (mod 16)

__global__ void __launch_bounds__(384) k_moments_mma(const DeviceTables t, const double *__restrict__ I, int frame, const double *__restrict__ fluid,
                                                     double *__restrict__ out, int depth) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int N = t.N, nk = (N + 3) >> 2, Np = mom_row_stride(N);
    double *sm = reinterpret_cast<double *>(smem_raw);
    double *sB = sm;                                              // [nk][32]: fragment order, columns 0..7
    double2 *sX = reinterpret_cast<double2 *>(sm + nk * 32);      // [nk][4]: columns 8, 9
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
    const int perWarp = depth * kMomCells * Np + kMomCells * 10 + kMomCells * kMomCellF + 2 * depth;
    double *slots = sm + nk * 40 + (size_t)w * perWarp, *tot = slots + depth * kMomCells * Np, *scell = tot + kMomCells * 10;
    const uint32_t bar0 = smem_u32(scell + kMomCells * kMomCellF);
    // the table: for angle n and column q = (a, b) of (00,01,02,03,11,12,13,22,23,33): dOmega_n ntil^a ntil^b
    for (int q = threadIdx.x; q < nk * 32; q += blockDim.x) {
        const int j = q >> 5, l = q & 31, n = 4 * j + (l & 3), col = l >> 2;
        double v = 0.0;
        if (n < N) {
            const double nt[4] = {1.0, t.nhat[3 * n], t.nhat[3 * n + 1], t.nhat[3 * n + 2]};
            const int ca[8] = {0, 0, 0, 0, 1, 1, 1, 2}, cb[8] = {0, 1, 2, 3, 1, 2, 3, 2};
            v = t.domega[n] * nt[ca[col]] * nt[cb[col]];
        }
        sB[q] = v;
    }
    for (int q = threadIdx.x; q < nk * 4; q += blockDim.x) {
        double2 v = make_double2(0.0, 0.0);
        if (q < N) { const double w0 = t.domega[q], n2 = t.nhat[3 * q + 1], n3 = t.nhat[3 * q + 2]; v = make_double2(w0 * n2 * n3, w0 * n3 * n3); }
        sX[q] = v;
    }
    for (int q = lane; q < depth * kMomCells * Np; q += 32) slots[q] = 0.0;  // the pad of every row stays zero
    if (lane == 0) {
        for (int d = 0; d < depth; d++) mbar_init(bar0 + 16u * d, 1);
        fence_mbar_init();
    }
    fence_proxy_async();
    __syncthreads();
    const int gpr = (t.n[0] + kMomCells - 1) / kMomCells;  // groups per row
    const long long ngroups = (long long)gpr * t.n[1] * t.n[2];
    const long long nwarp = (long long)gridDim.x * nwarps, wid = (long long)blockIdx.x * nwarps + w;
    const long long chunk = (ngroups + nwarp - 1) / nwarp, gbeg = wid * chunk, gend = min(ngroups, gbeg + chunk);
    if (gbeg >= gend) return;
    GroupIt cur = group_at(t, gbeg, gpr, kMomCells, 0), ahead = cur;
    long long gahead = gbeg;
    int sl_ahead = 0;
    auto issue = [&]() {  // the rows of group `ahead` into its ring slot, one bulk copy per cell
        const int cnt = min(kMomCells, t.n[0] - kMomCells * ahead.ig);
        const uint32_t bar = bar0 + 16u * sl_ahead;
        if (lane == 0) mbar_expect_tx(bar, (uint32_t)(cnt * N * 8));
        __syncwarp();
        if (lane < cnt) bulk_g2s(smem_u32(slots + (sl_ahead * kMomCells + lane) * Np), I + (ahead.c + lane) * N, (uint32_t)(N * 8), bar);
        group_next(t, ahead, gpr, kMomCells);
        gahead++;
        if (++sl_ahead == depth) sl_ahead = 0;
    };
    for (int d = 0; d < depth - 1 && gahead < gend; d++) issue();
    const int r = lane >> 2, kk = lane & 3;
    const int ncomp = (frame == 0 || frame == 2) ? 10 : 4;
    // the epilogue's per-cell scalars: item q = lane + 32 m = cell * 24 + field; offset relative to the group's first cell
    // (cell table: doubles past t.cell + c0 * RAD_NCELL; fluid: field * ncell + cell), kind 0 nothing, 1 cell table, 2 fluid
    int cvoff[6], cvkind[6];
#pragma unroll
    for (int m = 0; m < 6; m++) {
        const int q = lane + 32 * m, cl = q / kMomCellF, f = q - cl * kMomCellF;
        cvkind[m] = 0; cvoff[m] = cl;
        if (frame != 2) {
            if (f < 5) { cvkind[m] = 1; cvoff[m] = cl * RAD_NCELL + f; }                  // n^0, E_alphahat
            else if (f < 20) { cvkind[m] = 1; cvoff[m] = cl * RAD_NCELL + 30 + f; }       // beta^i (3), triad (6), co-triad (6)
            else if (f < 23 && frame == 3) { cvkind[m] = 2 + (f - 20); }                  // u^1', u^2', u^3' of cell cl
        }
    }
    int sl = 0, par = 0;
    for (long long g = gbeg; g < gend; g++) {
        const int cnt = min(kMomCells, t.n[0] - kMomCells * cur.ig);
        const long long c0 = cur.c;
        group_next(t, cur, gpr, kMomCells);
        if (gahead < gend) issue();  // into the slot read in the previous iteration
        double cv[6];
#pragma unroll
        for (int m = 0; m < 6; m++) {
            cv[m] = 0.0;
            const int cl = (lane + 32 * m) / kMomCellF;
            if (cl < cnt) {
                if (cvkind[m] == 1) cv[m] = __ldg(t.cell + c0 * RAD_NCELL + cvoff[m]);
                else if (cvkind[m] >= 2) cv[m] = __ldg(fluid + (long long)cvkind[m] * t.ncell + c0 + cl);
            }
        }
        mbar_wait(bar0 + 16u * sl, (uint32_t)par);
        const uint32_t aRow = smem_u32(slots + (sl * kMomCells + r) * Np) + 8u * kk;
        const uint32_t aB = smem_u32(sB) + 8u * lane, aX = smem_u32(sX) + 16u * kk;
        double d0 = 0.0, d1 = 0.0, e0 = 0.0, e1 = 0.0, x8 = 0.0, x9 = 0.0, y8 = 0.0, y9 = 0.0;
        int j = 0;
#pragma unroll 4
        for (; j + 1 < nk; j += 2) {
            const double a0 = lds(aRow + 32u * j), a1 = lds(aRow + 32u * j + 32u);
            const double b0 = lds(aB + 256u * j), b1 = lds(aB + 256u * j + 256u);
            const double2 p0 = lds2(aX + 64u * j), p1 = lds2(aX + 64u * j + 64u);
            dmma884(d0, d1, a0, b0);
            dmma884(e0, e1, a1, b1);
            x8 = fma(a0, p0.x, x8); x9 = fma(a0, p0.y, x9);
            y8 = fma(a1, p1.x, y8); y9 = fma(a1, p1.y, y9);
        }
        if (j < nk) {
            const double a0 = lds(aRow + 32u * j), b0 = lds(aB + 256u * j);
            const double2 p0 = lds2(aX + 64u * j);
            dmma884(d0, d1, a0, b0);
            x8 = fma(a0, p0.x, x8); x9 = fma(a0, p0.y, x9);
        }
        d0 += e0; d1 += e1; x8 += y8; x9 += y9;
        x8 += __shfl_xor_sync(0xffffffffu, x8, 1); x9 += __shfl_xor_sync(0xffffffffu, x9, 1);
        x8 += __shfl_xor_sync(0xffffffffu, x8, 2); x9 += __shfl_xor_sync(0xffffffffu, x9, 2);
        __syncwarp();  // the previous group's epilogue has read tot and scell; every lane is done with the slot
        tot[r * 10 + 2 * kk] = d0; tot[r * 10 + 2 * kk + 1] = d1;
        if (kk == 0) { tot[r * 10 + 8] = x8; tot[r * 10 + 9] = x9; }
#pragma unroll
        for (int m = 0; m < 6; m++) scell[lane + 32 * m] = cv[m];
        __syncwarp();
        // ---- epilogue.  Frame 0: lane = (cell, nu) forms W^a = M^{ab} e^nu_b and the outputs R^{mu nu} = e^mu_a W^a for mu <= nu
        // (R^{mu nu} = e^mu_a e^nu_b M^{ab}; e^0_0 = n^0, e^i_0 = -beta^i n^0, e^i_a = triad, upper triangular, R2)
        if (frame == 0) {
            const int cl = lane & 7, nu = lane >> 3;
            if (cl < cnt) {
                const double *M10 = tot + cl * 10, *ca = scell + cl * kMomCellF;
                const double nup0 = ca[0], b1 = -ca[5] * nup0, b2 = -ca[6] * nup0, b3 = -ca[7] * nup0;
                const double t11 = ca[8], t12 = ca[9], t13 = ca[10], t22 = ca[11], t23 = ca[12], t33 = ca[13];
                const double E0 = nu == 0 ? nup0 : (nu == 1 ? b1 : (nu == 2 ? b2 : b3));
                const double E1 = nu == 1 ? t11 : 0.0, E2 = nu == 1 ? t12 : (nu == 2 ? t22 : 0.0), E3 = nu == 1 ? t13 : (nu == 2 ? t23 : (nu == 3 ? t33 : 0.0));
                const double W0 = M10[0] * E0 + M10[1] * E1 + M10[2] * E2 + M10[3] * E3;
                const double W1 = M10[1] * E0 + M10[4] * E1 + M10[5] * E2 + M10[6] * E3;
                const double W2 = M10[2] * E0 + M10[5] * E1 + M10[7] * E2 + M10[8] * E3;
                const double W3 = M10[3] * E0 + M10[6] * E1 + M10[8] * E2 + M10[9] * E3;
                const long long c = c0 + cl;
                out[nu * t.ncell + c] = nup0 * W0;                                                                   // (0, nu)
                if (nu >= 1) out[(3 + nu) * t.ncell + c] = b1 * W0 + t11 * W1 + t12 * W2 + t13 * W3;                 // (1, nu)
                if (nu >= 2) out[(5 + nu) * t.ncell + c] = b2 * W0 + t22 * W2 + t23 * W3;                            // (2, nu)
                if (nu == 3) out[9 * t.ncell + c] = b3 * W0 + t33 * W3;                                              // (3, 3)
            }
        } else
        for (int o = lane; o < ncomp * kMomCells; o += 32) {
            const int li = o >> 3, cl = o & 7;
            if (cl >= cnt) continue;
            const long long c = c0 + cl;
            const double *M10 = tot + cl * 10, *ca = scell + cl * kMomCellF, *cb = ca + 16;
            // ca: [0] n^0, [1..4] E_alphahat, [5..7] beta^i, [8..13] triad (x1,x2,x3,y2,y3,z3), [14] theta 1x, [15] theta 1y; cb: [0] theta 1z, [1] 2y, [2] 2z, [3] 3z, [4..6] u^i'
            double v;
            if (frame == 2) {
                v = M10[li];
            } else if (frame == 1) {  // R^0_alpha = n^0 sum n_alpha I dOmega; n_0 = E_ahat ntil^ahat, n_i = theta^a_i n^a
                if (li == 0) v = ca[1] * M10[0] + ca[2] * M10[1] + ca[3] * M10[2] + ca[4] * M10[3];
                else if (li == 1) v = ca[14] * M10[1];
                else if (li == 2) v = ca[15] * M10[1] + cb[1] * M10[2];
                else v = cb[0] * M10[1] + cb[2] * M10[2] + cb[3] * M10[3];
                v *= ca[0];
            } else {
                const double M[4][4] = {{M10[0], M10[1], M10[2], M10[3]}, {M10[1], M10[4], M10[5], M10[6]}, {M10[2], M10[5], M10[7], M10[8]}, {M10[3], M10[6], M10[8], M10[9]}};
                {  // fluid frame (Eq.13-14 with G2): nbar^0 = u^0 - u_a n^a, nbar^a = n^a + u^a (u_b n^b / (1 + u^0) - 1)
                    const double th[6] = {ca[14], ca[15], cb[0], cb[1], cb[2], cb[3]};
                    double uh[4];
                    tetrad_velocity(th, cb[4], cb[5], cb[6], uh);
                    const double rr = 1.0 / (1.0 + uh[0]);
                    double Lm[4][4];
                    Lm[0][0] = uh[0]; Lm[0][1] = -uh[1]; Lm[0][2] = -uh[2]; Lm[0][3] = -uh[3];
#pragma unroll
                    for (int a2 = 1; a2 < 4; a2++) {
                        Lm[a2][0] = -uh[a2];
#pragma unroll
                        for (int b = 1; b < 4; b++) Lm[a2][b] = (a2 == b ? 1.0 : 0.0) + uh[a2] * uh[b] * rr;
                    }
                    double LM[4];  // Lambda^0_a M^{ab}
#pragma unroll
                    for (int b = 0; b < 4; b++) LM[b] = Lm[0][0] * M[0][b] + Lm[0][1] * M[1][b] + Lm[0][2] * M[2][b] + Lm[0][3] * M[3][b];
                    v = 0.0;
#pragma unroll
                    for (int q = 0; q < 4; q++) {
                        const double x = LM[0] * Lm[q][0] + LM[1] * Lm[q][1] + LM[2] * Lm[q][2] + LM[3] * Lm[q][3];
                        if (q == li) v = x;
                    }
                }
            }
            out[li * t.ncell + c] = v;
        }
        if (++sl == depth) { sl = 0; par ^= 1; }
    }
}

size_t couple_smem(int N, int warps) {
    const int npass = (N + kCA - 1) / kCA;
    return sizeof(double) * (4 * (size_t)npass * kCA + (size_t)warps * ((kDepth + 1) * kCG * couple_row_stride(N) + kCG * kCellF + 2 * kDepth));
}
size_t moments_smem(int N, int warps, int depth) {
    const int nk = (N + 3) / 4;
    return sizeof(double) * ((size_t)nk * 40 + (size_t)warps * (depth * kMomCells * mom_row_stride(N) + kMomCells * 10 + kMomCells * kMomCellF + 2 * depth));
}

}  // namespace

// 1 if the streaming kernels serve this angle grid and these arrays: rows must be multiples of 16 bytes (bulk copies).
// I == nullptr asks about the angle grid alone.
int stream_serves(const DeviceTables &t, const void *I) {
    return (t.N & 1) == 0 && ((uintptr_t)I & 15) == 0 && couple_smem(t.N, 2) <= (size_t)t.smem_optin;
}

// returns 1 (launched), 0 (not served), -1 (CUDA error)
int launch_couple_stream(const DeviceTables &t, const Params &p, double *I, const double *fluid, const double *aP, const double *aE, const double *aS,
                         double dt, double *T_out, double *dT0, unsigned long long *noroot, cudaStream_t s, int kz0, int kz1) {
    if (!stream_serves(t, I)) return 0;
    int warps = 12;  // as many as shared memory holds
    while (warps > 2 && couple_smem(t.N, warps) > (size_t)t.smem_optin) warps--;
    const size_t smem = couple_smem(t.N, warps);
    CoupleArgs a{I, fluid, aP, aE, aS, dt, T_out, dT0, noroot, kz0, kz1};
    const int per_sm = (int)std::max<size_t>(1, std::min<size_t>(4, (size_t)t.smem_optin / (smem + 1024)));
    const int grid = t.sms * per_sm;
    const int npass = (t.N + kCA - 1) / kCA;
#define RAD_COUPLE_LAUNCH(VEST, NP)                                                                                                                  \
    do {                                                                                                                                             \
        if (cudaFuncSetAttribute(k_couple_stream<VEST, NP>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return -1;       \
        k_couple_stream<VEST, NP><<<grid, warps * 32, smem, s>>>(t, p, a);                                                                            \
    } while (0)
    if (p.vel_estimate && p.couple) { if (npass == 21) RAD_COUPLE_LAUNCH(true, 21); else RAD_COUPLE_LAUNCH(true, 0); }
    else if (npass == 21) RAD_COUPLE_LAUNCH(false, 21);  // N = 161..168 (geodesic level 4)
    else if (npass == 12) RAD_COUPLE_LAUNCH(false, 12);  // N = 89..96 (geodesic level 3)
    else RAD_COUPLE_LAUNCH(false, 0);
#undef RAD_COUPLE_LAUNCH
    return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

int launch_moments_stream(const DeviceTables &t, const double *I, int frame, const double *fluid, double *out, cudaStream_t s) {
    if ((t.N & 1) || ((uintptr_t)I & 15)) return 0;
    // ring depth 2 and as many warps as shared memory holds (<= 12); deeper rings do not pay once ~100 KB are in flight per SM
    const int depth = 2;
    int warps = 12;
    while (warps > 2 && moments_smem(t.N, warps, depth) > (size_t)t.smem_optin) warps--;
    const size_t smem = moments_smem(t.N, warps, depth);
    if (smem > (size_t)t.smem_optin) return 0;
    const int per_sm = (int)std::max<size_t>(1, std::min<size_t>(4, (size_t)t.smem_optin / (smem + 1024)));
    if (cudaFuncSetAttribute(k_moments_mma, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return -1;
    k_moments_mma<<<t.sms * per_sm, warps * 32, smem, s>>>(t, I, frame, fluid, out, depth);
    return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

}  // namespace rad
