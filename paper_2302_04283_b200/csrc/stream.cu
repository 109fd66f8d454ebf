// stream.cu -- the per-cell angle reductions as streaming kernels: the locally implicit coupling (section 2.5, Eq.31-50, with
// the radiation-dominated velocity estimate of Eq.51-55), the ergosphere mask, the fluid increment, and the
// angular moments (Eq.45, Eq.38).
//
// Both kernels read every intensity once and are bound by HBM, so they are built around the memory system:
//   * a warp owns a ring of shared-memory slots; one bulk asynchronous copy (TMA, 1-D cp.async.bulk, mbarrier completion) brings
//     the rows of TWO cells that are neighbours along x (2 N contiguous doubles) into a slot, kDepth - 1 pairs ahead of the one
//     being worked on, so that the copies of all resident warps keep the memory system busy while the arithmetic runs;
//   * the 2 N intensities of a pair are one flat run: lane l takes the items f = l, l + 32, ... (for N = 162: 11 passes for 324
//     items, 92 % of the lanes busy, against 84 % with one cell per warp pass).  Passes that lie in one cell use that cell's
//     scalars from registers; the one pass that straddles the two cells selects per lane;
//   * angle sums: every lane accumulates the sums of both cells; the lanes' partial sums are transposed through shared memory
//     (lane q adds up row q), ~24 stores + 32 loads for all sums of both cells instead of a five-level shuffle butterfly each;
//   * per-cell scalar work (tetrad-frame fluid velocity, velocity estimate, quartic Eq.49) runs in the two half-warps, one cell each.
// The coupling makes two sweeps over the slot: sweep 1 forms the sums and leaves g1 I and g2 / n0bar^4 of Eq.40 in shared memory,
// sweep 2 is one fused multiply-add per intensity and the coalesced store.  The fluid increment needs no second reduction: with
// I_+ - I* = (g1 - 1) I* + src g2', its moments are P + src Q, and P, Q are sums of sweep 1.
#include <stdint.h>

#include <algorithm>

#include "async_copy.cuh"
#include "stage_math.cuh"

namespace rad {
namespace {

constexpr int kWarps = 4;   // warps per CTA
constexpr int kDepth = 3;   // ring slots per warp
constexpr int kCellF = 20;  // per-cell scalars fetched for the coupling: fluid (5), opacities (3), n^0, E_alphahat (4), co-triad (6), excised

__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// pairs of cells along x: position of a pair in the block and the flat index of its first cell; advancing is integer adds only
struct PairIt {
    int ip, j, k;  // pair number along x, interior row (j, k)
};
__device__ __forceinline__ PairIt pair_at(long long pid, int ppr, int n1, int kzb) {
    const long long row = pid / ppr;
    PairIt it;
    it.ip = (int)(pid - row * ppr);
    it.j = (int)(row % n1);
    it.k = (int)(row / n1) + kzb;
    return it;
}
__device__ __forceinline__ void pair_next(PairIt &it, int ppr, int n1) {
    if (++it.ip == ppr) { it.ip = 0; if (++it.j == n1) { it.j = 0; ++it.k; } }
}
__device__ __forceinline__ long long pair_cell(const DeviceTables &t, const PairIt &it, int &cnt) {
    cnt = min(2, t.n[0] - 2 * it.ip);
    return ((long long)(it.k + t.ng) * t.NJ + (it.j + t.ng)) * t.NI + (2 * it.ip + t.ng);
}

// sums over the warp of NS values per lane through shared memory: lane l writes its NS partial sums to red[q * 33 + l], lane q < NS
// adds up row q (odd row stride: the column reads of the NS lanes fall into different banks) and leaves the total in tot[q].
// red: NS * 33 doubles, tot: NS doubles, both private to the warp.  ~NS stores + 32 loads + 32 adds instead of a 5-level butterfly.
template <int NS>
__device__ __forceinline__ void warp_sums_smem(const double (&v)[NS], int lane, double *red, double *tot) {
    __syncwarp();
#pragma unroll
    for (int q = 0; q < NS; q++) red[q * 33 + lane] = v[q];
    __syncwarp();
    if (lane < NS) {
        const double *r = red + lane * 33;
        double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
#pragma unroll
        for (int i = 0; i < 32; i += 4) { s0 += r[i]; s1 += r[i + 1]; s2 += r[i + 2]; s3 += r[i + 3]; }
        tot[lane] = (s0 + s1) + (s2 + s3);
    }
    __syncwarp();
}

// per-cell scalars of the coupling, in registers
struct CellK {
    double uh0, uh1, uh2, uh3;  // tetrad-frame fluid four-velocity used in the coupling (R10; Eq.55 when the estimate applies)
    double aEdt, nup0;          // alpha_E beta dt (Eq.33b), n^0
    double E0, E1, E2, E3;      // E_alphahat: n_0 = E_0 + E_a n^a (mask)
    double live;                // 1: the cell takes part (not excised)
};
__device__ __forceinline__ CellK select(const CellK &a, const CellK &b, bool second) {
    CellK r;
    r.uh0 = second ? b.uh0 : a.uh0; r.uh1 = second ? b.uh1 : a.uh1; r.uh2 = second ? b.uh2 : a.uh2; r.uh3 = second ? b.uh3 : a.uh3;
    r.aEdt = second ? b.aEdt : a.aEdt; r.nup0 = second ? b.nup0 : a.nup0;
    r.E0 = second ? b.E0 : a.E0; r.E1 = second ? b.E1 : a.E1; r.E2 = second ? b.E2 : a.E2; r.E3 = second ? b.E3 : a.E3;
    r.live = second ? b.live : a.live;
    return r;
}

// sweep 1 for one intensity: fluid-frame factors (R11), the twelve summands, and the two numbers sweep 2 needs.
// With dd = n^0 + n^0bar alpha_E dt, rp = 1/(n^0bar dd):  dOmega_bar = dOmega / n^0bar^2, Ibar dOmega_bar = n^0bar^2 Ihat dOmega,
// A_1 = sum (n^0/dd) Ibar dOmega_bar, A_2 = dt/4pi sum dOmega rp (Eq.42), and Eq.40 back in the tetrad frame is
// Ihat_+ = g1 Ihat_- + src g2',  g1 = n^0 / dd,  g2' = 1 / (dd n^0bar^3).
__device__ __forceinline__ void sweep1_item(const CellK &c, double n0crit, const double4 an, double I, double (&acc)[12], double &a_out, double &b_out,
                                            bool &masked) {
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
    masked = n0crit > 0.0 && fabs(chain4(c.E0, c.E1, c.E2, c.E3, an.y, an.z, an.w)) < n0crit;  // |n_0| < n_0^crit (pinned chain)
    a_out = g1 * I;
    b_out = g2;
}

// ---------------------------------------------------------------------------------------------------------------------------------
// coupling.  VEST: the radiation-dominated velocity estimate of Eq.51-55 (NEXT-2; reading G8 in DESIGN.md).
// smem per warp: kDepth slots of 2 N doubles (intensities; sweep 1 leaves the masked intensities there), one buffer a[2 N], one
// buffer b[2 N], 2 x kCellF cell scalars, 8 doubles of per-cell results; per CTA: the angle table {dOmega, n^1, n^2, n^3}[N].
// ---------------------------------------------------------------------------------------------------------------------------------
struct CoupleArgs {
    double *I;
    const double *fluid, *aP, *aE, *aS;
    double dt;
    double *T_out, *dT0;
    unsigned long long *noroot;
    int kz0, kz1;  // interior planes kz0 <= k < kz1 (0-based, without ghosts); kz1 <= kz0 = the whole block
};

template <bool VEST>
__global__ void __launch_bounds__(kWarps * 32, 3) k_couple_stream(const DeviceTables t, const Params p, const CoupleArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int N = t.N, L2 = 2 * N;
    double *sm = reinterpret_cast<double *>(smem_raw);
    double4 *sAng = reinterpret_cast<double4 *>(sm);  // [N]
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int perWarp = (kDepth + 2) * L2 + 2 * kCellF + 12 * 33 + 24 + 2 * kDepth;  // doubles (the last 2 kDepth: mbarriers, 8 B each, 16 B apart)
    double *wbase = sm + 4 * N + (size_t)w * perWarp;
    double *slots = wbase, *abuf = wbase + kDepth * L2, *bbuf = abuf + L2, *scell = bbuf + L2, *red = scell + 2 * kCellF, *tot = red + 12 * 33;
    const uint32_t bar0 = smem_u32(tot + 24);
    for (int q = threadIdx.x; q < N; q += blockDim.x) sAng[q] = make_double4(t.domega[q], t.nhat[3 * q], t.nhat[3 * q + 1], t.nhat[3 * q + 2]);
    if (lane == 0) {
        for (int d = 0; d < kDepth; d++) mbar_init(bar0 + 16u * d, 1);
        fence_mbar_init();
    }
    __syncthreads();

    // pairs of cells along x: pairs per row ppr = ceil(n0 / 2); pair id -> (row, first cell)
    const int n0 = t.n[0], ppr = (n0 + 1) >> 1;
    const int kzb = a.kz1 > a.kz0 ? a.kz0 : 0, kze = a.kz1 > a.kz0 ? a.kz1 : t.n[2];
    const long long npairs = (long long)ppr * t.n[1] * (kze - kzb);
    const long long nwarp = (long long)gridDim.x * kWarps, wid = (long long)blockIdx.x * kWarps + w;
    // a warp takes a contiguous chunk of pairs (consecutive pairs are consecutive in memory)
    const long long chunk = (npairs + nwarp - 1) / nwarp, pbeg = wid * chunk, pend = min(npairs, pbeg + chunk);
    if (pbeg >= pend) return;
    PairIt cur = pair_at(pbeg, ppr, t.n[1], kzb), ahead = cur, nxt = cur;  // the pair worked on, the next pair to be copied, the next pair's scalars
    long long pahead = pbeg;
    auto issue = [&]() {  // the rows of pair `ahead` into its ring slot
        int cnt;
        const long long c = pair_cell(t, ahead, cnt);
        const int sl = (int)((pahead - pbeg) % kDepth);
        const uint32_t bar = bar0 + 16u * sl, bytes = (uint32_t)(cnt * N * 8);
        if (lane == 0) {
            fence_proxy_async();  // sweep 1 wrote into this slot through the generic proxy
            mbar_expect_tx(bar, bytes);
            bulk_g2s(smem_u32(slots + sl * L2), a.I + c * N, bytes, bar);
        }
        pair_next(ahead, ppr, t.n[1]);
        pahead++;
    };
    // the 20 per-cell scalars of a pair, fetched by the lanes one pair ahead: item q = cell * 20 + field -> lane q % 32, round q / 32
    auto fetch_cell = [&](double (&v)[2]) {  // of pair `nxt`
        int cnt;
        const long long c0 = pair_cell(t, nxt, cnt);
        pair_next(nxt, ppr, t.n[1]);
#pragma unroll
        for (int r = 0; r < 2; r++) {
            const int q = r * 32 + lane, cl = q / kCellF, f = q - cl * kCellF;
            double x = 0.0;
            if (q < 2 * kCellF && cl < cnt) {
                const long long c = c0 + cl;
                if (f < 5) x = __ldg(a.fluid + (long long)f * t.ncell + c);
                else if (f == 5) x = p.couple ? __ldg(a.aP + c) : 0.0;
                else if (f == 6) x = p.couple ? __ldg(a.aE + c) : 0.0;
                else if (f == 7) x = p.couple ? __ldg(a.aS + c) : 0.0;
                else if (f < 13) x = __ldg(t.cell + c * RAD_NCELL + (f - 8));  // n^0, E_0..3
                else if (f < 19) x = __ldg(t.cell + c * RAD_NCELL + 44 + (f - 13));  // co-triad
                else x = __ldg(t.cell + c * RAD_NCELL + 50);  // excised
            } else if (f == 19 || f == 8) x = 1.0;  // a missing second cell counts as excised (n^0 = 1 keeps its idle lanes finite)
            v[r] = x;
        }
    };
    for (int d = 0; d < kDepth - 1 && pahead < pend; d++) issue();
    double cellv[2];
    fetch_cell(cellv);
    const int s0 = N >> 5;                 // passes 0 .. s0-1 lie in cell 0
    const int s1 = (N + 31) >> 5;          // passes s1 .. lie in cell 1 (s0 == s1 when N is a multiple of 32)
    const int npass = (L2 + 31) >> 5;
    const uint32_t aS_ = smem_u32(slots), aA = smem_u32(abuf), aB = smem_u32(bbuf);

    for (long long pid = pbeg; pid < pend; pid++) {
        const int rel = (int)(pid - pbeg), sl = rel % kDepth;
        int cnt;
        const long long c0 = pair_cell(t, cur, cnt);
        pair_next(cur, ppr, t.n[1]);
        // cell scalars of this pair to shared memory, next pair's on their way
        __syncwarp();
#pragma unroll
        for (int r = 0; r < 2; r++) if (r * 32 + lane < 2 * kCellF) scell[r * 32 + lane] = cellv[r];
        if (pid + 1 < pend) fetch_cell(cellv);
        if (pahead < pend) issue();  // its slot was released at the end of the previous iteration
        __syncwarp();
        // ---- per-cell preparation: lanes 0..15 cell 0, lanes 16..31 cell 1 (all lanes of a half compute the same values)
        const int mycell = lane >> 4;
        const double *sc = scell + mycell * kCellF;
        const double rho = sc[0], Tm = sc[1], aPc = sc[5], aEc = sc[6], aSc = sc[7], nup0 = sc[8];
        const bool excised = sc[19] != 0.0, docouple = p.couple && !excised;
        CellK ck;
        ck.uh0 = 1.0; ck.uh1 = ck.uh2 = ck.uh3 = 0.0;
        ck.aEdt = docouple ? (aEc + aSc) * a.dt : 0.0;  // Eq.33b
        ck.nup0 = nup0; ck.E0 = sc[9]; ck.E1 = sc[10]; ck.E2 = sc[11]; ck.E3 = sc[12];
        ck.live = excised ? 0.0 : 1.0;
        if (docouple) {
            const double u1 = sc[2], u2 = sc[3], u3 = sc[4];
            ck.uh1 = sc[13] * u1 + sc[14] * u2 + sc[15] * u3; ck.uh2 = sc[16] * u2 + sc[17] * u3; ck.uh3 = sc[18] * u3;  // u^ahat = theta^ahat_j u^j' (R10)
            ck.uh0 = sqrt(1.0 + (ck.uh1 * ck.uh1 + ck.uh2 * ck.uh2 + ck.uh3 * ck.uh3));
        }
        mbar_wait(bar0 + 16u * sl, (uint32_t)((rel / kDepth) & 1));
        const uint32_t aSl = aS_ + (uint32_t)(sl * L2) * 8u;

        if (VEST) {
            // ---- Eq.51-55: tetrad-frame moments of I*, radiation velocity, force, clamped fractions, blended velocity
            double m[2][10];
#pragma unroll
            for (int q = 0; q < 10; q++) { m[0][q] = 0.0; m[1][q] = 0.0; }
            for (int it = 0; it < npass; it++) {
                const int f = it * 32 + lane;
                const bool second = f >= N, valid = f < cnt * N;
                const double4 an = sAng[valid ? (second ? f - N : f) : 0];
                const double w0 = valid ? lds(aSl + 8u * f) * an.x : 0.0;
                const double w1 = w0 * an.y, w2 = w0 * an.z, w3 = w0 * an.w;
                const double v10[10] = {w0, w1, w2, w3, w1 * an.y, w1 * an.z, w1 * an.w, w2 * an.z, w2 * an.w, w3 * an.w};
                if (it < s0) {
#pragma unroll
                    for (int q = 0; q < 10; q++) m[0][q] += v10[q];
                } else if (it >= s1) {
#pragma unroll
                    for (int q = 0; q < 10; q++) m[1][q] += v10[q];
                } else {
#pragma unroll
                    for (int q = 0; q < 10; q++) { m[0][q] += second ? 0.0 : v10[q]; m[1][q] += second ? v10[q] : 0.0; }
                }
            }
            warp_sums_smem<10>(m[0], lane, red, tot);
            warp_sums_smem<10>(m[1], lane, red, tot + 10);
            double M[10];
#pragma unroll
            for (int q = 0; q < 10; q++) M[q] = tot[mycell * 10 + q];
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
        // the two cells' scalars for the sweeps: cell 0's from lane 0, cell 1's from lane 16
        CellK k0, k1;
        {
            const unsigned full = 0xffffffffu;
#define RAD_BC(field) k0.field = __shfl_sync(full, ck.field, 0); k1.field = __shfl_sync(full, ck.field, 16)
            RAD_BC(uh0); RAD_BC(uh1); RAD_BC(uh2); RAD_BC(uh3); RAD_BC(aEdt); RAD_BC(nup0); RAD_BC(E0); RAD_BC(E1); RAD_BC(E2); RAD_BC(E3); RAD_BC(live);
#undef RAD_BC
        }
        // ---- sweep 1
        double acc[2][12];
#pragma unroll
        for (int q = 0; q < 12; q++) { acc[0][q] = 0.0; acc[1][q] = 0.0; }
        const double n0crit = p.n0_crit;
        auto pass1 = [&](int it, const CellK &c, double (&ac)[12], bool valid, int n) {
            const int f = it * 32 + lane;
            double4 an = sAng[n];
            double I = lds(aSl + 8u * f);
            if (!valid) { an.x = 0.0; I = 0.0; }  // an idle lane adds zeros
            double a_o, b_o;
            bool masked;
            sweep1_item(c, n0crit, an, I, ac, a_o, b_o, masked);
            if (valid) {
                if (masked && c.live != 0.0) { a_o = 0.0; b_o = 0.0; sts(aSl + 8u * f, 0.0); }
                sts(aA + 8u * f, a_o); sts(aB + 8u * f, b_o);
            }
        };
#pragma unroll 2
        for (int it = 0; it < s0; it++) pass1(it, k0, acc[0], true, it * 32 + lane);
        if (s1 > s0) {  // the straddling pass
            const int f = s0 * 32 + lane;
            const bool second = f >= N;
            const CellK ks = select(k0, k1, second);
            const bool valid = f < cnt * N;
            double tmpa[12];
#pragma unroll
            for (int q = 0; q < 12; q++) tmpa[q] = 0.0;
            pass1(s0, ks, tmpa, valid, valid ? (second ? f - N : f) : 0);
#pragma unroll
            for (int q = 0; q < 12; q++) { acc[0][q] += second ? 0.0 : tmpa[q]; acc[1][q] += second ? tmpa[q] : 0.0; }
        }
        if (cnt > 1) {
#pragma unroll 2
            for (int it = s1; it < npass; it++) {
                const int f = it * 32 + lane;
                const bool valid = f < L2;
                pass1(it, k1, acc[1], valid, valid ? f - N : 0);
            }
        }
        // ---- reduce: 24 sums -> lane l holds sum l (cell l / 16, sum l % 16)
        warp_sums_smem<12>(acc[0], lane, red, tot);
        warp_sums_smem<12>(acc[1], lane, red, tot + 12);
        double S[12];
#pragma unroll
        for (int q = 0; q < 12; q++) S[q] = tot[mycell * 12 + q];
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
        if ((lane & 15) == 0 && mycell < cnt) {
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
        // (src, coupled) of both cells to every lane
        const double src0 = __shfl_sync(0xffffffffu, coupled ? src : 0.0, 0), src1 = __shfl_sync(0xffffffffu, coupled ? src : 0.0, 16);
        const bool cp0 = __shfl_sync(0xffffffffu, (int)coupled, 0) != 0, cp1 = __shfl_sync(0xffffffffu, (int)coupled, 16) != 0;
        const bool ex0 = k0.live == 0.0, ex1 = k1.live == 0.0;
        // ---- sweep 2: Eq.40 in the tetrad frame, store
        __syncwarp();
        double *out = a.I + c0 * N;
        for (int it = 0; it < npass; it++) {
            const int f = it * 32 + lane;
            if (f >= cnt * N) break;
            const bool second = f >= N;
            if (second ? ex1 : ex0) continue;  // excised cells keep what the transport wrote (0)
            const double Iold = lds(aSl + 8u * f);
            double Inew = Iold;
            if (second ? cp1 : cp0) Inew = fma(second ? src1 : src0, lds(aB + 8u * f), lds(aA + 8u * f));
            out[f] = Inew;
        }
        __syncwarp();  // the slot is free for the copy issued at the top of the next iteration
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
    // position of a group in the block, advanced by integer adds only: (group along x, row j, plane k) and the flat index of its first cell
    struct GroupIt { int ig, j, k; long long c; };
    auto group_at = [&](long long g) {
        const long long row = g / gpr;
        GroupIt it;
        it.ig = (int)(g - row * gpr); it.j = (int)(row % t.n[1]); it.k = (int)(row / t.n[1]);
        it.c = ((long long)(it.k + t.ng) * t.NJ + (it.j + t.ng)) * t.NI + (kMomCells * it.ig + t.ng);
        return it;
    };
    auto group_next = [&](GroupIt &it) {
        it.c += kMomCells;
        if (++it.ig == gpr) {
            it.ig = 0; it.c += t.NI - (long long)kMomCells * gpr;
            if (++it.j == t.n[1]) { it.j = 0; ++it.k; it.c += (long long)t.NI * (t.NJ - t.n[1]); }
        }
    };
    GroupIt cur = group_at(gbeg), ahead = cur;
    long long gahead = gbeg;
    int sl_ahead = 0;
    auto issue = [&]() {  // the rows of group `ahead` into its ring slot, one bulk copy per cell
        const int cnt = min(kMomCells, t.n[0] - kMomCells * ahead.ig);
        const uint32_t bar = bar0 + 16u * sl_ahead;
        if (lane == 0) mbar_expect_tx(bar, (uint32_t)(cnt * N * 8));
        __syncwarp();
        if (lane < cnt) bulk_g2s(smem_u32(slots + (sl_ahead * kMomCells + lane) * Np), I + (ahead.c + lane) * N, (uint32_t)(N * 8), bar);
        group_next(ahead);
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
        group_next(cur);
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

size_t couple_smem(int N) { return sizeof(double) * (4 * (size_t)N + (size_t)kWarps * ((kDepth + 2) * 2 * N + 2 * kCellF + 12 * 33 + 24 + 2 * kDepth)); }
size_t moments_smem(int N, int warps, int depth) {
    const int nk = (N + 3) / 4;
    return sizeof(double) * ((size_t)nk * 40 + (size_t)warps * (depth * kMomCells * mom_row_stride(N) + kMomCells * 10 + kMomCells * kMomCellF + 2 * depth));
}

}  // namespace

// 1 if the streaming kernels serve this angle grid and these arrays: rows must be multiples of 16 bytes (bulk copies).
// I == nullptr asks about the angle grid alone.
int stream_serves(const DeviceTables &t, const void *I) {
    return (t.N & 1) == 0 && ((uintptr_t)I & 15) == 0 && couple_smem(t.N) <= (size_t)t.smem_optin;
}

// returns 1 (launched), 0 (not served), -1 (CUDA error)
int launch_couple_stream(const DeviceTables &t, const Params &p, double *I, const double *fluid, const double *aP, const double *aE, const double *aS,
                         double dt, double *T_out, double *dT0, unsigned long long *noroot, cudaStream_t s, int kz0, int kz1) {
    if (!stream_serves(t, I)) return 0;
    const size_t smem = couple_smem(t.N);
    CoupleArgs a{I, fluid, aP, aE, aS, dt, T_out, dT0, noroot, kz0, kz1};
    const int per_sm = (int)std::max<size_t>(1, std::min<size_t>(8, (size_t)t.smem_optin / (smem + 1024)));
    const int grid = t.sms * per_sm;
    if (p.vel_estimate && p.couple) {
        if (cudaFuncSetAttribute(k_couple_stream<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return -1;
        k_couple_stream<true><<<grid, kWarps * 32, smem, s>>>(t, p, a);
    } else {
        if (cudaFuncSetAttribute(k_couple_stream<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return -1;
        k_couple_stream<false><<<grid, kWarps * 32, smem, s>>>(t, p, a);
    }
    return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

int launch_moments_stream(const DeviceTables &t, const double *I, int frame, const double *fluid, double *out, cudaStream_t s) {
    if ((t.N & 1) || ((uintptr_t)I & 15)) return 0;
    // ring depth 3 and as many warps as shared memory holds (<= 8); deeper rings do not pay once ~100 KB are in flight per SM
    int depth = 2, warps = 12;
    while (warps > 2 && moments_smem(t.N, warps, depth) > (size_t)t.smem_optin) warps--;
    if (moments_smem(t.N, warps, depth) > (size_t)t.smem_optin) depth = 2;
    const size_t smem = moments_smem(t.N, warps, depth);
    if (smem > (size_t)t.smem_optin) return 0;
    const int per_sm = (int)std::max<size_t>(1, std::min<size_t>(4, (size_t)t.smem_optin / (smem + 1024)));
    if (cudaFuncSetAttribute(k_moments_mma, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return -1;
    k_moments_mma<<<t.sms * per_sm, warps * 32, smem, s>>>(t, I, frame, fluid, out, depth);
    return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

}  // namespace rad
