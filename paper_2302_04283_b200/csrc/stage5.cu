// stage5.cu -- the fused flux-divergence kernel (north_star subsystem 2), angle-resident version: spatial + angular flux
// divergence (Eq.22, 24, 25) and cons -> prim in ONE launch; the implicit coupling follows in its own streaming kernel
// (stream.cu; the two-kernel stage measured faster than the single launch that also held the coupling).
//
// Mapping:
//   * a CTA owns a TY x TZ tile of cell columns in the y-z plane and marches along x through KX cells.  A cell is served
//     by WPC warps; a thread keeps NITER FIXED angles for the whole march, so the angle's direction, solid angle and
//     edge-ownership record live in registers, and so does the x stencil (I of planes i-1 .. i+2 is rotated, one new
//     value per step) and the flux through the lower x face (carried).
//   * every face flux is computed ONCE: a cell computes the flux through its upper y and z faces and publishes it in
//     shared memory; the neighbour above takes it as its lower-face flux after the CTA barrier of the step (only the
//     cells on the low edges of the tile compute their lower faces themselves).
//   * shared memory is filled by bulk asynchronous copies (TMA, 1-D) two steps ahead, completion on two mbarriers, into one
//     of two PAGES (step parity): the tile's own rows and the 2-deep halo rows of the current plane, the own rows two planes
//     ahead (the x stencil's new value), the stored angular-edge coefficients of each cell (the owner of an edge overwrites
//     the coefficient with the edge flux, the partner angle pulls it from there) and the published face fluxes; the packed
//     per-cell geometry records have 4 buffers of their own.  Every address of a step is page base + a loop-invariant offset,
//     and the step loop is unrolled by two, so the page is a compile-time choice.  One __syncthreads per step.
//   * TAU (template): the optical-depth-aware spatial flux of Eq.26-29 -- a per-cell table (k_tau_table) of u^alphahat and f/2
//     of the upper faces comes in with the other copies for the tile's cells and the halo cells at distance 1.
#include <cstdio>

#include "async_copy.cuh"
#include "flux_math.cuh"
#include "stage_math.cuh"

namespace rad {
namespace {

constexpr int RECN = RAD_STAGE_RECN;  // packed per-cell record, see k_pack_rec
constexpr int USTR = 52;              // a cell's record slot in shared memory: [0..35] record, [36..43] lower y face, [44..51] lower z face

template <int TY_, int TZ_, int WPC_, bool TAU_ = false>
struct Tile {
    static constexpr int TY = TY_, TZ = TZ_, WPC = WPC_;
    static constexpr bool TAU = TAU_;  // optical-depth-aware flux (Eq.26-29): per-cell velocity records of the tile and its 1-deep halo
    static constexpr int NVH = 2 * TZ + 2 * TY;  // halo cells at distance 1 (no corners)
    static constexpr int NC = TY * TZ, NH = 4 * TZ + 4 * TY, NR0 = 4 * NC + NH + TY + TZ, NR = NR0 + (TAU ? NC + NVH : 0), NT = NC * WPC * 32;
    static constexpr int NFY = (TY - 1) * TZ, NFZ = TY * (TZ - 1);
};

// Shared memory: two PAGES (step parity), each holding everything that changes with the step and is dead after the step's CTA
// barrier -- the tile's own rows of plane s, the halo rows of plane s, the own rows of plane s + 2 (the x stencil's new value), the
// edge coefficients, the published face fluxes (TAU: the velocity records of the halo cells) -- so that every address of a step is
// (page base + thread offset) + a loop-invariant offset; then the packed records (4 buffers: read after the barrier too).
struct Layout5 {
    int Np, Kp, pHalo, pAhead, pE, pFy, pFz, pFx, pVh, PG, oPage, oU, oRole, oV, oBar, total;  // offsets in doubles (p*: inside a page)
};
template <class T>
__host__ __device__ inline Layout5 make_layout5(int N) {
    Layout5 L;
    L.Np = (N + 1) & ~1;
    L.Kp = (3 * N + 3) & ~1;  // 3 N coefficients / fluxes + the always-zero slot 3N
    L.pHalo = T::NC * L.Np;
    L.pAhead = L.pHalo + T::NH * L.Np;
    L.pE = L.pAhead + T::NC * L.Np;
    L.pFy = L.pE + T::NC * L.Kp;
    L.pFz = L.pFy + T::NFY * L.Np;
    L.pFx = L.pFz + T::NFZ * L.Np;  // the lower z face of cell (0,0), computed by cell (1,1) (load balance)
    L.pVh = L.pFx + L.Np;           // TAU: velocity records (8 doubles) of the halo cells at distance 1
    L.PG = L.pVh + (T::TAU ? T::NVH * 8 : 0);
    L.oPage = 0;
    L.oU = L.oPage + 2 * L.PG;
    L.oRole = L.oU + 4 * T::NC * USTR;
    L.oV = L.oRole + T::NR * 4;     // TAU: velocity records of the own cells, 4 buffers
    L.oBar = L.oV + (T::TAU ? 4 * T::NC * 8 : 0);
    L.total = L.oBar + 3;  // two mbarriers, then the bytes of one step's copies
    return L;
}

// one bulk copy per step: what thread `r` of the CTA brings in for step u (source advances by `stride` doubles per step,
// destination cycles through nbuf buffers `dstride` doubles apart)
struct Role {
    const double *src0;
    int stride, dst0, dstride, nbufm1, boff, bytes;
};
static_assert(sizeof(Role) == 32, "Role is stored as four doubles");

// TAU: G = -(1 + 1/n^0bar) of a cell for one angle, n^0bar = u^0hat - u^ahat n^ahat (Eq.29)
__device__ __forceinline__ double tau_G(double u0, double u1, double u2, double u3, double n1, double n2, double n3) {
    return -(1.0 + rcp3(u0 - (u1 * n1 + u2 * n2 + u3 * n3)));
}

// ------------------------------------------------------------------------------------------------------------------
template <int NITER, int WPC, int TY, int TZ, int MINB, bool PLM, bool TAU>
__global__ void __launch_bounds__(TY *TZ *WPC * 32, MINB)
    k_stage5(const DeviceTables t, const Params p, const StageArgs a, const Layout5 L, const int KX) {
    using T = Tile<TY, TZ, WPC, TAU>;
    constexpr int NC = T::NC, NH = T::NH, NR = T::NR;
    constexpr uint32_t ITB = WPC * 32 * 8;  // byte distance between a thread's consecutive angles
    extern __shared__ __align__(16) unsigned char smem_raw[];
    double *sm = reinterpret_cast<double *>(smem_raw);
    const uint32_t smb = smem_u32(sm);
    const int N = t.N;
    const int Np = L.Np, Kp = L.Kp;
    const int tid = threadIdx.x, lane = tid & 31;
    const int w = __shfl_sync(0xffffffffu, tid >> 5, 0);  // warp-uniform by construction
    const int cs = w / WPC, wc = w - cs * WPC;
    const int wy = cs % TY, wz = cs / TY;
    const uint32_t bar0 = smb + 8u * L.oBar;
    Role *roles = reinterpret_cast<Role *>(sm + L.oRole);

    const int ng = t.ng;
    const int kzb = a.kz1 > a.kz0 ? a.kz0 : 0, kze = a.kz1 > a.kz0 ? a.kz1 : t.n[2];  // the slab of interior planes this launch updates
    const int j0 = blockIdx.y * TY + ng, k0 = blockIdx.z * TZ + ng + kzb;
    const int j = j0 + wy, k = k0 + wz;
    const bool active = j < t.n[1] + ng && k < kze + ng;
    const int i_begin = blockIdx.x * KX + ng, i_end = min(i_begin + KX, t.n[0] + ng), nsteps = i_end - i_begin;
    const long long c_first = ((long long)k * t.NJ + j) * t.NI + i_begin;

    // ---- copy roles
    if (tid < NR) {
        Role r;
        r.src0 = nullptr; r.stride = 0; r.dst0 = 0; r.dstride = 0; r.nbufm1 = 0; r.boff = 0; r.bytes = 0;
        const int row_bytes = N * 8;
        if (tid < NC + NH) {
            int jj, kk;
            if (tid < NC) { jj = j0 + tid % TY; kk = k0 + tid / TY; }
            else {
                const int h = tid - NC;
                if (h < 4 * TZ) { const int hz = h >> 2, q = h & 3; kk = k0 + hz; jj = j0 + (q < 2 ? q - 2 : TY + q - 2); }
                else { const int hh = h - 4 * TZ, hy = hh >> 2, q = hh & 3; jj = j0 + hy; kk = k0 + (q < 2 ? q - 2 : TZ + q - 2); }
            }
            if (jj < t.NJ && kk < t.NK) {
                const long long c0 = ((long long)kk * t.NJ + jj) * t.NI + i_begin;
                r.stride = N; r.bytes = row_bytes;
                r.src0 = a.I_in + c0 * N; r.dstride = L.PG; r.nbufm1 = 1;
                r.dst0 = L.oPage + (tid < NC ? tid * Np : L.pHalo + (tid - NC) * Np);
            }
        } else if (TAU && tid >= T::NR0) {
            // velocity records (8 doubles: u^alphahat, f/2 of the three upper faces, pad) of plane u: the own cells (4 buffers) and
            // the halo cells at distance 1 (2 buffers; index: y halo wz * 2 + {below, above}, z halo 2 TZ + wy * 2 + {below, above})
            const int q = tid - T::NR0;
            int jj, kk;
            if (q < NC) { jj = j0 + q % TY; kk = k0 + q / TY; r.dst0 = L.oV + q * 8; r.dstride = NC * 8; r.nbufm1 = 3; }
            else {
                const int h = q - NC;
                if (h < 2 * TZ) { kk = k0 + (h >> 1); jj = (h & 1) ? j0 + TY : j0 - 1; }
                else { jj = j0 + ((h - 2 * TZ) >> 1); kk = ((h - 2 * TZ) & 1) ? k0 + TZ : k0 - 1; }
                r.dst0 = L.oPage + L.pVh + h * 8; r.dstride = L.PG; r.nbufm1 = 1;
            }
            if (jj < t.NJ && kk < t.NK) {
                r.src0 = a.vel8 + (((long long)kk * t.NJ + jj) * t.NI + i_begin) * 8; r.stride = 8; r.bytes = 64;
            }
        } else {
            const int q = tid - NC - NH;
            int kind, ccs;  // 0 edge coefficients, 1 cell record, 2 lower y face, 3 lower z face, 4 own row of plane u + 2
            if (q < NC) { kind = 0; ccs = q; }
            else if (q < 2 * NC) { kind = 1; ccs = q - NC; }
            else if (q < 2 * NC + TZ) { kind = 2; ccs = (q - 2 * NC) * TY; }
            else if (q < 2 * NC + TZ + TY) { kind = 3; ccs = q - 2 * NC - TZ; }
            else { kind = 4; ccs = q - 2 * NC - TZ - TY; }
            const int jj = j0 + ccs % TY, kk = k0 + ccs / TY;
            if (jj < t.n[1] + ng && kk < kze + ng) {
                const long long c0 = ((long long)kk * t.NJ + jj) * t.NI + i_begin;
                if (kind == 4) {
                    r.src0 = a.I_in + (c0 + 2) * N; r.stride = N; r.dst0 = L.oPage + L.pAhead + ccs * Np; r.dstride = L.PG; r.nbufm1 = 1; r.bytes = row_bytes;
                } else if (kind == 0) {
                    const long long ci = ((long long)(kk - ng) * t.n[1] + (jj - ng)) * t.n[0] + (i_begin - ng);
                    r.src0 = t.ke + ci * 3 * N; r.stride = 3 * N; r.dst0 = L.oPage + L.pE + ccs * Kp; r.dstride = L.PG; r.nbufm1 = 1; r.bytes = 3 * row_bytes;
                } else {
                    r.stride = RECN; r.dstride = NC * USTR; r.nbufm1 = 3;
                    if (kind == 1) { r.src0 = t.rec + c0 * RECN; r.dst0 = L.oU + ccs * USTR; r.bytes = RECN * 8; }
                    else if (kind == 2) { r.src0 = t.rec + (c0 - t.NI) * RECN + 8; r.dst0 = L.oU + ccs * USTR + 36; r.bytes = 64; }
                    else { r.src0 = t.rec + (c0 - (long long)t.NI * t.NJ) * RECN + 16; r.dst0 = L.oU + ccs * USTR + 44; r.bytes = 64; }
                }
            }
        }
        roles[tid] = r;
    }
    if (wc == 0 && lane < 2) {  // the always-zero flux slot of both coefficient buffers
        sm[L.oPage + lane * L.PG + L.pE + cs * Kp + 3 * N] = 0.0;
        if (3 * N + 1 < Kp) sm[L.oPage + lane * L.PG + L.pE + cs * Kp + 3 * N + 1] = 0.0;
    }
    if (tid == 0) {
        mbar_init(bar0, 1); mbar_init(bar0 + 8u, 1);
        fence_mbar_init();
    }
    __syncthreads();
    if (tid == 0) {
        uint32_t step_bytes = 0;
        for (int r = 0; r < NR; r++) step_bytes += (uint32_t)roles[r].bytes;
        mbar_expect_tx(bar0, step_bytes);
        if (nsteps > 1) mbar_expect_tx(bar0 + 8u, step_bytes);
        *reinterpret_cast<uint32_t *>(sm + L.oBar + 2) = step_bytes;
    }
    __syncthreads();
    // everything step u needs, signalled on full[u & 1]: own and halo rows of plane u, own rows of plane u + 2, coefficients and
    // records of the cells of plane u
    const int myrole = (tid >> 5) + (T::NT / 32) * lane;  // the copies of a step are spread over all warps (a warp issues its lanes' copies one by one)
    auto issue = [&](int u) {
        const Role r = roles[myrole];
        if (r.bytes) {
            const int buf = (u + r.boff) & r.nbufm1;
            bulk_g2s(smb + 8u * (uint32_t)(r.dst0 + buf * r.dstride), r.src0 + (long long)u * r.stride, (uint32_t)r.bytes, bar0 + 8u * (u & 1));
        }
    };
    if (myrole < NR) {
        issue(0);
        if (nsteps > 1) issue(1);
    }

    // ---- the thread's angles: n = lane + 32 wc + 32 WPC it.  Only the last one can fall past N; such a slot is idle:
    // it reads angle 0, has zero weights, pulls from the always-zero flux slot and stores nothing.
    const int nbase = wc * 32 + lane;
    const bool last_valid = nbase + (NITER - 1) * WPC * 32 < N;
    const uint32_t lane8 = (uint32_t)nbase * 8u;                                      // byte offset of angle it: lane8 + it * ITB ...
    const uint32_t last8 = last_valid ? lane8 + (NITER - 1) * ITB : 0u;              // ... except the last
    unsigned rx[NITER], ry[NITER], rz[NITER];
    double n1[NITER], n2[NITER], n3[NITER], winv[NITER];
#pragma unroll
    for (int it = 0; it < NITER; it++) {
        const bool v = it < NITER - 1 || last_valid;
        const int n = v ? nbase + it * WPC * 32 : 0;
        n1[it] = t.nhat[3 * n]; n2[it] = t.nhat[3 * n + 1]; n3[it] = t.nhat[3 * n + 2];
        winv[it] = v ? t.winv[n] : 0.0;
        const uint4 rec = reinterpret_cast<const uint4 *>(t.ang_rec)[n];
        const unsigned z = 24u * (unsigned)N;  // byte offset of the always-zero slot 3 N
        rx[it] = v ? rec.x : 0u; ry[it] = v ? rec.y : (z << 16); rz[it] = v ? rec.z : (z | (z << 16));
    }
#define OFF8(it) ((it) < NITER - 1 ? lane8 + (uint32_t)(it) * ITB : last8)

    // ---- x stencil and the flux through the lower x face of the first cell (carried from then on)
    double xm1[NITER], x0[NITER], xp1[NITER], carry[NITER];
#pragma unroll
    for (int it = 0; it < NITER; it++) { xm1[it] = 0.0; x0[it] = 0.0; xp1[it] = 0.0; carry[it] = 0.0; }
    if (active) {
        const double *Ic = a.I_in + c_first * N;
        const double *fr = t.rec + (c_first - 1) * RECN;
        const FaceRec f = {__ldg(fr), __ldg(fr + 1), __ldg(fr + 2), __ldg(fr + 3), __ldg(fr + 4), __ldg(fr + 5), __ldg(fr + 6), __ldg(fr + 7)};
#pragma unroll
        for (int it = 0; it < NITER; it++) {
            const int n = OFF8(it) >> 3;
            const double xm2 = PLM ? __ldg(Ic - 2 * N + n) : 0.0;
            xm1[it] = __ldg(Ic - N + n); x0[it] = __ldg(Ic + n); xp1[it] = __ldg(Ic + N + n);
            double GL = 0.0, GR = 0.0, fhx = 0.0;
            if (TAU) {
                const double *vL = a.vel8 + (c_first - 1) * 8, *vR = a.vel8 + c_first * 8;
                GL = tau_G(__ldg(vL), __ldg(vL + 1), __ldg(vL + 2), __ldg(vL + 3), n1[it], n2[it], n3[it]);
                GR = tau_G(__ldg(vR), __ldg(vR + 1), __ldg(vR + 2), __ldg(vR + 3), n1[it], n2[it], n3[it]);
                fhx = __ldg(vL + 4);
            }
            carry[it] = face_flux<PLM, TAU>(f, n1[it], n2[it], n3[it], xm2, xm1[it], x0[it], xp1[it], GL, GR, fhx);
        }
    }
    const int barid = 1 + cs;
    // loop-invariant byte offsets inside a page (warp-uniform): the eight stencil neighbours' rows, the cell's own row, its row two
    // planes ahead, its coefficients, where it publishes and takes face fluxes
    uint32_t nbOff[8];
#pragma unroll
    for (int q = 0; q < 8; q++) {
        const int dq = (q & 3) < 2 ? (q & 3) - 2 : (q & 3) - 1;  // -2, -1, +1, +2
        int row;
        if (q < 4) {
            const int yy = wy + dq;
            if (yy >= 0 && yy < TY) row = wz * TY + yy;
            else row = NC + wz * 4 + (yy < 0 ? yy + 2 : yy - TY + 2);
        } else {
            const int zz = wz + dq;
            if (zz >= 0 && zz < TZ) row = zz * TY + wy;
            else row = NC + 4 * TZ + wy * 4 + (zz < 0 ? zz + 2 : zz - TZ + 2);
        }
        nbOff[q] = (uint32_t)(row * Np) * 8u;  // (the halo rows follow the NC own rows)
    }
    const uint32_t ownOff = (uint32_t)(cs * Np) * 8u, aheadOff = 8u * (uint32_t)(L.pAhead + cs * Np), eOff = 8u * (uint32_t)(L.pE + cs * Kp);
    const uint32_t pubY = 8u * (uint32_t)(L.pFy + (wz * (TY - 1) + wy) * Np), pubZ = 8u * (uint32_t)(L.pFz + (wz * TY + wy) * Np), fxOff = 8u * (uint32_t)L.pFx;
    const uint32_t aPage = smb + 8u * L.oPage, pageB = 8u * (uint32_t)L.PG, N8p = 8u * (uint32_t)Np;
    const uint32_t aU0 = smb + 8u * (uint32_t)(L.oU + cs * USTR);
    // load balance: cell (0,0) would compute five faces (x, upper y and z, lower y and z), cell (1,1) three; cell (1,1)
    // takes over the lower z face of cell (0,0)
    const bool helped = TY >= 2 && TZ >= 2 && j0 + 1 < t.n[1] + ng && k0 + 1 < kze + ng;
    const bool is_helper = helped && cs == TY + 1, is_helpee = helped && cs == 0;
    const uint32_t N8 = (uint32_t)N * 8u;
    double *outp = a.I_out + c_first * N;
    const double *I0p = a.I0 ? a.I0 + c_first * N : nullptr;

#pragma unroll 2  // (with the pages, a step's parity becomes a compile-time constant: C3 5.07 -> 4.80 ms; unrolling by 4: 4.88)
    for (int s = 0; s < nsteps; s++) {
        const int b = s & 1;
        mbar_wait(bar0 + 8u * b, (s >> 1) & 1);
        if (TAU && s + 1 < nsteps) mbar_wait(bar0 + 8u * (b ^ 1), ((s + 1) >> 1) & 1);  // the velocity records of plane s+1 (x face above)
        if (tid == 0 && s + 2 < nsteps) mbar_expect_tx(bar0 + 8u * b, *reinterpret_cast<volatile uint32_t *>(sm + L.oBar + 2));  // re-armed for step s+2 (copies start after the barrier below)
        const uint32_t pg = aPage + (uint32_t)b * pageB;   // this step's page
        const uint32_t aEb = pg + eOff;
        uint32_t tb[NITER];                                // page base + the thread's angle offset
#pragma unroll
        for (int it = 0; it < NITER; it++) tb[it] = pg + OFF8(it);
        const uint32_t aUb = aU0 + (uint32_t)(s & 3) * (NC * USTR * 8u);
        double d[NITER], xp2[NITER];
#pragma unroll
        for (int it = 0; it < NITER; it++) asm volatile("" : "+r"(rx[it]), "+r"(ry[it]), "+r"(rz[it]));  // unpack per step: the unpacked offsets would be spilled

        if (active) {
            const uint32_t ownrow = pg + ownOff;
#pragma unroll
            for (int it = 0; it < NITER; it++) xp2[it] = lds(tb[it] + aheadOff);
            // ---- angular fluxes (Eq.25, donor cell in angle): owners turn q_e into the edge flux in place
#pragma unroll
            for (int it = 0; it < NITER; it++) {  // loads first, stores last: the volatile accesses keep their order
                const unsigned pj[3] = {rx[it] & 0xffffu, rx[it] >> 16, ry[it] & 0xffffu};
                const uint32_t qa = tb[it] + eOff;
                double q[3], G[3];
#pragma unroll
                for (int jj = 0; jj < 3; jj++) q[jj] = lds(qa + (uint32_t)jj * N8);  // unused slots have q = 0
#pragma unroll
                for (int jj = 0; jj < 3; jj++) {
                    const bool owner_up = (__double2loint(q[jj]) & 1) != 0;
                    G[jj] = lds_unless(ownrow + pj[jj], owner_up, x0[it]);  // the upwind intensity: the thread's own (in a register) or the partner's
                }
#pragma unroll
                for (int jj = 0; jj < 3; jj++) G[jj] *= q[jj];
                d[it] = (G[0] + G[1]) + G[2];
                if (it < NITER - 1 || last_valid) {
#pragma unroll
                    for (int jj = 0; jj < 3; jj++) sts(qa + (uint32_t)jj * N8, G[jj]);
                }
            }
            if (WPC > 1) named_bar_sync(barid, WPC * 32); else __syncwarp();
#pragma unroll
            for (int it = 0; it < NITER; it++) {
                const double pulled = (lds(aEb + (ry[it] >> 16)) + lds(aEb + (rz[it] & 0xffffu))) + lds(aEb + (rz[it] >> 16));  // unused -> slot 3N = 0
                d[it] = (d[it] - pulled) * winv[it];
            }
            // ---- spatial fluxes (Eq.24).  x: the upper face; the lower one is carried
            double G0[NITER];  // TAU: G of this cell per angle
            const uint32_t vOwn = smb + 8u * (uint32_t)(L.oV + ((s & 3) * NC + cs) * 8), vHal = pg + 8u * (uint32_t)L.pVh;
            double2 own46 = make_double2(0.0, 0.0);  // f/2 of the upper x and y faces
            double own6 = 0.0;                       // ... and of the upper z face
            if (TAU) {
                const double2 u01 = lds2(vOwn), u23 = lds2(vOwn + 16);
                own46 = lds2(vOwn + 32); own6 = lds(vOwn + 48);
#pragma unroll
                for (int it = 0; it < NITER; it++) G0[it] = tau_G(u01.x, u01.y, u23.x, u23.y, n1[it], n2[it], n3[it]);
            }
            {
                const FaceRec f = lds_face(aUb);
                double2 x01 = make_double2(1.0, 0.0), x23 = make_double2(0.0, 0.0);
                if (TAU) {
                    if (s + 1 < nsteps) { const uint32_t vXp = smb + 8u * (uint32_t)(L.oV + (((s + 1) & 3) * NC + cs) * 8); x01 = lds2(vXp); x23 = lds2(vXp + 16); }
                    else { const double *vg = a.vel8 + (c_first + s + 1) * 8; x01 = make_double2(__ldg(vg), __ldg(vg + 1)); x23 = make_double2(__ldg(vg + 2), __ldg(vg + 3)); }
                }
#pragma unroll
                for (int it = 0; it < NITER; it++) {
                    const double F = face_flux<PLM, TAU>(f, n1[it], n2[it], n3[it], xm1[it], x0[it], xp1[it], xp2[it], TAU ? G0[it] : 0.0,
                                                         TAU ? tau_G(x01.x, x01.y, x23.x, x23.y, n1[it], n2[it], n3[it]) : 0.0, own46.x);
                    d[it] += F - carry[it];
                    carry[it] = F;
                }
            }
            // y and z: the upper face, published for the neighbour above; the lower face only on the low edge of the tile
#pragma unroll
            for (int ax = 1; ax <= 2; ax++) {
                const int q0 = ax == 1 ? 0 : 4;
                const uint32_t rm2 = nbOff[q0], rm1 = nbOff[q0 + 1], rp1 = nbOff[q0 + 2], rp2 = nbOff[q0 + 3];  // (offsets: added to tb[it])
                const bool low_edge = (ax == 1 ? wy : wz) == 0, publish = ax == 1 ? wy < TY - 1 : wz < TZ - 1;
                const uint32_t pub = ax == 1 ? pubY : pubZ;
                const FaceRec fh = lds_face(aUb + 64 * ax);
                double2 q01 = make_double2(1.0, 0.0), q23 = make_double2(0.0, 0.0);  // TAU: velocity of the cell above along this axis
                if (TAU) {
                    const bool inside = ax == 1 ? wy + 1 < TY : wz + 1 < TZ;
                    const uint32_t vq = inside ? vOwn + (uint32_t)(ax == 1 ? 1 : TY) * 64u : vHal + (uint32_t)(ax == 1 ? wz * 2 + 1 : 2 * TZ + wy * 2 + 1) * 64u;
                    q01 = lds2(vq); q23 = lds2(vq + 16);
                }
                const double fhu = ax == 1 ? own46.y : own6;
                // the upper face lies between this cell (x0, in a register) and the cell above (p1); the cell behind the upwind one
                // (below: m1, above: p2) is loaded from the row the sign of n^a selects
                FaceGeom gu[NITER];
                double p1[NITER], far[NITER], F[NITER];
#pragma unroll
                for (int it = 0; it < NITER; it++) {
                    gu[it] = face_geom(fh, n1[it], n2[it], n3[it]);
                    p1[it] = lds(tb[it] + rp1);
                    far[it] = PLM ? lds(tb[it] + (gu[it].neg ? rp2 : rm1)) : 0.0;
                }
#pragma unroll
                for (int it = 0; it < NITER; it++) {
                    F[it] = face_value<PLM, TAU>(gu[it], gu[it].neg ? p1[it] : x0[it], far[it], p1[it] - x0[it], TAU ? G0[it] : 0.0,
                                                 TAU ? tau_G(q01.x, q01.y, q23.x, q23.y, n1[it], n2[it], n3[it]) : 0.0, fhu);
                    d[it] += F[it];
                }
                if (publish) {
#pragma unroll
                    for (int it = 0; it < NITER; it++)
                        if (it < NITER - 1 || last_valid) sts(tb[it] + pub, F[it]);
                }
                if (low_edge && !(ax == 2 && is_helpee)) {
                    const FaceRec fl = lds_face(aUb + (ax == 1 ? 8 * 36 : 8 * 44));
                    double2 l01 = make_double2(1.0, 0.0), l23 = make_double2(0.0, 0.0);
                    double fhl = 0.0;  // TAU: the cell below is a halo cell; f/2 of this face is its upper-face entry
                    if (TAU) {
                        const uint32_t vq = vHal + (uint32_t)(ax == 1 ? wz * 2 : 2 * TZ + wy * 2) * 64u;
                        l01 = lds2(vq); l23 = lds2(vq + 16); fhl = lds(vq + (ax == 1 ? 40 : 48));
                    }
#pragma unroll
                    for (int it = 0; it < NITER; it++) {  // the lower face: between the cell below (m1) and this one
                        const FaceGeom gl = face_geom(fl, n1[it], n2[it], n3[it]);
                        const double m1 = lds(tb[it] + rm1);
                        const double farl = PLM ? (gl.neg ? p1[it] : lds_unless(tb[it] + rm2, gl.neg, 0.0)) : 0.0;
                        d[it] -= face_value<PLM, TAU>(gl, gl.neg ? x0[it] : m1, farl, x0[it] - m1,
                                                      TAU ? tau_G(l01.x, l01.y, l23.x, l23.y, n1[it], n2[it], n3[it]) : 0.0, TAU ? G0[it] : 0.0, fhl);
                    }
                }
            }
        }
        if (is_helper) {  // lower z face of cell (0,0): rows z-2, z-1 of column 0 are halo rows, z and z+1 ring rows
            // (page offsets) rows z-2, z-1 of column 0: the first two z halo rows; z: own row 0; z+1: own row TY
            const uint32_t r_m2 = (uint32_t)((NC + 4 * TZ) * Np) * 8u, r_m1 = (uint32_t)((NC + 4 * TZ + 1) * Np) * 8u, r_0 = 0u, r_p1 = (uint32_t)(TY * Np) * 8u;
            const FaceRec fl = lds_face(aUb - (uint32_t)cs * (USTR * 8u) + 8 * 44);
            double2 l01 = make_double2(1.0, 0.0), l23 = make_double2(0.0, 0.0), r01 = l01, r23 = l23;
            double fhl = 0.0;
            if (TAU) {  // cell (0,0) and the halo cell below it in z
                const uint32_t vl = pg + 8u * (uint32_t)(L.pVh + 2 * TZ * 8), vr = smb + 8u * (uint32_t)(L.oV + ((s & 3) * NC) * 8);
                l01 = lds2(vl); l23 = lds2(vl + 16); fhl = lds(vl + 48); r01 = lds2(vr); r23 = lds2(vr + 16);
            }
            double q0[NITER];
#pragma unroll
            for (int it = 0; it < NITER; it++) {
                const FaceGeom gl = face_geom(fl, n1[it], n2[it], n3[it]);
                const double q1 = lds(tb[it] + r_m1), q2 = lds(tb[it] + r_0);
                const double farl = PLM ? lds(tb[it] + (gl.neg ? r_p1 : r_m2)) : 0.0;
                q0[it] = face_value<PLM, TAU>(gl, gl.neg ? q2 : q1, farl, q2 - q1, TAU ? tau_G(l01.x, l01.y, l23.x, l23.y, n1[it], n2[it], n3[it]) : 0.0,
                                              TAU ? tau_G(r01.x, r01.y, r23.x, r23.y, n1[it], n2[it], n3[it]) : 0.0, fhl);
            }
#pragma unroll
            for (int it = 0; it < NITER; it++)
                if (it < NITER - 1 || last_valid) sts(tb[it] + fxOff, q0[it]);
        }
        // the edge fluxes (written over the coefficients) and the published face fluxes went through the generic proxy; the copies of
        // step s + 2 overwrite the same bytes through the asynchronous proxy: every writer fences before the barrier
        fence_proxy_async();
        __syncthreads();  // the fluxes of this plane are published; nobody reads the rows, halo and coefficients of plane s any more
        if (s + 2 < nsteps && myrole < NR) issue(s + 2);
        if (!active) continue;

        if (is_helpee) {
#pragma unroll
            for (int it = 0; it < NITER; it++) d[it] -= lds(tb[it] + fxOff);
        }

        if (wy > 0) {
#pragma unroll
            for (int it = 0; it < NITER; it++) d[it] -= lds(tb[it] + (pubY - N8p));  // what the cell below in y published
        }
        if (wz > 0) {
#pragma unroll
            for (int it = 0; it < NITER; it++) d[it] -= lds(tb[it] + (pubZ - (uint32_t)TY * N8p));  // ... in z
        }
        // ---- flux-divergence update of C = n^0 n_0 I (Eq.22, stage form R8), cons -> prim
        const double2 c01 = lds2(aUb + 8 * 24);
        const bool excised = c01.y != 0.0;
        const double2 w01 = lds2(aUb + 8 * 26), w23 = lds2(aUb + 8 * 28);  // n^0 E_alphahat
        const double mbdt = -a.beta_dt;
        double Is[NITER];
#pragma unroll
        for (int it = 0; it < NITER; it++) {
            const double wgt = chain4(w01.x, w01.y, w23.x, w23.y, n1[it], n2[it], n3[it]);  // n^0 n_0 at the cell centre
            double v = a.gam1 * x0[it];
            if (I0p != nullptr) v = fma(a.gam0, __ldg(I0p + (OFF8(it) >> 3)), v);
            v = fma(mbdt * d[it], rcp3(wgt), v);
            Is[it] = (excised || !(it < NITER - 1 || last_valid)) ? 0.0 : v;
        }

#pragma unroll
        for (int it = 0; it < NITER; it++) {
            if (it < NITER - 1 || last_valid) outp[OFF8(it) >> 3] = Is[it];
            xm1[it] = x0[it]; x0[it] = xp1[it]; xp1[it] = xp2[it];
        }
        outp += N;
        if (I0p != nullptr) I0p += N;
    }
#undef OFF8
}

// ------------------------------------------------------------------------------------------------------------------
// packed per-cell record of the stage kernel, RECN doubles for EVERY cell of the array (ghosts included):
//   [0..7]   upper x face (= lower x face of cell c+1): e^x_alphahat (4), E_alphahat / dx (4)   (rad.h face record, R6)
//   [8..15]  upper y face, [16..23] upper z face, likewise with dy, dz
//   [24] n^0   [25] excised flag   [26..29] n^0 E_alphahat (cell centre)   [30..35] co-triad
// faces whose upper neighbour is outside the array are zero.
__global__ void __launch_bounds__(256) k_pack_rec(const DeviceTables t, double *__restrict__ rec) {
    const long long total = t.ncell * RECN;
    for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < total; idx += (long long)gridDim.x * blockDim.x) {
        const long long c = idx / RECN;
        const int m = (int)(idx - c * RECN);
        const int i = (int)(c % t.NI), j = (int)((c / t.NI) % t.NJ), k = (int)(c / ((long long)t.NI * t.NJ));
        double v = 0.0;
        if (m < 24) {
            const int ax = m >> 3, r = m & 7;
            const bool inside = ax == 0 ? i + 1 < t.NI : (ax == 1 ? j + 1 < t.NJ : k + 1 < t.NK);
            if (inside) {
                const long long cu = c + (ax == 0 ? 1 : (ax == 1 ? (long long)t.NI : (long long)t.NI * t.NJ));
                v = t.face[(cu * 3 + ax) * RAD_NFACE + r];
                if (r >= 4) v *= t.inv_dx[ax];
            }
        } else {
            const double *cg = t.cell + c * RAD_NCELL;
            if (m == 24) v = cg[0];
            else if (m == 25) v = cg[50];
            else if (m < 30) v = cg[1 + (m - 26)] * cg[0];
            else v = cg[44 + (m - 30)];
        }
        rec[idx] = v;
    }
}

// Parity helper: the upwind decision of the stage kernel itself for the three UPPER faces of every cell -- face_geom() on the packed
// records, exactly what k_stage5 evaluates -- as sgn n^a: -1 where the kernel takes the upper cell as upwind, +1 the lower, 0 for n^a = 0.
__global__ void __launch_bounds__(256) k_stage_face_signs(const DeviceTables t, signed char *__restrict__ out) {
    const long long total = t.ncell * 3 * t.N;
    for (long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x; q < total; q += (long long)gridDim.x * blockDim.x) {
        const int n = (int)(q % t.N);
        const long long cf = q / t.N;  // cell * 3 + axis
        const double *r = t.rec + (cf / 3) * RECN + (cf % 3) * 8;
        const FaceRec f = {r[0], r[1], r[2], r[3], r[4], r[5], r[6], r[7]};
        const FaceGeom g = face_geom(f, t.nhat[3 * n], t.nhat[3 * n + 1], t.nhat[3 * n + 2]);
        out[q] = g.na == 0.0 ? 0 : (g.neg ? -1 : 1);
    }
}

template <int NITER, int WPC, int TY, int TZ, int MINB, bool TAU>
int launch5t(const DeviceTables &t, const Params &p, const StageArgs &a, cudaStream_t s) {
    using T = Tile<TY, TZ, WPC, TAU>;
    const Layout5 L = make_layout5<T>(t.N);
    const size_t smem = sizeof(double) * (size_t)L.total;
    if (smem > (size_t)t.smem_optin) return 0;
    // run length along x: long runs amortise the prologue, short runs fill the SMs of small grids; pick the candidate
    // with the fewest CTA waves x (steps + prologue cost)
    const int nz = a.kz1 > a.kz0 ? a.kz1 - a.kz0 : t.n[2];
    const long long tiles = (long long)((t.n[1] + TY - 1) / TY) * ((nz + TZ - 1) / TZ);
    int KX = t.n[0];
    double best = 1e300;
    for (int cand = t.n[0];; cand = (cand + 1) / 2) {
        const long long ctas = tiles * ((t.n[0] + cand - 1) / cand);
        const double cost = (double)((ctas + t.sms - 1) / t.sms) * (cand + 3);
        if (cost < best) { best = cost; KX = cand; }
        if (cand <= 4) break;
    }
    dim3 grid((t.n[0] + KX - 1) / KX, (t.n[1] + TY - 1) / TY, (nz + TZ - 1) / TZ);
    if (grid.y > 65535 || grid.z > 65535) return 0;
#define RAD_LAUNCH5(PLM)                                                                                               \
    do {                                                                                                               \
        if (cudaFuncSetAttribute(k_stage5<NITER, WPC, TY, TZ, MINB, PLM, TAU>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return -1; \
        k_stage5<NITER, WPC, TY, TZ, MINB, PLM, TAU><<<grid, T::NT, smem, s>>>(t, p, a, L, KX);                         \
    } while (0)
    if (p.recon_space == 1) RAD_LAUNCH5(true); else RAD_LAUNCH5(false);
#undef RAD_LAUNCH5
    return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

template <int NITER, int WPC, int TY, int TZ, int MINB = 1>
int launch5(const DeviceTables &t, const Params &p, const StageArgs &a, cudaStream_t s) {
    if (a.vel8 != nullptr) return launch5t<NITER, WPC, TY, TZ, MINB, true>(t, p, a, s);
    return launch5t<NITER, WPC, TY, TZ, MINB, false>(t, p, a, s);
}

// TAU: per-cell record of the optical-depth-aware flux for EVERY cell (ghosts included), 8 doubles: tetrad-frame fluid velocity
// u^alphahat (R10), f/2 = -expm1(-tau^2)/2 of the cell's upper x, y, z faces (Eq.26-27 with R15, R16, R18, G1; 0 where the upper
// neighbour is outside the array), pad.  One launch per stage (the fluid state and beta dt change).
__device__ __forceinline__ void cell_u(const DeviceTables &t, const double *__restrict__ fluid, long long c, double (&u)[4]) {
    const double *th = t.cell + c * RAD_NCELL + 44;
    const double u1 = fluid[2 * t.ncell + c], u2 = fluid[3 * t.ncell + c], u3 = fluid[4 * t.ncell + c];
    u[1] = th[0] * u1 + th[1] * u2 + th[2] * u3; u[2] = th[3] * u2 + th[4] * u3; u[3] = th[5] * u3;
    u[0] = sqrt(1.0 + (u[1] * u[1] + u[2] * u[2] + u[3] * u[3]));
}
__global__ void __launch_bounds__(256) k_tau_table(const DeviceTables t, const double *__restrict__ fluid, const double *__restrict__ aE,
                                                   const double *__restrict__ aS, double tau_dt, double *__restrict__ vel8) {
    for (long long c = blockIdx.x * (long long)blockDim.x + threadIdx.x; c < t.ncell; c += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(c % t.NI), j = (int)((c / t.NI) % t.NJ), k = (int)(c / ((long long)t.NI * t.NJ));
        double u[4], un[4];
        cell_u(t, fluid, c, u);
        const double ae = aE[c] + aS[c];
        double out[8] = {u[0], u[1], u[2], u[3], 0.0, 0.0, 0.0, 0.0};
#pragma unroll
        for (int ax = 0; ax < 3; ax++) {
            const bool inside = ax == 0 ? i + 1 < t.NI : (ax == 1 ? j + 1 < t.NJ : k + 1 < t.NK);
            if (!inside) continue;
            const long long cu = c + (ax == 0 ? 1 : (ax == 1 ? (long long)t.NI : (long long)t.NI * t.NJ));
            cell_u(t, fluid, cu, un);
            const double tau = tau_dt * (0.5 * (ae + (aE[cu] + aS[cu]))) / (0.5 * (u[0] + un[0]));
            out[4 + ax] = -0.5 * expm1(-tau * tau);
        }
#pragma unroll
        for (int q = 0; q < 8; q++) vel8[c * 8 + q] = out[q];
    }
}

}  // namespace

// The tile shape per number of angles (the A/B runs behind these choices are in
// profiles/r1_k_stage5_ncu_full.md).  CALL(NITER, WPC, TY, TZ): NITER * WPC * 32 >= N angle slots per cell.
#define RAD_S5_DISPATCH(N, CALL)                 \
    do {                                         \
        if ((N) <= 32) CALL(1, 1, 4, 2);         \
        else if ((N) <= 64) CALL(1, 2, 4, 2);    \
        else if ((N) <= 96) CALL(3, 1, 4, 3);    \
        else if ((N) <= 128) CALL(2, 2, 4, 2);   \
        else if ((N) <= 192) CALL(3, 2, 4, 2);   \
        else CALL(4, 2, 2, 2);                   \
    } while (0)

// returns 1 (launched), 0 (this configuration is not served by this kernel), -1 (CUDA error)
int launch_stage_angle(const DeviceTables &t, const Params &p, const StageArgs &a, cudaStream_t s) {
    if (!stage_angle_serves(t, a.vel8 != nullptr)) return 0;
    if (((uintptr_t)a.I_in & 15) || ((uintptr_t)a.vel8 & 15)) return 0;  // rows are brought in by 16-byte bulk copies
#define RAD_S5_CALL(NITER, WPC, TY, TZ) return launch5<NITER, WPC, TY, TZ>(t, p, a, s)
    RAD_S5_DISPATCH(t.N, RAD_S5_CALL);
#undef RAD_S5_CALL
    return 0;
}

// the instance launch_stage_angle runs for this context, written as ncu prints it without casts and blanks (profiles/*.csv key)
int stage_angle_kernel_name(const DeviceTables &t, const Params &p, bool tau, char *buf, size_t n) {
    if (!stage_angle_serves(t, tau)) return snprintf(buf, n, "k_fluxdiv");
#define RAD_S5_CALL(NITER, WPC, TY, TZ) return snprintf(buf, n, "k_stage5<%d,%d,%d,%d,1,%d,%d>", NITER, WPC, TY, TZ, p.recon_space == 1 ? 1 : 0, tau ? 1 : 0)
    RAD_S5_DISPATCH(t.N, RAD_S5_CALL);
#undef RAD_S5_CALL
    return 0;
}

int stage_angle_serves(const DeviceTables &t, bool tau) {
    if (!t.fused_ok || t.ke == nullptr || t.rec == nullptr || (t.N & 1) || t.N > 256) return 0;  // rows must be multiples of 16 bytes
    if (((uintptr_t)t.ke & 15) || ((uintptr_t)t.rec & 15)) return 0;
    // the layout with the velocity records (TAU) is the larger one: N ~ 176..180 fits without them only
#define RAD_S5_CALL(NITER, WPC, TY, TZ)                                                                                           \
    return sizeof(double) * (size_t)(tau ? make_layout5<Tile<TY, TZ, WPC, true>>(t.N).total : make_layout5<Tile<TY, TZ, WPC, false>>(t.N).total) <= \
           (size_t)t.smem_optin
    RAD_S5_DISPATCH(t.N, RAD_S5_CALL);
#undef RAD_S5_CALL
    return 0;
}

int launch_tau_table(const DeviceTables &t, const double *fluid, const double *aE, const double *aS, double tau_dt, double *vel8, cudaStream_t s) {
    k_tau_table<<<t.sms * 4, 256, 0, s>>>(t, fluid, aE, aS, tau_dt, vel8);
    return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

int launch_stage_face_signs(const DeviceTables &t, signed char *out, cudaStream_t s) {
    if (t.rec == nullptr) return 0;
    k_stage_face_signs<<<t.sms * 8, 256, 0, s>>>(t, out);
    return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

int launch_pack_rec(const DeviceTables &t, double *rec, cudaStream_t s) {
    k_pack_rec<<<t.sms * 8, 256, 0, s>>>(t, rec);
    return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

}  // namespace rad
