// stage4.cu -- the fused stage kernel, tile-synchronous version: spatial + angular flux divergence (Eq.22, 24, 25),
// cons -> prim, locally implicit coupling (section 2.5), ergosphere mask, fluid increment
// in ONE launch, with every intensity row staged into shared memory by bulk asynchronous copies (TMA, 1-D).
//
// Mapping:
//   * a CTA owns a TY x TZ tile of cell columns in the y-z plane and marches along x through KX cells; one WARP per
//     cell, lanes over angles (intensities are I[cell][angle], angle innermost, so a row is one contiguous run).
//   * shared memory holds, for the plane x = i being updated: the tile's own rows of planes i-1 .. i+2 (a ring of
//     5 plane slots; the x stencil reads them, the y/z stencils of the neighbouring warps read plane i) and the
//     2-deep halo rows of plane i around the tile.  The rows of plane i+3 and the halo of plane i+1 are in flight
//     (cp.async.bulk global -> shared, completion on an mbarrier) while plane i is computed: no warp waits on a
//     global load of intensities, and every row crosses L2 -> SM once per tile that needs it.
//   * the stored angular-edge coefficients of a cell (3 N doubles) are bulk-copied into a warp-private buffer one
//     step ahead; the owner of an edge overwrites the coefficient with the edge flux in place, the partner angle
//     pulls it from there (__syncwarp only).
//   * FP64 is the scarce resource: the x flux is carried, grid spacings and n^0 are folded
//     into the per-cell records, flux differences are accumulated by FMA, the van Leer slope uses one Newton step,
//     sign tests are integer tests of the high word.
//   * the warp holds all N post-transport intensities of its cell in registers: the coupling's angle reductions
//     are warp shuffles, the quartic is solved in registers, I* never goes to memory.
#include <cstdint>

#include "stage_math.cuh"

namespace rad {
namespace {

constexpr int TY = 4, TZ = 3, NW = TY * TZ, NH = 4 * TZ + 4 * TY, RING = 5;

// ---- shared-memory layout (offsets in doubles) -------------------------------------------------------------------
struct Layout {
    int Np;   // row stride of intensity rows (even, >= N)
    int Kp;   // stride of the per-warp coefficient/flux buffers: 3 N + 2 (slot 3N is the always-zero flux)
    int Nt;   // length of the per-angle tables, padded to a whole number of warp iterations (lanes past N read benign entries)
    int oR, oH, oK, oU, oUraw, oN, oW, oD, oRec, oBar, total;
};
__host__ __device__ inline Layout make_layout(int N) {
    Layout L;
    L.Np = (N + 1) & ~1;
    L.Kp = 3 * N + 2;
    L.Nt = ((N + 31) / 32) * 32;
    L.oR = 0;
    L.oH = L.oR + RING * NW * L.Np;
    L.oK = L.oH + 2 * NH * L.Np;
    L.oU = L.oK + NW * L.Kp;
    L.oUraw = L.oU + NW * 64;
    L.oN = L.oUraw + NW * 64;
    L.oW = L.oN + 3 * L.Nt;
    L.oD = L.oW + L.Nt;
    L.oRec = L.oD + L.Nt;          // uint4 per angle = 2 doubles
    L.oBar = L.oRec + 2 * L.Nt;    // 2 + NW mbarriers (8 bytes each)
    L.total = L.oBar + 2 + NW;
    return L;
}

// ---- PTX helpers: mbarrier, bulk copy --------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(bar), "r"(parity)
        : "memory");
}
// global -> shared bulk copy (TMA, 1-D); bytes multiple of 16, both addresses 16-byte aligned
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst), "l"(src), "r"(bytes),
                 "r"(bar)
                 : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }

__device__ __forceinline__ int hi32(double x) { return __double2hiint(x); }

// 1/d to ~2^-40 (hardware seed 2^-20 + one Newton step): enough for the limited slope, which is a correction term
__device__ __forceinline__ double rcp_1n(double d) {
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(d));
    const double e = fma(-d, r, 1.0);
    return fma(r, e, r);
}

struct FaceRec {  // e: n^a = e0 + e_b n^b; E: (1/dx_a) n_0 = E0 + E_b n^b (the grid spacing is folded in)
    double e0, e1, e2, e3, E0, E1, E2, E3;
};
__device__ __forceinline__ FaceRec load_face_s(const double *f) {  // shared memory, warp-uniform address
    const double2 a = *reinterpret_cast<const double2 *>(f), b = *reinterpret_cast<const double2 *>(f + 2),
                  c = *reinterpret_cast<const double2 *>(f + 4), d = *reinterpret_cast<const double2 *>(f + 6);
    return {a.x, a.y, b.x, b.y, c.x, c.y, d.x, d.y};
}

// The same through volatile loads: the record is re-read at every use instead of being kept in 16 registers for the whole
// step (five face records in registers are what made the kernel spill; a warp-uniform shared-memory read is one wavefront).
__device__ __forceinline__ double2 lds_v2(uint32_t addr) {
    double2 v;
    asm volatile("ld.volatile.shared.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr));
    return v;
}
__device__ __forceinline__ FaceRec load_face_v(uint32_t addr) {
    const double2 a = lds_v2(addr), b = lds_v2(addr + 16), c = lds_v2(addr + 32), d = lds_v2(addr + 48);
    return {a.x, a.y, b.x, b.y, c.x, c.y, d.x, d.y};
}

// Upwind flux through a face (Eq.24), split into weight and face value: returns w = n^a n_0 / dx_a and sets
// `up` to the reconstructed upwind intensity.  PLM: van Leer limited slope of the upwind cell (R7): with (far, mid, oth)
// = (LL, L, R) for n^a > 0 and (RR, R, L) otherwise, the face value is mid + dl dr / (dl + dr), dl = mid - far,
// dr = oth - mid (the harmonic mean is odd under reversal, so one formula serves both signs).  Branch free.
template <bool PLM>
__device__ __forceinline__ double face_w(const FaceRec &f, double n1, double n2, double n3, double qLL, double qL, double qR, double qRR,
                                         double &up) {
    const double na = chain4(f.e0, f.e1, f.e2, f.e3, n1, n2, n3);
    const double n0 = chain4(f.E0, f.E1, f.E2, f.E3, n1, n2, n3);
    const bool pos = hi32(na) > 0;  // na > 0 (na = +-0 -> false; the flux is then 0 either way)
    up = pos ? qL : qR;
    if (PLM) {
        const double far = pos ? qLL : qRR, oth = pos ? qR : qL;
        const double dl = up - far, dr = oth - up, pr = dl * dr;
        const double h = pr * fast_rcp(dl + dr);
        up += hi32(pr) > 0 ? h : 0.0;
    }
    return __dmul_rn(na, n0);
}

// 8-byte asynchronous copy global -> shared (LDGSTS): the per-cell records are fetched one step ahead without holding
// registers (a register prefetch would be spilled and the spill would wait for the load)
__device__ __forceinline__ void cp_async8(uint32_t dst, const void *src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// sums of four values over the warp, all lanes get all four: the first two butterfly steps halve the number of values a
// lane carries instead of adding four values each (6 adds and 10 64-bit shuffles instead of 20 and 20)
__device__ __forceinline__ void warp_sum4(double &a, double &b, double &c, double &d, int lane) {
    const unsigned full = 0xffffffffu;
    const bool u16 = (lane & 16) != 0;
    double k0 = u16 ? c : a, k1 = u16 ? d : b;
    k0 += __shfl_xor_sync(full, u16 ? a : c, 16);
    k1 += __shfl_xor_sync(full, u16 ? b : d, 16);
    const bool u8 = (lane & 8) != 0;
    double k = u8 ? k1 : k0;
    k += __shfl_xor_sync(full, u8 ? k0 : k1, 8);
    k += __shfl_xor_sync(full, k, 4);
    k += __shfl_xor_sync(full, k, 2);
    k += __shfl_xor_sync(full, k, 1);
    a = __shfl_sync(full, k, 0); b = __shfl_sync(full, k, 8); c = __shfl_sync(full, k, 16); d = __shfl_sync(full, k, 24);
}

// ------------------------------------------------------------------------------------------------------------------
template <int NITER, bool PLM, bool COUPLE>
__global__ void __launch_bounds__(NW * 32, 1) k_stage4(const DeviceTables t, const Params p, const StageArgs a, const int KX) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int N = t.N;
    const Layout L = make_layout(N);
    const int Np = L.Np, Kp = L.Kp, Nt = L.Nt;
    double *sm = reinterpret_cast<double *>(smem_raw);
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const int wy = w % TY, wz = w / TY;
    double *sR = sm + L.oR, *sH = sm + L.oH, *sK = sm + L.oK + w * Kp, *sU = sm + L.oU + w * 64, *sUraw = sm + L.oUraw + w * 64;
    double *sN = sm + L.oN, *sWinv = sm + L.oW, *sDom = sm + L.oD;
    uint4 *sRec = reinterpret_cast<uint4 *>(sm + L.oRec);
    const uint32_t bar0 = smem_u32(sm + L.oBar);           // full[0], full[1], then kbar[w]
    const uint32_t kbar = bar0 + 8u * (2 + w);
    const uint32_t row_bytes = (uint32_t)N * 8u, ke_bytes = 3u * (uint32_t)N * 8u;

    // per-angle tables; entries past N (read by the idle lanes of the last iteration) are benign: direction of angle 0,
    // zero weights, partner 0, pulls from the always-zero flux slot
    for (int q = tid; q < Nt; q += blockDim.x) {
        const int qa = q < N ? q : 0;
        sWinv[q] = q < N ? t.winv[qa] : 0.0;
        sDom[q] = q < N ? t.domega[qa] : 0.0;
        uint4 rec = reinterpret_cast<const uint4 *>(t.ang_rec)[qa];
        if (q >= N) { const unsigned z = 3u * (unsigned)N; rec = make_uint4(0u, z << 16, z | (z << 16), 0u); }
        sRec[q] = rec;
        sN[q] = t.nhat[3 * qa]; sN[Nt + q] = t.nhat[3 * qa + 1]; sN[2 * Nt + q] = t.nhat[3 * qa + 2];
    }
    if (lane == 0) { sK[3 * N] = 0.0; sK[3 * N + 1] = 0.0; }
    sU[lane] = 0.0; sU[32 + lane] = 0.0;
    if (tid == 0) {
        for (int q = 0; q < 2 + NW; q++) mbar_init(bar0 + 8u * q, 1);
        fence_mbar_init();
    }
    __syncthreads();

    const int ng = t.ng;
    const int j0 = blockIdx.y * TY + ng, k0 = blockIdx.z * TZ + ng;
    const int j = j0 + wy, k = k0 + wz;
    const bool active = j < t.n[1] + ng && k < t.n[2] + ng;
    const int i_begin = blockIdx.x * KX + ng, i_end = min(i_begin + KX, t.n[0] + ng), nsteps = i_end - i_begin;

    // ---- copy roles: lane 0 of a warp brings in the warp's own rows (also for a cell column outside the interior, as
    // long as it is inside the array: active neighbours read it), lanes 1..3 bring in halo rows
    int role = 0;                 // 0 none, 1 own row, 2 halo row
    long long src_cell0 = 0;      // cell index at i = 0 of the pencil this lane copies from
    int dst_row = 0;              // own: w; halo: halo index
    if (lane == 0 && j < t.NJ && k < t.NK) { role = 1; src_cell0 = ((long long)k * t.NJ + j) * t.NI; dst_row = w; }
    if (lane >= 1 && lane <= 3) {
        const int h = w + NW * (lane - 1);
        if (h < NH) {
            int jj, kk;
            if (h < 4 * TZ) { const int hz = h >> 2, q = h & 3; kk = k0 + hz; jj = j0 + (q < 2 ? q - 2 : TY + q - 2); }
            else { const int hh = h - 4 * TZ, hy = hh >> 2, q = hh & 3; jj = j0 + hy; kk = k0 + (q < 2 ? q - 2 : TZ + q - 2); }
            if (jj < t.NJ && kk < t.NK) { role = 2; src_cell0 = ((long long)kk * t.NJ + jj) * t.NI; dst_row = h; }
        }
    }
    const int n_own = __syncthreads_count(role == 1), n_halo = __syncthreads_count(role == 2);
    const uint32_t tx_step = (uint32_t)(n_own + n_halo) * row_bytes;

    // ---- prologue: planes i_begin-2 .. i_begin+2 of the own rows (slot of plane d = (d + 2) % 5), halo of plane i_begin
    if (tid == 0) mbar_expect_tx(bar0, (uint32_t)(5 * n_own + n_halo) * row_bytes);
    __syncthreads();
    if (role == 1) {
        for (int d = -2; d <= 2; d++)
            bulk_g2s(smem_u32(sR + ((d + 2) * NW + dst_row) * Np), a.I_in + (src_cell0 + i_begin + d) * N, row_bytes, bar0);
    } else if (role == 2) {
        bulk_g2s(smem_u32(sH + dst_row * Np), a.I_in + (src_cell0 + i_begin) * N, row_bytes, bar0);
    }
    const long long c_first = ((long long)k * t.NJ + j) * t.NI + i_begin;
    const long long cint_first = ((long long)(k - ng) * t.n[1] + (j - ng)) * t.n[0] + (i_begin - ng);
    if (lane == 0 && active) {
        mbar_expect_tx(kbar, ke_bytes);
        bulk_g2s(smem_u32(sK), t.ke + cint_first * 3 * N, ke_bytes, kbar);
    }

    // ---- where the 8 stencil neighbours of this warp's cell live: ring (own rows of another warp) or halo buffer
    int nbOff[8];      // row offset in doubles inside a ring plane slot / a halo buffer
    unsigned nbHalo = 0;
#pragma unroll
    for (int q = 0; q < 8; q++) {
        const int d = (q & 3) < 2 ? (q & 3) - 2 : (q & 3) - 1;  // -2, -1, +1, +2
        if (q < 4) {
            const int yy = wy + d;
            if (yy >= 0 && yy < TY) nbOff[q] = (wz * TY + yy) * Np;
            else { nbOff[q] = (wz * 4 + (yy < 0 ? yy + 2 : yy - TY + 2)) * Np; nbHalo |= 1u << q; }
        } else {
            const int zz = wz + d;
            if (zz >= 0 && zz < TZ) nbOff[q] = (zz * TY + wy) * Np;
            else { nbOff[q] = (4 * TZ + wy * 4 + (zz < 0 ? zz + 2 : zz - TZ + 2)) * Np; nbHalo |= 1u << q; }
        }
    }

    const double idx0 = t.inv_dx[0], idx1 = t.inv_dx[1], idx2 = t.inv_dx[2];
    const bool last_valid = (NITER - 1) * 32 + lane < N;

    // Warp-uniform records of a cell, gathered two per lane (cp.async, one step ahead) and broadcast through shared memory:
    //   sU[0..7] x face above, [8..15] y face below, [16..23] y face above, [24..31] z face below, [32..39] z face above
    //            (E parts multiplied by 1/dx of the face's axis),
    //   [40] n^0, [41] excised flag, [42..45] n^0 E_0..E_3, [46..51] co-triad, [52..56] rho, T, u1', u2', u3',
    //   [57..59] alpha_P, alpha_E, alpha_s
    const double *ptrA = t.face, *ptrB = t.cell;
    int strideB = 0;
    double sclA = 1.0;
    bool sclB_n0 = false, haveB = false;
    if (active) {
        const long long c = c_first, cz = (long long)t.NI * t.NJ;
        const int g = lane >> 3, r = lane & 7;
        ptrA = t.face + ((g == 0 ? c + 1 : (g == 2 ? c + t.NI : c)) * 3 + (g == 0 ? 0 : (g == 3 ? 2 : 1))) * RAD_NFACE + r;
        if (r >= 4) sclA = g == 0 ? idx0 : (g == 3 ? idx2 : idx1);
        ptrB = t.cell + c * RAD_NCELL;
        strideB = RAD_NCELL;
        haveB = lane < 20;
        if (lane < 8) { ptrB = t.face + ((c + cz) * 3 + 2) * RAD_NFACE + lane; strideB = 3 * RAD_NFACE; }
        else if (lane == 8) ;                                            // n^0
        else if (lane == 9) ptrB += 50;                                  // excised flag
        else if (lane < 14) { ptrB += lane - 9; sclB_n0 = true; }        // E_0..E_3, stored multiplied by n^0
        else if (lane < 20) ptrB += 44 + (lane - 14);
        else if (COUPLE && p.couple && lane < 28) {
            ptrB = lane < 25 ? a.fluid + (long long)(lane - 20) * t.ncell + c : (lane == 25 ? a.aP : (lane == 26 ? a.aE : a.aS)) + c;
            strideB = 1; haveB = true;
        } else if (COUPLE && lane == 21) { ptrB = a.fluid + t.ncell + c; strideB = 1; haveB = true; }  // T_- is reported even when not coupling
    }
    const uint32_t rawA = smem_u32(sUraw + lane), rawB = smem_u32(sUraw + 32 + lane);
    if (active) {
        cp_async8(rawA, ptrA); ptrA += 3 * RAD_NFACE;
        if (haveB) { cp_async8(rawB, ptrB); ptrB += strideB; }
    }
    cp_async_commit();

    // ---- flux through the lower x face of the first cell of this run (carried from then on)
    double carry[NITER];
    mbar_wait(bar0, 0);
    if (active) {
        FaceRec f;
        {
            const double *fr = t.face + (c_first * 3 + 0) * RAD_NFACE;
            f = {__ldg(fr), __ldg(fr + 1), __ldg(fr + 2), __ldg(fr + 3), __ldg(fr + 4) * idx0, __ldg(fr + 5) * idx0, __ldg(fr + 6) * idx0,
                 __ldg(fr + 7) * idx0};
        }
        const double *r0 = sR + (0 * NW + w) * Np + lane, *r1 = sR + (1 * NW + w) * Np + lane, *r2 = sR + (2 * NW + w) * Np + lane,
                     *r3 = sR + (3 * NW + w) * Np + lane;
#pragma unroll
        for (int it = 0; it < NITER; it++) {
            const int n = it * 32 + lane;
            double up;
            const double wgt = face_w<PLM>(f, sN[n], sN[Nt + n], sN[2 * Nt + n], PLM ? r0[it * 32] : 0.0, r1[it * 32], r2[it * 32],
                                           PLM ? r3[it * 32] : 0.0, up);
            carry[it] = __dmul_rn(wgt, up);
        }
    }

    for (int s = 0; s < nsteps; s++) {
        const int i = i_begin + s;
        const bool more = s + 1 < nsteps;
        if (tid == 0 && more) mbar_expect_tx(bar0 + 8u * ((s + 1) & 1), tx_step);
        __syncthreads();  // every warp is done with step s-1: its ring slot and halo buffer can be refilled
        if (more) {
            if (role == 1) bulk_g2s(smem_u32(sR + (((s + 5) % RING) * NW + dst_row) * Np), a.I_in + (src_cell0 + i + 3) * N, row_bytes, bar0 + 8u * ((s + 1) & 1));
            else if (role == 2) bulk_g2s(smem_u32(sH + (((s + 1) & 1) * NH + dst_row) * Np), a.I_in + (src_cell0 + i + 1) * N, row_bytes, bar0 + 8u * ((s + 1) & 1));
        }
        mbar_wait(bar0 + 8u * (s & 1), (s >> 1) & 1);
        if (!active) continue;

        const long long c = c_first + s;
        // ring slots of planes i-1, i, i+1, i+2 (plane i_begin + d lives in slot (d + 2) % 5); all pointers include the lane
        const double *R0 = sR + (((s + 2) % RING) * NW) * Np + lane;
        const double *Hc = sH + ((s & 1) * NH) * Np + lane;
        const double *own = R0 + w * Np;
        const double *xm1 = sR + (((s + 1) % RING) * NW + w) * Np + lane, *xp1 = sR + (((s + 3) % RING) * NW + w) * Np + lane,
                     *xp2 = sR + (((s + 4) % RING) * NW + w) * Np + lane;

        // ---- uniform records of this cell: raw (landed by cp.async) -> scaled -> sU; fetch the next cell's
        {
            cp_async_wait_all();
            const double vA = sUraw[lane], vB = sUraw[32 + lane];
            const double nup0 = __shfl_sync(0xffffffffu, vB, 8);
            __syncwarp();  // the previous step's readers of sU are done
            sU[lane] = vA * sclA;
            sU[32 + lane] = lane < 8 ? vB * ((lane >= 4) ? idx2 : 1.0) : (sclB_n0 ? vB * nup0 : vB);
            if (more) {
                cp_async8(rawA, ptrA); ptrA += 3 * RAD_NFACE;
                if (haveB) { cp_async8(rawB, ptrB); ptrB += strideB; }
            }
            cp_async_commit();
        }

        // ---- angular fluxes (Eq.25, donor cell in angle): owners turn q_e into the edge flux in place
        double div[NITER];
        mbar_wait(kbar, s & 1);
        {
            const double *ownrow = own - lane;
#pragma unroll
            for (int it = 0; it < NITER; it++) {
                const int n = it * 32 + lane;
                const uint4 rec = sRec[n];
                const unsigned pj[3] = {rec.x & 0xffffu, rec.x >> 16, rec.y & 0xffffu};
                double asum = 0.0;
#pragma unroll
                for (int jj = 0; jj < 3; jj++) {  // unused slots have q = 0
                    const double q = sK[jj * N + n];
                    const bool owner_up = (__double2loint(q) & 1) != 0;
                    const double G = q * ownrow[owner_up ? (unsigned)n : pj[jj]];
                    asum += G;
                    if (it < NITER - 1 || last_valid) sK[jj * N + n] = G;
                }
                div[it] = asum;
            }
        }
        __syncwarp();
#pragma unroll
        for (int it = 0; it < NITER; it++) {
            const int n = it * 32 + lane;
            const uint4 rec = sRec[n];
            const double asum = div[it] - ((sK[rec.y >> 16] + sK[rec.z & 0xffffu]) + sK[rec.z >> 16]);  // unused -> sK[3N] = 0
            div[it] = asum * sWinv[n];
        }
        __syncwarp();  // all pulls done: the buffer can take the next cell's coefficients
        if (lane == 0 && more) {
            fence_proxy_async();
            mbar_expect_tx(kbar, ke_bytes);
            bulk_g2s(smem_u32(sK), t.ke + (cint_first + s + 1) * 3 * N, ke_bytes, kbar);
        }

        // ---- spatial fluxes (Eq.24), flux-divergence update of C = n^0 n_0 I (Eq.22, stage form R8), cons -> prim
        const double2 c01 = *reinterpret_cast<const double2 *>(sU + 40);
        const double nup0 = c01.x;
        const bool excised = c01.y != 0.0;
        const double *nb[8];
#pragma unroll
        for (int q = 0; q < 8; q++) nb[q] = ((nbHalo >> q) & 1u ? Hc : R0) + nbOff[q];
        const double mbdt = -a.beta_dt, thr = p.n0_crit * nup0;  // |n_0| < n0_crit  <=>  |n^0 n_0| < n0_crit n^0
        double Is[NITER];
        unsigned maskbits = 0;
        const uint32_t sUa = smem_u32(sU);
#pragma unroll
        for (int it = 0; it < NITER; it++) {
            const int n = it * 32 + lane, o = it * 32;
            const double n1 = sN[n], n2 = sN[Nt + n], n3 = sN[2 * Nt + n];
            const double Iown = own[o];
            double d = div[it], up;
            {   // x: flux through the upper face (the lower x face of cell i+1); the lower one is carried
                const FaceRec fx = load_face_v(sUa);
                const double wgt = face_w<PLM>(fx, n1, n2, n3, PLM ? xm1[o] : 0.0, Iown, xp1[o], PLM ? xp2[o] : 0.0, up);
                const double F = __dmul_rn(wgt, up);
                d += F - carry[it];
                carry[it] = F;
            }
            {   // y: rows -2, -1, +1, +2 serve both faces
                const double m2 = PLM ? nb[0][o] : 0.0, m1 = nb[1][o], p1 = nb[2][o], p2 = PLM ? nb[3][o] : 0.0;
                const FaceRec fl = load_face_v(sUa + 64);
                const double wl = face_w<PLM>(fl, n1, n2, n3, m2, m1, Iown, p1, up);
                d = fma(-wl, up, d);
                const FaceRec fh = load_face_v(sUa + 128);
                const double wh = face_w<PLM>(fh, n1, n2, n3, m1, Iown, p1, p2, up);
                d = fma(wh, up, d);
            }
            {   // z
                const double m2 = PLM ? nb[4][o] : 0.0, m1 = nb[5][o], p1 = nb[6][o], p2 = PLM ? nb[7][o] : 0.0;
                const FaceRec fl = load_face_v(sUa + 192);
                const double wl = face_w<PLM>(fl, n1, n2, n3, m2, m1, Iown, p1, up);
                d = fma(-wl, up, d);
                const FaceRec fh = load_face_v(sUa + 256);
                const double wh = face_w<PLM>(fh, n1, n2, n3, m1, Iown, p1, p2, up);
                d = fma(wh, up, d);
            }
            const double2 w01 = lds_v2(sUa + 8 * 42), w23 = lds_v2(sUa + 8 * 44);
            const double wgt = chain4(w01.x, w01.y, w23.x, w23.y, n1, n2, n3);  // n^0 n_0 at the cell centre (sU[42..45] = n^0 E)
            if (fabs(wgt) < thr) maskbits |= 1u << it;
            double v = a.gam1 * Iown;
            if (a.I0 != nullptr) v = fma(a.gam0, __ldg(a.I0 + c * N + min(n, N - 1)), v);
            v = fma(mbdt * d, fast_rcp(wgt), v);
            Is[it] = (excised || (it == NITER - 1 && !last_valid)) ? 0.0 : v;
        }

        if (COUPLE) {
            // ---- locally implicit coupling (section 2.5, Eq.31-50), fluid increment, mask
            const bool enable = !excised;
            double th[6], uh[4] = {1.0, 0.0, 0.0, 0.0};
            {
                const double2 t0 = *reinterpret_cast<const double2 *>(sU + 46), t1 = *reinterpret_cast<const double2 *>(sU + 48),
                              t2 = *reinterpret_cast<const double2 *>(sU + 50);
                th[0] = t0.x; th[1] = t0.y; th[2] = t1.x; th[3] = t1.y; th[4] = t2.x; th[5] = t2.y;
            }
            const double2 f0 = *reinterpret_cast<const double2 *>(sU + 52), f1 = *reinterpret_cast<const double2 *>(sU + 54),
                          f2 = *reinterpret_cast<const double2 *>(sU + 56), f3 = *reinterpret_cast<const double2 *>(sU + 58);
            const double rho = f0.x, Tm = f0.y, aP = f2.y, aS = f3.y, aE = f3.x + f3.y;  // Eq.33b
            if (p.couple && enable) tetrad_velocity(th, f1.x, f1.y, f2.x, uh);
            const double aEdt = aE * a.beta_dt;
            // sweep 1.  With d = n^0 + n^0bar alpha_E dt, rp = 1/(n^0bar d):  dOmega_bar = dOmega / n^0bar^2 (R11),
            // Ibar dOmega_bar = n^0bar^2 Ihat dOmega,  A_1 = sum (n^0/d) Ibar dOmega_bar, A_2 = dt/4pi sum dOmega rp (Eq.42),
            // and Eq.40 back in the tetrad frame is  Ihat_+ = g1 Ihat_- + src / (d n^0bar^3),  g1 = n^0 / d.
            double g1[NITER], g2r4[NITER];
            double Wsum = 0.0, A1 = 0.0, A2 = 0.0, Em = 0.0;
#pragma unroll
            for (int it = 0; it < NITER; it++) {
                const int n = it * 32 + lane;
                const double n1 = sN[n], n2 = sN[Nt + n], n3 = sN[2 * Nt + n];
                const double dom = sDom[n];  // 0 for idle lanes
                const double nbar = uh[0] - fma(uh[3], n3, fma(uh[2], n2, uh[1] * n1));  // n^0bar = -u_alpha n^alpha
                const double dd = fma(nbar, aEdt, nup0);
                const double rp = fast_rcp(nbar * dd);
                const double rd = nbar * rp, rn = dd * rp, rn2 = rn * rn;
                const double x = (nbar * nbar) * (Is[it] * dom);                            // Ibar dOmega_bar (Eq.38 summand)
                g1[it] = nup0 * rd;
                g2r4[it] = rn2 * rp;
                Em += x;
                A1 = fma(g1[it], x, A1);                                                    // Eq.42a
                A2 = fma(dom, rp, A2);                                                      // Eq.42b
                Wsum = fma(dom, rn2, Wsum);
            }
            warp_sum4(Wsum, A1, A2, Em, lane);
            double Tp = Tm, src = 0.0;
            bool coupled = false, noroot = false;
            if (p.couple && enable) {
                const double scale = p.renorm ? kFourPi / Wsum : 1.0;                       // R12
                A1 *= scale; Em *= scale; A2 *= scale * a.beta_dt / kFourPi;
                const double Cv = rho / (p.gamma_gas - 1.0);
                const double B4 = A2 * aP * p.a_rad, om = 1.0 - A2 * aS;                   // Eq.50
                const double B1 = Cv * om, Bp = A1 - om * Em;
                double dTemp = 0.0;
                if (!quartic_delta(B4, B1, Bp, Tm, dTemp)) {
                    noroot = true;
                } else {
                    coupled = true;
                    Tp = Tm + dTemp;
                    const double Ep = Em - Cv * dTemp;                                      // Eq.48
                    const double T2 = Tp * Tp;
                    src = (aP * p.a_rad * T2 * T2 + aS * Ep) * a.beta_dt / kFourPi;
                }
            }
            // sweep 2: Eq.40, fluid increment through the tetrad-frame first moments of the change, mask
            double M0 = 0.0, M1 = 0.0, M2 = 0.0, M3 = 0.0;
#pragma unroll
            for (int it = 0; it < NITER; it++) {
                const int n = it * 32 + lane;
                const double n1 = sN[n], n2 = sN[Nt + n], n3 = sN[2 * Nt + n];
                const double dom = sDom[n];
                const double Iold = Is[it];
                double Inew = coupled ? fma(src, g2r4[it], g1[it] * Iold) : Iold;
                const double wI = dom * (Inew - Iold);
                M0 += wI; M1 = fma(wI, n1, M1); M2 = fma(wI, n2, M2); M3 = fma(wI, n3, M3);
                if (thr > 0.0 && enable && ((maskbits >> it) & 1u)) Inew = 0.0;
                Is[it] = Inew;
            }
            warp_sum4(M0, M1, M2, M3, lane);
            if (lane == 0) {
                if (noroot && a.noroot) atomicAdd(a.noroot, 1ull);
                if (a.T_out) a.T_out[c] = Tp;
                if (a.dT0) {  // R^0_alpha = sum n^0 n_alpha I dOmega; n^0 n_0 = W_ahat n^ahat, n_i = theta^a_i n^a
                    const double2 w01 = *reinterpret_cast<const double2 *>(sU + 42), w23 = *reinterpret_cast<const double2 *>(sU + 44);
                    a.dT0[c] = -(w01.x * M0 + w01.y * M1 + w23.x * M2 + w23.y * M3);
                    a.dT0[t.ncell + c] = -(nup0 * (th[0] * M1));
                    a.dT0[2 * t.ncell + c] = -(nup0 * (th[1] * M1 + th[3] * M2));
                    a.dT0[3 * t.ncell + c] = -(nup0 * (th[2] * M1 + th[4] * M2 + th[5] * M3));
                }
            }
        }
        double *out = a.I_out + c * N + lane;
#pragma unroll
        for (int it = 0; it < NITER; it++)
            if (it < NITER - 1 || last_valid) out[it * 32] = Is[it];
    }
}

template <int NITER>
int launch_niter4(const DeviceTables &t, const Params &p, const StageArgs &a, bool couple, dim3 grid, size_t smem, int KX, cudaStream_t s) {
#define RAD_LAUNCH4(PLM, CPL)                                                                                          \
    do {                                                                                                               \
        if (cudaFuncSetAttribute(k_stage4<NITER, PLM, CPL>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return -1; \
        k_stage4<NITER, PLM, CPL><<<grid, NW * 32, smem, s>>>(t, p, a, KX);                                             \
    } while (0)
    if (p.recon_space == 1) { if (couple) RAD_LAUNCH4(true, true); else RAD_LAUNCH4(true, false); }
    else { if (couple) RAD_LAUNCH4(false, true); else RAD_LAUNCH4(false, false); }
#undef RAD_LAUNCH4
    return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

}  // namespace

// returns 1 (launched), 0 (this configuration is not served by the tile kernel), -1 (CUDA error)
int launch_stage_tile(const DeviceTables &t, const Params &p, const StageArgs &a, bool couple, cudaStream_t s) {
    if (!t.fused_ok || t.ke == nullptr) return 0;
    if (t.N & 1) return 0;  // rows must be multiples of 16 bytes for the bulk copies
    const int niter = (t.N + 31) / 32;
    if (niter > 6) return 0;
    const Layout L = make_layout(t.N);
    const size_t smem = sizeof(double) * (size_t)L.total;
    if (smem > 227 * 1024) return 0;
    // 16-byte alignment of every row the copies touch
    if (((uintptr_t)a.I_in & 15) || ((uintptr_t)t.ke & 15)) return 0;
    // run length along x: long runs amortise the prologue (5 planes), short runs fill the SMs of small grids; pick the
    // candidate with the fewest CTA waves x (steps + prologue cost)
    const long long tiles = (long long)((t.n[1] + TY - 1) / TY) * ((t.n[2] + TZ - 1) / TZ);
    int KX = t.n[0];
    double best = 1e300;
    for (int cand = t.n[0]; cand >= 4; cand = (cand + 1) / 2) {
        const long long ctas = tiles * ((t.n[0] + cand - 1) / cand);
        const double cost = (double)((ctas + 147) / 148) * (cand + 3);
        if (cost < best) { best = cost; KX = cand; }
        if (cand == 4) break;
    }
    dim3 grid((t.n[0] + KX - 1) / KX, (t.n[1] + TY - 1) / TY, (t.n[2] + TZ - 1) / TZ);
    if (grid.y > 65535 || grid.z > 65535) return 0;
    switch (niter) {
        case 1: return launch_niter4<1>(t, p, a, couple, grid, smem, KX, s);
        case 2: return launch_niter4<2>(t, p, a, couple, grid, smem, KX, s);
        case 3: return launch_niter4<3>(t, p, a, couple, grid, smem, KX, s);
        case 4: return launch_niter4<4>(t, p, a, couple, grid, smem, KX, s);
        case 5: return launch_niter4<5>(t, p, a, couple, grid, smem, KX, s);
        default: return launch_niter4<6>(t, p, a, couple, grid, smem, KX, s);
    }
}

}  // namespace rad
