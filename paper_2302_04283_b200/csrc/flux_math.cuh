// flux_math.cuh -- the spatial face flux of Eq.24 (and its optical-depth-aware form Eq.26-29) as the tile kernels evaluate it.
#pragma once
#include "async_copy.cuh"
#include "stage_math.cuh"

namespace rad {

struct FaceRec {  // n^a = e0 + e_b n^b;  n_0 / dx_a = E0 + E_b n^b (the grid spacing is folded in)
    double e0, e1, e2, e3, E0, E1, E2, E3;
};
// Upwind flux n^a n_0 I / dx_a (Eq.24) through the face between cells L and R; qLL, qL, qR, qRR are the
// intensities of the four cells around it.  PLM: van Leer limited slope of the upwind cell (R7): with (far, up, oth)
// = (LL, L, R) for n^a >= 0 and (RR, R, L) otherwise, the face value is up + dl dr / (dl + dr), dl = up - far,
// dr = oth - up (the harmonic mean is odd under reversal, so one formula serves both signs).  oth - up = +-(qR - qL): the
// difference is formed once and its sign bit flipped with the sign bit of n^a.  Branch free; sign tests are integer tests
// of the high word (n^a = +-0 -> the flux is 0 either way).  The limited slope is added under a predicate, so a slope
// that is not used (dl dr <= 0, where dl + dr may be 0) never reaches the result.
// TAU (Eq.26-29; readings R15-R18, G1 in DESIGN.md): with G = -(1 + 1/n^0bar) of the two cells for this angle and fh = f/2 of the
// face, the factor 1 - g_up + g of Eq.28 is 1 + fh (G_R - G_L) for n^a > 0 and 1 + fh (G_L - G_R) otherwise.
struct FaceGeom {  // n^a and n_0 / dx_a of one face for one angle
    double na, n0;
    bool neg;       // n^a < 0 (or -0): the upper cell is upwind
    int flip;       // the sign bit of n^a
};
__device__ __forceinline__ FaceGeom face_geom(const FaceRec &f, double n1, double n2, double n3) {
    FaceGeom g;
    g.na = chain4(f.e0, f.e1, f.e2, f.e3, n1, n2, n3);
    g.n0 = chain4(f.E0, f.E1, f.E2, f.E3, n1, n2, n3);
    g.neg = hi32(g.na) < 0;
    g.flip = hi32(g.na) & (int)0x80000000;
    return g;
}
// up = the upwind one of (qL, qR), far = the cell behind it, D = qR - qL
template <bool PLM, bool TAU = false>
__device__ __forceinline__ double face_value(const FaceGeom &g, double up, double far, double D, double GL = 0.0, double GR = 0.0, double fh = 0.0) {
    if (PLM) {
        const double dl = up - far, dr = __hiloint2double(__double2hiint(D) ^ g.flip, __double2loint(D)), pr = dl * dr;
        const double h = div3(pr, dl + dr);  // only used where pr > 0, i.e. dl + dr != 0
        if (hi32(pr) > 0) up += h;
    }
    if (TAU) up *= fma(fh, g.neg ? GL - GR : GR - GL, 1.0);
    return __dmul_rn(__dmul_rn(g.na, g.n0), up);
}
// all four intensities in registers (x faces)
template <bool PLM, bool TAU = false>
__device__ __forceinline__ double face_flux(const FaceRec &f, double n1, double n2, double n3, double qLL, double qL, double qR, double qRR,
                                            double GL = 0.0, double GR = 0.0, double fh = 0.0) {
    const FaceGeom g = face_geom(f, n1, n2, n3);
    const double up = g.neg ? qR : qL, far = PLM ? (g.neg ? qRR : qLL) : 0.0;
    return face_value<PLM, TAU>(g, up, far, qR - qL, GL, GR, fh);
}

__device__ __forceinline__ FaceRec lds_face(uint32_t addr) {  // warp-uniform address
    const double2 a = lds2(addr), b = lds2(addr + 16), c = lds2(addr + 32), d = lds2(addr + 48);
    return {a.x, a.y, b.x, b.y, c.x, c.y, d.x, d.y};
}

}  // namespace rad
