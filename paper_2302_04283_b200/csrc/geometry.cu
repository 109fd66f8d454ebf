// geometry.cu -- subsystem 1: geometry / tetrad precompute (paper section 2.1-2.2).
//
// One thread per (cell, evaluation point): the cell centre and the centres of its lower x, y, z faces.
// Everything is stationary (Eq.4, Eq.12), so this runs once in rad_create.  Spatial derivatives are
// carried by forward-mode dual numbers through metric -> 3+1 split -> tetrad; d/dt = 0.
//
//   3+1 split (Eq.5) done the standard way round: gamma_ab = g_ab, beta_a = g_0a,
//   beta^a = gamma^ab beta_b, alpha^2 = beta_a beta^a - g_00.
//   Tetrad (R2): e_0hat = (1/alpha, -beta^a/alpha) (Eq.11), triad = Gram-Schmidt of d_x, d_y, d_z.
//   Ricci rotation coefficients (Eq.17) with the first index lowered,
//     omega_{c a b} = e^lam_c e^del_b ( g_{lam eps} d_del e^eps_a + Gamma_{lam del sig} e^sig_a ),
//     Gamma_{lam del sig} = (d_del g_{lam sig} + d_sig g_{lam del} - d_lam g_{del sig}) / 2,
//   which needs no inverse metric; omega^c_{ab} = eta^{cc} omega_{cab}.
#include <math.h>

#include "rad_internal.h"

namespace rad {
namespace {

struct D3 {  // value and gradient
    double v, x, y, z;
};
__device__ __forceinline__ D3 cst(double c) { return {c, 0.0, 0.0, 0.0}; }
__device__ __forceinline__ D3 operator+(D3 a, D3 b) { return {a.v + b.v, a.x + b.x, a.y + b.y, a.z + b.z}; }
__device__ __forceinline__ D3 operator-(D3 a, D3 b) { return {a.v - b.v, a.x - b.x, a.y - b.y, a.z - b.z}; }
__device__ __forceinline__ D3 operator-(D3 a) { return {-a.v, -a.x, -a.y, -a.z}; }
__device__ __forceinline__ D3 operator*(D3 a, D3 b) {
    return {a.v * b.v, a.x * b.v + a.v * b.x, a.y * b.v + a.v * b.y, a.z * b.v + a.v * b.z};
}
__device__ __forceinline__ D3 operator*(double s, D3 a) { return {s * a.v, s * a.x, s * a.y, s * a.z}; }
__device__ __forceinline__ D3 operator/(D3 a, D3 b) {
    const double q = a.v / b.v, r = 1.0 / b.v;
    return {q, (a.x - q * b.x) * r, (a.y - q * b.y) * r, (a.z - q * b.z) * r};
}
__device__ __forceinline__ D3 dsqrt(D3 a) {
    const double s = sqrt(a.v), h = 0.5 / s;
    return {s, h * a.x, h * a.y, h * a.z};
}
__device__ __forceinline__ double grad(const D3 &a, int d) { return d == 1 ? a.x : (d == 2 ? a.y : (d == 3 ? a.z : 0.0)); }

// covariant metric, symmetric 4x4
__device__ void metric(int kind, double M, double a, double px, double py, double pz, D3 g[4][4]) {
    for (int m = 0; m < 4; m++)
        for (int n = 0; n < 4; n++) g[m][n] = cst(m == n ? (m == 0 ? -1.0 : 1.0) : 0.0);
    if (kind == 0) return;
    // Cartesian Kerr-Schild: g = eta + f l l,  f = 2 M r^3 / (r^4 + a^2 z^2),  l = (1, (r x + a y)/(r^2+a^2), (r y - a x)/(r^2+a^2), z/r)
    const D3 x = {px, 1.0, 0.0, 0.0}, y = {py, 0.0, 1.0, 0.0}, z = {pz, 0.0, 0.0, 1.0};
    const D3 a2 = cst(a * a);
    const D3 w = x * x + y * y + z * z - a2;
    const D3 r2 = 0.5 * (w + dsqrt(w * w + 4.0 * (a2 * z * z)));
    const D3 r = dsqrt(r2);
    const D3 f = (2.0 * M) * (r2 * r) / (r2 * r2 + a2 * z * z);
    D3 l[4];
    l[0] = cst(1.0);
    l[1] = (r * x + a * y) / (r2 + a2);
    l[2] = (r * y - a * x) / (r2 + a2);
    l[3] = z / r;
    for (int m = 0; m < 4; m++)
        for (int n = 0; n < 4; n++) g[m][n] = g[m][n] + f * l[m] * l[n];
}

struct PointGeom {
    double alpha;
    double beta_up[3];
    double e[4][4];      // e[mu][ahat]
    double E[4];         // g_{0 mu} e^mu_ahat
    double omega[4][4][4];  // omega^c_{ab}
    double g[4][4];
};

__device__ void point_geometry(int kind, double M, double a, double px, double py, double pz, bool want_omega, PointGeom &out) {
    D3 g[4][4];
    metric(kind, M, a, px, py, pz, g);
    // inverse spatial metric by cofactors
    D3 gm[3][3];
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) gm[i][j] = g[i + 1][j + 1];
    D3 cof[3][3];
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) {
            const int i1 = (i + 1) % 3, i2 = (i + 2) % 3, j1 = (j + 1) % 3, j2 = (j + 2) % 3;
            cof[i][j] = gm[i1][j1] * gm[i2][j2] - gm[i1][j2] * gm[i2][j1];
        }
    const D3 det = gm[0][0] * cof[0][0] + gm[0][1] * cof[0][1] + gm[0][2] * cof[0][2];
    D3 beta_up[3];
    for (int i = 0; i < 3; i++) {
        D3 s = cst(0.0);
        for (int j = 0; j < 3; j++) s = s + (cof[j][i] / det) * g[0][j + 1];  // gamma^{ij} beta_j
        beta_up[i] = s;
    }
    D3 b2 = cst(0.0);
    for (int i = 0; i < 3; i++) b2 = b2 + g[0][i + 1] * beta_up[i];
    const D3 alpha = dsqrt(b2 - g[0][0]);
    D3 e[4][4];
    e[0][0] = cst(1.0) / alpha;
    for (int i = 0; i < 3; i++) e[i + 1][0] = -(beta_up[i] / alpha);
    for (int ah = 1; ah < 4; ah++) {
        D3 v[4] = {cst(0.0), cst(0.0), cst(0.0), cst(0.0)};
        v[ah] = cst(1.0);
        for (int bh = 1; bh < ah; bh++) {
            D3 pr = cst(0.0);
            for (int i = 1; i < 4; i++) pr = pr + g[ah][i] * e[i][bh];
            for (int i = 1; i < 4; i++) v[i] = v[i] - pr * e[i][bh];
        }
        D3 n2 = cst(0.0);
        for (int i = 1; i < 4; i++)
            for (int j = 1; j < 4; j++) n2 = n2 + g[i][j] * v[i] * v[j];
        const D3 nr = dsqrt(n2);
        e[0][ah] = cst(0.0);
        for (int i = 1; i < 4; i++) e[i][ah] = v[i] / nr;
    }
    out.alpha = alpha.v;
    for (int i = 0; i < 3; i++) out.beta_up[i] = beta_up[i].v;
    for (int m = 0; m < 4; m++)
        for (int n = 0; n < 4; n++) { out.e[m][n] = e[m][n].v; out.g[m][n] = g[m][n].v; }
    for (int ah = 0; ah < 4; ah++) {
        double s = 0.0;
        for (int m = 0; m < 4; m++) s += g[0][m].v * e[m][ah].v;
        out.E[ah] = s;
    }
    out.E[0] = -alpha.v;  // g_{0 mu} e^mu_0hat = (g_00 - beta_i beta^i)/alpha = -alpha exactly
    if (!want_omega) return;
    for (int c = 0; c < 4; c++)
        for (int ah = 0; ah < 4; ah++)
            for (int bh = 0; bh < 4; bh++) {
                double s = 0.0;
                for (int lam = 0; lam < 4; lam++) {
                    const double ec = e[lam][c].v;
                    if (ec == 0.0) continue;
                    for (int del = 1; del < 4; del++) {  // e^0_bhat * d_0(...) = 0 and Gamma_{lam 0 sig} handled below
                        const double eb = e[del][bh].v;
                        if (eb == 0.0) continue;
                        double cov = 0.0;
                        for (int eps = 0; eps < 4; eps++) cov += g[lam][eps].v * grad(e[eps][ah], del);
                        for (int sig = 0; sig < 4; sig++)
                            cov += 0.5 * (grad(g[lam][sig], del) + grad(g[lam][del], sig) - grad(g[del][sig], lam)) * e[sig][ah].v;
                        s += ec * eb * cov;
                    }
                    {   // del = 0: d_0 e = 0; Gamma_{lam 0 sig} = (d_sig g_{lam 0} - d_lam g_{0 sig}) / 2
                        const double eb = e[0][bh].v;
                        if (eb != 0.0) {
                            double cov = 0.0;
                            for (int sig = 0; sig < 4; sig++) cov += 0.5 * (grad(g[lam][0], sig) - grad(g[0][sig], lam)) * e[sig][ah].v;
                            s += ec * eb * cov;
                        }
                    }
                }
                out.omega[c][ah][bh] = (c == 0 ? -s : s);
            }
}

// xfx, xfy, xfz: face coordinates of a stretched axis (device), or nullptr = uniform spacing from (x0, y0, z0)
__global__ void k_geometry(int kind, double M, double a, double excise_r, int NI, int NJ, int NK, int ng, double x0, double y0,
                           double z0, double dx, double dy, double dz, const double *__restrict__ xfx, const double *__restrict__ xfy,
                           const double *__restrict__ xfz, double *__restrict__ cell, double *__restrict__ face) {
    const long long ncell = (long long)NI * NJ * NK;
    const long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (t >= 4 * ncell) return;
    const long long c = t >> 2;
    const int pt = (int)(t & 3);  // 0 centre, 1..3 lower face along axis pt-1
    const int i = (int)(c % NI), j = (int)((c / NI) % NJ), k = (int)(c / ((long long)NI * NJ));
    double px = xfx ? 0.5 * (xfx[i] + xfx[i + 1]) : x0 + (i - ng + 0.5) * dx, py = xfy ? 0.5 * (xfy[j] + xfy[j + 1]) : y0 + (j - ng + 0.5) * dy,
           pz = xfz ? 0.5 * (xfz[k] + xfz[k + 1]) : z0 + (k - ng + 0.5) * dz;
    if (pt == 1) px = xfx ? xfx[i] : x0 + (i - ng) * dx;
    if (pt == 2) py = xfy ? xfy[j] : y0 + (j - ng) * dy;
    if (pt == 3) pz = xfz ? xfz[k] : z0 + (k - ng) * dz;
    PointGeom G;
    point_geometry(kind, M, a, px, py, pz, pt == 0, G);
    if (pt == 0) {
        double *o = cell + c * RAD_NCELL;
        o[0] = G.e[0][0];
        for (int q = 0; q < 4; q++) o[1 + q] = G.E[q];
        int w = 5;
        for (int ch = 1; ch < 4; ch++)
            for (int al = 0; al < 4; al++)
                for (int be = al; be < 4; be++) o[w++] = (al == be) ? G.omega[ch][al][al] : G.omega[ch][al][be] + G.omega[ch][be][al];
        for (int q = 0; q < 3; q++) o[35 + q] = G.beta_up[q];
        o[38] = G.e[1][1]; o[39] = G.e[1][2]; o[40] = G.e[1][3]; o[41] = G.e[2][2]; o[42] = G.e[2][3]; o[43] = G.e[3][3];
        // co-triad theta^a_i = g_{i mu} e^mu_a (spatial part of the inverse tetrad, Eq.9)
        double th[3][3];
        for (int ah = 0; ah < 3; ah++)
            for (int q = 0; q < 3; q++) {
                double s = 0.0;
                for (int m = 1; m < 4; m++) s += G.g[q + 1][m] * G.e[m][ah + 1];
                th[ah][q] = s;
            }
        o[44] = th[0][0]; o[45] = th[0][1]; o[46] = th[0][2]; o[47] = th[1][1]; o[48] = th[1][2]; o[49] = th[2][2];
        double ex = 0.0;
        if (kind == 1 && excise_r > 0.0) {
            const double R2 = px * px + py * py + pz * pz, ww = R2 - a * a;
            const double r = sqrt(0.5 * (ww + sqrt(ww * ww + 4.0 * a * a * pz * pz)));
            ex = (r < excise_r) ? 1.0 : 0.0;
        }
        o[50] = ex;
        o[51] = 0.0;
    } else {
        double *o = face + (c * 3 + (pt - 1)) * RAD_NFACE;
        for (int q = 0; q < 4; q++) { o[q] = G.e[pt][q]; o[4 + q] = G.E[q]; }
    }
}

}  // namespace

int launch_geometry(const rad_metric &m, const rad_grid &g, const double *const xf_dev[3], double *cell, double *face, long long ncell, cudaStream_t s) {
    const int NI = g.n[0] + 2 * g.ng, NJ = g.n[1] + 2 * g.ng, NK = g.n[2] + 2 * g.ng;
    const int threads = 128;
    const long long blocks = (4 * ncell + threads - 1) / threads;
    k_geometry<<<(unsigned)blocks, threads, 0, s>>>(m.kind, m.M, m.a, m.excise_r, NI, NJ, NK, g.ng, g.x0[0], g.x0[1], g.x0[2],
                                                    g.dx[0], g.dx[1], g.dx[2], xf_dev[0], xf_dev[1], xf_dev[2], cell, face);
    return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

}  // namespace rad
