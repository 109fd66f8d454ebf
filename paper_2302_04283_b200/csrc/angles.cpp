// angles.cpp -- host-side construction of the angular grids of section 2.6.
//
// Latitude-longitude grid: P:L478-480, centres per reading R1.  Geodesic grid: P:L482-495 gives the
// concept (icosahedron, N_lev^2 triangles per face, projected triangle centres joined by geodesic arcs);
// the complete specification -- vertex placement, index order, neighbour order -- is reading R3 in
// DESIGN.md.  Index and neighbour tables are integer data compared bit for bit with the oracle's, and
// nhat is built with a fixed operation order so that upwind signs agree exactly as well.
#include <algorithm>
#include <array>
#include <cmath>
#include <map>
#include <tuple>

#include "rad_internal.h"

namespace rad {
namespace {

using V3 = std::array<double, 3>;
const double kPi = 3.14159265358979323846;

inline double dot(const V3 &a, const V3 &b) { return (a[0] * b[0] + a[1] * b[1]) + a[2] * b[2]; }
inline V3 cross(const V3 &a, const V3 &b) {
    return {a[1] * b[2] - a[2] * b[1], a[2] * b[0] - a[0] * b[2], a[0] * b[1] - a[1] * b[0]};
}
inline V3 normalized(const V3 &p) {
    double r = std::sqrt((p[0] * p[0] + p[1] * p[1]) + p[2] * p[2]);
    return {p[0] / r, p[1] / r, p[2] / r};
}

void reserve(AngleTables &t, int N) {
    t.N = N;
    t.E = 0;
    t.nhat.assign(3 * N, 0.0);
    t.domega.assign(N, 0.0);
    t.nnbr.assign(N, 0);
    t.nbr.assign(RAD_MAXNBR * N, -1);
    t.nbr_edge.assign(RAD_MAXNBR * N, -1);
    t.edge_lo.clear(); t.edge_hi.clear(); t.edge_len.clear(); t.edge_mid.clear(); t.edge_nrm.clear();
}

// register the edge shared by angle n (slot sn) and angle m (slot sm); `nrm` points from n to m
void push_edge(AngleTables &t, int n, int sn, int m, int sm, double len, const V3 &mid, const V3 &nrm) {
    int e = t.E++;
    bool fwd = n < m;
    t.edge_lo.push_back(fwd ? n : m);
    t.edge_hi.push_back(fwd ? m : n);
    t.edge_len.push_back(len);
    for (int c = 0; c < 3; c++) {
        t.edge_mid.push_back(mid[c]);
        t.edge_nrm.push_back(fwd ? nrm[c] : -nrm[c]);
    }
    t.nbr[n * RAD_MAXNBR + sn] = m; t.nbr_edge[n * RAD_MAXNBR + sn] = e;
    t.nbr[m * RAD_MAXNBR + sm] = n; t.nbr_edge[m * RAD_MAXNBR + sm] = e;
}

}  // namespace

bool build_latlon(int nzeta, int npsi, AngleTables &t, std::string &err) {
    if (nzeta < 1 || npsi < 1) { err = "latlon grid needs nzeta >= 1 and npsi >= 1"; return false; }
    const int N = nzeta * npsi;
    reserve(t, N);
    const double dpsi = 2.0 * kPi / npsi;
    auto mu_face = [&](int l) { return 1.0 - 2.0 * l / nzeta; };  // equally spaced in cos(zeta) from +1 to -1
    for (int l = 0; l < nzeta; l++) {
        const double mu = 0.5 * (mu_face(l) + mu_face(l + 1));      // R1: centre in cos(zeta)
        const double s = std::sqrt(1.0 - mu * mu);
        for (int m = 0; m < npsi; m++) {
            const int n = l * npsi + m;
            const double psi = (m + 0.5) * dpsi;                   // R1: centre in psi
            t.nhat[3 * n + 0] = s * std::cos(psi);                  // Eq.15b-d
            t.nhat[3 * n + 1] = s * std::sin(psi);
            t.nhat[3 * n + 2] = mu;
            t.domega[n] = 4.0 * kPi / N;                            // equal solid angles
            t.nnbr[n] = 4;                                          // slots: zeta-, zeta+, psi-, psi+
        }
    }
    // zeta-faces (parallels) between rows l and l+1; weight sin(zeta_f) dpsi (Eq.20f); normal = e_zeta so that
    // the edge coefficient is n^zeta of Eq.16b
    for (int l = 0; l + 1 < nzeta; l++) {
        const double muf = mu_face(l + 1), sf = std::sqrt(1.0 - muf * muf);
        for (int m = 0; m < npsi; m++) {
            const double psi = (m + 0.5) * dpsi, cp = std::cos(psi), sp = std::sin(psi);
            push_edge(t, l * npsi + m, 1, (l + 1) * npsi + m, 0, sf * dpsi, {sf * cp, sf * sp, muf},
                      {muf * cp, muf * sp, -sf});
        }
    }
    // psi-faces (meridian arcs) between columns m and m+1; weight Delta(cos zeta); normal = e_psi / sin(zeta_c) so
    // that the edge coefficient is n^psi of Eq.16c
    if (npsi > 1) {
        for (int l = 0; l < nzeta; l++) {
            const double mu = 0.5 * (mu_face(l) + mu_face(l + 1)), s = std::sqrt(1.0 - mu * mu);
            for (int m = 0; m < npsi; m++) {
                const double psif = (m + 1) * dpsi, cp = std::cos(psif), sp = std::sin(psif);
                push_edge(t, l * npsi + m, 3, l * npsi + (m + 1) % npsi, 2, mu_face(l) - mu_face(l + 1),
                          {s * cp, s * sp, mu}, {-sp / s, cp / s, 0.0});
            }
        }
    }
    return true;
}

bool build_geodesic(int nlev, AngleTables &t, std::string &err) {
    if (nlev < 1 || nlev > 64) { err = "geodesic grid needs 1 <= nlev <= 64"; return false; }
    const int L = nlev, N = 10 * L * L + 2;
    reserve(t, N);
    // icosahedron with a vertex at each pole: V0 north, V1..5 upper ring, V6..10 lower ring (offset by 36 deg), V11 south
    std::array<V3, 12> V;
    const double ring_r = 2.0 / std::sqrt(5.0), ring_z = 1.0 / std::sqrt(5.0);
    V[0] = {0.0, 0.0, 1.0};
    V[11] = {0.0, 0.0, -1.0};
    for (int k = 0; k < 5; k++) {
        V[1 + k] = {ring_r * std::cos(2.0 * kPi * k / 5.0), ring_r * std::sin(2.0 * kPi * k / 5.0), ring_z};
        V[6 + k] = {ring_r * std::cos(2.0 * kPi * (k + 0.5) / 5.0), ring_r * std::sin(2.0 * kPi * (k + 0.5) / 5.0), -ring_z};
    }
    std::array<std::array<int, 3>, 20> F;
    for (int k = 0; k < 5; k++) {
        const int k1 = (k + 1) % 5;
        F[4 * k + 0] = {0, 1 + k, 1 + k1};
        F[4 * k + 1] = {1 + k, 6 + k, 1 + k1};
        F[4 * k + 2] = {6 + k, 6 + k1, 1 + k1};
        F[4 * k + 3] = {11, 6 + k1, 6 + k};
    }
    // lattice points; identity is combinatorial; index = order of first occurrence over (face, i, j)
    using Key = std::tuple<int, int, int, int>;
    std::map<Key, int> ids;
    std::vector<V3> planar;  // canonical planar position (first occurrence)
    std::vector<std::array<int, 3>> tris;
    std::vector<int> lat((L + 1) * (L + 1));
    for (int f = 0; f < 20; f++) {
        const int va = F[f][0], vb = F[f][1], vc = F[f][2];
        auto edge_key = [&](int p, int q, int steps_from_p) {
            return p < q ? Key{1, p, q, steps_from_p} : Key{1, q, p, L - steps_from_p};
        };
        for (int i = 0; i <= L; i++)
            for (int j = 0; j <= L - i; j++) {
                Key key;
                if (i == 0 && j == 0) key = Key{0, va, 0, 0};
                else if (i == L) key = Key{0, vb, 0, 0};
                else if (j == L) key = Key{0, vc, 0, 0};
                else if (j == 0) key = edge_key(va, vb, i);
                else if (i == 0) key = edge_key(va, vc, j);
                else if (i + j == L) key = edge_key(vb, vc, j);
                else key = Key{2, f, i, j};
                auto it = ids.find(key);
                int id;
                if (it == ids.end()) {
                    id = (int)planar.size();
                    ids.emplace(key, id);
                    V3 p;
                    for (int c = 0; c < 3; c++) {  // fixed order: (A + (B-A) i/L) + (C-A) j/L
                        const double t1 = (V[vb][c] - V[va][c]) * ((double)i / L);
                        const double t2 = (V[vc][c] - V[va][c]) * ((double)j / L);
                        p[c] = (V[va][c] + t1) + t2;
                    }
                    planar.push_back(p);
                    const V3 u = normalized(p);
                    for (int c = 0; c < 3; c++) t.nhat[3 * id + c] = u[c];
                } else {
                    id = it->second;
                }
                lat[i * (L + 1) + j] = id;
            }
        for (int i = 0; i < L; i++)
            for (int j = 0; j < L - i; j++) {
                tris.push_back({lat[i * (L + 1) + j], lat[(i + 1) * (L + 1) + j], lat[i * (L + 1) + j + 1]});
                if (i + j < L - 1)
                    tris.push_back({lat[(i + 1) * (L + 1) + j], lat[(i + 1) * (L + 1) + j + 1], lat[i * (L + 1) + j + 1]});
            }
    }
    if ((int)planar.size() != N || (int)tris.size() != 20 * L * L) { err = "geodesic grid: internal count mismatch"; return false; }
    // cell corners = projected planar centroids of the small triangles
    std::vector<V3> corner(tris.size());
    std::vector<std::vector<int>> tris_of(N);
    for (size_t q = 0; q < tris.size(); q++) {
        V3 c;
        for (int d = 0; d < 3; d++) c[d] = ((planar[tris[q][0]][d] + planar[tris[q][1]][d]) + planar[tris[q][2]][d]) / 3.0;
        corner[q] = normalized(c);
        for (int s = 0; s < 3; s++) tris_of[tris[q][s]].push_back((int)q);
    }
    auto nh = [&](int n) { return V3{t.nhat[3 * n], t.nhat[3 * n + 1], t.nhat[3 * n + 2]}; };
    std::vector<std::array<int, RAD_MAXNBR>> corner_of(N);  // corner k of cell n lies between neighbours k and k+1
    for (int n = 0; n < N; n++) {
        // neighbours = the other vertices of the incident triangles, sorted counter-clockwise seen from outside
        std::vector<int> nb;
        for (int q : tris_of[n])
            for (int s = 0; s < 3; s++) {
                const int m = tris[q][s];
                if (m != n && std::find(nb.begin(), nb.end(), m) == nb.end()) nb.push_back(m);
            }
        if (nb.size() != tris_of[n].size() || nb.size() > RAD_MAXNBR) { err = "geodesic grid: bad vertex degree"; return false; }
        const V3 c = nh(n);
        int ax = 0;
        for (int d = 1; d < 3; d++) if (std::fabs(c[d]) < std::fabs(c[ax])) ax = d;
        V3 ref = {0.0, 0.0, 0.0};
        ref[ax] = 1.0;
        const double pr = dot(ref, c);
        const V3 e1 = normalized({ref[0] - pr * c[0], ref[1] - pr * c[1], ref[2] - pr * c[2]});
        const V3 e2 = cross(c, e1);
        std::vector<std::pair<double, int>> by_angle;
        for (int m : nb) by_angle.push_back({std::atan2(dot(nh(m), e2), dot(nh(m), e1)), m});
        std::sort(by_angle.begin(), by_angle.end());
        const int deg = (int)nb.size();
        int start = 0;
        for (int q = 1; q < deg; q++) if (by_angle[q].second < by_angle[start].second) start = q;
        t.nnbr[n] = deg;
        for (int q = 0; q < deg; q++) t.nbr[n * RAD_MAXNBR + q] = by_angle[(start + q) % deg].second;
        double omega = 0.0;
        for (int k = 0; k < deg; k++) {
            const int m0 = t.nbr[n * RAD_MAXNBR + k], m1 = t.nbr[n * RAD_MAXNBR + (k + 1) % deg];
            int found = -1;
            for (int q : tris_of[n]) {
                bool h0 = false, h1 = false;
                for (int s = 0; s < 3; s++) { h0 |= tris[q][s] == m0; h1 |= tris[q][s] == m1; }
                if (h0 && h1) found = q;
            }
            if (found < 0) { err = "geodesic grid: corner lookup failed"; return false; }
            corner_of[n][k] = found;
        }
        for (int k = 0; k < deg; k++) {  // fan of spherical triangles (centre, corner_k, corner_{k+1})
            const V3 &b = corner[corner_of[n][k]], &d = corner[corner_of[n][(k + 1) % deg]];
            omega += 2.0 * std::atan2(std::fabs(dot(c, cross(b, d))), 1.0 + dot(c, b) + dot(b, d) + dot(d, c));
        }
        t.domega[n] = omega;
    }
    // unique edges, enumerated by (n ascending, slot ascending) with the neighbour index above n
    for (int n = 0; n < N; n++) {
        const int deg = t.nnbr[n];
        for (int k = 0; k < deg; k++) {
            const int m = t.nbr[n * RAD_MAXNBR + k];
            if (m < n) continue;
            const V3 &c1 = corner[corner_of[n][(k + deg - 1) % deg]], &c2 = corner[corner_of[n][k]];
            const V3 cx = cross(c1, c2);
            const double len = std::atan2(std::sqrt(dot(cx, cx)), dot(c1, c2));
            const V3 mid = normalized({c1[0] + c2[0], c1[1] + c2[1], c1[2] + c2[2]});
            V3 nrm = normalized(cx);
            const V3 a = nh(n), b = nh(m);
            if (dot(nrm, {b[0] - a[0], b[1] - a[1], b[2] - a[2]}) < 0) nrm = {-nrm[0], -nrm[1], -nrm[2]};
            int sm = -1;
            for (int q = 0; q < t.nnbr[m]; q++) if (t.nbr[m * RAD_MAXNBR + q] == n) sm = q;
            push_edge(t, n, k, m, sm, len, mid, nrm);
        }
    }
    return true;
}

// Explicit angle grid (rad_angles kind 2: any grid of cells with centres, solid angles and edges): the caller gives per
// angle the direction, the solid angle, the neighbour list, and per (angle, slot) the edge's arc length, unit midpoint and in-sphere
// normal pointing from the angle to that neighbour.  Unique edges are enumerated by (n ascending, slot ascending) with the neighbour
// index above n (the order of the geodesic builder); an edge's data are taken from its lower angle's entry.
bool build_explicit(int N, const double *nhat, const double *domega, const int *nnbr, const int *nbr, const double *edge_len,
                    const double *edge_mid, const double *edge_nrm, AngleTables &t, std::string &err) {
    if (N < 1 || !nhat || !domega || !nnbr || !nbr || !edge_len || !edge_mid || !edge_nrm) { err = "explicit angle grid: missing table"; return false; }
    reserve(t, N);
    for (int n = 0; n < N; n++) {
        double r2 = 0.0;
        for (int c = 0; c < 3; c++) { t.nhat[3 * n + c] = nhat[3 * n + c]; r2 += nhat[3 * n + c] * nhat[3 * n + c]; }
        if (!(std::fabs(r2 - 1.0) < 1e-12) || !(domega[n] > 0.0) || !std::isfinite(domega[n])) { err = "explicit angle grid: nhat must be unit vectors and domega positive"; return false; }
        t.domega[n] = domega[n];
        if (nnbr[n] < 0 || nnbr[n] > RAD_MAXNBR) { err = "explicit angle grid: nnbr out of range"; return false; }
        t.nnbr[n] = nnbr[n];
        for (int s = 0; s < RAD_MAXNBR; s++) {
            const int m = nbr[n * RAD_MAXNBR + s];
            if (m < -1 || m >= N || m == n || (s >= nnbr[n] && m != -1)) { err = "explicit angle grid: bad neighbour index"; return false; }
        }
    }
    for (int n = 0; n < N; n++)
        for (int s = 0; s < RAD_MAXNBR; s++) {
            const int m = nbr[n * RAD_MAXNBR + s];
            if (m < 0 || m < n) continue;
            int sm = -1;  // the neighbour's matching slot: the first one that lists n and is not paired yet
            for (int q = 0; q < RAD_MAXNBR && sm < 0; q++)
                if (nbr[m * RAD_MAXNBR + q] == n && t.nbr_edge[m * RAD_MAXNBR + q] < 0) sm = q;
            if (sm < 0) { err = "explicit angle grid: neighbour lists are not symmetric"; return false; }
            const size_t q = (size_t)n * RAD_MAXNBR + s;
            if (!std::isfinite(edge_len[q]) || edge_len[q] < 0.0) { err = "explicit angle grid: bad edge length"; return false; }
            double m2 = 0.0, k2 = 0.0;  // a NaN here would reach every stored coefficient of every cell without any error
            for (int c = 0; c < 3; c++) { m2 += edge_mid[3 * q + c] * edge_mid[3 * q + c]; k2 += edge_nrm[3 * q + c] * edge_nrm[3 * q + c]; }
            // (edge_nrm carries the metric factor of its coordinate: 1 / sin zeta on the psi edges of a latitude-longitude grid, Eq.16c)
            if (!(std::fabs(m2 - 1.0) < 1e-6) || !std::isfinite(k2) || !(k2 > 0.0)) { err = "explicit angle grid: edge_mid must be finite unit vectors, edge_nrm finite and non-zero"; return false; }
            push_edge(t, n, s, m, sm, edge_len[q], {edge_mid[3 * q], edge_mid[3 * q + 1], edge_mid[3 * q + 2]},
                      {edge_nrm[3 * q], edge_nrm[3 * q + 1], edge_nrm[3 * q + 2]});
        }
    for (int n = 0; n < N; n++)
        for (int s = 0; s < RAD_MAXNBR; s++)
            if (nbr[n * RAD_MAXNBR + s] >= 0 && t.nbr_edge[n * RAD_MAXNBR + s] < 0) { err = "explicit angle grid: neighbour lists are not symmetric"; return false; }
    return true;
}

}  // namespace rad
