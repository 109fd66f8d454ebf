/* oracle/rad_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain FP64 CPU statement of the explicit-plus-locally-implicit radiation stage of
 * White et al., arXiv 2302.04283 ("the paper"), written from the paper's equations in the
 * paper's order and notation.  P:L<n> = /root/reference/PAPER.md line n.  R#/G# = readings
 * listed in DESIGN.md (and SURVEY.md 8(c)) where the paper is silent / garbled.
 *
 * No blocking, fusion or reordering: every function is the formula written out.  The only
 * fused multiply-adds are the explicit fma() chains that pin the arithmetic deciding the
 * upwind signs (n^a at faces, c_e at angular edges), so that integer sign tables can be
 * compared bit for bit.  Compile: gcc -O2 -ffp-contract=off -fopenmp.
 *
 * Parity unpinned (no external anchor; the oracle IS the definition): R1 lat-lon centres,
 * R3 geodesic index order, R2 triad order, R6 face-centre evaluation, R7 limiter form,
 * R12 renorm flag, R13 failure policy, R14 mask placement; and in the optical-depth-aware flux
 * (face_flux with vel != NULL, Eq.26-29): the sign and form of g_L/R (Eq.29) and the readings
 * R15-R17 -- its limits (tau = 0, tau -> 0 quadratically, uniform flow, saturation) and
 * conservation ARE pinned (tests/test_oracle_tauflux.py).  Everything else is pinned by
 * tests/test_oracle_*.py (-m "not gpu").
 */
#include "rad_oracle.h"
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

static const double PI = 3.14159265358979323846;

/* ======================================================================================
 * O1. Angle grids
 * ==================================================================================== */
struct orc_angles {
    int N, E;
    int kind, nzeta, npsi; /* 0 latitude-longitude (nzeta x npsi), 1 geodesic */
    double *nhat;    /* [N][3]  unit directions n^ahat, Eq.15b-d */
    double *domega;  /* [N]     Delta Omega */
    int *nnbr;       /* [N] */
    int *nbr;        /* [N][6] neighbour angle index or -1 */
    int *nbr_edge;   /* [N][6] unique edge id or -1 */
    int *edge_lo, *edge_hi; /* [E] lo < hi */
    double *edge_len;       /* [E] Delta lambda_e (Eq.20f) */
    double *edge_mid;       /* [E][3] unit vector to edge midpoint */
    double *edge_nrm;       /* [E][3] in-sphere normal of the edge, pointing lo -> hi */
    double *edge_T;         /* [E][3][10] pinned products T[c][k] = N^c * q_k, q = n^alpha n^beta */
};

static void ang_alloc(orc_angles *A, int N, int Emax) {
    A->N = N; A->E = 0;
    A->nhat = calloc((size_t)N * 3, sizeof(double));
    A->domega = calloc(N, sizeof(double));
    A->nnbr = calloc(N, sizeof(int));
    A->nbr = malloc(sizeof(int) * N * ORC_MAXNBR);
    A->nbr_edge = malloc(sizeof(int) * N * ORC_MAXNBR);
    for (int i = 0; i < N * ORC_MAXNBR; i++) { A->nbr[i] = -1; A->nbr_edge[i] = -1; }
    A->edge_lo = calloc(Emax, sizeof(int));
    A->edge_hi = calloc(Emax, sizeof(int));
    A->edge_len = calloc(Emax, sizeof(double));
    A->edge_mid = calloc((size_t)Emax * 3, sizeof(double));
    A->edge_nrm = calloc((size_t)Emax * 3, sizeof(double));
    A->edge_T = calloc((size_t)Emax * 30, sizeof(double));
}

/* T[c][k] = N^c * q_k with q_k = n^alpha n^beta over (00,01,02,03,11,12,13,22,23,33), n^0hat = 1.
 * Each entry is two roundings: q_k = n^alpha*n^beta, then N^c*q_k.  (pinned) */
static void edge_fill_T(orc_angles *A, int e) {
    const double *m = &A->edge_mid[3 * e], *Nn = &A->edge_nrm[3 * e];
    double n4[4] = {1.0, m[0], m[1], m[2]}, q[10];
    int k = 0;
    for (int a = 0; a < 4; a++)
        for (int b = a; b < 4; b++) q[k++] = n4[a] * n4[b];
    for (int c = 0; c < 3; c++)
        for (k = 0; k < 10; k++) A->edge_T[30 * e + 10 * c + k] = Nn[c] * q[k];
}

void orc_angles_free(orc_angles *A) {
    if (!A) return;
    free(A->nhat); free(A->domega); free(A->nnbr); free(A->nbr); free(A->nbr_edge);
    free(A->edge_lo); free(A->edge_hi); free(A->edge_len); free(A->edge_mid); free(A->edge_nrm);
    free(A->edge_T); free(A);
}
int orc_angles_nang(const orc_angles *A) { return A->N; }
int orc_angles_nedge(const orc_angles *A) { return A->E; }

void orc_angles_tables(const orc_angles *A, double *nhat, double *domega, int *nnbr, int *nbr,
                       int *nbr_edge, int *edge_lo, int *edge_hi, double *edge_len,
                       double *edge_mid, double *edge_nrm, double *edge_T) {
    int N = A->N, E = A->E;
    if (nhat) memcpy(nhat, A->nhat, sizeof(double) * 3 * N);
    if (domega) memcpy(domega, A->domega, sizeof(double) * N);
    if (nnbr) memcpy(nnbr, A->nnbr, sizeof(int) * N);
    if (nbr) memcpy(nbr, A->nbr, sizeof(int) * N * ORC_MAXNBR);
    if (nbr_edge) memcpy(nbr_edge, A->nbr_edge, sizeof(int) * N * ORC_MAXNBR);
    if (edge_lo) memcpy(edge_lo, A->edge_lo, sizeof(int) * E);
    if (edge_hi) memcpy(edge_hi, A->edge_hi, sizeof(int) * E);
    if (edge_len) memcpy(edge_len, A->edge_len, sizeof(double) * E);
    if (edge_mid) memcpy(edge_mid, A->edge_mid, sizeof(double) * 3 * E);
    if (edge_nrm) memcpy(edge_nrm, A->edge_nrm, sizeof(double) * 3 * E);
    if (edge_T) memcpy(edge_T, A->edge_T, sizeof(double) * 30 * E);
}

/* add the unique edge (n,slot_n)-(m,slot_m); nrm points n -> m on entry */
static void ang_add_edge(orc_angles *A, int n, int sn, int m, int sm, double len, const double mid[3],
                         const double nrm_n_to_m[3]) {
    int e = A->E++;
    int lo = n < m ? n : m, hi = n < m ? m : n;
    double s = (n < m) ? 1.0 : -1.0;
    A->edge_lo[e] = lo; A->edge_hi[e] = hi; A->edge_len[e] = len;
    for (int c = 0; c < 3; c++) { A->edge_mid[3 * e + c] = mid[c]; A->edge_nrm[3 * e + c] = s * nrm_n_to_m[c]; }
    A->nbr[n * ORC_MAXNBR + sn] = m; A->nbr_edge[n * ORC_MAXNBR + sn] = e;
    A->nbr[m * ORC_MAXNBR + sm] = n; A->nbr_edge[m * ORC_MAXNBR + sm] = e;
    edge_fill_T(A, e);
}

/* Latitude/longitude grid: N_zeta+1 lines of latitude equally spaced in cos(zeta)
 * from +1 to -1, N_psi+1 lines of longitude equally spaced in psi; equal solid angles
 * 4 pi/(N_zeta N_psi).  R1: centres at the midpoint of the face cosines and of the face psi.
 * Index n = l*N_psi + m.  Slots: 0 zeta-, 1 zeta+, 2 psi-, 3 psi+.
 * Edge weights Eq.20f: zeta-face Delta lambda = sin(zeta_f) Delta psi, psi-face
 * Delta lambda = Delta(cos zeta).  Edge "normal" Ntilde such that c_e = a . Ntilde equals the
 * paper's n^zeta (Eq.16b) resp. n^psi (Eq.16c): e_zeta resp. e_psi / sin(zeta_centre). */
orc_angles *orc_angles_latlon(int nzeta, int npsi) {
    if (nzeta < 1 || npsi < 1) return NULL;
    orc_angles *A = calloc(1, sizeof(*A));
    int N = nzeta * npsi;
    ang_alloc(A, N, 2 * N + 4);
    A->kind = 0; A->nzeta = nzeta; A->npsi = npsi;
    double dpsi = 2.0 * PI / npsi;
    for (int l = 0; l < nzeta; l++) {
        double muf0 = 1.0 - 2.0 * l / nzeta, muf1 = 1.0 - 2.0 * (l + 1) / nzeta;
        double mu = 0.5 * (muf0 + muf1), s = sqrt(1.0 - mu * mu);
        for (int m = 0; m < npsi; m++) {
            int n = l * npsi + m;
            double psi = (m + 0.5) * dpsi;
            A->nhat[3 * n + 0] = s * cos(psi);
            A->nhat[3 * n + 1] = s * sin(psi);
            A->nhat[3 * n + 2] = mu;
            A->domega[n] = 4.0 * PI / N;
            A->nnbr[n] = 4;
        }
    }
    /* zeta-faces between l and l+1 at fixed m (none at the poles: sin(zeta_f)=0 there) */
    for (int l = 0; l + 1 < nzeta; l++) {
        double muf = 1.0 - 2.0 * (l + 1) / nzeta, sf = sqrt(1.0 - muf * muf);
        for (int m = 0; m < npsi; m++) {
            double psi = (m + 0.5) * dpsi;
            double mid[3] = {sf * cos(psi), sf * sin(psi), muf};
            double ez[3] = {muf * cos(psi), muf * sin(psi), -sf}; /* unit vector of increasing zeta */
            ang_add_edge(A, l * npsi + m, 1, (l + 1) * npsi + m, 0, sf * dpsi, mid, ez);
        }
    }
    /* psi-faces between m and m+1 (periodic) at fixed l */
    if (npsi > 1)
        for (int l = 0; l < nzeta; l++) {
            double muf0 = 1.0 - 2.0 * l / nzeta, muf1 = 1.0 - 2.0 * (l + 1) / nzeta;
            double mu = 0.5 * (muf0 + muf1), s = sqrt(1.0 - mu * mu);
            for (int m = 0; m < npsi; m++) {
                int m1 = (m + 1) % npsi;
                double psif = (m + 1) * dpsi;
                double mid[3] = {s * cos(psif), s * sin(psif), mu};
                double ep[3] = {-sin(psif) / s, cos(psif) / s, 0.0}; /* e_psi / s_c, increasing psi */
                ang_add_edge(A, l * npsi + m, 3, l * npsi + m1, 2, muf0 - muf1, mid, ep);
            }
        }
    return A;
}

/* ---- small 3-vector helpers ---- */
static double dot3(const double *a, const double *b) { return (a[0] * b[0] + a[1] * b[1]) + a[2] * b[2]; }
static void cross3(const double *a, const double *b, double *c) {
    c[0] = a[1] * b[2] - a[2] * b[1];
    c[1] = a[2] * b[0] - a[0] * b[2];
    c[2] = a[0] * b[1] - a[1] * b[0];
}
static void unit3(const double *p, double *u) {
    double r = sqrt((p[0] * p[0] + p[1] * p[1]) + p[2] * p[2]);
    u[0] = p[0] / r; u[1] = p[1] / r; u[2] = p[2] / r;
}
/* spherical triangle area, tan(Omega/2) = |a.(b x c)| / (1 + a.b + b.c + c.a) */
static double sph_tri_area(const double *a, const double *b, const double *c) {
    double bc[3];
    cross3(b, c, bc);
    return 2.0 * atan2(fabs(dot3(a, bc)), 1.0 + dot3(a, b) + dot3(b, c) + dot3(c, a));
}

/* Geodesic grid: icosahedron, each face triangulated into N_lev^2 triangles,
 * triangle centres projected onto the sphere are the cell CORNERS; cells are the lattice
 * points (10 N_lev^2 + 2 of them, 12 pentagons).  Full specification = reading R3. */
typedef struct { int kind, a, b, c; } lat_key; /* 0: vertex a; 1: edge (a<b), step c from a; 2: face a, (i,j)=(b,c) */

orc_angles *orc_angles_geodesic(int nlev) {
    if (nlev < 1) return NULL;
    int L = nlev, N = 10 * L * L + 2, NT = 20 * L * L;
    orc_angles *A = calloc(1, sizeof(*A));
    ang_alloc(A, N, 3 * N);
    A->kind = 1;
    /* icosahedron: north pole V0, upper ring U_k = V_{1+k}, lower ring L_k = V_{6+k}, south pole V11 */
    double V[12][3];
    double cr = 2.0 / sqrt(5.0), sr = 1.0 / sqrt(5.0);
    V[0][0] = 0; V[0][1] = 0; V[0][2] = 1;
    V[11][0] = 0; V[11][1] = 0; V[11][2] = -1;
    for (int k = 0; k < 5; k++) {
        V[1 + k][0] = cr * cos(2.0 * PI * k / 5.0); V[1 + k][1] = cr * sin(2.0 * PI * k / 5.0); V[1 + k][2] = sr;
        V[6 + k][0] = cr * cos(2.0 * PI * (k + 0.5) / 5.0); V[6 + k][1] = cr * sin(2.0 * PI * (k + 0.5) / 5.0); V[6 + k][2] = -sr;
    }
    int F[20][3];
    for (int k = 0; k < 5; k++) {
        int k1 = (k + 1) % 5;
        int f0[3] = {0, 1 + k, 1 + k1}, f1[3] = {1 + k, 6 + k, 1 + k1}, f2[3] = {6 + k, 6 + k1, 1 + k1}, f3[3] = {11, 6 + k1, 6 + k};
        memcpy(F[4 * k + 0], f0, sizeof f0); memcpy(F[4 * k + 1], f1, sizeof f1);
        memcpy(F[4 * k + 2], f2, sizeof f2); memcpy(F[4 * k + 3], f3, sizeof f3);
    }
    lat_key *keys = malloc(sizeof(lat_key) * N);
    double *P = malloc(sizeof(double) * 3 * N); /* canonical planar lattice point (first occurrence) */
    int *idx = malloc(sizeof(int) * 20 * (L + 1) * (L + 1));
    int *tri = malloc(sizeof(int) * 3 * NT);
    int nk = 0, nt = 0;
#define IDX(f, i, j) idx[((f) * (L + 1) + (i)) * (L + 1) + (j)]
    for (int f = 0; f < 20; f++) {
        int va = F[f][0], vb = F[f][1], vc = F[f][2];
        for (int i = 0; i <= L; i++)
            for (int j = 0; j <= L - i; j++) {
                lat_key key;
                if (i == 0 && j == 0) { key = (lat_key){0, va, 0, 0}; }
                else if (i == L) { key = (lat_key){0, vb, 0, 0}; }
                else if (j == L) { key = (lat_key){0, vc, 0, 0}; }
                else if (j == 0) { /* edge A-B, i steps from A */
                    key = (va < vb) ? (lat_key){1, va, vb, i} : (lat_key){1, vb, va, L - i};
                } else if (i == 0) { /* edge A-C, j steps from A */
                    key = (va < vc) ? (lat_key){1, va, vc, j} : (lat_key){1, vc, va, L - j};
                } else if (i + j == L) { /* edge B-C, j steps from B */
                    key = (vb < vc) ? (lat_key){1, vb, vc, j} : (lat_key){1, vc, vb, L - j};
                } else { key = (lat_key){2, f, i, j}; }
                int id = -1;
                for (int q = 0; q < nk; q++)
                    if (keys[q].kind == key.kind && keys[q].a == key.a && keys[q].b == key.b && keys[q].c == key.c) { id = q; break; }
                if (id < 0) {
                    id = nk++;
                    keys[id] = key;
                    for (int c = 0; c < 3; c++) { /* p = (A + (B-A) i/L) + (C-A) j/L  (pinned order) */
                        double t1 = (V[vb][c] - V[va][c]) * ((double)i / L);
                        double t2 = (V[vc][c] - V[va][c]) * ((double)j / L);
                        P[3 * id + c] = (V[va][c] + t1) + t2;
                    }
                    unit3(&P[3 * id], &A->nhat[3 * id]);
                }
                IDX(f, i, j) = id;
            }
        for (int i = 0; i < L; i++)
            for (int j = 0; j < L - i; j++) {
                tri[3 * nt + 0] = IDX(f, i, j); tri[3 * nt + 1] = IDX(f, i + 1, j); tri[3 * nt + 2] = IDX(f, i, j + 1); nt++;
                if (i + j < L - 1) {
                    tri[3 * nt + 0] = IDX(f, i + 1, j); tri[3 * nt + 1] = IDX(f, i + 1, j + 1); tri[3 * nt + 2] = IDX(f, i, j + 1); nt++;
                }
            }
    }
#undef IDX
    if (nk != N || nt != NT) { fprintf(stderr, "orc_angles_geodesic: count mismatch %d %d\n", nk, nt); abort(); }
    /* cell corners: planar centroid of each small triangle, radially projected */
    double *corner = malloc(sizeof(double) * 3 * NT);
    for (int t = 0; t < NT; t++) {
        double c[3];
        for (int d = 0; d < 3; d++) c[d] = ((P[3 * tri[3 * t] + d] + P[3 * tri[3 * t + 1] + d]) + P[3 * tri[3 * t + 2] + d]) / 3.0;
        unit3(c, &corner[3 * t]);
    }
    /* neighbours of n = lattice points sharing a small triangle with n, ordered counter-clockwise
     * seen from outside, starting at the smallest-index neighbour */
    for (int n = 0; n < N; n++) {
        int nb[8], nnb = 0;
        for (int t = 0; t < NT; t++)
            for (int s = 0; s < 3; s++)
                if (tri[3 * t + s] == n)
                    for (int s2 = 0; s2 < 3; s2++) {
                        int m = tri[3 * t + s2], seen = (m == n);
                        for (int q = 0; q < nnb; q++) seen |= (nb[q] == m);
                        if (!seen) nb[nnb++] = m;
                    }
        const double *nh = &A->nhat[3 * n];
        double ax[3] = {0, 0, 0}, e1[3], e2[3], phi[8];
        int amin = 0;
        for (int c = 1; c < 3; c++) if (fabs(nh[c]) < fabs(nh[amin])) amin = c;
        ax[amin] = 1.0;
        double d = dot3(ax, nh), t1[3] = {ax[0] - d * nh[0], ax[1] - d * nh[1], ax[2] - d * nh[2]};
        unit3(t1, e1); cross3(nh, e1, e2);
        for (int q = 0; q < nnb; q++) phi[q] = atan2(dot3(&A->nhat[3 * nb[q]], e2), dot3(&A->nhat[3 * nb[q]], e1));
        for (int q = 0; q < nnb; q++) /* insertion sort by angle */
            for (int r = q; r > 0 && phi[r] < phi[r - 1]; r--) {
                double tp = phi[r]; phi[r] = phi[r - 1]; phi[r - 1] = tp;
                int ti = nb[r]; nb[r] = nb[r - 1]; nb[r - 1] = ti;
            }
        int start = 0;
        for (int q = 1; q < nnb; q++) if (nb[q] < nb[start]) start = q;
        A->nnbr[n] = nnb;
        for (int q = 0; q < nnb; q++) A->nbr[n * ORC_MAXNBR + q] = nb[(start + q) % nnb];
    }
    /* corner k of cell n = the triangle (n, nbr_k, nbr_{k+1}); solid angle = fan of spherical triangles */
    int *cornid = malloc(sizeof(int) * N * ORC_MAXNBR);
    for (int n = 0; n < N; n++) {
        int nn = A->nnbr[n];
        for (int k = 0; k < nn; k++) {
            int m0 = A->nbr[n * ORC_MAXNBR + k], m1 = A->nbr[n * ORC_MAXNBR + (k + 1) % nn], found = -1;
            for (int t = 0; t < NT && found < 0; t++) {
                int has = 0;
                for (int s = 0; s < 3; s++) has += (tri[3 * t + s] == n) + 2 * (tri[3 * t + s] == m0) + 4 * (tri[3 * t + s] == m1);
                if (has == 7) found = t;
            }
            if (found < 0) { fprintf(stderr, "orc_angles_geodesic: corner not found\n"); abort(); }
            cornid[n * ORC_MAXNBR + k] = found;
        }
        double om = 0.0;
        for (int k = 0; k < nn; k++)
            om += sph_tri_area(&A->nhat[3 * n], &corner[3 * cornid[n * ORC_MAXNBR + k]], &corner[3 * cornid[n * ORC_MAXNBR + (k + 1) % nn]]);
        A->domega[n] = om;
    }
    /* unique edges: between n and its neighbour in slot k lie corners k-1 and k */
    for (int n = 0; n < N; n++) {
        int nn = A->nnbr[n];
        for (int k = 0; k < nn; k++) {
            int m = A->nbr[n * ORC_MAXNBR + k];
            if (m < n) continue;
            const double *c1 = &corner[3 * cornid[n * ORC_MAXNBR + (k + nn - 1) % nn]], *c2 = &corner[3 * cornid[n * ORC_MAXNBR + k]];
            double cx[3], sum[3] = {c1[0] + c2[0], c1[1] + c2[1], c1[2] + c2[2]}, mid[3], nrm[3], dn[3];
            cross3(c1, c2, cx);
            double len = atan2(sqrt(dot3(cx, cx)), dot3(c1, c2));
            unit3(sum, mid); unit3(cx, nrm);
            for (int c = 0; c < 3; c++) dn[c] = A->nhat[3 * m + c] - A->nhat[3 * n + c];
            if (dot3(nrm, dn) < 0) { nrm[0] = -nrm[0]; nrm[1] = -nrm[1]; nrm[2] = -nrm[2]; }
            int sm = -1;
            for (int q = 0; q < A->nnbr[m]; q++) if (A->nbr[m * ORC_MAXNBR + q] == n) sm = q;
            ang_add_edge(A, n, k, m, sm, len, mid, nrm);
        }
    }
    free(keys); free(P); free(idx); free(tri); free(corner); free(cornid);
    return A;
}

/* ======================================================================================
 * O2. Geometry: metric, 3+1 split, tetrad, Ricci rotation coefficients
 *     Derivatives by forward-mode dual numbers (value + d/dx, d/dy, d/dz); d/dt = 0 (Eq.4, 12).
 * ==================================================================================== */
typedef struct { double v, d[3]; } dual;
static dual dc(double c) { dual r = {c, {0, 0, 0}}; return r; }
static dual dadd(dual a, dual b) { dual r = {a.v + b.v, {a.d[0] + b.d[0], a.d[1] + b.d[1], a.d[2] + b.d[2]}}; return r; }
static dual dsub(dual a, dual b) { dual r = {a.v - b.v, {a.d[0] - b.d[0], a.d[1] - b.d[1], a.d[2] - b.d[2]}}; return r; }
static dual dmul(dual a, dual b) {
    dual r = {a.v * b.v, {a.d[0] * b.v + a.v * b.d[0], a.d[1] * b.v + a.v * b.d[1], a.d[2] * b.v + a.v * b.d[2]}};
    return r;
}
static dual ddiv(dual a, dual b) {
    double q = a.v / b.v;
    dual r = {q, {(a.d[0] - q * b.d[0]) / b.v, (a.d[1] - q * b.d[1]) / b.v, (a.d[2] - q * b.d[2]) / b.v}};
    return r;
}
static dual dsqrt(dual a) {
    double s = sqrt(a.v);
    dual r = {s, {0.5 * a.d[0] / s, 0.5 * a.d[1] / s, 0.5 * a.d[2] / s}};
    return r;
}
static dual dneg(dual a) { dual r = {-a.v, {-a.d[0], -a.d[1], -a.d[2]}}; return r; }

/* covariant metric g_{mu nu}(x).  kind 0: Minkowski eta.  kind 1: Cartesian Kerr-Schild
 * (named at P:L1002; textbook closed form g = eta + f l l). */
static void metric_dual(int kind, double M, double a, const dual X[3], dual g[4][4]) {
    for (int m = 0; m < 4; m++) for (int n = 0; n < 4; n++) g[m][n] = dc(m == n ? (m == 0 ? -1.0 : 1.0) : 0.0);
    if (kind == 0) return;
    dual x = X[0], y = X[1], z = X[2];
    dual R2 = dadd(dadd(dmul(x, x), dmul(y, y)), dmul(z, z));
    dual A2 = dc(a * a);
    dual w = dsub(R2, A2);
    dual r2 = dmul(dc(0.5), dadd(w, dsqrt(dadd(dmul(w, w), dmul(dc(4.0 * a * a), dmul(z, z))))));
    dual r = dsqrt(r2);
    dual f = ddiv(dmul(dc(2.0 * M), dmul(r2, r)), dadd(dmul(r2, r2), dmul(A2, dmul(z, z))));
    dual l[4];
    l[0] = dc(1.0);
    l[1] = ddiv(dadd(dmul(r, x), dmul(dc(a), y)), dadd(r2, A2));
    l[2] = ddiv(dsub(dmul(r, y), dmul(dc(a), x)), dadd(r2, A2));
    l[3] = ddiv(z, r);
    for (int m = 0; m < 4; m++) for (int n = 0; n < 4; n++) g[m][n] = dadd(g[m][n], dmul(f, dmul(l[m], l[n])));
}

/* 4x4 inverse by Gauss-Jordan with partial pivoting, in dual arithmetic */
static void inverse4_dual(dual A[4][4], dual Ai[4][4]) {
    dual W[4][8];
    for (int i = 0; i < 4; i++) for (int j = 0; j < 4; j++) { W[i][j] = A[i][j]; W[i][4 + j] = dc(i == j ? 1.0 : 0.0); }
    for (int c = 0; c < 4; c++) {
        int p = c;
        for (int r = c + 1; r < 4; r++) if (fabs(W[r][c].v) > fabs(W[p][c].v)) p = r;
        if (p != c) for (int j = 0; j < 8; j++) { dual t = W[c][j]; W[c][j] = W[p][j]; W[p][j] = t; }
        dual piv = W[c][c];
        for (int j = 0; j < 8; j++) W[c][j] = ddiv(W[c][j], piv);
        for (int r = 0; r < 4; r++) {
            if (r == c) continue;
            dual fct = W[r][c];
            for (int j = 0; j < 8; j++) W[r][j] = dsub(W[r][j], dmul(fct, W[c][j]));
        }
    }
    for (int i = 0; i < 4; i++) for (int j = 0; j < 4; j++) Ai[i][j] = W[i][4 + j];
}

/* out[ORC_NPOINT]: alpha, beta^i[3], g[4][4], ginv[4][4], e[mu][ahat], elow[ahat][mu], omega[c][a][b] */
void orc_geometry_point(int kind, double M, double a, const double xx[3], double *out) {
    dual X[3];
    for (int i = 0; i < 3; i++) { X[i] = dc(xx[i]); X[i].d[i] = 1.0; }
    dual g[4][4], gi[4][4];
    metric_dual(kind, M, a, X, g);
    inverse4_dual(g, gi);
    /* Eq.5a,c: alpha = (-g^00)^(-1/2), beta^a = alpha^2 g^0a */
    dual alpha = ddiv(dc(1.0), dsqrt(dneg(gi[0][0])));
    dual beta[3];
    for (int i = 0; i < 3; i++) beta[i] = dmul(dmul(alpha, alpha), gi[0][i + 1]);
    /* tetrad e^mu_ahat, stored e[mu][ahat].  Eq.11: e^mu_0hat = -alpha g^{0 mu}. */
    dual e[4][4];
    for (int m = 0; m < 4; m++) e[m][0] = dneg(dmul(alpha, gi[0][m]));
    /* R2: spatial triad = Gram-Schmidt of d_x, d_y, d_z (in that order) w.r.t. gamma_ab = g_ab
     * (Eq.5d).  d_i are tangent to the slice, hence already orthogonal to e_0hat. */
    for (int ah = 1; ah <= 3; ah++) {
        dual v[4] = {dc(0), dc(0), dc(0), dc(0)};
        v[ah] = dc(1.0);
        for (int bh = 1; bh < ah; bh++) {
            dual pr = dc(0); /* gamma(d_ah, e_bh) */
            for (int i = 1; i < 4; i++) pr = dadd(pr, dmul(g[ah][i], e[i][bh]));
            for (int i = 0; i < 4; i++) v[i] = dsub(v[i], dmul(pr, e[i][bh]));
        }
        dual nrm2 = dc(0);
        for (int i = 1; i < 4; i++) for (int j = 1; j < 4; j++) nrm2 = dadd(nrm2, dmul(g[i][j], dmul(v[i], v[j])));
        dual nrm = dsqrt(nrm2);
        for (int i = 0; i < 4; i++) e[i][ah] = ddiv(v[i], nrm);
    }
    /* Eq.9: e^ahat_mu = eta^{ahat chat} g_{mu delta} e^delta_chat, stored elow[ahat][mu] */
    double elow[4][4];
    for (int ah = 0; ah < 4; ah++)
        for (int m = 0; m < 4; m++) {
            double s = 0;
            for (int dl = 0; dl < 4; dl++) s += g[m][dl].v * e[dl][ah].v;
            elow[ah][m] = (ah == 0 ? -1.0 : 1.0) * s;
        }
    /* Christoffel symbols Gamma^eps_{delta sigma} = 1/2 g^{eps lam}(d_delta g_{lam sigma} + d_sigma g_{lam delta} - d_lam g_{delta sigma}) */
    double dg[4][4][4]; /* dg[mu][nu][delta] = d_delta g_{mu nu}; d_0 = 0 (Eq.4) */
    for (int m = 0; m < 4; m++) for (int n = 0; n < 4; n++) { dg[m][n][0] = 0.0; for (int i = 0; i < 3; i++) dg[m][n][i + 1] = g[m][n].d[i]; }
    double Gam[4][4][4];
    for (int ep = 0; ep < 4; ep++) for (int dl = 0; dl < 4; dl++) for (int sg = 0; sg < 4; sg++) {
        double s = 0;
        for (int lm = 0; lm < 4; lm++) s += gi[ep][lm].v * (dg[lm][sg][dl] + dg[lm][dl][sg] - dg[dl][sg][lm]);
        Gam[ep][dl][sg] = 0.5 * s;
    }
    /* Eq.17: omega^chat_{ahat bhat} = e^chat_eps e^delta_bhat (d_delta e^eps_ahat + Gamma^eps_{delta sigma} e^sigma_ahat) */
    double *om = out + 68;
    for (int ch = 0; ch < 4; ch++) for (int ah = 0; ah < 4; ah++) for (int bh = 0; bh < 4; bh++) {
        double s = 0;
        for (int ep = 0; ep < 4; ep++) for (int dl = 0; dl < 4; dl++) {
            double cov = (dl == 0) ? 0.0 : e[ep][ah].d[dl - 1]; /* d_0 e = 0 (Eq.12) */
            for (int sg = 0; sg < 4; sg++) cov += Gam[ep][dl][sg] * e[sg][ah].v;
            s += elow[ch][ep] * e[dl][bh].v * cov;
        }
        om[(ch * 4 + ah) * 4 + bh] = s;
    }
    out[0] = alpha.v;
    for (int i = 0; i < 3; i++) out[1 + i] = beta[i].v;
    for (int m = 0; m < 4; m++) for (int n = 0; n < 4; n++) {
        out[4 + 4 * m + n] = g[m][n].v;
        out[20 + 4 * m + n] = gi[m][n].v;
        out[36 + 4 * m + n] = e[m][n].v;
        out[52 + 4 * m + n] = elow[m][n];
    }
}

/* ======================================================================================
 * Problem: uniform Cartesian grid + metric + angle grid + parameters
 * ==================================================================================== */
struct orc_problem {
    int kind; double M, a, excise_r;
    int n[3], ng, NI, NJ, NK;
    double x0[3], dx[3];
    double *xf[3];   /* R22: face coordinates of a stretched grid, [n + 2 ng + 1] per axis, or NULL (uniform: x0 + (i - ng) dx) */
    int bc_lo[3], bc_hi[3];
    const orc_angles *ang;
    double gamma_gas, a_rad, n0_crit;
    int recon_space, renorm, couple;
    double tau_factor; /* constant of Eq.26; 0 = free-streaming flux Eq.24 */
    int recon_angle;   /* 0 donor cell, 1 PLM on the latitude-longitude grid incl. across the poles */
    int vel_estimate;  /* 1: radiation-dominated velocity estimate Eq.51-55 */
    int dt0_literal;   /* 0: dT^0_alpha = -sum n^0 n_alpha (I_+ - I*) dOmega; 1: -(R^0_alpha[I_+] - R^0_alpha[I*]) formed from two sums */
    int *mirror;       /* [3][N] angle whose direction is n with component a flipped (reflecting boundary, bc code 3), or -1 */
    long long ncell;
    double *cell; /* [ncell][ORC_NCELL] */
    double *face; /* [ncell][3][ORC_NFACE]: lower face of each cell along each axis */
    int *excised; /* [ncell] */
};

static long long cidx(const orc_problem *P, int k, int j, int i) { return ((long long)k * P->NJ + j) * P->NI + i; }

/* pack what the stage needs at a point: (cell) alpha, e[mu][ahat], L[mu][ahat] = g_{mu nu} e^nu_ahat,
 * S[c][k] = omega^c_{alpha beta} + omega^c_{beta alpha} (alpha<beta) or omega^c_{alpha alpha},
 * k over (00,01,02,03,11,12,13,22,23,33), c = 1..3 */
static void pack_cell(const double *pt, double *c) {
    c[0] = pt[0];
    const double *g = pt + 4, *e = pt + 36, *om = pt + 68;
    for (int m = 0; m < 4; m++) for (int ah = 0; ah < 4; ah++) {
        c[1 + 4 * m + ah] = e[4 * m + ah];
        double s = 0;
        for (int nu = 0; nu < 4; nu++) s += g[4 * m + nu] * e[4 * nu + ah];
        c[17 + 4 * m + ah] = s;
    }
    for (int ch = 1; ch < 4; ch++) {
        int k = 0;
        for (int al = 0; al < 4; al++) for (int be = al; be < 4; be++) {
            double w = om[(ch * 4 + al) * 4 + be];
            if (be != al) w += om[(ch * 4 + be) * 4 + al];
            c[33 + 10 * (ch - 1) + k++] = w;
        }
    }
    for (int p = 0; p < 3; p++) c[63 + p] = pt[1 + p]; /* beta^a (Eq.5c) */
    int q = 0;
    for (int p = 0; p < 3; p++) for (int r = p; r < 3; r++) c[66 + q++] = g[4 * (p + 1) + (r + 1)]; /* gamma_ab = g_ab (Eq.5d): xx,xy,xz,yy,yz,zz */
}
static void pack_face(const double *pt, int axis, double *f) {
    const double *g = pt + 4, *e = pt + 36;
    for (int ah = 0; ah < 4; ah++) {
        f[ah] = e[4 * (axis + 1) + ah];
        double s = 0;
        for (int nu = 0; nu < 4; nu++) s += g[nu] * e[4 * nu + ah]; /* g_{0 nu} e^nu_ahat */
        f[4 + ah] = s;
    }
}

/* coordinate of the lower face of cell `i` along axis d, and the cell's centre and width (Eq.20b,c with sqrt(-g) = 1 on a Cartesian
 * tensor-product grid: Delta A_a / Delta V = 1 / Delta x^a of the cell) */
static double face_coord(const orc_problem *P, int d, int i) { return P->xf[d] ? P->xf[d][i] : P->x0[d] + (i - P->ng) * P->dx[d]; }
static double centre_coord(const orc_problem *P, int d, int i) {
    return P->xf[d] ? 0.5 * (P->xf[d][i] + P->xf[d][i + 1]) : P->x0[d] + (i - P->ng + 0.5) * P->dx[d];
}
static double cell_width(const orc_problem *P, int d, int i) { return P->xf[d] ? P->xf[d][i + 1] - P->xf[d][i] : P->dx[d]; }

/* xf0, xf1, xf2: face coordinates of a stretched Cartesian grid along x, y, z (NEXT-4, Eq.20b,c; reading R22), each with
 * n + 2 ng + 1 entries (ghost cells included), or NULL for the uniform spacing dx from x0 */
orc_problem *orc_create_stretched(int kind, double M, double a, double excise_r, const int n[3], int ng, const double x0[3],
                                  const double dx[3], const int bc_lo[3], const int bc_hi[3], const orc_angles *ang,
                                  double gamma_gas, double a_rad, double n0_crit, int recon_space, int renorm, int couple,
                                  const double *xf0, const double *xf1, const double *xf2) {
    orc_problem *P = calloc(1, sizeof(*P));
    {
        const double *src[3] = {xf0, xf1, xf2};
        for (int d = 0; d < 3; d++) {
            P->xf[d] = NULL;
            if (src[d]) {
                P->xf[d] = malloc(sizeof(double) * (n[d] + 2 * ng + 1));
                memcpy(P->xf[d], src[d], sizeof(double) * (n[d] + 2 * ng + 1));
            }
        }
    }
    P->kind = kind; P->M = M; P->a = a; P->excise_r = excise_r; P->ng = ng; P->ang = ang;
    for (int d = 0; d < 3; d++) { P->n[d] = n[d]; P->x0[d] = x0[d]; P->dx[d] = dx[d]; P->bc_lo[d] = bc_lo[d]; P->bc_hi[d] = bc_hi[d]; }
    P->NI = n[0] + 2 * ng; P->NJ = n[1] + 2 * ng; P->NK = n[2] + 2 * ng;
    P->gamma_gas = gamma_gas; P->a_rad = a_rad; P->n0_crit = n0_crit;
    P->recon_space = recon_space; P->renorm = renorm; P->couple = couple;
    P->ncell = (long long)P->NI * P->NJ * P->NK;
    P->cell = malloc(sizeof(double) * P->ncell * ORC_NCELL);
    P->face = malloc(sizeof(double) * P->ncell * 3 * ORC_NFACE);
    P->excised = calloc(P->ncell, sizeof(int));
    /* R20 (reflecting wall): the image of direction n under a reflection that flips tetrad component a is the grid
     * angle whose direction vector equals n-hat with that component negated; -1 where the grid has no such angle */
    P->mirror = malloc(sizeof(int) * 3 * ang->N);
    for (int ax = 0; ax < 3; ax++)
        for (int n = 0; n < ang->N; n++) {
            double want[3] = {ang->nhat[3 * n], ang->nhat[3 * n + 1], ang->nhat[3 * n + 2]};
            want[ax] = -want[ax];
            int found = -1;
            for (int m = 0; m < ang->N && found < 0; m++) {
                double d0 = ang->nhat[3 * m] - want[0], d1 = ang->nhat[3 * m + 1] - want[1], d2 = ang->nhat[3 * m + 2] - want[2];
                if (fabs(d0) < 1e-12 && fabs(d1) < 1e-12 && fabs(d2) < 1e-12) found = m;
            }
            P->mirror[ax * ang->N + n] = found;
        }
#pragma omp parallel for schedule(static)
    for (int k = 0; k < P->NK; k++)
        for (int j = 0; j < P->NJ; j++)
            for (int i = 0; i < P->NI; i++) {
                long long c = cidx(P, k, j, i);
                int id[3] = {i, j, k};
                double xc[3], pt[ORC_NPOINT];
                for (int d = 0; d < 3; d++) xc[d] = centre_coord(P, d, id[d]);
                orc_geometry_point(kind, M, a, xc, pt);
                pack_cell(pt, &P->cell[c * ORC_NCELL]);
                if (kind == 1 && excise_r > 0) { /* Kerr-Schild radius of the cell centre */
                    double R2 = xc[0] * xc[0] + xc[1] * xc[1] + xc[2] * xc[2], w = R2 - a * a;
                    double r = sqrt(0.5 * (w + sqrt(w * w + 4 * a * a * xc[2] * xc[2])));
                    P->excised[c] = (r < excise_r);
                }
                for (int ax = 0; ax < 3; ax++) { /* R6: face quantities at the face centre */
                    double xf[3] = {xc[0], xc[1], xc[2]};
                    xf[ax] = face_coord(P, ax, id[ax]);
                    orc_geometry_point(kind, M, a, xf, pt);
                    pack_face(pt, ax, &P->face[(c * 3 + ax) * ORC_NFACE]);
                }
            }
    return P;
}
orc_problem *orc_create(int kind, double M, double a, double excise_r, const int n[3], int ng, const double x0[3],
                        const double dx[3], const int bc_lo[3], const int bc_hi[3], const orc_angles *ang,
                        double gamma_gas, double a_rad, double n0_crit, int recon_space, int renorm, int couple) {
    return orc_create_stretched(kind, M, a, excise_r, n, ng, x0, dx, bc_lo, bc_hi, ang, gamma_gas, a_rad, n0_crit, recon_space, renorm, couple,
                                NULL, NULL, NULL);
}
void orc_destroy(orc_problem *P) {
    if (!P) return;
    free(P->cell); free(P->face); free(P->excised); free(P->mirror);
    for (int d = 0; d < 3; d++) free(P->xf[d]);
    free(P);
}
long long orc_ncells_total(const orc_problem *P) { return P->ncell; }
void orc_get_geometry(const orc_problem *P, double *cell, double *face, int *excised) {
    if (cell) memcpy(cell, P->cell, sizeof(double) * P->ncell * ORC_NCELL);
    if (face) memcpy(face, P->face, sizeof(double) * P->ncell * 3 * ORC_NFACE);
    if (excised) memcpy(excised, P->excised, sizeof(int) * P->ncell);
}

/* ======================================================================================
 * a7. Ghost fill: 0 caller-filled (no-op), 1 periodic, 2 outflow (copy of the
 * nearest interior cell).  Axis by axis x, y, z; later axes see earlier axes' ghosts, so
 * edges and corners are filled too.
 * ==================================================================================== */
void orc_fill_ghosts(const orc_problem *P, double *I) {
    int N = P->ang->N, ng = P->ng, dims[3] = {P->NI, P->NJ, P->NK};
    for (int ax = 0; ax < 3; ax++)
        for (int k = 0; k < P->NK; k++) for (int j = 0; j < P->NJ; j++) for (int i = 0; i < P->NI; i++) {
            int id[3] = {i, j, k}, src[3] = {i, j, k}, q = id[ax], nint = P->n[ax], bc;
            int wrap = ng + (((q - ng) % nint) + nint) % nint; /* periodic image inside the interior (also for nint < ng) */
            if (q < ng) {
                bc = P->bc_lo[ax];
                if (bc == 1) src[ax] = wrap; else if (bc == 2) src[ax] = ng; else if (bc == 3) src[ax] = 2 * ng - 1 - q; else continue;
            } else if (q >= dims[ax] - ng) {
                bc = P->bc_hi[ax];
                if (bc == 1) src[ax] = wrap; else if (bc == 2) src[ax] = ng + nint - 1; else if (bc == 3) src[ax] = 2 * (dims[ax] - ng) - 1 - q; else continue;
            } else continue;
            double *dst = &I[cidx(P, k, j, i) * N];
            const double *sp = &I[cidx(P, src[2], src[1], src[0]) * N];
            if (bc == 3) { /* R20: mirror cell across the wall, direction with the normal component flipped */
                for (int n = 0; n < N; n++) { int m = P->mirror[ax * N + n]; dst[n] = (m >= 0) ? sp[m] : 0.0; }
            } else memcpy(dst, sp, sizeof(double) * N);
        }
}
/* 1 if every angle has its mirror image under the flip of component ax on this angle grid */
int orc_has_mirror(const orc_problem *P, int ax) {
    for (int n = 0; n < P->ang->N; n++) if (P->mirror[ax * P->ang->N + n] < 0) return 0;
    return 1;
}

/* ======================================================================================
 * O3. Transport
 * ==================================================================================== */
/* pinned: n^a = fma(e^a_3,n^3, fma(e^a_2,n^2, fma(e^a_1,n^1, e^a_0)))  (n^0hat = 1, Eq.15a) */
static double contract4(const double *row, const double *nh) {
    return fma(row[3], nh[2], fma(row[2], nh[1], fma(row[1], nh[0], row[0])));
}
/* R7: van Leer (1974) harmonic-mean limited slope on uniform spacing */
static double vl_slope(double qm, double q0, double qp) {
    double dl = q0 - qm, dr = qp - q0, pr = dl * dr;
    return (pr > 0.0) ? 2.0 * pr / (dl + dr) : 0.0;
}
/* PPM (Colella & Woodward 1984, cited P:L276) on uniform spacing, as used for cell-centred variables without characteristic
 * tracing: the monotonised parabola of cell 0 from the five values q[-2..2]; returns its values at the lower (qm) and upper (qp)
 * face.  CW84 Eq.1.6-1.8: interface value q_{1/2} = q_0 + (q_1 - q_0)/2 - (dq_1 - dq_0)/6 with van Leer-limited average slopes
 * dq = min(|q_{+1} - q_{-1}|/2, 2|q_{+1} - q_0|, 2|q_0 - q_{-1}|) sgn(q_{+1} - q_{-1}) at non-extrema, 0 at extrema;
 * CW84 Eq.1.10: flatten at extrema, pull the far face in where the parabola overshoots. */
static double ppm_dq(double qm, double q0, double qp) {
    double dl = q0 - qm, dr = qp - q0;
    if (dl * dr <= 0.0) return 0.0;
    double d = 0.5 * (qp - qm), lim = fmin(2.0 * fabs(dl), 2.0 * fabs(dr));
    return (d > 0.0 ? 1.0 : -1.0) * fmin(fabs(d), lim);
}
static void ppm_states(const double q[5], double *qm_out, double *qp_out) {
    double dqm = ppm_dq(q[0], q[1], q[2]), dq0 = ppm_dq(q[1], q[2], q[3]), dqp = ppm_dq(q[2], q[3], q[4]);
    double qm = q[1] + 0.5 * (q[2] - q[1]) - (dq0 - dqm) / 6.0; /* value at the lower face */
    double qp = q[2] + 0.5 * (q[3] - q[2]) - (dqp - dq0) / 6.0; /* value at the upper face */
    double q0 = q[2];
    if ((qp - q0) * (q0 - qm) <= 0.0) { qm = q0; qp = q0; }
    else {
        double dq = qp - qm, q6 = 6.0 * (q0 - 0.5 * (qm + qp));
        if (dq * q6 > dq * dq) qm = 3.0 * q0 - 2.0 * qp;
        else if (-dq * dq > dq * q6) qp = 3.0 * q0 - 2.0 * qm;
    }
    *qm_out = qm; *qp_out = qp;
}

/* Eq.24: flux of n^a n_0 I through the LOWER face of cell id[] along axis ax, angle n.
 * With vel != NULL (tau_factor != 0): the optical-depth-aware flux of Eq.26-29.  vel[cell][5] holds the
 * tetrad-frame fluid velocity u^alphahat (4) of each cell (its own cell-centre tetrad, R10) and alpha_E = alpha^a_E + alpha^s.
 * Readings: R15 "interpolated to the interface" = arithmetic mean of the two adjacent cells; R16 the undefined
 * v^0hat of Eq.26 = mean of the two cells' u^0hat; R17 g = (g_L + g_R)/2; R18 Delta t = beta dt of the stage, tau =
 * tau_factor * alpha_E dt / v^0hat; G1 f = -expm1(-tau^2) (the sentence after Eq.27 defines expm1; Eq.27 as printed lacks it). */
static double face_flux(const orc_problem *P, const double *I, int ax, int i, int j, int k, int n, const double *vel, double tau_dt) {
    int N = P->ang->N, st[3] = {0, 0, 0};
    st[ax] = 1;
    long long cR = cidx(P, k, j, i), cL = cidx(P, k - st[2], j - st[1], i - st[0]);
    long long cLL = cidx(P, k - 2 * st[2], j - 2 * st[1], i - 2 * st[0]), cRR = cidx(P, k + st[2], j + st[1], i + st[0]);
    const double *f = &P->face[(cR * 3 + ax) * ORC_NFACE], *nh = &P->ang->nhat[3 * n];
    double na = contract4(f, nh), n0 = contract4(f + 4, nh);
    double qL = I[cL * N + n], qR = I[cR * N + n], Iup;
    if (na > 0.0) {
        Iup = qL;
        if (P->recon_space == 1) Iup = qL + 0.5 * vl_slope(I[cLL * N + n], qL, qR);
        else if (P->recon_space == 2) { /* upper-face value of the parabola of cell L */
            long long c3 = cidx(P, k - 3 * st[2], j - 3 * st[1], i - 3 * st[0]);
            double q[5] = {I[c3 * N + n], I[cLL * N + n], qL, qR, I[cRR * N + n]}, qm;
            ppm_states(q, &qm, &Iup);
        }
    } else if (na < 0.0) {
        Iup = qR;
        if (P->recon_space == 1) Iup = qR - 0.5 * vl_slope(qL, qR, I[cRR * N + n]);
        else if (P->recon_space == 2) { /* lower-face value of the parabola of cell R */
            long long c3 = cidx(P, k + 2 * st[2], j + 2 * st[1], i + 2 * st[0]);
            double q[5] = {I[cLL * N + n], qL, qR, I[cRR * N + n], I[c3 * N + n]}, qp;
            ppm_states(q, &Iup, &qp);
        }
    } else return 0.0;
    if (vel) {
        const double *vL = &vel[cL * 5], *vR = &vel[cR * 5];
        double aE = 0.5 * (vL[4] + vR[4]), v0 = 0.5 * (vL[0] + vR[0]);               /* R15, R16 */
        double tau = tau_dt * aE / v0;                                                /* Eq.26 */
        double fint = -expm1(-tau * tau);                                             /* Eq.27 with G1 */
        double nbL = vL[0] - (vL[1] * nh[0] + vL[2] * nh[1] + vL[3] * nh[2]);         /* n^0bar_L = -(u_alpha n^alpha)_L */
        double nbR = vR[0] - (vR[1] * nh[0] + vR[2] * nh[1] + vR[3] * nh[2]);
        double gL = -fint * (1.0 + 1.0 / nbL), gR = -fint * (1.0 + 1.0 / nbR);        /* Eq.29 */
        double g = 0.5 * (gL + gR);                                                   /* R17 */
        Iup *= (na > 0.0) ? (1.0 - gL + g) : (1.0 - gR + g);                          /* Eq.28 */
    }
    return na * n0 * Iup;
}
/* R21: PLM in angle on the latitude-longitude grid.  "Reconstruction on latitude/longitude grids uses the same
 * algorithms as spatial reconstruction": the van Leer slope of R7 in index space along zeta and along psi.  The neighbours of
 * cell (l, m) along zeta are (l -+ 1, m); beyond a pole the row continues on the far side of the sphere, in cell
 * (l, m + N_psi/2) of the same row l (the paper's example: (0,4), (0,0), (1,0), (2,0) for N_psi = 8); along psi the grid is
 * periodic.  I is a scalar: no sign change across the poles.  Returns the value of cell u at its face in slot `slot`
 * (0 zeta-, 1 zeta+, 2 psi-, 3 psi+). */
static double latlon_face_value(const orc_angles *A, const double *Ic, int u, int slot) {
    int np = A->npsi, l = u / np, m = u % np, lo, hi;
    if (slot < 2) {
        int across = l * np + (m + np / 2) % np;
        lo = (l > 0) ? (l - 1) * np + m : across;
        hi = (l + 1 < A->nzeta) ? (l + 1) * np + m : across;
    } else {
        lo = l * np + (m + np - 1) % np;
        hi = l * np + (m + 1) % np;
    }
    double s = vl_slope(Ic[lo], Ic[u], Ic[hi]);
    return (slot & 1) ? Ic[u] + 0.5 * s : Ic[u] - 0.5 * s;
}
/* for the pins: value of cell u at its face in `slot`, from the row Ic[N] of one spatial cell */
double orc_latlon_face_value(const orc_angles *A, const double *Ic, int u, int slot) { return latlon_face_value(A, Ic, u, slot); }

/* pinned: c_e = -sum_{c=1..3} sum_{k=0..9} S[c][k] T_e[c][k], accumulated by fma from 0 in that order.
 * = a(n_e) . N_e with a^c = -omega^c_{alpha beta} n^alpha n^beta  (R5; Eq.16b,c) */
static double edge_coeff(const double *S, const double *T) {
    double acc = 0.0;
    for (int q = 0; q < 30; q++) acc = fma(S[q], T[q], acc);
    return -acc;
}

static void transport_impl(const orc_problem *P, const double *I_in, const double *I0, double gam0, double gam1,
                           double beta_dt, const double *vel, double tau_dt, double *I_out) {
    const orc_angles *A = P->ang;
    int N = A->N, E = A->E, ng = P->ng;
#pragma omp parallel
    {
        double *Fe = malloc(sizeof(double) * (E > 0 ? E : 1));
#pragma omp for schedule(static)
        for (int k = ng; k < P->NK - ng; k++)
            for (int j = ng; j < P->NJ - ng; j++)
                for (int i = ng; i < P->NI - ng; i++) {
                    long long c = cidx(P, k, j, i);
                    const double *cg = &P->cell[c * ORC_NCELL];
                    if (P->excised[c]) { for (int n = 0; n < N; n++) I_out[c * N + n] = 0.0; continue; }
                    /* Eq.25 angular fluxes, DC reconstruction, once per unique edge */
                    for (int e = 0; e < E; e++) {
                        double ce = edge_coeff(cg + 33, &A->edge_T[30 * e]);
                        double n0e = contract4(cg + 17, &A->edge_mid[3 * e]); /* n_0 at the edge direction, cell-centre tetrad */
                        int up = (ce > 0.0) ? A->edge_lo[e] : A->edge_hi[e];
                        double Iup = I_in[c * N + up];
                        if (P->recon_angle == 1 && ce != 0.0) { /* R21: the upwind cell's PLM value at this edge */
                            int slot = 0;
                            while (A->nbr_edge[up * ORC_MAXNBR + slot] != e) slot++;
                            Iup = latlon_face_value(A, &I_in[c * N], up, slot);
                        }
                        Fe[e] = (ce == 0.0) ? 0.0 : ce * n0e * Iup;
                    }
                    for (int n = 0; n < N; n++) {
                        const double *nh = &A->nhat[3 * n];
                        double nup0 = contract4(cg + 1, nh);  /* n^0 */
                        double nlo0 = contract4(cg + 17, nh); /* n_0 */
                        /* Eq.22: spatial flux divergence; uniform Cartesian grid with sqrt(-g)=1 => dA/dV = 1/dx */
                        double div = 0.0;
                        div += (face_flux(P, I_in, 0, i + 1, j, k, n, vel, tau_dt) - face_flux(P, I_in, 0, i, j, k, n, vel, tau_dt)) / cell_width(P, 0, i);
                        div += (face_flux(P, I_in, 1, i, j + 1, k, n, vel, tau_dt) - face_flux(P, I_in, 1, i, j, k, n, vel, tau_dt)) / cell_width(P, 1, j);
                        div += (face_flux(P, I_in, 2, i, j, k + 1, n, vel, tau_dt) - face_flux(P, I_in, 2, i, j, k, n, vel, tau_dt)) / cell_width(P, 2, k);
                        /* angular flux divergence: (1/dOmega) sum_e +-dlambda_e F_e, + where the edge normal points out of n */
                        double adiv = 0.0;
                        for (int s = 0; s < A->nnbr[n]; s++) {
                            int e = A->nbr_edge[n * ORC_MAXNBR + s];
                            if (e < 0) continue;
                            double sgn = (A->edge_lo[e] == n) ? 1.0 : -1.0;
                            adiv += sgn * A->edge_len[e] * Fe[e];
                        }
                        div += adiv / A->domega[n];
                        /* R8 stage form: C* = gam0 C0 + gam1 C - beta dt div, C = n^0 n_0 I; Eq.79 prim = C/(n^0 n_0) */
                        double w = nup0 * nlo0;
                        double C = gam1 * (w * I_in[c * N + n]);
                        if (I0) C += gam0 * (w * I0[c * N + n]);
                        I_out[c * N + n] = (C - beta_dt * div) / w;
                    }
                }
        free(Fe);
    }
}

void orc_transport(const orc_problem *P, const double *I_in, const double *I0, double gam0, double gam1,
                   double beta_dt, double *I_out) {
    transport_impl(P, I_in, I0, gam0, gam1, beta_dt, NULL, 0.0, I_out);
}

/* ======================================================================================
 * O4/O5. Locally implicit coupling (Eq.31-50), fluid increment, mask
 * ==================================================================================== */
/* R13: unique positive root of the quartic Eq.49, B4 T^4 + B1 T + B0 = 0, for B4 >= 0, B1 > 0, B0 < 0.
 * Eq.48 then needs T_+ - T_-, and in a gas-dominated cell (C_v T >> Ebar) forming that difference from a
 * rounded T_+ would lose log10(C_v T / Ebar) digits of Ebar_+.  So the SAME quartic is solved for the change
 * d = T_+ - T_-:   g(d) = B4 (T_- + d)^4 + B1 d + Bp = 0,  Bp = B0 + B1 T_- = A1 - (1 - A2 alpha_s) Ebar_-,
 * by Newton from the upper bound T_ub = min(-B0/B1, (-B0/B4)^(1/4)) (g is convex and increasing: monotone
 * convergence from the right).  Stop when the step is below 1e-15 of |d| plus the rounding scale of g/g'.
 * returns 0 and *d_out if a positive root exists, -1 otherwise (B0 >= 0 or non-finite coefficients). */
static int quartic_delta(double B4, double B1, double Bp, double Tm, double *d_out) {
    double B0 = Bp - B1 * Tm;
    if (!(B0 < 0.0) || !(B1 > 0.0) || !(B4 >= 0.0) || !isfinite(B0) || !isfinite(B1) || !isfinite(B4)) return -1;
    if (B4 == 0.0) { *d_out = -Bp / B1; return 0; }
    double d = fmin(-B0 / B1, sqrt(sqrt(-B0 / B4))) - Tm;
    for (int it = 0; it < 60; it++) {
        double T = Tm + d, T3 = T * T * T;
        double g = B4 * T3 * T + B1 * d + Bp, gp = 4.0 * B4 * T3 + B1;
        double dd = g / gp;
        d -= dd;
        if (fabs(dd) <= 1e-15 * (fabs(d) + (fabs(Bp) + B4 * T3 * T) / gp)) break;
    }
    *d_out = d;
    return 0;
}

/* R10: coordinate-frame u^mu from the normal-frame spatial velocity u^a': gamma = sqrt(1 +
 * gamma_ab u^a' u^b'), u^0 = gamma/alpha, u^a = u^a' - beta^a gamma/alpha (inverse of Eq.7) */
static void fluid_four_velocity(const double *cg, const double unorm[3], double ucon[4]) {
    double alpha = cg[0];
    const double *beta = cg + 63, *gm = cg + 66;
    double gam_ab[3][3] = {{gm[0], gm[1], gm[2]}, {gm[1], gm[3], gm[4]}, {gm[2], gm[4], gm[5]}};
    double u2 = 0;
    for (int p = 0; p < 3; p++) for (int q = 0; q < 3; q++) u2 += gam_ab[p][q] * unorm[p] * unorm[q];
    double gam = sqrt(1.0 + u2);
    ucon[0] = gam / alpha;
    for (int p = 0; p < 3; p++) ucon[p + 1] = unorm[p] - beta[p] * gam / alpha;
}

void orc_set_tau_factor(orc_problem *P, double tau_factor) { P->tau_factor = tau_factor; }
/* options: 0 recon_angle (0 DC, 1 lat-lon PLM; returns -1 if the angle grid is not lat-lon with even N_psi), 1 vel_estimate,
 * 2 dt0_literal */
int orc_set_option(orc_problem *P, int which, int value) {
    if (which == 0) {
        if (value == 1 && (P->ang->kind != 0 || (P->ang->npsi & 1))) return -1;
        P->recon_angle = value;
    } else if (which == 1) P->vel_estimate = value;
    else if (which == 2) P->dt0_literal = value;
    else return -1;
    return 0;
}

/* vel[cell][5] for EVERY cell of the array (ghosts included: the faces of the outermost interior cells need their
 * neighbours): tetrad-frame fluid velocity u^alphahat (R10, with the cell's own cell-centre tetrad; the same lines as in
 * orc_coupling) and alpha_E = alpha^a_E + alpha^s (Eq.33b) */
void orc_cell_velocity(const orc_problem *P, const double *fluid, const double *opac, double *vel) {
    long long nc = P->ncell;
#pragma omp parallel for schedule(static)
    for (long long c = 0; c < nc; c++) {
        const double *cg = &P->cell[c * ORC_NCELL], *Lw = cg + 17;
        double unorm[3] = {fluid[2 * nc + c], fluid[3 * nc + c], fluid[4 * nc + c]}, ucon[4];
        fluid_four_velocity(cg, unorm, ucon);
        for (int ah = 0; ah < 4; ah++) {
            double s = 0;
            for (int b = 0; b < 4; b++) s += Lw[4 * b + ah] * ucon[b];
            vel[c * 5 + ah] = (ah == 0 ? -1.0 : 1.0) * s;
        }
        vel[c * 5 + 4] = opac[1 * nc + c] + opac[2 * nc + c];
    }
}

/* transport with the optical-depth-aware spatial flux of Eq.26-29 when tau_factor != 0 (else Eq.24) */
void orc_transport_tau(const orc_problem *P, const double *I_in, const double *I0, double gam0, double gam1,
                       double beta_dt, const double *fluid, const double *opac, double *I_out) {
    if (P->tau_factor == 0.0 || !fluid || !opac) { transport_impl(P, I_in, I0, gam0, gam1, beta_dt, NULL, 0.0, I_out); return; }
    double *vel = malloc(sizeof(double) * 5 * P->ncell);
    orc_cell_velocity(P, fluid, opac, vel);
    transport_impl(P, I_in, I0, gam0, gam1, beta_dt, vel, P->tau_factor * beta_dt, I_out);
    free(vel);
}

/* NEXT-2: radiation-dominated velocity estimate (Eq.51-55).  Inputs: the tetrad-frame intensities of one cell
 * (after transport), the gas four-velocity uh[4] in the tetrad frame, rho, T, the absorptivities, dt.  If Ebar (fluid-frame
 * radiation energy density for the gas velocity, Eq.38 in covariant form u_a u_b R^{ab}) exceeds rho + u_gas, uh is
 * replaced by the blend of Eq.55 and 1 is returned; else uh is left alone and 0 is returned.
 * Readings: G8 -- Eq.54 as printed has u^ahat in the denominator; taken as f^a = G^a dt / (T_rad^{0a} - T_gas^{0a}),
 * the fraction of the momentum gap the force closes in dt (the printed form diverges for a gas at rest and lets the sign of
 * u^a decide the clamp); a vanishing denominator gives f^a = 0.  R19 -- |v_rad|^2 is capped at 1 - 1e-12 so that the
 * "associated four-velocity" exists for a single beam; u^0hat of the blend from normalisation.  T in Eq.53 is the
 * pre-coupling gas temperature.  Optional outputs for the pins: G[4] (Eq.53), fr[3] (Eq.54, clamped), Rt[10] (R^{ahat bhat}). */
static int velocity_estimate(const orc_problem *P, const double *Ic, double uh[4], double rho, double Tm, double aP, double aEa,
                             double aS, double dt, double *G_out, double *fr_out, double *R_out) {
    const orc_angles *A = P->ang;
    int N = A->N;
    double R[4][4] = {{0}};
    for (int n = 0; n < N; n++) {
        const double *nh = &A->nhat[3 * n];
        double n4[4] = {1.0, nh[0], nh[1], nh[2]}, w = Ic[n] * A->domega[n];
        for (int a = 0; a < 4; a++) for (int b = 0; b < 4; b++) R[a][b] += w * n4[a] * n4[b]; /* Eq.45 in the tetrad frame */
    }
    if (R_out) { int q = 0; for (int a = 0; a < 4; a++) for (int b = a; b < 4; b++) R_out[q++] = R[a][b]; }
    double ul[4] = {-uh[0], uh[1], uh[2], uh[3]}; /* u_ahat */
    double uR[4], Ebar = 0;
    for (int a = 0; a < 4; a++) { uR[a] = 0; for (int b = 0; b < 4; b++) uR[a] += ul[b] * R[a][b]; }
    for (int a = 0; a < 4; a++) Ebar += ul[a] * uR[a];
    double ugas = rho * Tm / (P->gamma_gas - 1.0), pgas = rho * Tm; /* k_B/(mu m_p) = 1 */
    double emis = aP * P->a_rad * Tm * Tm * Tm * Tm + aS * Ebar, aE = aEa + aS;
    double G[4];
    for (int a = 0; a < 4; a++) G[a] = -emis * uh[a] - aE * uR[a]; /* Eq.53 */
    if (G_out) for (int a = 0; a < 4; a++) G_out[a] = G[a];
    if (fr_out) for (int a = 0; a < 3; a++) fr_out[a] = 0.0;
    if (!(Ebar > rho + ugas) || !(R[0][0] > 0.0)) return 0;
    double v[3] = {R[0][1] / R[0][0], R[0][2] / R[0][0], R[0][3] / R[0][0]}; /* Eq.51 */
    double vv = v[0] * v[0] + v[1] * v[1] + v[2] * v[2];
    if (vv > 1.0 - 1e-12) vv = 1.0 - 1e-12; /* R19 */
    double W = 1.0 / sqrt(1.0 - vv), ur[4] = {W, W * v[0], W * v[1], W * v[2]};
    double wgas = rho + ugas + pgas, un[4];
    for (int a = 1; a < 4; a++) {
        double Tgas = wgas * uh[0] * uh[a], Trad = wgas * ur[0] * ur[a]; /* Eq.52 */
        double den = Trad - Tgas, f = (den != 0.0) ? G[a] * dt / den : 0.0; /* Eq.54 with G8 */
        if (!(f > 0.0)) f = 0.0;
        if (f > 1.0) f = 1.0;
        if (fr_out) fr_out[a - 1] = f;
        un[a] = (1.0 - f) * uh[a] + f * ur[a]; /* Eq.55 */
    }
    uh[1] = un[1]; uh[2] = un[2]; uh[3] = un[3];
    uh[0] = sqrt(1.0 + (un[1] * un[1] + un[2] * un[2] + un[3] * un[3]));
    return 1;
}

long long orc_coupling(const orc_problem *P, double *I, const double *fluid, const double *opac, double dt,
                       double *T_out, double *dT0) {
    const orc_angles *A = P->ang;
    int N = A->N, ng = P->ng;
    long long nc = P->ncell, nfail = 0;
#pragma omp parallel reduction(+ : nfail)
    {
        double *n0bar = malloc(sizeof(double) * N), *dOmb = malloc(sizeof(double) * N), *Ibm = malloc(sizeof(double) * N);
#pragma omp for schedule(static)
        for (int k = ng; k < P->NK - ng; k++)
            for (int j = ng; j < P->NJ - ng; j++)
                for (int i = ng; i < P->NI - ng; i++) {
                    long long c = cidx(P, k, j, i);
                    const double *cg = &P->cell[c * ORC_NCELL], *e = cg + 1, *Lw = cg + 17;
                    double rho = fluid[0 * nc + c], Tm = fluid[1 * nc + c];
                    double unorm[3] = {fluid[2 * nc + c], fluid[3 * nc + c], fluid[4 * nc + c]};
                    double aP = opac[0 * nc + c], aEa = opac[1 * nc + c], aS = opac[2 * nc + c];
                    double *Ic = &I[c * N];
                    if (T_out) T_out[c] = Tm;
                    if (dT0) for (int m = 0; m < 4; m++) dT0[m * nc + c] = 0.0;
                    if (P->excised[c]) continue;
                    int coupled = 0;
                    double Tp = Tm;
                    if (P->couple) {
                        /* R10: gamma = sqrt(1 + gamma_ab u^a' u^b'), u^0 = gamma/alpha, u^a = u^a' - beta^a gamma/alpha
                         * (inverse of Eq.7) */
                        double ucon[4];
                        fluid_four_velocity(cg, unorm, ucon);
                        /* u^ahat = e^ahat_beta u^beta = eta^{ahat ahat} L[beta][ahat] u^beta (Eq.8b, 9) */
                        double uh[4];
                        for (int ah = 0; ah < 4; ah++) {
                            double s = 0;
                            for (int b = 0; b < 4; b++) s += Lw[4 * b + ah] * ucon[b];
                            uh[ah] = (ah == 0 ? -1.0 : 1.0) * s;
                        }
                        if (P->vel_estimate) velocity_estimate(P, Ic, uh, rho, Tm, aP, aEa, aS, dt, NULL, NULL, NULL); /* Eq.51-55 */
                        /* per angle: n^0bar = -u_alpha n^alpha = u^0hat - u^ahat n^ahat (Eq.14a,b);
                         * R11: Ibar = (n^0bar)^4 Ihat, dOmega_bar = dOmega / (n^0bar)^2 */
                        double W = 0;
                        for (int n = 0; n < N; n++) {
                            const double *nh = &A->nhat[3 * n];
                            n0bar[n] = uh[0] - (uh[1] * nh[0] + uh[2] * nh[1] + uh[3] * nh[2]);
                            dOmb[n] = A->domega[n] / (n0bar[n] * n0bar[n]);
                            double n2 = n0bar[n] * n0bar[n];
                            Ibm[n] = n2 * n2 * Ic[n];
                            W += dOmb[n];
                        }
                        if (P->renorm) for (int n = 0; n < N; n++) dOmb[n] = 4.0 * PI * dOmb[n] / W; /* R12 */
                        double aE = aEa + aS; /* Eq.33b */
                        double nup0 = contract4(e, &A->nhat[0]); /* n^0 = 1/alpha for every angle (e^0_ahat = 0) */
                        double A1 = 0, A2 = 0, Em = 0;
                        for (int n = 0; n < N; n++) {
                            double dn = nup0 + n0bar[n] * aE * dt;
                            A1 += (nup0 / dn) * Ibm[n] * dOmb[n];          /* Eq.42a */
                            A2 += (n0bar[n] / dn) * dOmb[n];                /* Eq.42b (x dt/4pi below) */
                            Em += Ibm[n] * dOmb[n];                         /* Eq.38 */
                        }
                        A2 *= dt / (4.0 * PI);
                        double Cv = rho / (P->gamma_gas - 1.0);            /* k_B/(mu m_p) = 1 */
                        double B4 = A2 * aP * P->a_rad;                    /* Eq.50a */
                        double B1 = Cv * (1.0 - A2 * aS);                  /* Eq.50b */
                        double Bp = A1 - (1.0 - A2 * aS) * Em;             /* Eq.50c: B0 = Bp - B1 T_- */
                        double dT = 0.0;
                        if (quartic_delta(B4, B1, Bp, Tm, &dT) != 0) { nfail++; Tp = Tm; }
                        else {
                            coupled = 1;
                            Tp = Tm + dT;
                            double Ep = Em - Cv * dT;                      /* Eq.48 */
                            double src = aP * P->a_rad * Tp * Tp * Tp * Tp + aS * Ep;
                            /* subtract the change of R^0_alpha from T^0_alpha.  SURVEY O5: the change is formed angle by angle,
                             * dT^0_alpha = -sum_n n^0 n_alpha (Ihat_+ - I*) dOmega_n; with dt0_literal the two sums R^0_alpha[I*] and
                             * R^0_alpha[Ihat_+] are formed first and subtracted (the same number up to the rounding of two N-term sums). */
                            double Rb[4] = {0, 0, 0, 0}, Ra[4] = {0, 0, 0, 0}, dR[4] = {0, 0, 0, 0};
                            for (int n = 0; n < N; n++) {
                                const double *nh = &A->nhat[3 * n];
                                double dn = nup0 + n0bar[n] * aE * dt;
                                double Ibp = (nup0 * Ibm[n] + n0bar[n] * dt / (4.0 * PI) * src) / dn; /* Eq.40 */
                                double n2 = n0bar[n] * n0bar[n];
                                double Inew = Ibp / (n2 * n2), Iold = Ic[n];
                                for (int m = 0; m < 4; m++) {
                                    double wgt = nup0 * contract4(Lw + 4 * m, nh) * A->domega[n]; /* n^0 n_alpha dOmega */
                                    Rb[m] += wgt * Iold; Ra[m] += wgt * Inew;
                                    dR[m] += wgt * (Inew - Iold);
                                }
                                Ic[n] = Inew;
                            }
                            if (dT0) for (int m = 0; m < 4; m++) dT0[m * nc + c] = P->dt0_literal ? -(Ra[m] - Rb[m]) : -dR[m];
                        }
                    }
                    (void)coupled;
                    if (T_out) T_out[c] = Tp;
                    /* R14 / P:L329: zero I wherever |n_0| < n_0^crit (cell-centre n_0) */
                    for (int n = 0; n < N; n++) {
                        double n0 = contract4(Lw, &A->nhat[3 * n]);
                        if (fabs(n0) < P->n0_crit) Ic[n] = 0.0;
                    }
                }
        free(n0bar); free(dOmb); free(Ibm);
    }
    return nfail;
}

/* Eq.51-55 for one cell, for the pins: u_inout[4] tetrad-frame gas velocity in, estimate out; G[4], fr[3], R[10] as in
 * velocity_estimate.  returns 1 if the cell is radiation dominated (the blend was applied) */
int orc_velocity_estimate_cell(const orc_problem *P, const double *Icell, double *u_inout, double rho, double Tm, double aP, double aEa,
                               double aS, double dt, double *G, double *fr, double *R) {
    return velocity_estimate(P, Icell, u_inout, rho, Tm, aP, aEa, aS, dt, G, fr, R);
}

long long orc_stage(const orc_problem *P, double *I_in, double *I_out, const double *I0, const double *fluid,
                    const double *opac, double gam0, double gam1, double beta_dt, double *T_out, double *dT0) {
    orc_fill_ghosts(P, I_in);
    orc_transport_tau(P, I_in, I0, gam0, gam1, beta_dt, fluid, opac, I_out);
    return orc_coupling(P, I_out, fluid, opac, beta_dt, T_out, dT0);
}

/* ======================================================================================
 * O6. Moments (Eq.45, Eq.71d, Eq.38)
 * ==================================================================================== */
void orc_moments(const orc_problem *P, const double *I, int frame, const double *fluid, double *out) {
    const orc_angles *A = P->ang;
    int N = A->N, ng = P->ng;
    long long nc = P->ncell;
#pragma omp parallel for schedule(static)
    for (int k = ng; k < P->NK - ng; k++)
        for (int j = ng; j < P->NJ - ng; j++)
            for (int i = ng; i < P->NI - ng; i++) {
                long long c = cidx(P, k, j, i);
                const double *cg = &P->cell[c * ORC_NCELL], *e = cg + 1, *Lw = cg + 17;
                double acc[10] = {0};
                double uh[4] = {1, 0, 0, 0};
                if (frame == 3) {
                    double unorm[3] = {fluid[2 * nc + c], fluid[3 * nc + c], fluid[4 * nc + c]}, ucon[4];
                    fluid_four_velocity(cg, unorm, ucon);
                    for (int ah = 0; ah < 4; ah++) {
                        double s = 0;
                        for (int b = 0; b < 4; b++) s += Lw[4 * b + ah] * ucon[b];
                        uh[ah] = (ah == 0 ? -1.0 : 1.0) * s;
                    }
                }
                for (int n = 0; n < N; n++) {
                    const double *nh = &A->nhat[3 * n];
                    double w = I[c * N + n] * A->domega[n];
                    double nh4[4] = {1.0, nh[0], nh[1], nh[2]}, nup[4], nlo0;
                    for (int m = 0; m < 4; m++) nup[m] = contract4(e + 4 * m, nh);
                    nlo0 = contract4(Lw, nh);
                    if (frame == 0) { int q = 0; for (int a = 0; a < 4; a++) for (int b = a; b < 4; b++) acc[q++] += w * nup[a] * nup[b]; }
                    else if (frame == 1) { for (int m = 0; m < 4; m++) acc[m] += w * nup[0] * contract4(Lw + 4 * m, nh); (void)nlo0; }
                    else if (frame == 2) { int q = 0; for (int a = 0; a < 4; a++) for (int b = a; b < 4; b++) acc[q++] += w * nh4[a] * nh4[b]; }
                    else { /* Eq.13-14 with G2 (denominator 1 + u^0hat); Eq.38: dOmega_bar Ibar = (n^0bar)^2 Ihat dOmega_hat */
                        double nb[4];
                        nb[0] = uh[0] - (uh[1] * nh[0] + uh[2] * nh[1] + uh[3] * nh[2]);
                        double udotn = uh[1] * nh[0] + uh[2] * nh[1] + uh[3] * nh[2];
                        for (int p = 1; p < 4; p++) nb[p] = -uh[p] + nh[p - 1] + uh[p] * udotn / (1.0 + uh[0]);
                        /* R^{0bar abar} = oint Ibar nbar^0 nbar^a dOmega_bar with unit-length fluid-frame direction nbar^a/nbar^0:
                         * Ibar dOmega_bar = (n^0bar)^2 Ihat dOmega_hat, direction cosines nb[p]/nb[0] */
                        acc[0] += w * nb[0] * nb[0];
                        for (int p = 1; p < 4; p++) acc[p] += w * nb[0] * nb[p];
                    }
                }
                int ncomp = (frame == 0 || frame == 2) ? 10 : 4;
                for (int q = 0; q < ncomp; q++) out[q * nc + c] = acc[q];
            }
}

/* ======================================================================================
 * Upwind sign tables and signal speed
 * ==================================================================================== */
static signed char sgn(double x) { return (signed char)((x > 0.0) - (x < 0.0)); }

void orc_upwind_tables(const orc_problem *P, signed char *face_sign, signed char *edge_sign) {
    const orc_angles *A = P->ang;
    int N = A->N, E = A->E;
    for (long long c = 0; c < P->ncell; c++) {
        if (face_sign)
            for (int ax = 0; ax < 3; ax++)
                for (int n = 0; n < N; n++)
                    face_sign[(c * 3 + ax) * N + n] = sgn(contract4(&P->face[(c * 3 + ax) * ORC_NFACE], &A->nhat[3 * n]));
        if (edge_sign)
            for (int e = 0; e < E; e++) edge_sign[c * E + e] = sgn(edge_coeff(&P->cell[c * ORC_NCELL + 33], &A->edge_T[30 * e]));
    }
}

/* c_e (pinned chain) and n_0 at the edge direction for every unique edge of one cell */
void orc_edge_coeffs(const orc_problem *P, long long cell, double *ce, double *n0e) {
    const orc_angles *A = P->ang;
    const double *cg = &P->cell[cell * ORC_NCELL];
    for (int e = 0; e < A->E; e++) {
        if (ce) ce[e] = edge_coeff(cg + 33, &A->edge_T[30 * e]);
        if (n0e) n0e[e] = contract4(cg + 17, &A->edge_mid[3 * e]);
    }
}

double orc_max_speed(const orc_problem *P, double out_axis[3]) {
    const orc_angles *A = P->ang;
    double mx[3] = {0, 0, 0};
    for (long long c = 0; c < P->ncell; c++)
        for (int ax = 0; ax < 3; ax++) {
            const double *f = &P->face[(c * 3 + ax) * ORC_NFACE];
            /* n^0 at the face: e^0_0hat = -E_0hat^{-1}... use 1/alpha_face = -1/L[0][0] (E_0hat = -alpha) */
            double n0up = -1.0 / f[4];
            for (int n = 0; n < A->N; n++) {
                double v = fabs(contract4(f, &A->nhat[3 * n]) / n0up);
                if (v > mx[ax]) mx[ax] = v;
            }
        }
    if (out_axis) for (int d = 0; d < 3; d++) out_axis[d] = mx[d];
    return fmax(mx[0], fmax(mx[1], mx[2]));
}
