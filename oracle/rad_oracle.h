/* oracle/rad_oracle.h -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, FP64 CPU statement of the radiation stage of White et al.
 * (arXiv 2302.04283), written from the paper's equations.  Cited as
 * P:L<line> = /root/reference/PAPER.md line.  Only tests/, the smoke check
 * and bench.py's cpu_baseline / --impl reference legs may load this library.
 * It shares no code with paper_2302_04283_b200/csrc (the CUDA path).
 *
 * All functions use plain pointers to host memory; layouts are stated per
 * function.  Compile with -O2 -ffp-contract=off (the only fused operations
 * are the explicit fma() calls that pin the upwind-sign arithmetic).
 */
#ifndef RAD_ORACLE_H
#define RAD_ORACLE_H

#ifdef __cplusplus
extern "C" {
#endif

/* ---- sizes of the oracle's own geometry records (doubles) ---- */
#define ORC_NPOINT 132 /* orc_geometry_point: alpha, beta^i[3], g[16], ginv[16], e[16], elow[16], omega[64] */
#define ORC_NCELL 72   /* per cell centre: alpha, e[mu][ahat] (16), L[mu][ahat]=g_{mu nu}e^nu_ahat (16), S[c][k] (30), beta^a (3), gamma_ab (6) */
#define ORC_NFACE 8    /* per face centre: e[a][0..3] (row of the face's axis), L[0][0..3] */
#define ORC_MAXNBR 6

typedef struct orc_angles orc_angles;
typedef struct orc_problem orc_problem;

/* ---- O1: angle grids (SURVEY 8(c) R1,R3) ---- */
orc_angles *orc_angles_latlon(int nzeta, int npsi);
orc_angles *orc_angles_geodesic(int nlev);
void orc_angles_free(orc_angles *);
int orc_angles_nang(const orc_angles *);
int orc_angles_nedge(const orc_angles *);
/* copy out tables: nhat[N][3], domega[N], nnbr[N], nbr[N][6] (-1 = none),
 * nbr_edge[N][6] (unique edge id, -1), edge_lo[E], edge_hi[E] (lo<hi angle ids),
 * edge_len[E] (Delta lambda), edge_mid[E][3] (unit), edge_nrm[E][3] (points lo->hi),
 * edge_T[E][30] (pinned products N^c q_k).  Any pointer may be NULL. */
void orc_angles_tables(const orc_angles *, double *nhat, double *domega, int *nnbr, int *nbr,
                       int *nbr_edge, int *edge_lo, int *edge_hi, double *edge_len,
                       double *edge_mid, double *edge_nrm, double *edge_T);

/* ---- O2: geometry at one point ---- */
/* kind 0 Minkowski, 1 Cartesian Kerr-Schild(M,a).  out[ORC_NPOINT]. */
void orc_geometry_point(int kind, double M, double a, const double x[3], double *out);

/* ---- problem = grid + metric + angles + parameters ---- */
orc_problem *orc_create(int metric_kind, double M, double a, double excise_r, const int n[3], int ng,
                        const double x0[3], const double dx[3], const int bc_lo[3],
                        const int bc_hi[3], const orc_angles *ang, double gamma_gas, double a_rad,
                        double n0_crit, int recon_space, int renorm, int couple);
/* the same on a stretched Cartesian grid (NEXT-4; Eq.20b,c with sqrt(-g) = 1: Delta A_a / Delta V = 1 / Delta x^a of the cell; reading R22:
 * reconstruction in index space): xf0, xf1, xf2 = face coordinates along x, y, z incl. ghost cells (n + 2 ng + 1 entries), or NULL = uniform */
orc_problem *orc_create_stretched(int kind, double M, double a, double excise_r, const int n[3], int ng, const double x0[3],
                                  const double dx[3], const int bc_lo[3], const int bc_hi[3], const orc_angles *ang,
                                  double gamma_gas, double a_rad, double n0_crit, int recon_space, int renorm, int couple,
                                  const double *xf0, const double *xf1, const double *xf2);
void orc_destroy(orc_problem *);
long long orc_ncells_total(const orc_problem *);
/* geometry tables built at create: cell[ncells_total][ORC_NCELL], face[ncells_total][3][ORC_NFACE],
 * excised[ncells_total] (0/1) */
void orc_get_geometry(const orc_problem *, double *cell, double *face, int *excised);

/* ---- a7: ghost fill. I[k][j][i][n] with ng ghosts per side ---- */
void orc_fill_ghosts(const orc_problem *, double *I);

/* ---- a1-a3: transport (Eq.22,24,25). Writes interior of I_out. ---- */
void orc_transport(const orc_problem *, const double *I_in, const double *I0, double gam0, double gam1,
                   double beta_dt, double *I_out);

/* ---- NEXT-1: optical-depth-aware spatial flux (Eq.26-29).  tau_factor = the constant of Eq.26; 0 (default)
 * = Eq.24.  orc_stage uses it through orc_transport_tau; fluid and opac must then be valid in the ghost cells too. ---- */
void orc_set_tau_factor(orc_problem *, double tau_factor);
void orc_cell_velocity(const orc_problem *, const double *fluid, const double *opac, double *vel /* [ncells_total][5] */);
void orc_transport_tau(const orc_problem *, const double *I_in, const double *I0, double gam0, double gam1,
                       double beta_dt, const double *fluid, const double *opac, double *I_out);

/* ---- options set after create: which = 0 recon_angle (0 donor cell, 1 PLM on the latitude-longitude grid incl. across the poles,
 * P:L280; -1 is returned if the grid is not lat-lon with even N_psi), 1 vel_estimate (Eq.51-55), 2 dt0_literal
 * (dT^0_alpha as the difference of two sums instead of the sum of differences).  recon_space = 2 (PPM) needs ng = 3.
 * Boundary code 3 = reflecting wall with the angle-mirror permutation (R20). ---- */
int orc_set_option(orc_problem *, int which, int value);
int orc_has_mirror(const orc_problem *, int axis);
double orc_latlon_face_value(const orc_angles *, const double *Icell, int u, int slot /* 0 zeta-, 1 zeta+, 2 psi-, 3 psi+ */);
int orc_velocity_estimate_cell(const orc_problem *, const double *Icell, double *u_inout, double rho, double Tm, double aP, double aEa,
                               double aS, double dt, double *G, double *fr, double *R);

/* ---- a4-a6: coupling (Eq.31-50) in place on I (interior), then the n_0 mask.
 * fluid: SoA [5][ncells_total] = rho, T, u1', u2', u3'.  opac: SoA [3][ncells_total] =
 * alpha_a_planck, alpha_a_energy, alpha_s.  T_out[ncells_total], dT0[4][ncells_total] (may be NULL).
 * returns number of cells whose quartic had no positive root. */
long long orc_coupling(const orc_problem *, double *I, const double *fluid, const double *opac,
                       double dt, double *T_out, double *dT0);

/* full stage = fill ghosts of I_in (per bc; in place), transport, coupling, mask. */
long long orc_stage(const orc_problem *, double *I_in, double *I_out, const double *I0,
                    const double *fluid, const double *opac, double gam0, double gam1, double beta_dt,
                    double *T_out, double *dT0);

/* ---- O6: moments (Eq.45, 38). frame 0: R^{ab} coord (10: 00,01,02,03,11,12,13,22,23,33),
 * 1: R^0_a (4), 2: tetrad R^{ahat bhat} (10), 3: fluid frame Ebar, F^abar (4).
 * out SoA [ncomp][ncells_total]; interior cells only are written. */
void orc_moments(const orc_problem *, const double *I, int frame, const double *fluid, double *out);

/* ---- upwind sign tables (bit-exact parity). face_sign[ncells_total][3][N] = sgn n^a at the
 * lower face of each cell; edge_sign[ncells_total][E] = sgn c_e (cell-centre). int8. ---- */
void orc_upwind_tables(const orc_problem *, signed char *face_sign, signed char *edge_sign);

/* c_e = a(n_e).N_e (R5; pinned fma chain) and n_0 at the edge direction, for the E unique edges of one cell */
void orc_edge_coeffs(const orc_problem *, long long cell, double *ce, double *n0e);

/* max over cells and angles of |n^a / n^0| at faces (for the CFL-limited dt) */
double orc_max_speed(const orc_problem *, double out_axis[3]);

#ifdef __cplusplus
}
#endif
#endif
