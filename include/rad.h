/* rad.h -- C ABI of librad.so: the explicit-plus-locally-implicit radiation stage of the
 * finite-solid-angle GR transport of White et al., arXiv 2302.04283, for one NVIDIA B200 (sm_100a).
 *
 * Citations: P:L<n> = line n of the paper text; "R#" = a reading listed in DESIGN.md.
 *
 * Conventions
 *  - Plain C types only.  Every pointer is marked HOST or DEVICE.  DEVICE pointers must live on the
 *    device given to rad_create.  The library owns only what it builds (angle tables, geometry tables,
 *    scratch); the caller owns intensity, fluid, opacity and output buffers.
 *  - No exceptions or aborts cross the ABI: every call returns a rad_status; rad_last_error() gives text.
 *  - Work is enqueued on the caller's CUDA stream (a cudaStream_t passed as void*; NULL = default
 *    stream).  No implicit synchronisation except where stated.
 *  - There is no CPU fallback: if no CUDA device is usable, rad_create returns RAD_ECUDA.
 *
 * Arrays
 *  - Grid: uniform Cartesian, n[0..2] interior cells along x,y,z, ng = 2 ghost cells per side
 *    (PLM needs two; PPM three).  NI = n[0]+2ng etc.  Cell (k,j,i) has flat index c = (k*NJ + j)*NI + i.
 *  - Intensity I[c][n]: angle index n innermost (contiguous), N = number of angles.  FP64.
 *  - Per-cell scalars are SoA: field[f][c].
 */
#ifndef RAD_H
#define RAD_H
#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct rad_ctx rad_ctx; /* opaque, owned by the library */

typedef enum {
    RAD_OK = 0,
    RAD_EINVAL = 1,       /* bad argument (NULL, non-finite, bad shape, aliasing) */
    RAD_ENOMEM = 2,       /* host or device allocation failed */
    RAD_ECUDA = 3,        /* CUDA runtime error (text in rad_last_error) */
    RAD_EUNSUPPORTED = 4, /* valid request the library does not implement */
    RAD_ESTATE = 5        /* call not valid in this state */
} rad_status;

/* ---- geometry record layouts (doubles), also the input format of metric kind 2 ------------------
 * Cell centre record, RAD_NCELL doubles:
 *   [0]      n^0 = e^0_0hat = 1/alpha   (Eq.5a, Eq.11; the same for every angle because e^0_ahat = 0, R2)
 *   [1..4]   E_alphahat = g_{0 mu} e^mu_alphahat, alphahat = 0..3  (E_0hat = -alpha);  n_0 = E_0 + E_a n^a
 *   [5..34]  S[c][k], c = 1..3, k over (00,01,02,03,11,12,13,22,23,33):
 *            S = omega^c_{ab} + omega^c_{ba} (a<b), omega^c_{aa} (a=b); Ricci rotation coefficients Eq.17
 *   [35..37] beta^i (Eq.5c)
 *   [38..43] triad e^i_ahat, upper triangular (R2): (x1,x2,x3,y2,y3,z3)
 *   [44..49] co-triad theta^ahat_i = e^ahat_i, upper triangular: (1x,1y,1z,2y,2z,3z); n_i = theta^a_i n^a
 *   [50]     1.0 if the cell is excised, else 0.0;  [51] unused
 * Face centre record, RAD_NFACE doubles, three per cell (the LOWER x, y, z face of the cell), R6:
 *   [0..3]   e^a_alphahat for the face's own axis a (alphahat = 0..3);  n^a = e^a_0 + e^a_b n^b
 *   [4..7]   E_alphahat at the face centre
 */
#define RAD_NCELL 52
#define RAD_NFACE 8
#define RAD_MAXNBR 6

typedef struct {
    int kind;        /* 0 Minkowski, 1 Cartesian Kerr-Schild, 2 tabulated */
    double M, a;     /* kind 1: mass and spin */
    double excise_r; /* kind 1: cells whose centre has Kerr-Schild radius r < excise_r are excised
                        (I_out = 0, T and fluid increments untouched); 0 = none */
    const double *cell_tab; /* kind 2, DEVICE, [ncells_total][RAD_NCELL]; copied at create */
    const double *face_tab; /* kind 2, DEVICE, [ncells_total][3][RAD_NFACE]; copied at create */
} rad_metric;

typedef struct {
    int n[3], ng;           /* interior cells per axis; ghost cells per side: 2, or 3 (needed by recon_space = 2, PPM) */
    double x0[3], dx[3];    /* lower corner of the interior and cell sizes */
    int bc_lo[3], bc_hi[3]; /* 0 caller-filled, 1 periodic, 2 outflow (copy of nearest interior cell),
                               3 reflecting wall: ghost cell = mirror cell across the wall, with the intensity of
                               the direction whose wall-normal tetrad component is flipped (reading R20); needs an angle
                               grid that is symmetric under that flip (every lat-lon grid with even npsi; the geodesic
                               grid for the y axis only), else rad_create returns RAD_EUNSUPPORTED */
    const double *xf[3];    /* stretched Cartesian grid (NEXT-4; Eq.20b,c): per axis NULL (uniform: faces at x0 + i dx) or
                               HOST array of the n + 2 ng + 1 face coordinates of that axis, ghost cells included, strictly
                               increasing; copied at create.  With sqrt(-g) = 1 the area-to-volume ratio of a cell is
                               Delta A_a / Delta V = 1 / (its width along a); geometry is evaluated at the true cell and face
                               centres; reconstruction works in index space (reading R22).  A stretched axis sends the stage
                               through the generic flux-divergence kernel (the tile kernel shares face fluxes divided by one dx) */
} rad_grid;

typedef struct {
    int kind; /* 0 latitude-longitude (nzeta x npsi), 1 geodesic (level nlev),
                 2 explicit tables (any grid the paper allows) */
    int nzeta, npsi, nlev;
    /* kind 2, all HOST, copied at create.  nang angles; per angle: unit direction nhat[nang][3] (Eq.15b-d), solid angle
     * domega[nang], number of neighbours nnbr[nang] (<= RAD_MAXNBR), neighbour list nbr[nang][RAD_MAXNBR] (-1 = none; both
     * angles of an edge must list each other); per (angle, slot): the edge's arc length edge_len[nang][RAD_MAXNBR]
     * (Delta lambda, Eq.20f), unit vector to its midpoint edge_mid[nang][RAD_MAXNBR][3] and in-sphere unit normal
     * edge_nrm[nang][RAD_MAXNBR][3] pointing from the angle to that neighbour.  An edge's data are read from the entry of
     * its lower-numbered angle.  Errors: RAD_EINVAL (NULL, non-unit nhat, non-positive domega, asymmetric lists, negative or
     * non-finite edge_len, edge_mid that is not a finite unit vector, edge_nrm that is not finite or is zero; edge_nrm need
     * not be unit: it carries the metric factor of its coordinate, 1 / sin zeta on the psi edges of a lat-lon grid, Eq.16c). */
    int nang;
    const double *nhat, *domega, *edge_len, *edge_mid, *edge_nrm;
    const int *nnbr, *nbr;
} rad_angles;

typedef struct { /* fluid-frame absorptivities, DEVICE, each [ncells_total], NOT owned;
                    contents may change between stages */
    const double *alpha_a_planck, *alpha_a_energy, *alpha_s;
} rad_opac;

typedef struct {
    double gamma_gas;         /* adiabatic index Gamma (Eq.48); k_B/(mu m_p) = 1 */
    double a_rad;             /* radiation constant (Eq.34) */
    double n0_crit;           /* Ihat is zeroed where |n_0| < n0_crit; <= 0 disables */
    int recon_space;          /* 0 donor cell, 1 PLM van Leer, 2 PPM Colella & Woodward (needs ng = 3; runs in the
                                 generic flux-divergence kernel) */
    int recon_angle;          /* 0 donor cell; 1 PLM on the latitude-longitude grid, across the poles as P:L280 spells
                                 out (reading R21; lat-lon grids with even npsi only, else RAD_EUNSUPPORTED; generic kernel).
                                 MAPR on the geodesic grid is not implemented: its sources are not in the paper */
    int renorm_fluid_weights; /* R12: 1 = rescale fluid-frame solid angles to sum to 4 pi */
    int couple;               /* 0 = transport only, 1 = with implicit coupling (section 2.5) */
    double tau_factor;        /* constant of Eq.26: 0 = free-streaming spatial flux (Eq.24); > 0 = optical-depth-aware flux
                                 (Eq.26-29; readings R15-R18, G1 in DESIGN.md).  Then rad_stage reads fluid and opacities in the first
                                 ghost layer too, runs as a per-cell table kernel plus the stage kernel, and
                                 rad_transport returns RAD_ESTATE (the flux needs the fluid state) */
    int recompute_edge_coeffs; /* stored-versus-recomputed angular geometry:
                                  0 = the angular-edge coefficients dlambda_e c_e n_0e (Eq.16-17, Eq.25) are built once
                                      in rad_create and stored, 3 N doubles per interior cell (adds 24 B per
                                      intensity update of HBM traffic, removes ~100 FP64 operations per update);
                                  1 = not stored: every stage recomputes them from the Ricci rotation coefficients
                                      (no extra memory; the generic flux-divergence kernel recomputes them and is FP64-bound). */
    int vel_estimate;          /* radiation-dominated velocity estimate (Eq.51-55; reading G8 in DESIGN.md):
                                  1 = in cells where Ebar exceeds rho + u_gas the coupling uses the fluid velocity of Eq.55
                                      (blend of the gas velocity and the radiation velocity of Eq.51 with the clamped
                                      fractions of Eq.54) instead of the pre-coupling velocity; 0 = always the pre-coupling velocity.
                                  Restrictions (the estimate lives in the streaming coupling kernel only): with couple = 1, rad_create returns
                                  RAD_EUNSUPPORTED for an odd number of angles or one whose rows do not fit that kernel's shared memory, and
                                  rad_stage / rad_couple return RAD_EUNSUPPORTED at run time for an intensity array that is not 16-byte aligned */
} rad_params;

/* Build a context: angle tables on the host (section 2.6), geometry tables on the device (section 2.1-2.2,
 * one kernel launch; synchronises the device once).  `device` is the CUDA ordinal.
 * Errors: RAD_EINVAL (NULL, ng not 2 or 3, PPM with ng = 2, n < 1, non-finite or non-positive dx, bad enum, tau_factor < 0),
 * RAD_EUNSUPPORTED (recon_angle = 1 or a reflecting wall on an angle grid that does not allow it), RAD_ENOMEM, RAD_ECUDA.
 * On error *out is NULL. */
rad_status rad_create(const rad_metric *, const rad_grid *, const rad_angles *, const rad_opac *,
                      const rad_params *, int device, rad_ctx **out);

/* One radiation stage (P:L69-81 tasks 1,3,4,7,8; Eq.22,24,25, Eq.31-50):
 *   ghost fill of I_in per bc (writes I_in's ghost cells; no-op for caller-filled)
 *   C_new = gam0 C0 + gam1 C - beta_dt (spatial + angular flux divergence),  C = n^0 n_0 I;  I_new = C_new / (n^0 n_0)
 *   coupling over beta_dt (if params.couple): I_new -> I_+, gas temperature T_+, fluid increment
 *   mask |n_0| < n0_crit
 * I_in, I_out, I0: DEVICE [ncells_total][N]; I_out must not alias I_in or I0 (RAD_EINVAL); only the
 *   interior of I_out is written.  I0 may be NULL (then the gam0 term is absent).
 * fluid: DEVICE SoA [5][ncells_total] = rho, T, u^1', u^2', u^3' (normal-frame velocity).
 * T_out: DEVICE [ncells_total] or NULL.  dT0: DEVICE [4][ncells_total] or NULL: increment of the
 *   fluid's T^0_alpha = -(change of R^0_alpha in the coupling).  Interior cells only.
 * n_noroot: HOST or NULL.  If given, the call synchronises the stream and stores the number of cells
 *   whose quartic (Eq.49) had no positive root (those cells are left uncoupled, R13).
 * Forward Euler is (gam0, gam1, beta_dt) = (0, 1, dt). */
rad_status rad_stage(rad_ctx *, double *I_in, double *I_out, const double *I0, const double *fluid,
                     double gam0, double gam1, double beta_dt, double *T_out, double *dT0,
                     long long *n_noroot, void *cuda_stream);

/* rad_stage for callers that cannot ask the CUDA allocator for memory once their run is under way.
 *
 * Who that is: a time integrator that calls the stage thousands of times from inside its step loop, after it has
 *   (a) handed all remaining device memory to a pool of its own (a torch caching allocator sized to the card, an AMR framework's
 *       arena), so that a late cudaMalloc inside the library fails or evicts the pool, or
 *   (b) put the fluid solver, the halo copies and the radiation stage on different streams: cudaMalloc and cudaFree wait for the
 *       whole device, so one allocation in the middle of a step stalls every stream of the application, or
 *   (c) promised its users a device-memory footprint that is fixed once set-up is over.
 * rad_stage itself allocates in one situation: with the optical-depth-aware flux (tau_factor > 0, Eq.26-29) its first call on a
 * context takes a per-cell table (8 doubles per cell) from cudaMalloc, which the table kernel writes and the flux-divergence
 * kernel reads.  rad_stage_static computes the same stage -- same kernels, same arguments, same results bit for bit -- with that
 * table in an array that is part of librad.so's device image instead: RAD_STATIC_MAX_CELLS x 8 doubles = 4 MiB, resident on every
 * GPU that loads the library from the load until the process exits, whether or not this entry point is ever called.
 * It calls no cudaMalloc, cudaFree or other allocating routine, on any call, for any tau_factor (with tau_factor = 0 the array is
 * not touched and the call is rad_stage under another name).
 *
 *  - Limit: the block, ghost layers included, may have at most RAD_STATIC_MAX_CELLS cells (65 536: e.g. 36 x 36 x 36 interior
 *    cells with ng = 2, which covers the paper's 32^3 blocks).  A larger context gets RAD_EUNSUPPORTED and a message
 *    that names both numbers; nothing is launched.  Use rad_stage for those.
 *  - First call on a device: looks up where the array sits in that device's memory (one cudaGetSymbolAddress, result cached per
 *    device ordinal).  The look-up is not a stream operation: make this first call during set-up, before any stream capture.
 *  - One array for everybody: all contexts, streams and host threads of the process share it on a given device.  Two calls
 *    whose kernels can overlap on the GPU (different streams without an event between them, or two host threads) overwrite
 *    each other's table and both results are garbage.  Calls on one stream, or ordered by events, are safe.
 *  - Nothing needs clearing between calls: every call rewrites the table entries of all its cells before reading any, and
 *    reads no others; the rest of the array keeps stale values of earlier, larger blocks.
 * Arguments, outputs, aliasing rules and the other status codes are those of rad_stage. */
#define RAD_STATIC_MAX_CELLS 65536
rad_status rad_stage_static(rad_ctx *, double *I_in, double *I_out, const double *I0, const double *fluid,
                            double gam0, double gam1, double beta_dt, double *T_out, double *dT0,
                            long long *n_noroot, void *cuda_stream);

/* Same stage with HOST buffers (same shapes): copies I_in, fluid and the three opacity arrays
 * host->device into library-owned scratch, runs the stage, copies I_out, T_out, dT0 back, and
 * synchronises.  With caller-filled boundaries and an angle grid the tile kernel serves, the block is
 * processed in slabs of z planes on three streams, so that the copy-in of the next slab and the
 * copy-out of the previous one overlap the stage of the current one (pinned host memory needed for
 * the overlap); otherwise copy-in, rad_stage, copy-out run one after the other.  Ghost cells of
 * I_out_host receive the values of I_in_host; T_out_host / dT0_host are defined in interior cells.  opac_host: HOST SoA [3][ncells_total] = alpha_a_planck, alpha_a_energy, alpha_s.
 * I0 is not supported here (forward-Euler style stages only).  Pinned host memory makes the copies faster
 * but is not required. */
rad_status rad_stage_host(rad_ctx *, const double *I_in_host, double *I_out_host, const double *fluid_host,
                          const double *opac_host, double gam0, double gam1, double beta_dt,
                          double *T_out_host, double *dT0_host, long long *n_noroot);

/* The two halves of a stage, separately (used by tests and profiling):
 * rad_transport = ghost fill + flux-divergence kernel; rad_couple = coupling + mask in place on I. */
rad_status rad_fill_ghosts(rad_ctx *, double *I, void *cuda_stream);
rad_status rad_transport(rad_ctx *, double *I_in, double *I_out, const double *I0, double gam0, double gam1,
                         double beta_dt, void *cuda_stream);
rad_status rad_couple(rad_ctx *, double *I, const double *fluid, double dt, double *T_out, double *dT0,
                      long long *n_noroot, void *cuda_stream);

/* Angular moments of I (Eq.45, Eq.38) for interior cells, DEVICE out SoA [ncomp][ncells_total]:
 * frame 0: coordinate R^{ab} (10: 00,01,02,03,11,12,13,22,23,33); 1: mixed R^0_a (4);
 * frame 2: tetrad R^{ahat bhat} (10); 3: fluid frame Ebar, F^abar (4; needs fluid, Eq.13-14). */
rad_status rad_moments(rad_ctx *, const double *I, int frame, const double *fluid, double *out, void *cuda_stream);

/* Tables for parity checks.  Copies `nbytes` (must equal the table's size) to HOST memory; synchronises. */
typedef enum {
    RAD_TAB_NANG = 0,       /* int[1] */
    RAD_TAB_NEDGE = 1,      /* int[1] */
    RAD_TAB_NHAT = 2,       /* double[N][3] */
    RAD_TAB_DOMEGA = 3,     /* double[N] */
    RAD_TAB_NNBR = 4,       /* int[N] */
    RAD_TAB_NBR = 5,        /* int[N][6], -1 = none; geodesic: counter-clockwise from outside starting at the
                               smallest index (R3); lat-lon: zeta-, zeta+, psi-, psi+ */
    RAD_TAB_NBR_EDGE = 6,   /* int[N][6] unique edge id */
    RAD_TAB_EDGE_LO = 7,    /* int[E]  lower angle index of each unique edge */
    RAD_TAB_EDGE_HI = 8,    /* int[E] */
    RAD_TAB_EDGE_LEN = 9,   /* double[E] Delta lambda_e (Eq.20f) */
    RAD_TAB_EDGE_MID = 10,  /* double[E][3] unit vector to the edge midpoint */
    RAD_TAB_EDGE_NRM = 11,  /* double[E][3] in-sphere edge normal, pointing lo -> hi */
    RAD_TAB_CELL = 12,      /* double[ncells_total][RAD_NCELL] */
    RAD_TAB_FACE = 13,      /* double[ncells_total][3][RAD_NFACE] */
    RAD_TAB_FACE_SIGN = 14, /* signed char[ncells_total][3][N]: sgn n^a at each cell's lower faces (upwind index, Eq.24) */
    RAD_TAB_EDGE_SIGN = 15, /* signed char[ncells_total][E]: sgn c_e (upwind index, Eq.25) */
    RAD_TAB_MAXSPEED = 16,  /* double[3]: max over faces and angles of |n^a / n^0| per axis (for the CFL step, R9) */
    /* the upwind decisions as the stage kernel itself takes them (RAD_ESTATE if the context does not run the tile kernel): */
    RAD_TAB_OWN_EDGE = 17,  /* int[N][3]: unique edge id owned by angle n in slot j, -1 = none (balanced ownership) */
    RAD_TAB_KE = 18,        /* double[n2][n1][n0][3][N] (interior cells): stored edge coefficient of the edge angle n owns in slot j,
                               +-dlambda_e c_e n_0e; its lowest mantissa bit = 1 if the owner is the upwind end (Eq.25) */
    RAD_TAB_STAGE_FACE_SIGN = 19 /* signed char[ncells_total][3][N]: sgn n^a at each cell's UPPER faces, from the kernel's own face
                                    evaluation on its packed records (Eq.24) */
} rad_table;
rad_status rad_get_table(rad_ctx *, int which, void *host_out, size_t nbytes);

/* number of cells including ghosts, = NI*NJ*NK */
long long rad_ncells_total(const rad_ctx *);
/* kernels launched by this context so far (bench.py's gpu_launches) */
long long rad_launch_count(const rad_ctx *);

/* Host-only helper (needs no device): the angle grid's unique edges and the ownership tables the tile kernel works with (edges.cpp).
 * Every unique edge e = (edge_lo[e], edge_hi[e]) is owned by one of its two angles, at most three per angle, in a slot 0..2
 * (own_edge[n][slot] = e or -1, own_partner[n][slot] = the angle at the other end); the slots are a colouring under which the edges an
 * angle RECEIVES have different slots too: pull_pos[n][k] = k * nang + owner of the edge angle n receives from slot k, or -1.
 * nang, nedge: HOST out.  The arrays are HOST, int, optional (NULL = not wanted), each with room for `capacity` entries: edge_lo / edge_hi
 * need nedge, the others 3 * nang; with all five NULL only the sizes are returned.  RAD_EUNSUPPORTED if the grid has an angle with
 * more than six edges. */
rad_status rad_edge_ownership(const rad_angles *, int *nang, int *nedge, int *edge_lo, int *edge_hi, int *own_edge, int *own_partner, int *pull_pos,
                              size_t capacity);

/* Halo exchange between two blocks on the same device that touch along `axis` (0 x, 1 y, 2 z), block `hi` above block `lo`: the
 * communication task of a stage for a domain cut into blocks, one context per block.  The upper ghost layers of I_lo
 * receive the first ng interior layers of I_hi and the lower ghost layers of I_hi the last ng interior layers of I_lo, over the
 * full extent (ghosts included) of the other two axes.  Both contexts must agree in angle grid size, ghost depth and the extents
 * across the axis (RAD_EINVAL otherwise); the touching boundaries should carry boundary code 0 (caller-filled) so that rad_stage
 * leaves the exchanged layers alone.  Call it for x, then y, then z before rad_stage, like the ghost fill, so that edges and corners
 * are consistent.  I_lo, I_hi: DEVICE, each laid out for its own context.  Enqueued on `stream` (2 launches); no sync. */
rad_status rad_exchange_halo(rad_ctx *lo, double *I_lo, rad_ctx *hi, double *I_hi, int axis, void *cuda_stream);

/* Names of the kernels one rad_stage launches on this context after the ghost fill, "flux-divergence kernel;coupling kernel", each
 * written as ncu prints the instance without casts and blanks, e.g. "k_stage5<3,2,4,2,1,1,0>;k_couple_stream<0,21>".  bench.py keys
 * the committed ncu summaries (the .csv files under profiles/) with them and prints no profile figure for a kernel whose name it does not find.
 * buf: HOST, nbytes >= 128.  RAD_EINVAL if the buffer is too small. */
rad_status rad_stage_kernels(rad_ctx *, char *buf /* HOST */, size_t nbytes);

/* Measurement helper (not part of the stage): the device's FP64 fused-multiply-add rate, in lane-level DFMA
 * operations per second (x2 = flop/s), from a register-only kernel timed with CUDA events; synchronises.
 * bench.py uses it as the denominator of the FP64 ("alu") roofline of the stage kernel. */
rad_status rad_probe_fp64(rad_ctx *, double *dfma_per_sec /* HOST */);

/* Text of the last error on this context (or of the last failed rad_create if ctx is NULL).  Never NULL. */
const char *rad_last_error(const rad_ctx *);

void rad_destroy(rad_ctx *);

#ifdef __cplusplus
}
#endif
#endif
