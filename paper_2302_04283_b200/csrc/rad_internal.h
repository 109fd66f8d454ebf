// rad_internal.h -- shared declarations of librad.so's translation units (not part of the ABI).
#pragma once
#include <cuda_runtime.h>

#include <string>
#include <vector>

#include "rad.h"

namespace rad {

// Angle grid tables, built on the host (section 2.6 of the paper).
struct AngleTables {
    int N = 0, E = 0;
    std::vector<double> nhat;      // [N][3]
    std::vector<double> domega;    // [N]
    std::vector<int> nnbr;         // [N]
    std::vector<int> nbr;          // [N][6]
    std::vector<int> nbr_edge;     // [N][6]
    std::vector<int> edge_lo, edge_hi;  // [E]
    std::vector<double> edge_len;  // [E]
    std::vector<double> edge_mid;  // [E][3]
    std::vector<double> edge_nrm;  // [E][3]
};
// Balanced ownership of the unique angular edges (edges.cpp): every angle owns <= kMaxOwn of its edges and
// receives the flux of <= kMaxOwn others.
constexpr int kMaxOwn = 3;
struct EdgeOwnership {
    std::vector<int> own_edge;     // [N][3] unique edge id owned in slot j, or -1
    std::vector<int> own_partner;  // [N][3] angle at the far end of that edge, or -1
    std::vector<int> pull_pos;     // [N][3] entry k: position k*N + owner of the flux this angle receives from slot k of its owner, or -1
};
bool build_edge_ownership(const AngleTables &a, EdgeOwnership &out, std::string &err);

bool build_latlon(int nzeta, int npsi, AngleTables &out, std::string &err);
bool build_geodesic(int nlev, AngleTables &out, std::string &err);
bool build_explicit(int N, const double *nhat, const double *domega, const int *nnbr, const int *nbr, const double *edge_len,
                    const double *edge_mid, const double *edge_nrm, AngleTables &out, std::string &err);

// Everything the kernels read besides the caller's arrays (device pointers).
struct DeviceTables {
    int N, E;
    int n[3], ng, NI, NJ, NK;
    long long ncell;
    int sms, smem_optin;  // device: SM count and the opt-in shared memory per CTA (bytes), queried once in rad_create
    double inv_dx[3];
    const double *xf[3];     // stretched grid: face coordinates of axis d (n + 2 ng + 1), or nullptr (uniform)
    const double *inv_w[3];  // ... and 1 / width of every cell of that axis (n + 2 ng), or nullptr
    // angle tables
    const double *nhat;      // [N][3]
    const double *domega;    // [N]
    const int *nnbr;         // [N]
    const int *nbr_edge;     // [N][6]
    const int *edge_lo, *edge_hi;  // [E]
    const double *edge_len;  // [E]
    const double *edge_mid;  // [E][3]
    const double *edge_T;    // [E][30]  pinned products N^c * (n^a n^b)
    // per angle: signed weights of its edges, sgn * dlambda_e / dOmega_n, [N][6] (0 where no edge)
    const double *nbr_w;
    // the same per-angle tables angle-innermost, for kernels whose lanes run over angles (coalesced: k_fluxdiv's update phase)
    const double *nhat_t;    // [3][N]
    const int *nbr_edge_t;   // [6][N]
    const double *nbr_w_t;   // [6][N]
    // geometry
    const double *cell;  // [ncell][RAD_NCELL]
    const double *face;  // [ncell][3][RAD_NFACE]
    // fused stage kernel (stage5.cu): per-angle record {8 own_partner[3], 8 pull_pos[3], 0, 0} (byte offsets) as 8 x uint16 (16 B),
    // 1/dOmega, the owned edge ids, and the stored edge coefficients
    const short *ang_rec;    // [N][8]
    const double *winv;      // [N]
    const int *own_edge;     // [N][3]
    const double *ke;        // [n2][n1][n0][3][N] interior cells only, or nullptr (not stored)
    int fused_ok;            // 1 if the fused kernel can serve this angle grid
    const int *mirror;       // [3][N] angle image under the flip of tetrad component a (reflecting walls, R20), or nullptr
    int recon_angle;         // 0 donor cell, 1 PLM on the latitude-longitude grid (R21)
    int nzeta, npsi;         // latitude-longitude grid shape (recon_angle == 1)
    const double *rec;       // [ncell][RAD_STAGE_RECN] packed per-cell record of the angle-resident stage kernel (stage5.cu), or nullptr
};
#define RAD_STAGE_RECN 36

// arguments of one stage (device pointers are the caller's)
struct StageArgs {
    const double *I_in, *I0;
    double *I_out;
    double gam0, gam1, beta_dt;
    const double *vel8; // optical-depth-aware flux (Eq.26-29): per cell {u^alphahat (4), f/2 of the upper x, y, z faces, pad}, or nullptr (Eq.24)
    int kz0, kz1;  // stage5 only: update the interior planes kz0 <= k < kz1 (0-based, without ghosts); kz1 <= kz0 = the whole block
};

struct Params {
    double gamma_gas, a_rad, n0_crit;
    double rgm1;  // 1 / (gamma_gas - 1)
    double tau_factor;  // constant of Eq.26; 0 = free-streaming flux (Eq.24)
    int recon_space, renorm, couple;
    int vel_estimate;  // 1: radiation-dominated velocity estimate Eq.51-55 in the coupling (NEXT-2)
};

// kernel launchers (each returns the number of kernels it launched, or -1 after setting a CUDA error)
int launch_geometry(const rad_metric &m, const rad_grid &g, const double *const xf_dev[3], double *cell, double *face, long long ncell,
                    cudaStream_t s);
int launch_exchange_halo(const DeviceTables &lo, double *I_lo, const DeviceTables &hi, double *I_hi, int axis, cudaStream_t s);
int launch_fill_ghosts(const DeviceTables &t, const int bc_lo[3], const int bc_hi[3], double *I, cudaStream_t s);
int launch_fluxdiv(const DeviceTables &t, const Params &p, const double *I_in, const double *I0, double gam0,
                   double gam1, double beta_dt, double *I_out, cudaStream_t s, const double *vel = nullptr, double tau_dt = 0.0);
// optical-depth-aware flux (NEXT-1, Eq.26-29): per-cell {u^alphahat, alpha_E} of every cell, vel[ncell][5]
int launch_cell_velocity(const DeviceTables &t, const double *fluid, const double *aE, const double *aS, double *vel, cudaStream_t s);
int launch_coupling(const DeviceTables &t, const Params &p, double *I, const double *fluid, const double *aP,
                    const double *aE, const double *aS, double dt, double *T_out, double *dT0,
                    unsigned long long *noroot, cudaStream_t s);
int launch_moments(const DeviceTables &t, const double *I, int frame, const double *fluid, double *out,
                   cudaStream_t s);
// streaming versions (stream.cu; even N, 16-byte aligned I): 1 launched, 0 not served, -1 CUDA error
int stream_serves(const DeviceTables &t, const void *I);
int launch_couple_stream(const DeviceTables &t, const Params &p, double *I, const double *fluid, const double *aP, const double *aE, const double *aS,
                         double dt, double *T_out, double *dT0, unsigned long long *noroot, cudaStream_t s, int kz0 = 0, int kz1 = 0);
int launch_moments_stream(const DeviceTables &t, const double *I, int frame, const double *fluid, double *out, cudaStream_t s);
// angle-resident fused flux-divergence kernel (stage5.cu): 1 launched, 0 this configuration is not served (caller falls back to
// launch_fluxdiv), -1 CUDA error; and its record builder
int launch_stage_angle(const DeviceTables &t, const Params &p, const StageArgs &a, cudaStream_t s);
int stage_angle_kernel_name(const DeviceTables &t, const Params &p, bool tau, char *buf, size_t n);
// 1 if launch_stage_angle serves this context (so that a stage can be run slab by slab along z); tau: with the velocity records of
// the optical-depth-aware flux in shared memory (a larger layout: some angle counts fit without them only)
int stage_angle_serves(const DeviceTables &t, bool tau = false);
// TAU table of the angle-resident kernel: vel8[ncell][8], see k_tau_table (stage5.cu)
int launch_tau_table(const DeviceTables &t, const double *fluid, const double *aE, const double *aS, double tau_dt, double *vel8, cudaStream_t s);
int launch_pack_rec(const DeviceTables &t, double *rec, cudaStream_t s);
int launch_stage_face_signs(const DeviceTables &t, signed char *out, cudaStream_t s);  // 0 if the context has no stage records
int launch_build_ke(const DeviceTables &t, double *ke, cudaStream_t s);
int launch_sign_tables(const DeviceTables &t, signed char *face_sign, signed char *edge_sign, cudaStream_t s);
int launch_maxspeed(const DeviceTables &t, double *out3, cudaStream_t s);
// probe.cu: measured FP64 FMA rate of the current device (lane operations per second); 0 on success
int probe_dfma_rate(double *dfma_per_sec, long long *launches);

}  // namespace rad
