// api.cu -- the C ABI of librad.so (include/rad.h): argument checking, context ownership, launches.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "rad_internal.h"

struct rad_ctx {
    int device = 0;
    rad_metric metric{};
    rad_grid grid{};
    rad_angles angles{};
    rad_opac opac{};
    rad_params params{};
    rad::AngleTables host;
    rad::EdgeOwnership own;
    double *ke = nullptr;  // stored edge coefficients (owned)
    double *rec = nullptr; // packed per-cell records of the stage kernel (owned)
    double *vel8 = nullptr; // optical-depth-aware flux in the tile kernel: {u^alphahat, f/2 of the upper faces} per cell (owned, allocated on first use)
    double *vel = nullptr; // optical-depth-aware flux: {u^alphahat, alpha_E} per cell (owned, allocated on first use)
    rad::DeviceTables dev{};
    rad::Params kp{};
    std::vector<void *> owned;  // device allocations to free
    double *scratch_I[2] = {nullptr, nullptr};  // rad_stage_host
    double *scratch_small = nullptr;            // fluid[5] + opac[3] + T[1] + dT0[4] per cell
    unsigned long long *d_noroot = nullptr;
    cudaStream_t hs[3] = {nullptr, nullptr, nullptr};  // rad_stage_host: copy-in, compute, copy-out
    long long launches = 0;
    std::string err;
};

namespace {
thread_local std::string g_create_err;  // text of the last failed rad_create of the calling thread

struct DeviceGuard {
    int prev = -1;
    bool ok;
    explicit DeviceGuard(int dev) { ok = cudaGetDevice(&prev) == cudaSuccess && cudaSetDevice(dev) == cudaSuccess; }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

rad_status fail(rad_ctx *c, rad_status st, const std::string &msg) {
    if (c) c->err = msg; else g_create_err = msg;
    return st;
}
rad_status cuda_fail(rad_ctx *c, const char *where) {
    cudaError_t e = cudaGetLastError();
    return fail(c, RAD_ECUDA, std::string(where) + ": " + cudaGetErrorString(e));
}

template <class T>
bool upload(rad_ctx *c, const std::vector<T> &h, const T **dptr) {
    void *p = nullptr;
    const size_t bytes = std::max<size_t>(h.size(), 1) * sizeof(T);
    if (cudaMalloc(&p, bytes) != cudaSuccess) return false;
    c->owned.push_back(p);
    if (!h.empty() && cudaMemcpy(p, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice) != cudaSuccess) return false;
    *dptr = static_cast<const T *>(p);
    return true;
}

bool finite_pos(double v) { return std::isfinite(v) && v > 0.0; }

// the count of cells without a root (R13) back to the host, if asked for: synchronises the stream
rad_status read_noroot(rad_ctx *c, long long *n_noroot, cudaStream_t s, const char *where) {
    if (!n_noroot) return RAD_OK;
    unsigned long long v = 0;
    if (cudaMemcpyAsync(&v, c->d_noroot, sizeof(v), cudaMemcpyDeviceToHost, s) != cudaSuccess || cudaStreamSynchronize(s) != cudaSuccess)
        return cuda_fail(c, where);
    *n_noroot = (long long)v;
    return RAD_OK;
}

}  // namespace

extern "C" {

rad_status rad_create(const rad_metric *m, const rad_grid *g, const rad_angles *a, const rad_opac *o, const rad_params *p,
                      int device, rad_ctx **out) {
    if (out) *out = nullptr;
    if (!m || !g || !a || !p || !out) return fail(nullptr, RAD_EINVAL, "rad_create: NULL argument");
    if (g->ng != 2 && g->ng != 3) return fail(nullptr, RAD_EINVAL, "rad_create: ng must be 2 or 3");
    for (int d = 0; d < 3; d++) {
        if (g->n[d] < 1) return fail(nullptr, RAD_EINVAL, "rad_create: n[d] must be >= 1");
        if (!finite_pos(g->dx[d]) || !std::isfinite(g->x0[d])) return fail(nullptr, RAD_EINVAL, "rad_create: bad x0/dx");
        if (g->bc_lo[d] < 0 || g->bc_lo[d] > 3 || g->bc_hi[d] < 0 || g->bc_hi[d] > 3) return fail(nullptr, RAD_EINVAL, "rad_create: bad boundary code");
        if ((g->bc_lo[d] == 3 || g->bc_hi[d] == 3) && g->n[d] < g->ng) return fail(nullptr, RAD_EINVAL, "rad_create: a reflecting wall needs n[d] >= ng");
    }
    bool stretched = false;
    for (int d = 0; d < 3; d++) {
        if (!g->xf[d]) continue;
        stretched = true;
        for (int i = 0; i < g->n[d] + 2 * g->ng; i++)
            if (!std::isfinite(g->xf[d][i]) || !std::isfinite(g->xf[d][i + 1]) || !(g->xf[d][i + 1] > g->xf[d][i]))
                return fail(nullptr, RAD_EINVAL, "rad_create: xf must be finite and strictly increasing");
    }
    if (stretched && m->kind == 2) return fail(nullptr, RAD_EINVAL, "rad_create: a tabulated metric carries its own positions: xf must be NULL");
    if (m->kind < 0 || m->kind > 2) return fail(nullptr, RAD_EINVAL, "rad_create: bad metric kind");
    if (m->kind == 1 && (!finite_pos(m->M) || !std::isfinite(m->a) || std::fabs(m->a) > m->M)) return fail(nullptr, RAD_EINVAL, "rad_create: bad M or a");
    if (m->kind == 2 && (!m->cell_tab || !m->face_tab)) return fail(nullptr, RAD_EINVAL, "rad_create: tabulated metric needs cell_tab and face_tab");
    if (!(p->gamma_gas > 1.0) || !std::isfinite(p->gamma_gas) || !std::isfinite(p->a_rad) || p->a_rad < 0.0 || !std::isfinite(p->n0_crit))
        return fail(nullptr, RAD_EINVAL, "rad_create: bad gamma_gas / a_rad / n0_crit");
    if (p->recon_space < 0 || p->recon_space > 2) return fail(nullptr, RAD_EINVAL, "rad_create: recon_space must be 0 (DC), 1 (PLM) or 2 (PPM)");
    if (p->recon_space == 2 && g->ng < 3) return fail(nullptr, RAD_EINVAL, "rad_create: PPM needs ng = 3");
    if (p->recon_angle < 0 || p->recon_angle > 1) return fail(nullptr, RAD_EINVAL, "rad_create: recon_angle must be 0 (DC) or 1 (lat-lon PLM)");
    if (p->recon_angle == 1 && (a->kind != 0 || (a->npsi & 1)))
        return fail(nullptr, RAD_EUNSUPPORTED, "rad_create: PLM in angle needs a latitude-longitude grid with even npsi (MAPR on the geodesic grid is not implemented)");
    if (!std::isfinite(p->tau_factor) || p->tau_factor < 0.0) return fail(nullptr, RAD_EINVAL, "rad_create: tau_factor must be finite and >= 0");
    if (p->tau_factor != 0.0 && (!o || !o->alpha_a_energy || !o->alpha_s)) return fail(nullptr, RAD_EINVAL, "rad_create: tau_factor != 0 needs opacities");
    if (p->couple && (!o || !o->alpha_a_planck || !o->alpha_a_energy || !o->alpha_s)) return fail(nullptr, RAD_EINVAL, "rad_create: coupling needs opacities");

    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) {
        cudaGetLastError();
        return fail(nullptr, RAD_ECUDA, "rad_create: no usable CUDA device (there is no CPU fallback)");
    }
    DeviceGuard guard(device);
    if (!guard.ok) return cuda_fail(nullptr, "rad_create: cudaSetDevice");

    rad_ctx *c = new (std::nothrow) rad_ctx;
    if (!c) return fail(nullptr, RAD_ENOMEM, "rad_create: out of host memory");
    c->device = device; c->metric = *m; c->grid = *g; c->angles = *a; c->params = *p;
    if (o) c->opac = *o;
    c->kp.gamma_gas = p->gamma_gas; c->kp.a_rad = p->a_rad; c->kp.n0_crit = p->n0_crit; c->kp.rgm1 = 1.0 / (p->gamma_gas - 1.0); c->kp.tau_factor = p->tau_factor;
    c->kp.recon_space = p->recon_space; c->kp.renorm = p->renorm_fluid_weights; c->kp.couple = p->couple;
    c->kp.vel_estimate = p->vel_estimate;
    std::string err;
    bool ok = (a->kind == 0) ? rad::build_latlon(a->nzeta, a->npsi, c->host, err)
            : (a->kind == 1) ? rad::build_geodesic(a->nlev, c->host, err)
            : (a->kind == 2) ? rad::build_explicit(a->nang, a->nhat, a->domega, a->nnbr, a->nbr, a->edge_len, a->edge_mid, a->edge_nrm, c->host, err)
                             : (err = "bad angle grid kind", false);
    if (!ok) { delete c; return fail(nullptr, RAD_EINVAL, "rad_create: " + err); }

    c->angles.nhat = c->angles.domega = c->angles.edge_len = c->angles.edge_mid = c->angles.edge_nrm = nullptr;  // the caller's tables are not kept
    c->angles.nnbr = c->angles.nbr = nullptr;
    rad::DeviceTables &t = c->dev;
    const rad::AngleTables &h = c->host;
    t.N = h.N; t.E = h.E; t.ng = g->ng;
    t.recon_angle = p->recon_angle; t.nzeta = a->kind == 0 ? a->nzeta : 0; t.npsi = a->kind == 0 ? a->npsi : 0;
    // reflecting walls (R20): the angle whose direction is n-hat with component a flipped, for every axis that has such a wall
    std::vector<int> mirror((size_t)3 * h.N, 0);
    bool any_wall = false;
    for (int d = 0; d < 3; d++) {
        if (g->bc_lo[d] != 3 && g->bc_hi[d] != 3) continue;
        any_wall = true;
        for (int n = 0; n < h.N; n++) {
            double want[3] = {h.nhat[3 * n], h.nhat[3 * n + 1], h.nhat[3 * n + 2]};
            want[d] = -want[d];
            int found = -1;
            for (int m = 0; m < h.N && found < 0; m++)
                if (std::fabs(h.nhat[3 * m] - want[0]) < 1e-12 && std::fabs(h.nhat[3 * m + 1] - want[1]) < 1e-12 && std::fabs(h.nhat[3 * m + 2] - want[2]) < 1e-12) found = m;
            if (found < 0) { delete c; return fail(nullptr, RAD_EUNSUPPORTED, "rad_create: reflecting wall: the angle grid is not symmetric under the flip of that direction component"); }
            mirror[(size_t)d * h.N + n] = found;
        }
    }
    for (int d = 0; d < 3; d++) { t.n[d] = g->n[d]; t.inv_dx[d] = 1.0 / g->dx[d]; t.xf[d] = nullptr; t.inv_w[d] = nullptr; }
    c->grid.xf[0] = c->grid.xf[1] = c->grid.xf[2] = nullptr;  // the caller's arrays are not kept
    for (int d = 0; d < 3 && ok; d++) {
        if (!g->xf[d]) continue;
        const int m = g->n[d] + 2 * g->ng;
        std::vector<double> f(g->xf[d], g->xf[d] + m + 1), iw(m);
        for (int i = 0; i < m; i++) iw[i] = 1.0 / (f[i + 1] - f[i]);
        ok = upload(c, f, &t.xf[d]) && upload(c, iw, &t.inv_w[d]);
    }
    t.NI = g->n[0] + 2 * g->ng; t.NJ = g->n[1] + 2 * g->ng; t.NK = g->n[2] + 2 * g->ng;
    if (cudaDeviceGetAttribute(&t.sms, cudaDevAttrMultiProcessorCount, device) != cudaSuccess ||
        cudaDeviceGetAttribute(&t.smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, device) != cudaSuccess) {
        delete c;
        return cuda_fail(nullptr, "rad_create: device attributes");
    }
    t.ncell = (long long)t.NI * t.NJ * t.NK;
    // derived angle tables: pinned products T[e][c][k] = N^c * (n^alpha n^beta), and per-angle signed edge weights
    std::vector<double> edge_T((size_t)h.E * 30), nbr_w((size_t)h.N * RAD_MAXNBR, 0.0);
    for (int e = 0; e < h.E; e++) {
        const double n4[4] = {1.0, h.edge_mid[3 * e], h.edge_mid[3 * e + 1], h.edge_mid[3 * e + 2]};
        double q[10];
        int w = 0;
        for (int al = 0; al < 4; al++) for (int be = al; be < 4; be++) q[w++] = n4[al] * n4[be];
        for (int ch = 0; ch < 3; ch++) for (int k = 0; k < 10; k++) edge_T[(size_t)e * 30 + ch * 10 + k] = h.edge_nrm[3 * e + ch] * q[k];
    }
    for (int n = 0; n < h.N; n++)
        for (int s = 0; s < RAD_MAXNBR; s++) {
            const int e = h.nbr_edge[n * RAD_MAXNBR + s];
            if (e >= 0) nbr_w[n * RAD_MAXNBR + s] = (h.edge_lo[e] == n ? 1.0 : -1.0) / h.domega[n];
        }
    std::vector<double> nhat_t((size_t)3 * h.N), nbr_w_t((size_t)RAD_MAXNBR * h.N);
    std::vector<int> nbr_edge_t((size_t)RAD_MAXNBR * h.N);
    for (int n = 0; n < h.N; n++) {
        for (int d = 0; d < 3; d++) nhat_t[(size_t)d * h.N + n] = h.nhat[3 * n + d];
        for (int s = 0; s < RAD_MAXNBR; s++) {
            nbr_edge_t[(size_t)s * h.N + n] = h.nbr_edge[n * RAD_MAXNBR + s];
            nbr_w_t[(size_t)s * h.N + n] = nbr_w[n * RAD_MAXNBR + s];
        }
    }
    ok = ok && upload(c, nhat_t, &t.nhat_t) && upload(c, nbr_edge_t, &t.nbr_edge_t) && upload(c, nbr_w_t, &t.nbr_w_t);
    ok = ok && upload(c, h.nhat, &t.nhat) && upload(c, h.domega, &t.domega) && upload(c, h.nnbr, &t.nnbr) && upload(c, h.nbr_edge, &t.nbr_edge) &&
         upload(c, h.edge_lo, &t.edge_lo) && upload(c, h.edge_hi, &t.edge_hi) && upload(c, h.edge_len, &t.edge_len) &&
         upload(c, h.edge_mid, &t.edge_mid) && upload(c, edge_T, &t.edge_T) && upload(c, nbr_w, &t.nbr_w);
    t.mirror = nullptr;
    if (ok && any_wall) ok = upload(c, mirror, &t.mirror);
    // tile kernel (stage5.cu): balanced and coloured edge ownership, per-angle records, 1/dOmega
    t.fused_ok = 0; t.ang_rec = nullptr; t.winv = nullptr; t.own_edge = nullptr; t.ke = nullptr; t.rec = nullptr;
    const bool tile_cfg = g->ng == 2 && p->recon_space <= 1 && p->recon_angle == 0 && !stretched;  // what the tile kernel (stage5.cu) implements
    if (ok && h.N <= 256 && tile_cfg) {
        std::string oerr;
        if (rad::build_edge_ownership(h, c->own, oerr)) {
            std::vector<short> rec((size_t)h.N * 8, 0);
            std::vector<double> winv(h.N);
            for (int n = 0; n < h.N; n++) {
                for (int q = 0; q < 3; q++) {  // unused slots: partner 0 (its q_e is 0) and the always-zero flux slot 3N
                    const int pa = c->own.own_partner[(size_t)n * 3 + q], pu = c->own.pull_pos[(size_t)n * 3 + q];
                    rec[(size_t)n * 8 + q] = (short)(unsigned short)(8 * (pa >= 0 ? pa : 0));          // byte offsets in a row of doubles
                    rec[(size_t)n * 8 + 3 + q] = (short)(unsigned short)(8 * (pu >= 0 ? pu : 3 * h.N));
                }
                winv[n] = 1.0 / h.domega[n];
            }
            ok = upload(c, rec, &t.ang_rec) && upload(c, winv, &t.winv) && upload(c, c->own.own_edge, &t.own_edge);
            t.fused_ok = ok ? 1 : 0;
        }
    }
    double *cell = nullptr, *face = nullptr;
    if (ok) ok = cudaMalloc((void **)&cell, sizeof(double) * t.ncell * RAD_NCELL) == cudaSuccess;
    if (ok) c->owned.push_back(cell);
    if (ok) ok = cudaMalloc((void **)&face, sizeof(double) * t.ncell * 3 * RAD_NFACE) == cudaSuccess;
    if (ok) c->owned.push_back(face);
    if (ok) ok = cudaMalloc((void **)&c->d_noroot, sizeof(unsigned long long)) == cudaSuccess;
    if (ok) c->owned.push_back(c->d_noroot);
    if (!ok) {
        cudaError_t e = cudaGetLastError();
        std::string msg = std::string("rad_create: device allocation/upload failed: ") + cudaGetErrorString(e);
        rad_destroy(c);
        return fail(nullptr, e == cudaErrorMemoryAllocation ? RAD_ENOMEM : RAD_ECUDA, msg);
    }
    t.cell = cell; t.face = face;
    if (m->kind == 2) {
        ok = cudaMemcpy(cell, m->cell_tab, sizeof(double) * t.ncell * RAD_NCELL, cudaMemcpyDeviceToDevice) == cudaSuccess &&
             cudaMemcpy(face, m->face_tab, sizeof(double) * t.ncell * 3 * RAD_NFACE, cudaMemcpyDeviceToDevice) == cudaSuccess;
    } else {
        int nl = rad::launch_geometry(*m, *g, t.xf, cell, face, t.ncell, 0);
        ok = nl > 0 && cudaDeviceSynchronize() == cudaSuccess;
        if (ok) c->launches += nl;
    }
    if (!ok) {
        std::string msg = std::string("rad_create: geometry: ") + cudaGetErrorString(cudaGetLastError());
        rad_destroy(c);
        return fail(nullptr, RAD_ECUDA, msg);
    }
    c->metric.cell_tab = nullptr; c->metric.face_tab = nullptr;
    if (p->vel_estimate && p->couple && !rad::stream_serves(t, nullptr)) {
        rad_destroy(c);
        return fail(nullptr, RAD_EUNSUPPORTED, "rad_create: vel_estimate needs an even number of angles that fits the streaming coupling kernel's shared memory");
    }
    // stored edge coefficients q_e per (interior cell, owned edge): 3 N doubles per cell
    if (t.fused_ok && !p->recompute_edge_coeffs) {
        const size_t bytes = sizeof(double) * (size_t)g->n[0] * g->n[1] * g->n[2] * 3 * h.N;
        if (cudaMalloc((void **)&c->ke, bytes) != cudaSuccess) {
            cudaGetLastError();
            rad_destroy(c);
            return fail(nullptr, RAD_ENOMEM, "rad_create: no device memory for the stored edge coefficients (set recompute_edge_coeffs = 1)");
        }
        int nl = rad::launch_build_ke(t, c->ke, 0);
        if (nl < 0 || cudaDeviceSynchronize() != cudaSuccess) {
            std::string msg = std::string("rad_create: edge coefficients: ") + cudaGetErrorString(cudaGetLastError());
            rad_destroy(c);
            return fail(nullptr, RAD_ECUDA, msg);
        }
        c->launches += nl;
        t.ke = c->ke;
        // packed per-cell records of the angle-resident stage kernel (stage5.cu)
        if (cudaMalloc((void **)&c->rec, sizeof(double) * (size_t)t.ncell * RAD_STAGE_RECN) == cudaSuccess) {
            nl = rad::launch_pack_rec(t, c->rec, 0);
            if (nl < 0 || cudaDeviceSynchronize() != cudaSuccess) {
                std::string msg = std::string("rad_create: stage records: ") + cudaGetErrorString(cudaGetLastError());
                rad_destroy(c);
                return fail(nullptr, RAD_ECUDA, msg);
            }
            c->launches += nl;
            t.rec = c->rec;
        } else {
            cudaGetLastError();  // not fatal: without the records the generic flux-divergence kernel (transport.cu) serves the context
        }
    }
    *out = c;
    return RAD_OK;
}

void rad_destroy(rad_ctx *c) {
    if (!c) return;
    DeviceGuard guard(c->device);
    for (void *p : c->owned) cudaFree(p);
    for (int q = 0; q < 2; q++) if (c->scratch_I[q]) cudaFree(c->scratch_I[q]);
    if (c->scratch_small) cudaFree(c->scratch_small);
    for (int q = 0; q < 3; q++) if (c->hs[q]) cudaStreamDestroy(c->hs[q]);
    if (c->ke) cudaFree(c->ke);
    if (c->rec) cudaFree(c->rec);
    if (c->vel) cudaFree(c->vel);
    if (c->vel8) cudaFree(c->vel8);
    delete c;
}

const char *rad_last_error(const rad_ctx *c) { return c ? c->err.c_str() : g_create_err.c_str(); }
long long rad_ncells_total(const rad_ctx *c) { return c ? c->dev.ncell : 0; }
long long rad_launch_count(const rad_ctx *c) { return c ? c->launches : 0; }

rad_status rad_fill_ghosts(rad_ctx *c, double *I, void *stream) {
    if (!c || !I) return fail(c, RAD_EINVAL, "rad_fill_ghosts: NULL argument");
    DeviceGuard guard(c->device);
    int nl = rad::launch_fill_ghosts(c->dev, c->grid.bc_lo, c->grid.bc_hi, I, (cudaStream_t)stream);
    if (nl < 0) return cuda_fail(c, "rad_fill_ghosts");
    c->launches += nl;
    return RAD_OK;
}

rad_status rad_edge_ownership(const rad_angles *a, int *nang, int *nedge, int *edge_lo, int *edge_hi, int *own_edge, int *own_partner, int *pull_pos,
                              size_t capacity) {
    if (!a || !nang || !nedge) return fail(nullptr, RAD_EINVAL, "rad_edge_ownership: NULL argument");
    rad::AngleTables h;
    rad::EdgeOwnership o;
    std::string err;
    const bool ok = (a->kind == 0) ? rad::build_latlon(a->nzeta, a->npsi, h, err)
                  : (a->kind == 1) ? rad::build_geodesic(a->nlev, h, err)
                  : (a->kind == 2) ? rad::build_explicit(a->nang, a->nhat, a->domega, a->nnbr, a->nbr, a->edge_len, a->edge_mid, a->edge_nrm, h, err)
                                   : (err = "bad angle grid kind", false);
    if (!ok) return fail(nullptr, RAD_EINVAL, "rad_edge_ownership: " + err);
    *nang = h.N; *nedge = h.E;
    if (!rad::build_edge_ownership(h, o, err)) return fail(nullptr, RAD_EUNSUPPORTED, "rad_edge_ownership: " + err);
    if (!edge_lo && !edge_hi && !own_edge && !own_partner && !pull_pos) return RAD_OK;  // sizes only
    if ((size_t)h.E > capacity || (size_t)3 * h.N > capacity) return fail(nullptr, RAD_EINVAL, "rad_edge_ownership: capacity too small");
    if (edge_lo) memcpy(edge_lo, h.edge_lo.data(), sizeof(int) * h.E);
    if (edge_hi) memcpy(edge_hi, h.edge_hi.data(), sizeof(int) * h.E);
    if (own_edge) memcpy(own_edge, o.own_edge.data(), sizeof(int) * 3 * h.N);
    if (own_partner) memcpy(own_partner, o.own_partner.data(), sizeof(int) * 3 * h.N);
    if (pull_pos) memcpy(pull_pos, o.pull_pos.data(), sizeof(int) * 3 * h.N);
    return RAD_OK;
}

rad_status rad_exchange_halo(rad_ctx *lo, double *I_lo, rad_ctx *hi, double *I_hi, int axis, void *stream) {
    if (!lo || !hi || !I_lo || !I_hi) return fail(lo ? lo : hi, RAD_EINVAL, "rad_exchange_halo: NULL argument");
    if (axis < 0 || axis > 2) return fail(lo, RAD_EINVAL, "rad_exchange_halo: axis must be 0, 1 or 2");
    const rad::DeviceTables &a = lo->dev, &b = hi->dev;
    if (lo->device != hi->device || a.N != b.N || a.ng != b.ng) return fail(lo, RAD_EINVAL, "rad_exchange_halo: the blocks differ in device, angle count or ghost depth");
    for (int d = 0; d < 3; d++)
        if (d != axis && a.n[d] != b.n[d]) return fail(lo, RAD_EINVAL, "rad_exchange_halo: the blocks differ in an extent across the axis");
    if (a.n[axis] < a.ng || b.n[axis] < b.ng) return fail(lo, RAD_EINVAL, "rad_exchange_halo: a block is thinner than the ghost depth");
    if (I_lo == I_hi) return fail(lo, RAD_EINVAL, "rad_exchange_halo: the two blocks share an array");
    DeviceGuard guard(lo->device);
    const int nl = rad::launch_exchange_halo(a, I_lo, b, I_hi, axis, (cudaStream_t)stream);
    if (nl < 0) return cuda_fail(lo, "rad_exchange_halo");
    lo->launches += nl;
    return RAD_OK;
}

// The two halves of a stage on one stream (no argument checks: the callers did them).
// transport: ghost fill, then the tile kernel (stage5.cu) where it serves the context, else the generic flux-divergence kernel
// (transport.cu).  `fluid` != nullptr with tau_factor != 0 selects the optical-depth-aware flux (Eq.26-29).
static rad_status run_transport(rad_ctx *c, double *I_in, double *I_out, const double *I0, const double *fluid, double gam0, double gam1,
                                double beta_dt, cudaStream_t s, int kz0 = 0, int kz1 = 0, bool fill = true) {
    if (fill) {
        rad_status st = rad_fill_ghosts(c, I_in, s);
        if (st != RAD_OK) return st;
    }
    const bool tau = c->kp.tau_factor != 0.0;
    rad::StageArgs a{};
    a.I_in = I_in; a.I0 = I0; a.I_out = I_out; a.gam0 = gam0; a.gam1 = gam1; a.beta_dt = beta_dt; a.kz0 = kz0; a.kz1 = kz1;
    if (rad::stage_angle_serves(c->dev, tau)) {  // decided once: the table below is built for the kernel that will read it
        if (tau) {  // per-cell table {u^alphahat, f/2 of the upper faces}
            if (!c->vel8 && cudaMalloc((void **)&c->vel8, sizeof(double) * 8 * (size_t)c->dev.ncell) != cudaSuccess) {
                cudaGetLastError();
                return fail(c, RAD_ENOMEM, "rad_stage: no device memory for the velocity table");
            }
            const int nt = rad::launch_tau_table(c->dev, fluid, c->opac.alpha_a_energy, c->opac.alpha_s, c->kp.tau_factor * beta_dt, c->vel8, s);
            if (nt < 0) return cuda_fail(c, "rad_stage (velocity table)");
            c->launches += nt;
            a.vel8 = c->vel8;
        }
        const int nl = rad::launch_stage_angle(c->dev, c->kp, a, s);
        if (nl < 0) return cuda_fail(c, "rad_stage (tile kernel)");
        if (nl > 0) { c->launches += nl; return RAD_OK; }
    }
    if (kz1 > kz0) return fail(c, RAD_EUNSUPPORTED, "slab-wise transport needs the tile kernel");
    const double *vel = nullptr;
    if (tau) {  // generic path: per-cell {u^alphahat, alpha_E}
        if (!c->vel && cudaMalloc((void **)&c->vel, sizeof(double) * 5 * (size_t)c->dev.ncell) != cudaSuccess) {
            cudaGetLastError();
            return fail(c, RAD_ENOMEM, "rad_stage: no device memory for the velocity table");
        }
        const int nv = rad::launch_cell_velocity(c->dev, fluid, c->opac.alpha_a_energy, c->opac.alpha_s, c->vel, s);
        if (nv < 0) return cuda_fail(c, "rad_stage (velocity table)");
        c->launches += nv;
        vel = c->vel;
    }
    const int nl = rad::launch_fluxdiv(c->dev, c->kp, I_in, I0, gam0, gam1, beta_dt, I_out, s, vel, c->kp.tau_factor * beta_dt);
    if (nl < 0) return cuda_fail(c, "rad_stage (flux divergence)");
    c->launches += nl;
    return RAD_OK;
}

// coupling + mask + fluid increment in place on I: the streaming kernel (stream.cu) where it serves, else the generic one (coupling.cu)
static rad_status run_coupling(rad_ctx *c, double *I, const double *fluid, double dt, double *T_out, double *dT0, bool count, cudaStream_t s,
                               int kz0 = 0, int kz1 = 0) {
    unsigned long long *cnt = count ? c->d_noroot : nullptr;
    int nl = rad::launch_couple_stream(c->dev, c->kp, I, fluid, c->opac.alpha_a_planck, c->opac.alpha_a_energy, c->opac.alpha_s, dt, T_out, dT0, cnt, s, kz0, kz1);
    if (nl == 0 && kz1 > kz0) return fail(c, RAD_EUNSUPPORTED, "slab-wise coupling needs the streaming kernel");
    if (nl == 0 && c->kp.vel_estimate && c->kp.couple)
        return fail(c, RAD_EUNSUPPORTED, "the velocity estimate (Eq.51-55) runs in the streaming coupling kernel: it needs a 16-byte aligned intensity array");
    if (nl == 0) nl = rad::launch_coupling(c->dev, c->kp, I, fluid, c->opac.alpha_a_planck, c->opac.alpha_a_energy, c->opac.alpha_s, dt, T_out, dT0, cnt, s);
    if (nl < 0) return cuda_fail(c, "rad_couple");
    c->launches += nl;
    return RAD_OK;
}

rad_status rad_transport(rad_ctx *c, double *I_in, double *I_out, const double *I0, double gam0, double gam1, double beta_dt, void *stream) {
    if (!c || !I_in || !I_out) return fail(c, RAD_EINVAL, "rad_transport: NULL argument");
    if (I_in == I_out || I0 == I_out) return fail(c, RAD_EINVAL, "rad_transport: I_out must not alias I_in or I0 (the stencil reads old values)");
    if (!std::isfinite(gam0) || !std::isfinite(gam1) || !std::isfinite(beta_dt)) return fail(c, RAD_EINVAL, "rad_transport: non-finite weights");
    if (c->kp.tau_factor != 0.0) return fail(c, RAD_ESTATE, "rad_transport: with tau_factor != 0 the spatial flux needs the fluid state (Eq.26-29): use rad_stage");
    DeviceGuard guard(c->device);
    return run_transport(c, I_in, I_out, I0, nullptr, gam0, gam1, beta_dt, (cudaStream_t)stream);
}

rad_status rad_couple(rad_ctx *c, double *I, const double *fluid, double dt, double *T_out, double *dT0, long long *n_noroot, void *stream) {
    if (!c || !I || !fluid) return fail(c, RAD_EINVAL, "rad_couple: NULL argument");
    if (!std::isfinite(dt)) return fail(c, RAD_EINVAL, "rad_couple: non-finite dt");
    if (c->kp.couple && (!c->opac.alpha_a_planck || !c->opac.alpha_a_energy || !c->opac.alpha_s)) return fail(c, RAD_ESTATE, "rad_couple: context has no opacities");
    DeviceGuard guard(c->device);
    cudaStream_t s = (cudaStream_t)stream;
    if (n_noroot && cudaMemsetAsync(c->d_noroot, 0, sizeof(unsigned long long), s) != cudaSuccess) return cuda_fail(c, "rad_couple: memset");
    rad_status st = run_coupling(c, I, fluid, dt, T_out, dT0, n_noroot != nullptr, s);
    if (st != RAD_OK) return st;
    return read_noroot(c, n_noroot, s, "rad_couple: readback");
}

rad_status rad_stage(rad_ctx *c, double *I_in, double *I_out, const double *I0, const double *fluid, double gam0, double gam1,
                     double beta_dt, double *T_out, double *dT0, long long *n_noroot, void *stream) {
    if (!c || !fluid || !I_in || !I_out) return fail(c, RAD_EINVAL, "rad_stage: NULL argument");
    if (I_in == I_out || I0 == I_out) return fail(c, RAD_EINVAL, "rad_stage: I_out must not alias I_in or I0 (the stencil reads old values)");
    if (!std::isfinite(gam0) || !std::isfinite(gam1) || !std::isfinite(beta_dt)) return fail(c, RAD_EINVAL, "rad_stage: non-finite weights");
    if ((c->kp.couple || c->kp.tau_factor != 0.0) && (!c->opac.alpha_a_planck || !c->opac.alpha_a_energy || !c->opac.alpha_s))
        return fail(c, RAD_ESTATE, "rad_stage: context has no opacities");
    DeviceGuard guard(c->device);
    cudaStream_t s = (cudaStream_t)stream;
    if (n_noroot && cudaMemsetAsync(c->d_noroot, 0, sizeof(unsigned long long), s) != cudaSuccess) return cuda_fail(c, "rad_stage: memset");
    rad_status st = run_transport(c, I_in, I_out, I0, fluid, gam0, gam1, beta_dt, s);
    if (st != RAD_OK) return st;
    st = run_coupling(c, I_out, fluid, beta_dt, T_out, dT0, n_noroot != nullptr, s);
    if (st != RAD_OK) return st;
    return read_noroot(c, n_noroot, s, "rad_stage: readback");
}

// rad_stage_host, pipelined: the block is cut into slabs of planes along z; while slab j is computed, the input planes of
// slab j+1 travel host -> device and the output planes of slab j-1 device -> host (three streams, PCIe in both directions at
// once).  Used when the angle-resident stage kernel serves the context and all boundaries are caller-filled (a periodic or
// outflow fill in z needs the far end of the array first).  Returns RAD_EUNSUPPORTED if it does not apply.
static rad_status stage_host_pipelined(rad_ctx *c, const double *I_in_host, double *I_out_host, const double *fluid_host, const double *opac_host,
                                       double gam0, double gam1, double beta_dt, double *T_out_host, double *dT0_host, long long *n_noroot) {
    const rad::DeviceTables &t = c->dev;
    if (!rad::stage_angle_serves(t) || !rad::stream_serves(t, c->scratch_I[1]) || c->kp.tau_factor != 0.0) return RAD_EUNSUPPORTED;
    for (int d = 0; d < 3; d++)
        if (c->grid.bc_lo[d] != 0 || c->grid.bc_hi[d] != 0) return RAD_EUNSUPPORTED;
    const int nz = t.n[2], ng = t.ng;
    if (nz < 8) return RAD_EUNSUPPORTED;
    cudaStream_t *st = c->hs;
    for (int q = 0; q < 3; q++)
        if (!st[q] && cudaStreamCreateWithFlags(&st[q], cudaStreamNonBlocking) != cudaSuccess) return cuda_fail(c, "rad_stage_host: stream");
    const long long nc = t.ncell, plane = (long long)t.NI * t.NJ;  // cells per z plane
    const size_t pbytes = sizeof(double) * plane * t.N;
    double *dI = c->scratch_I[0], *dO = c->scratch_I[1];
    double *dfl = c->scratch_small, *dop = dfl + 5 * nc, *dT = dop + 3 * nc, *ddT0 = dT + nc;
    int nslab = (nz + 7) / 8;  // thin slabs: the first copy-in and the last copy-out are not overlapped
    if (nslab > 48) nslab = 48;
    const int per = (((nz + nslab - 1) / nslab) + 11) / 12 * 12;  // planes per slab, a multiple of every tile height (TZ = 2, 3)
    nslab = (nz + per - 1) / per;
    std::vector<cudaEvent_t> evH(nslab, nullptr), evK(nslab, nullptr);
    cudaEvent_t ev0 = nullptr;
    bool ok = cudaEventCreateWithFlags(&ev0, cudaEventDisableTiming) == cudaSuccess;
    for (int j = 0; j < nslab && ok; j++)
        ok = cudaEventCreateWithFlags(&evH[j], cudaEventDisableTiming) == cudaSuccess && cudaEventCreateWithFlags(&evK[j], cudaEventDisableTiming) == cudaSuccess;
    // the caller's earlier work on these buffers (legacy default stream) is ordered before the pipeline
    ok = ok && cudaEventRecord(ev0, 0) == cudaSuccess;
    for (int q = 0; q < 3 && ok; q++) ok = cudaStreamWaitEvent(st[q], ev0, 0) == cudaSuccess;
    if (ok && n_noroot) ok = cudaMemsetAsync(c->d_noroot, 0, sizeof(unsigned long long), st[1]) == cudaSuccess;
    const rad_opac saved = c->opac;
    c->opac.alpha_a_planck = dop; c->opac.alpha_a_energy = dop + nc; c->opac.alpha_s = dop + 2 * nc;
    bool launch_failed = false;
    int p_done = 0;  // array planes [0, p_done) are on their way to the device
    for (int j = 0; j < nslab && ok; j++) {
        const int kb = j * per, ke = kb + per < nz ? kb + per : nz;      // interior planes of the slab
        const int need = (j == nslab - 1) ? t.NK : ke + 2 * ng;          // array planes [0, need) must be resident: interior plane k is array plane k + ng
        if (need > p_done) {
            ok = cudaMemcpyAsync(dI + (size_t)p_done * plane * t.N, I_in_host + (size_t)p_done * plane * t.N, pbytes * (need - p_done), cudaMemcpyHostToDevice, st[0]) == cudaSuccess;
            p_done = need;
        }
        {   // fluid and opacities of the slab's own planes (read for interior cells only)
            const size_t fo = (size_t)(kb + ng) * plane, fb = sizeof(double) * plane * (ke - kb);
            for (int m = 0; m < 5 && ok; m++) ok = cudaMemcpyAsync(dfl + m * nc + fo, fluid_host + m * nc + fo, fb, cudaMemcpyHostToDevice, st[0]) == cudaSuccess;
            for (int m = 0; m < 3 && ok && opac_host; m++) ok = cudaMemcpyAsync(dop + m * nc + fo, opac_host + m * nc + fo, fb, cudaMemcpyHostToDevice, st[0]) == cudaSuccess;
        }
        ok = ok && cudaEventRecord(evH[j], st[0]) == cudaSuccess && cudaStreamWaitEvent(st[1], evH[j], 0) == cudaSuccess;
        // output planes of this slab start as a copy of the input (only interior cells are written by the stage: the ghost
        // cells of the returned array are those of the input); the ghost planes below / above go with the first / last slab
        const int ob = (j == 0) ? 0 : kb + ng, oe = (j == nslab - 1) ? t.NK : ke + ng;
        ok = ok && cudaMemcpyAsync(dO + (size_t)ob * plane * t.N, dI + (size_t)ob * plane * t.N, pbytes * (oe - ob), cudaMemcpyDeviceToDevice, st[1]) == cudaSuccess;
        if (!ok) break;
        // the slab's stage: flux divergence in the tile kernel, then the streaming coupling
        if (run_transport(c, dI, dO, nullptr, dfl, gam0, gam1, beta_dt, st[1], kb, ke, false) != RAD_OK ||
            run_coupling(c, dO, dfl, beta_dt, dT, ddT0, n_noroot != nullptr, st[1], kb, ke) != RAD_OK) { launch_failed = true; break; }
        ok = cudaEventRecord(evK[j], st[1]) == cudaSuccess && cudaStreamWaitEvent(st[2], evK[j], 0) == cudaSuccess;
        ok = ok && cudaMemcpyAsync(I_out_host + (size_t)ob * plane * t.N, dO + (size_t)ob * plane * t.N, pbytes * (oe - ob), cudaMemcpyDeviceToHost, st[2]) == cudaSuccess;
        const size_t cb = sizeof(double) * plane * (oe - ob), co = (size_t)ob * plane;
        if (ok && T_out_host) ok = cudaMemcpyAsync(T_out_host + co, dT + co, cb, cudaMemcpyDeviceToHost, st[2]) == cudaSuccess;
        for (int m = 0; m < 4 && ok && dT0_host; m++) ok = cudaMemcpyAsync(dT0_host + m * nc + co, ddT0 + m * nc + co, cb, cudaMemcpyDeviceToHost, st[2]) == cudaSuccess;
    }
    c->opac = saved;
    unsigned long long v = 0;
    if (ok && n_noroot) ok = cudaMemcpyAsync(&v, c->d_noroot, sizeof(v), cudaMemcpyDeviceToHost, st[2]) == cudaSuccess;
    for (int q = 0; q < 3; q++) ok = (cudaStreamSynchronize(st[q]) == cudaSuccess) && ok;
    for (int j = 0; j < nslab; j++) { if (evH[j]) cudaEventDestroy(evH[j]); if (evK[j]) cudaEventDestroy(evK[j]); }
    if (ev0) cudaEventDestroy(ev0);
    if (launch_failed) return RAD_ECUDA;  // text already set by the failing launch
    if (!ok) return cuda_fail(c, "rad_stage_host: pipelined copies");
    if (n_noroot) *n_noroot = (long long)v;
    return RAD_OK;
}

rad_status rad_stage_host(rad_ctx *c, const double *I_in_host, double *I_out_host, const double *fluid_host, const double *opac_host,
                          double gam0, double gam1, double beta_dt, double *T_out_host, double *dT0_host, long long *n_noroot) {
    if (!c || !I_in_host || !I_out_host || !fluid_host) return fail(c, RAD_EINVAL, "rad_stage_host: NULL argument");
    if (c->kp.couple && !opac_host) return fail(c, RAD_EINVAL, "rad_stage_host: coupling needs opac_host");
    if (!std::isfinite(gam0) || !std::isfinite(gam1) || !std::isfinite(beta_dt)) return fail(c, RAD_EINVAL, "rad_stage_host: non-finite weights");
    DeviceGuard guard(c->device);
    const long long nc = c->dev.ncell;
    const size_t ibytes = sizeof(double) * nc * c->dev.N, cb = sizeof(double) * nc;
    for (int q = 0; q < 2; q++)
        if (!c->scratch_I[q] && cudaMalloc((void **)&c->scratch_I[q], ibytes) != cudaSuccess) return fail(c, RAD_ENOMEM, "rad_stage_host: device scratch");
    if (!c->scratch_small) {
        if (cudaMalloc((void **)&c->scratch_small, 13 * cb) != cudaSuccess) return fail(c, RAD_ENOMEM, "rad_stage_host: device scratch");
        if (cudaMemset(c->scratch_small, 0, 13 * cb) != cudaSuccess) return cuda_fail(c, "rad_stage_host: memset");  // ghost entries of T_out / dT0 are returned as 0
    }
    if (c->kp.couple || opac_host) {
        if (opac_host) {
            const rad_status ps = stage_host_pipelined(c, I_in_host, I_out_host, fluid_host, opac_host, gam0, gam1, beta_dt, T_out_host, dT0_host, n_noroot);
            if (ps != RAD_EUNSUPPORTED) return ps;
        }
    }
    double *dfl = c->scratch_small, *dop = dfl + 5 * nc, *dT = dop + 3 * nc, *ddT0 = dT + nc;
    cudaStream_t s = 0;
    bool ok = cudaMemcpyAsync(c->scratch_I[0], I_in_host, ibytes, cudaMemcpyHostToDevice, s) == cudaSuccess &&
              cudaMemcpyAsync(dfl, fluid_host, 5 * cb, cudaMemcpyHostToDevice, s) == cudaSuccess;
    if (ok && opac_host) ok = cudaMemcpyAsync(dop, opac_host, 3 * cb, cudaMemcpyHostToDevice, s) == cudaSuccess;
    if (!ok) return cuda_fail(c, "rad_stage_host: H2D");
    // interior-only writes: start I_out from I_in so that ghost cells of the returned array are defined
    if (cudaMemcpyAsync(c->scratch_I[1], c->scratch_I[0], ibytes, cudaMemcpyDeviceToDevice, s) != cudaSuccess) return cuda_fail(c, "rad_stage_host: D2D");
    const rad_opac saved = c->opac;
    c->opac.alpha_a_planck = dop; c->opac.alpha_a_energy = dop + nc; c->opac.alpha_s = dop + 2 * nc;
    rad_status st = rad_stage(c, c->scratch_I[0], c->scratch_I[1], nullptr, dfl, gam0, gam1, beta_dt, dT, ddT0, n_noroot, s);
    c->opac = saved;
    if (st != RAD_OK) return st;
    ok = cudaMemcpyAsync(I_out_host, c->scratch_I[1], ibytes, cudaMemcpyDeviceToHost, s) == cudaSuccess;
    if (ok && T_out_host) ok = cudaMemcpyAsync(T_out_host, dT, cb, cudaMemcpyDeviceToHost, s) == cudaSuccess;
    if (ok && dT0_host) ok = cudaMemcpyAsync(dT0_host, ddT0, 4 * cb, cudaMemcpyDeviceToHost, s) == cudaSuccess;
    if (!ok || cudaStreamSynchronize(s) != cudaSuccess) return cuda_fail(c, "rad_stage_host: D2H");
    return RAD_OK;
}

rad_status rad_moments(rad_ctx *c, const double *I, int frame, const double *fluid, double *out, void *stream) {
    if (!c || !I || !out) return fail(c, RAD_EINVAL, "rad_moments: NULL argument");
    if (frame < 0 || frame > 3) return fail(c, RAD_EINVAL, "rad_moments: frame must be 0..3");
    if (frame == 3 && !fluid) return fail(c, RAD_EINVAL, "rad_moments: fluid frame needs fluid");
    DeviceGuard guard(c->device);
    int nl = rad::launch_moments_stream(c->dev, I, frame, fluid, out, (cudaStream_t)stream);
    if (nl == 0) nl = rad::launch_moments(c->dev, I, frame, fluid, out, (cudaStream_t)stream);
    if (nl < 0) return cuda_fail(c, "rad_moments");
    c->launches += nl;
    return RAD_OK;
}

rad_status rad_stage_kernels(rad_ctx *c, char *buf, size_t nbytes) {
    if (!c || !buf || nbytes == 0) return fail(c, RAD_EINVAL, "rad_stage_kernels: NULL argument");
    char a[96];
    rad::stage_angle_kernel_name(c->dev, c->kp, c->kp.tau_factor != 0.0, a, sizeof a);
    const bool stream = rad::stream_serves(c->dev, nullptr) != 0;
    char b[64];
    const int npass = (c->dev.N + 7) / 8;  // the pass counts the streaming kernel is instantiated for (stream.cu: launch_couple_stream)
    if (!stream) snprintf(b, sizeof b, "k_coupling");
    else if (c->kp.vel_estimate && c->kp.couple) snprintf(b, sizeof b, "k_couple_stream<1,%d>", npass == 21 ? 21 : 0);
    else snprintf(b, sizeof b, "k_couple_stream<0,%d>", (npass == 21 || npass == 12) ? npass : 0);
    const int w = snprintf(buf, nbytes, "%s;%s", a, b);
    if (w < 0 || (size_t)w >= nbytes) return fail(c, RAD_EINVAL, "rad_stage_kernels: buffer too small");
    return RAD_OK;
}

rad_status rad_probe_fp64(rad_ctx *c, double *dfma_per_sec) {
    if (!c || !dfma_per_sec) return fail(c, RAD_EINVAL, "rad_probe_fp64: NULL argument");
    DeviceGuard guard(c->device);
    if (rad::probe_dfma_rate(dfma_per_sec, &c->launches) != 0) return cuda_fail(c, "rad_probe_fp64");
    return RAD_OK;
}

rad_status rad_get_table(rad_ctx *c, int which, void *host_out, size_t nbytes) {
    if (!c || !host_out) return fail(c, RAD_EINVAL, "rad_get_table: NULL argument");
    DeviceGuard guard(c->device);
    const rad::AngleTables &h = c->host;
    const rad::DeviceTables &t = c->dev;
    const void *src = nullptr;
    size_t need = 0;
    int nang = h.N, nedge = h.E;
    switch (which) {
        case RAD_TAB_NANG: src = &nang; need = sizeof(int); break;
        case RAD_TAB_NEDGE: src = &nedge; need = sizeof(int); break;
        case RAD_TAB_NHAT: src = h.nhat.data(); need = sizeof(double) * 3 * h.N; break;
        case RAD_TAB_DOMEGA: src = h.domega.data(); need = sizeof(double) * h.N; break;
        case RAD_TAB_NNBR: src = h.nnbr.data(); need = sizeof(int) * h.N; break;
        case RAD_TAB_NBR: src = h.nbr.data(); need = sizeof(int) * RAD_MAXNBR * h.N; break;
        case RAD_TAB_NBR_EDGE: src = h.nbr_edge.data(); need = sizeof(int) * RAD_MAXNBR * h.N; break;
        case RAD_TAB_EDGE_LO: src = h.edge_lo.data(); need = sizeof(int) * h.E; break;
        case RAD_TAB_EDGE_HI: src = h.edge_hi.data(); need = sizeof(int) * h.E; break;
        case RAD_TAB_EDGE_LEN: src = h.edge_len.data(); need = sizeof(double) * h.E; break;
        case RAD_TAB_EDGE_MID: src = h.edge_mid.data(); need = sizeof(double) * 3 * h.E; break;
        case RAD_TAB_EDGE_NRM: src = h.edge_nrm.data(); need = sizeof(double) * 3 * h.E; break;
        case RAD_TAB_CELL: need = sizeof(double) * t.ncell * RAD_NCELL; break;
        case RAD_TAB_FACE: need = sizeof(double) * t.ncell * 3 * RAD_NFACE; break;
        case RAD_TAB_FACE_SIGN: need = (size_t)t.ncell * 3 * t.N; break;
        case RAD_TAB_EDGE_SIGN: need = (size_t)t.ncell * t.E; break;
        case RAD_TAB_MAXSPEED: need = 3 * sizeof(double); break;
        case RAD_TAB_OWN_EDGE:
            if (!t.fused_ok) return fail(c, RAD_ESTATE, "rad_get_table: this context does not run the tile kernel");
            src = c->own.own_edge.data(); need = sizeof(int) * 3 * h.N; break;
        case RAD_TAB_KE:
            if (!t.ke) return fail(c, RAD_ESTATE, "rad_get_table: this context stores no edge coefficients");
            need = sizeof(double) * (size_t)t.n[0] * t.n[1] * t.n[2] * 3 * h.N; break;
        case RAD_TAB_STAGE_FACE_SIGN:
            if (!t.rec) return fail(c, RAD_ESTATE, "rad_get_table: this context does not run the tile kernel");
            need = (size_t)t.ncell * 3 * t.N; break;
        default: return fail(c, RAD_EINVAL, "rad_get_table: unknown table");
    }
    if (nbytes != need) {
        char buf[128];
        snprintf(buf, sizeof buf, "rad_get_table: table %d has %zu bytes, caller gave %zu", which, need, nbytes);
        return fail(c, RAD_EINVAL, buf);
    }
    if (src) { memcpy(host_out, src, need); return RAD_OK; }
    if (which == RAD_TAB_CELL || which == RAD_TAB_FACE || which == RAD_TAB_KE) {
        const void *dsrc = which == RAD_TAB_CELL ? (const void *)t.cell : (which == RAD_TAB_FACE ? (const void *)t.face : (const void *)t.ke);
        if (cudaMemcpy(host_out, dsrc, need, cudaMemcpyDeviceToHost) != cudaSuccess) return cuda_fail(c, "rad_get_table");
        return RAD_OK;
    }
    void *tmp = nullptr;
    if (cudaMalloc(&tmp, need) != cudaSuccess) { cudaGetLastError(); return fail(c, RAD_ENOMEM, "rad_get_table: device scratch"); }
    int nl = 0;
    if (which == RAD_TAB_FACE_SIGN) nl = rad::launch_sign_tables(t, (signed char *)tmp, nullptr, 0);
    else if (which == RAD_TAB_EDGE_SIGN) nl = rad::launch_sign_tables(t, nullptr, (signed char *)tmp, 0);
    else if (which == RAD_TAB_STAGE_FACE_SIGN) nl = rad::launch_stage_face_signs(t, (signed char *)tmp, 0);
    else nl = rad::launch_maxspeed(t, (double *)tmp, 0);
    bool ok = nl >= 0 && cudaMemcpy(host_out, tmp, need, cudaMemcpyDeviceToHost) == cudaSuccess;
    cudaFree(tmp);
    if (!ok) return cuda_fail(c, "rad_get_table");
    c->launches += nl;
    return RAD_OK;
}


// ------------------------------------------------------------------------------------------------
// rad_stage_static: the stage of rad_stage for callers that must not allocate (see include/rad.h).
//
// With the optical-depth-aware flux (tau_factor > 0, Eq.26-29) a stage needs a per-cell table between its first kernel (which
// writes it from the fluid state) and the flux-divergence kernel (which reads it): scratch, neither input nor output.  rad_stage
// takes that table from cudaMalloc on its first call.  Here it lives in the array below, which is part of the library image:
// the driver places it when the library is loaded on a device and nothing is requested from the allocator afterwards.
// ------------------------------------------------------------------------------------------------
#define RAD_STATIC_DOUBLES_PER_CELL 8
static __device__ __align__(256) double g_static_table[(size_t)RAD_STATIC_MAX_CELLS * RAD_STATIC_DOUBLES_PER_CELL];  // 4 MiB on every device that loads librad.so

namespace {
constexpr int kMaxStaticDevices = 64;
double *g_static_addr[kMaxStaticDevices];  // per device ordinal: where g_static_table sits in that device's memory (nullptr = not asked yet)
std::mutex g_static_mutex;

// In host code `g_static_table` names a host-side shadow of the symbol, not device memory: handing it to a kernel would make the
// kernel touch the wrong address.  The device address has to be asked for, once per device and with that device current.
cudaError_t static_table_address(int device, double **out) {
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_addr[device]) {
        void *p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_static_table);
        if (e != cudaSuccess) return e;
        g_static_addr[device] = static_cast<double *>(p);
    }
    *out = g_static_addr[device];
    return cudaSuccess;
}
}  // namespace

rad_status rad_stage_static(rad_ctx *c, double *I_in, double *I_out, const double *I0, const double *fluid, double gam0, double gam1,
                            double beta_dt, double *T_out, double *dT0, long long *n_noroot, void *stream) {
    if (!c || !fluid || !I_in || !I_out) return fail(c, RAD_EINVAL, "rad_stage_static: NULL argument");
    if (I_in == I_out || I0 == I_out) return fail(c, RAD_EINVAL, "rad_stage_static: I_out must not alias I_in or I0 (the stencil reads old values)");
    if (!std::isfinite(gam0) || !std::isfinite(gam1) || !std::isfinite(beta_dt)) return fail(c, RAD_EINVAL, "rad_stage_static: non-finite weights");
    if ((c->kp.couple || c->kp.tau_factor != 0.0) && (!c->opac.alpha_a_planck || !c->opac.alpha_a_energy || !c->opac.alpha_s))
        return fail(c, RAD_ESTATE, "rad_stage_static: context has no opacities");
    if (c->dev.ncell > (long long)RAD_STATIC_MAX_CELLS) {
        char buf[192];
        snprintf(buf, sizeof buf, "rad_stage_static: the block has %lld cells with its ghost layers, the built-in table holds RAD_STATIC_MAX_CELLS = %d; use rad_stage",
                 c->dev.ncell, (int)RAD_STATIC_MAX_CELLS);
        return fail(c, RAD_EUNSUPPORTED, buf);
    }
    if (c->device < 0 || c->device >= kMaxStaticDevices) return fail(c, RAD_EUNSUPPORTED, "rad_stage_static: device ordinal beyond the per-device address table");
    DeviceGuard guard(c->device);
    if (!guard.ok) return cuda_fail(c, "rad_stage_static: cudaSetDevice");
    double *table = nullptr;
    if (static_table_address(c->device, &table) != cudaSuccess) return cuda_fail(c, "rad_stage_static: cudaGetSymbolAddress");
    cudaStream_t s = (cudaStream_t)stream;
    if (n_noroot && cudaMemsetAsync(c->d_noroot, 0, sizeof(unsigned long long), s) != cudaSuccess) return cuda_fail(c, "rad_stage_static: memset");
    rad_status st = rad_fill_ghosts(c, I_in, s);
    if (st != RAD_OK) return st;
    // flux divergence.  Both table builders write every one of the block's cells, so nothing of an earlier call is read and
    // nothing has to be cleared; the array's tail beyond this block keeps whatever the last larger block left there.
    const bool tau = c->kp.tau_factor != 0.0;
    rad::StageArgs a{};
    a.I_in = I_in; a.I0 = I0; a.I_out = I_out; a.gam0 = gam0; a.gam1 = gam1; a.beta_dt = beta_dt;
    int nl = 0;
    if (rad::stage_angle_serves(c->dev, tau)) {  // tile kernel: {u^alphahat, f/2 of the upper faces}, 8 doubles per cell
        if (tau) {
            const int nt = rad::launch_tau_table(c->dev, fluid, c->opac.alpha_a_energy, c->opac.alpha_s, c->kp.tau_factor * beta_dt, table, s);
            if (nt < 0) return cuda_fail(c, "rad_stage_static (velocity table)");
            c->launches += nt;
            a.vel8 = table;
        }
        nl = rad::launch_stage_angle(c->dev, c->kp, a, s);
        if (nl < 0) return cuda_fail(c, "rad_stage_static (tile kernel)");
    }
    if (nl == 0) {  // generic kernel: {u^alphahat, alpha_E}, 5 doubles per cell
        if (tau) {
            const int nv = rad::launch_cell_velocity(c->dev, fluid, c->opac.alpha_a_energy, c->opac.alpha_s, table, s);
            if (nv < 0) return cuda_fail(c, "rad_stage_static (velocity table)");
            c->launches += nv;
        }
        nl = rad::launch_fluxdiv(c->dev, c->kp, I_in, I0, gam0, gam1, beta_dt, I_out, s, tau ? table : nullptr, c->kp.tau_factor * beta_dt);
        if (nl < 0) return cuda_fail(c, "rad_stage_static (flux divergence)");
    }
    c->launches += nl;
    st = run_coupling(c, I_out, fluid, beta_dt, T_out, dT0, n_noroot != nullptr, s);
    if (st != RAD_OK) return st;
    return read_noroot(c, n_noroot, s, "rad_stage_static: readback");
}

}  // extern "C"
