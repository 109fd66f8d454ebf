"""Shared helpers of the GPU parity tests: build the same problem on both sides, convert the oracle's
geometry records to the library's tabulated-metric layout (rad.h), compare."""
import numpy as np

from paper_2302_04283_b200 import workloads as W

TOL_I, TOL_FLUID = 1e-11, 1e-10   # north_star: max relative error per intensity / on fluid energy after one stage


def dt0_floor(N):
    """dT^0_alpha is compared relative to max(|dT^0_alpha|, dt0_floor(N) * |R^0_0|) per cell.  Both sides form it
    as a sum over N angles of n^0 n_alpha dOmega (I_+ - I*) (the oracle literally, the coupling kernel as P + src Q with
    the sums P, Q of the two parts of I_+ - I*).  Every term carries a rounding of eps |I| dOmega whatever the size of the increment
    itself (a cell in equilibrium has dT^0_alpha = 0 in exact arithmetic), so two correct evaluations in different orders differ by
    a random walk of N such roundings: ~ sqrt(N) eps |R^0_0|.  The absolute bar is four of those: TOL_FLUID * floor = 4 sqrt(N) 2^-53 |R^0_0|
    (N = 92: floor 4.3e-5, N = 162: 5.7e-5, N = 362: 8.4e-5)."""
    return 4.0 * np.sqrt(N) * 2.0 ** -53 / TOL_FLUID



def oracle_tables_to_rad(cell, face, excised):
    """oracle cell record (alpha, e[4][4], L[4][4], S[30], beta[3], gamma[6]) -> rad.h RAD_NCELL layout"""
    nc = cell.shape[0]
    e = cell[:, 1:17].reshape(nc, 4, 4); L = cell[:, 17:33].reshape(nc, 4, 4)
    out = np.zeros((nc, 52))
    out[:, 0] = e[:, 0, 0]
    out[:, 1:5] = L[:, 0, :]
    out[:, 5:35] = cell[:, 33:63]
    out[:, 35:38] = cell[:, 63:66]
    out[:, 38:44] = np.stack([e[:, 1, 1], e[:, 1, 2], e[:, 1, 3], e[:, 2, 2], e[:, 2, 3], e[:, 3, 3]], 1)
    out[:, 44:50] = np.stack([L[:, 1, 1], L[:, 2, 1], L[:, 3, 1], L[:, 2, 2], L[:, 3, 2], L[:, 3, 3]], 1)
    out[:, 50] = excised
    return out, face.copy()


def make_oracle(oracle, cfg, n=None, **kw):
    c = W.CONFIGS[cfg]
    A = oracle.Angles(*c["angles"])
    nn, ng, x0, dx = W.grid(cfg, n)
    args = dict(metric_kind=c["metric"], M=c["M"], a=c["a"], excise_r=W.excise_radius(cfg), bc_lo=(c["bc"],) * 3, bc_hi=(c["bc"],) * 3,
                gamma_gas=W.GAMMA_GAS, a_rad=W.A_RAD, n0_crit=W.N0_CRIT, recon_space=1, renorm=1, couple=1)
    args.update(kw)
    return A, oracle.Problem(A, nn, x0, dx, **args)


def make_rad(B, cfg, opac, n=None, tabulated=None, device=0, **kw):
    """rad_create for config cfg; opac = CUDA tensor [3, ncell]; tabulated = (cell_tab, face_tab) CUDA tensors or None"""
    c = W.CONFIGS[cfg]
    nn, ng, x0, dx = W.grid(cfg, n)
    metric = dict(kind=c["metric"], M=c["M"], a=c["a"], excise_r=W.excise_radius(cfg))
    if tabulated is not None:
        metric = dict(kind=2, cell_tab=tabulated[0], face_tab=tabulated[1])
    grid = dict(n=nn, x0=x0, dx=dx, bc_lo=(c["bc"],) * 3, bc_hi=(c["bc"],) * 3)
    params = dict(gamma_gas=W.GAMMA_GAS, a_rad=W.A_RAD, n0_crit=W.N0_CRIT, recon_space=1, renorm_fluid_weights=1, couple=1)
    params.update(kw)
    op = None if opac is None else (opac[0], opac[1], opac[2])
    return B.rad_create(metric, grid, c["angles"], op, params, device)


def rel_err_I(got, ref):
    """max over interior (cell, angle) of |dI| / max(|I_ref|, 1e-12 * mean_n |I_ref| of the cell)"""
    den = np.maximum(np.abs(ref), 1e-12 * np.abs(ref).mean(-1, keepdims=True))
    den = np.where(den == 0, 1.0, den)
    return float((np.abs(got - ref) / den).max())


def rel_err(got, ref, floor):
    den = np.maximum(np.abs(ref), floor)
    den = np.where(den == 0, 1.0, den)
    return float((np.abs(got - ref) / den).max())


def err_dT0(P, dT0_got, dT0_ref, out_ref):
    """max over the four components of the relative error of the fluid increment with the floor dt0_floor(N) |R^0_0|; also returns the
    fraction of interior cells whose increment sits below the floor in every component"""
    R0 = np.abs(P.interior(P.moments(out_ref, 1)[0]))
    fl = dt0_floor(P.N)
    e = max(rel_err(P.interior(dT0_got[m]), P.interior(dT0_ref[m]), fl * R0 + 1e-300) for m in range(4))
    on_floor = np.all([np.abs(P.interior(dT0_ref[m])) < fl * R0 for m in range(4)], axis=0)
    return e, float(on_floor.mean())
