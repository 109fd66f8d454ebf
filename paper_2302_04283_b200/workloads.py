"""Seeded synthetic workloads C1-C5 (BASELINE.json `configs`).

This module holds NONE of the method's arithmetic: no metric, tetrad, flux or coupling
formula.  It only turns (config, seed, the angle grid's unit directions handed in by the
caller) into input arrays -- intensities, fluid primitives, absorptivities -- and is the
one module that both the oracle's tests and the CUDA path's tests/bench import.  The
arrays stand in for the Kerr-Schild accretion blocks of the paper's section 4,
whose actual torus data are not available.

Random numbers: counter-based, splitmix64(seed ^ (field_id << 40) + linear index) ->
U(0,1); Box-Muller for normals.  Integer hashing is exact on any device; the float
post-processing (log, cos, exp) may differ in the last bits between CPU and GPU, so a
parity test generates ONCE (on CPU) and hands the same array to both sides.
"""
import math

import torch

# field ids for the counter-based generator
_F_I, _F_RHO, _F_T, _F_V, _F_KAPPA, _F_Q, _F_MODES = 1, 2, 3, 4, 7, 8, 9

CONFIGS = {
    # name: metric kind (0 Minkowski, 1 Cartesian Kerr-Schild), spin, cells per axis, box, angles, bc, seed
    "C1": dict(metric=0, M=1.0, a=0.0, n=16, box=(0.0, 1.0), angles=("latlon", 5, 16), bc=1, seed=1001, excise=0.0),
    "C2": dict(metric=1, M=1.0, a=0.9, n=64, box=(4.0, 12.0), angles=("geodesic", 3), bc=0, seed=1002, excise=0.0),
    "C3": dict(metric=1, M=1.0, a=0.9, n=128, box=(2.5, 20.0), angles=("geodesic", 4), bc=0, seed=1003, excise=1.2),
    "C4": dict(metric=1, M=1.0, a=0.5, n=96, box=(3.0, 15.0), angles=("geodesic", 4), bc=0, seed=1004, excise=0.0),
    "C5": dict(metric=1, M=1.0, a=0.9, n=256, box=(2.0, 30.0), angles=("geodesic", 3), bc=0, seed=1005, excise=0.0),
}
NG = 2
GAMMA_GAS, A_RAD, N0_CRIT, CFL = 5.0 / 3.0, 1.0, 0.1, 0.3


def n_angles(cfg):
    a = CONFIGS[cfg]["angles"] if isinstance(cfg, str) else cfg["angles"]
    return a[1] * a[2] if a[0] == "latlon" else 10 * a[1] * a[1] + 2


def grid(cfg, n=None, sub=None, ng=None):
    """(n, ng, x0, dx) of a config; `n` overrides the cell count (same box: a coarser block); `sub` keeps the
    spacing of the n-cell block but takes only the sub^3 cells at its low corner (a bounded sample)."""
    c = CONFIGS[cfg] if isinstance(cfg, str) else cfg
    n = c["n"] if n is None else n
    lo, hi = c["box"]
    dx = (hi - lo) / n
    m = n if sub is None else sub
    return (m, m, m), (NG if ng is None else ng), (lo, lo, lo), (dx, dx, dx)


def excise_radius(cfg):
    """r < 1.2 r_h excision of config C3 (BASELINE.json); r_h = M + sqrt(M^2 - a^2)."""
    c = CONFIGS[cfg] if isinstance(cfg, str) else cfg
    if not c["excise"]:
        return 0.0
    return c["excise"] * (c["M"] + math.sqrt(c["M"] ** 2 - c["a"] ** 2))


# ----------------------------------------------------------------------------- random numbers
_MASK = (1 << 64) - 1


def _i64(x):
    x &= _MASK
    return x - (1 << 64) if x >= (1 << 63) else x


def _lsr(x, k):
    """logical right shift of an int64 tensor"""
    return (x >> k) & ((1 << (64 - k)) - 1)


def _splitmix(idx, seed, field):
    z = idx + _i64((seed ^ (field << 40)) * 0x9E3779B97F4A7C15 + 0x9E3779B97F4A7C15)
    z = z * _i64(0x9E3779B97F4A7C15)  # spread consecutive counters
    z = (z ^ _lsr(z, 30)) * _i64(0xBF58476D1CE4E5B9)
    z = (z ^ _lsr(z, 27)) * _i64(0x94D049BB133111EB)
    return z ^ _lsr(z, 31)


def uniform(count, seed, field, device="cpu", offset=0):
    """U(0,1) (never exactly 0) for counters offset .. offset+count-1"""
    idx = torch.arange(offset, offset + count, dtype=torch.int64, device=device)
    bits = _lsr(_splitmix(idx, seed, field), 11)
    return (bits.to(torch.float64) + 0.5) * (1.0 / 9007199254740992.0)


def normal(count, seed, field, device="cpu"):
    u1 = uniform(count, seed, field, device)
    u2 = uniform(count, seed, field, device, offset=1 << 38)
    return torch.sqrt(-2.0 * torch.log(u1)) * torch.cos(2.0 * math.pi * u2)


# ----------------------------------------------------------------------------- smooth fields
def _coords(n, ng, x0, dx, device):
    ax = [x0[d] + (torch.arange(n[d] + 2 * ng, dtype=torch.float64, device=device) - ng + 0.5) * dx[d] for d in range(3)]
    z, y, x = torch.meshgrid(ax[2], ax[1], ax[0], indexing="ij")  # arrays are [k][j][i]
    return x, y, z


def _smooth(x, y, z, box, seed, tag, nmodes=8, kmax=3):
    """unit-variance sum of `nmodes` random cosine modes with integer wavevectors |k_i| <= kmax"""
    lo, hi = box
    L = hi - lo
    u = uniform(4 * nmodes, seed, _F_MODES + 16 * tag, "cpu").tolist()
    out = torch.zeros_like(x)
    for m in range(nmodes):
        k = [int(u[4 * m + d] * (2 * kmax + 1)) - kmax for d in range(3)]
        if k == [0, 0, 0]:
            k = [1, 0, 0]
        ph = 2.0 * math.pi * u[4 * m + 3]
        out += torch.cos(2.0 * math.pi * (k[0] * (x - lo) + k[1] * (y - lo) + k[2] * (z - lo)) / L + ph)
    return out * math.sqrt(2.0 / nmodes)


def _solenoidal(x, y, z, box, seed, vmax, nmodes=24, kmax=8):
    """random-phase divergence-free velocity field, |k| <= kmax, amplitude ~ k^(-11/6) (E(k) ~ k^-5/3)"""
    lo, hi = box
    L = hi - lo
    u = uniform(8 * nmodes, seed, _F_MODES + 16 * 5, "cpu").tolist()
    v = [torch.zeros_like(x) for _ in range(3)]
    for m in range(nmodes):
        k = [int(u[8 * m + d] * (2 * kmax + 1)) - kmax for d in range(3)]
        if k == [0, 0, 0]:
            k = [1, 1, 0]
        kk = math.sqrt(sum(q * q for q in k))
        r = [u[8 * m + 3 + d] - 0.5 for d in range(3)]
        a = [r[1] * k[2] - r[2] * k[1], r[2] * k[0] - r[0] * k[2], r[0] * k[1] - r[1] * k[0]]  # r x k: perpendicular to k
        an = math.sqrt(sum(q * q for q in a)) or 1.0
        amp = kk ** (-11.0 / 6.0)
        ph = 2.0 * math.pi * u[8 * m + 6]
        c = torch.cos(2.0 * math.pi * (k[0] * (x - lo) + k[1] * (y - lo) + k[2] * (z - lo)) / L + ph)
        for d in range(3):
            v[d] += (amp * a[d] / an) * c
    vmag = torch.sqrt(v[0] ** 2 + v[1] ** 2 + v[2] ** 2).max()
    return [q * (vmax / vmag) for q in v]


# ----------------------------------------------------------------------------- the recipes
def make_inputs(cfg, nhat, n=None, device="cpu", sub=None, ng=None):
    """Inputs of one stage for config `cfg` ("C1".."C5").

    nhat: [N,3] unit directions of the angle grid (from the implementation under test).
    Returns dict: I [NK,NJ,NI,N] (ghosts included, generated like the interior),
    fluid [5,NK,NJ,NI] = rho, T, u1', u2', u3' (normal-frame spatial velocity),
    opac [3,NK,NJ,NI] = alpha_a_planck, alpha_a_energy, alpha_s (absorptivities).
    Velocities: a flat-space 3-velocity v (|v|<1) is turned into u' = v / sqrt(1 - v.v);
    any 3-vector is a valid u'.  "Thermal" intensities use the flat-space Doppler factor
    gamma (1 - v.n) of that v as a stand-in for n^0bar; this is an input recipe, not the
    method's frame transformation.
    """
    c = CONFIGS[cfg]
    seed = c["seed"]
    nn, ng, x0, dx = grid(cfg, n, sub, ng)  # (ng = 3: the ghost depth PPM needs; the default 2 is the workload's)
    nhat = torch.as_tensor(nhat, dtype=torch.float64, device=device)
    N = nhat.shape[0]
    NI, NJ, NK = nn[0] + 2 * ng, nn[1] + 2 * ng, nn[2] + 2 * ng
    ncell = NI * NJ * NK
    shp = (NK, NJ, NI)
    x, y, z = _coords(nn, ng, x0, dx, device)
    U = lambda f: uniform(ncell, seed, f, device).reshape(shp)
    M, a = c["M"], c["a"]

    def doppler(v):
        v2 = v[0] ** 2 + v[1] ** 2 + v[2] ** 2
        gam = 1.0 / torch.sqrt(1.0 - v2)
        vn = v[0][..., None] * nhat[:, 0] + v[1][..., None] * nhat[:, 1] + v[2][..., None] * nhat[:, 2]
        return gam[..., None] * (1.0 - vn)

    def thermal(T, v, noise):
        xi = 2.0 * uniform(ncell * N, seed, _F_I, device).reshape(shp + (N,)) - 1.0
        return (A_RAD * T ** 4 / (4.0 * math.pi))[..., None] / doppler(v) ** 4 * (1.0 + noise * xi)

    if cfg == "C1":
        rho = 0.5 + 1.5 * U(_F_RHO)
        T = 0.5 + 1.5 * U(_F_T)
        v = [-0.3 + 0.6 * uniform(ncell, seed, _F_V + d, device).reshape(shp) for d in range(3)]
        I = torch.exp(normal(ncell * N, seed, _F_I, device)).reshape(shp + (N,))
        aa, asc = 1.0 * rho, 0.5 * rho
    elif cfg in ("C2", "C5"):
        rcyl = torch.sqrt(x * x + y * y)
        r = torch.sqrt(x * x + y * y + z * z)
        Om = math.sqrt(M) / (rcyl ** 1.5 + a * math.sqrt(M))
        if cfg == "C2":
            rho = torch.exp(0.5 * _smooth(x, y, z, c["box"], seed, 1))
            T = 0.05 * (r / 4.0) ** (-1.0) * (1.0 + 0.1 * _smooth(x, y, z, c["box"], seed, 2))
            f = 1.0 + 0.05 * _smooth(x, y, z, c["box"], seed, 3)
            v = [-Om * y * f, Om * x * f, torch.zeros_like(x)]
            I = thermal(T, v, 0.2)
            aa, asc = 10.0 * rho, 1.0 * rho
        else:
            rho = torch.exp(-z * z / (2.0 * (0.1 * rcyl) ** 2)) * rcyl ** (-1.5) + 1e-6
            T = 0.02 * (r / 6.0) ** (-0.75)
            v = [-Om * y, Om * x, torch.zeros_like(x)]
            I = thermal(T, v, 0.01)
            aa, asc = 10.0 * rho, 4.0 * rho
    elif cfg == "C3":
        rho = torch.exp(_smooth(x, y, z, c["box"], seed, 1))
        T = 10.0 ** (-2.0 + 2.0 * U(_F_T))
        v = _solenoidal(x, y, z, c["box"], seed, 0.5)
        I = thermal(T, v, 0.2)
        aa = rho * 10.0 ** (-2.0 + 4.0 * U(_F_KAPPA))
        asc = 0.4 * rho
    elif cfg == "C4":
        T = 10.0 ** (-3.0 + 3.0 * U(_F_T))
        q = 10.0 ** (-2.0 + 5.0 * U(_F_Q))
        rho = A_RAD * T ** 3 / (3.0 * q)  # P_rad / P_gas = (a T^4 / 3) / (rho T) = q
        s = [_smooth(x, y, z, c["box"], seed, 10 + d) for d in range(3)]
        smax = torch.sqrt(s[0] ** 2 + s[1] ** 2 + s[2] ** 2).max()
        v = [q_ * (0.2 / smax) for q_ in s]
        I = thermal(T, v, 0.2)
        aa = torch.full_like(rho, 1.0e4)
        asc = torch.full_like(rho, 1.0e3)
    else:
        raise ValueError(cfg)
    v2 = v[0] ** 2 + v[1] ** 2 + v[2] ** 2
    gam = 1.0 / torch.sqrt(1.0 - v2)
    fluid = torch.stack([rho, T, gam * v[0], gam * v[1], gam * v[2]]).contiguous()
    opac = torch.stack([aa, aa, asc]).contiguous()
    return dict(I=I.contiguous(), fluid=fluid, opac=opac)
