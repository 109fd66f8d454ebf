"""Pins P7, P8, P13 and the stationary-solution pin of the oracle's transport step
(paper section 2.2-2.4, Eq.22, 24, 25; tests of section 3.1, 3.4)."""
import numpy as np
import pytest


def mink(oracle, A, n, recon=1, bc=1, dx=None, x0=(0.0, 0.0, 0.0)):
    dx = dx or tuple(1.0 / v for v in n)
    return oracle.Problem(A, n, x0, dx, metric_kind=0, bc_lo=(bc,) * 3, bc_hi=(bc,) * 3, recon_space=recon, couple=0)


@pytest.mark.parametrize("recon", [0, 1])
def test_uniform_isotropic_is_fixed_point(oracle, recon):
    """P7 / north_star: an isotropic field stays isotropic in Minkowski -- bit for bit"""
    A = oracle.Angles("geodesic", 2)
    P = mink(oracle, A, (6, 5, 4), recon)
    I = np.full((P.ncell, A.N), 0.7312)
    out = P.transport(I, 0.03)
    assert np.array_equal(P.interior(out), P.interior(I))


@pytest.mark.parametrize("grid", [("latlon", 4, 8), ("geodesic", 2)])
def test_beam_centroid_moves_along_straight_line(oracle, grid):
    """P7 / section 3.1: free streaming in flat space.  For donor-cell upwinding the intensity-weighted
    centroid of a single-angle beam moves by exactly n dt per step (summation by parts), and the total is kept."""
    A = oracle.Angles(*grid)
    n = (12, 10, 8)
    P = mink(oracle, A, n, recon=0)
    rng = np.random.default_rng(3)
    dx = np.array([1.0 / v for v in n])
    k, j, i = np.meshgrid(*(np.arange(v + 4) for v in n[::-1]), indexing="ij")
    X = np.stack([(i - 2 + 0.5) * dx[0], (j - 2 + 0.5) * dx[1], (k - 2 + 0.5) * dx[2]], -1).reshape(-1, 3)
    for ang in (0, A.N // 3, A.N - 2):
        I = np.zeros((P.ncell, A.N))
        blob = np.zeros(P.shape)
        blob[5:8, 6:9, 6:10] = rng.uniform(0.5, 2.0, (3, 3, 4))  # compact, away from the boundary
        I[:, ang] = blob.ravel()
        dt = 0.3 * dx.min()
        out = P.transport(I, dt)
        w0, w1 = I[:, ang], out[:, ang]
        assert abs(w1.sum() - w0.sum()) < 1e-13 * w0.sum()
        shift = (X * w1[:, None]).sum(0) / w1.sum() - (X * w0[:, None]).sum(0) / w0.sum()
        assert np.abs(shift - A.nhat[ang] * dt).max() < 1e-14
        # other angles untouched: no angular transport with a Cartesian tetrad in flat space
        other = np.delete(np.arange(A.N), ang)
        assert (P.interior(out)[..., other] == 0).all()
        assert (w1 >= 0).all()


def test_plm_is_exact_for_linear_profiles(oracle):
    """P7: second-order reconstruction advects a linear profile exactly: I* = I - dt n.grad I"""
    A = oracle.Angles("latlon", 3, 6)
    n = (8, 7, 6)
    P = mink(oracle, A, n, recon=1, bc=0)
    dx = np.array([1.0 / v for v in n])
    k, j, i = np.meshgrid(*(np.arange(v + 4) for v in n[::-1]), indexing="ij")
    X = np.stack([(i - 2 + 0.5) * dx[0], (j - 2 + 0.5) * dx[1], (k - 2 + 0.5) * dx[2]], -1).reshape(-1, 3)
    grad = np.array([0.7, -0.4, 0.25])
    I = np.repeat((3.0 + X @ grad)[:, None], A.N, 1) * (1.0 + 0.1 * np.arange(A.N))[None, :]
    dt = 0.02
    out = P.transport(I, dt)
    expect = I - dt * (A.nhat @ grad)[None, :] * (1.0 + 0.1 * np.arange(A.N))[None, :]
    assert np.abs(P.interior(out) - P.interior(expect)).max() < 1e-13


def test_limiter_is_van_leer(oracle):
    """R7: harmonic-mean slope; at an extremum the scheme falls back to donor cell"""
    A = oracle.Angles("latlon", 1, 4)  # directions (+-1,+-1,0)/sqrt2 rotated by pi/4
    P = mink(oracle, A, (8, 1, 1), recon=1, bc=1, dx=(1.0, 1.0, 1.0))
    q = np.array([1.0, 2.0, 4.0, 3.0, 3.0, 7.0, 1.0, 0.5])
    I = np.zeros(P.shape + (A.N,))
    I[2:-2, 2:-2, 2:-2, :] = q[None, None, :, None]
    I = I.reshape(-1, A.N)
    P.fill_ghosts(I)
    dt = 0.1
    out = P.interior(P.transport(I, dt))[0, 0]
    qq = np.concatenate([q[-2:], q, q[:2]])
    dl, dr = qq[1:-1] - qq[:-2], qq[2:] - qq[1:-1]
    with np.errstate(divide="ignore", invalid="ignore"):
        s = np.where(dl * dr > 0, 2 * dl * dr / (dl + dr), 0.0)   # slopes of cells -1..8
    for ang in range(4):
        nx = A.nhat[ang, 0]
        if nx > 0:
            face = qq[1:-1] + 0.5 * s          # upper-face state of cells -1..8
            flux = nx * face                    # flux through upper face of cell i-1.. ; F(i+1/2) = nx * face[i]
            new = q - dt * (flux[1:-1] - flux[0:-2])
        else:
            face = qq[1:-1] - 0.5 * s          # lower-face state of cells -1..8
            flux = nx * face
            new = q - dt * (flux[2:] - flux[1:-1])
        assert np.abs(out[:, ang] - new).max() < 1e-14


def test_beams_cross_unaffected(oracle):
    """section 3.1: beams cross without affecting one another: donor-cell transport is linear"""
    A = oracle.Angles("latlon", 4, 8)
    P = mink(oracle, A, (8, 8, 4), recon=0)
    rng = np.random.default_rng(5)
    I1 = np.zeros((P.ncell, A.N)); I2 = np.zeros((P.ncell, A.N))
    I1[:, 9] = rng.uniform(0, 1, P.ncell); I2[:, 22] = rng.uniform(0, 1, P.ncell)
    o12 = P.transport(I1 + I2, 0.02); o1 = P.transport(I1, 0.02); o2 = P.transport(I2, 0.02)
    assert np.abs(P.interior(o12) - P.interior(o1) - P.interior(o2)).max() < 1e-15


@pytest.mark.parametrize("kind,a,grid", [(0, 0.0, ("geodesic", 2)), (1, 0.9, ("geodesic", 2)), (1, 0.5, ("latlon", 4, 8))])
@pytest.mark.parametrize("recon", [0, 1])
def test_energy_conservation_sources_off(oracle, kind, a, grid, recon):
    """P8: the scheme conserves sum n^0 n_0 I dOmega dV: spatial fluxes telescope between cells,
    angular fluxes telescope between angles -- in flat AND curved spacetime."""
    A = oracle.Angles(*grid)
    n = (10, 9, 8)
    dx = (0.3, 0.3, 0.3)
    P = oracle.Problem(A, n, (3.0, 2.5, 2.0), dx, metric_kind=kind, M=1.0, a=a, recon_space=recon, couple=0)
    cell, _, _ = P.geometry()
    n4 = np.concatenate([np.ones((A.N, 1)), A.nhat], 1)
    w = (cell[:, 1:5] @ n4.T) * (cell[:, 17:21] @ n4.T)     # n^0 n_0 per (cell, angle)
    rng = np.random.default_rng(11)
    I = np.zeros(P.shape + (A.N,))
    I[5:-5, 5:-5, 5:-5] = np.exp(rng.normal(size=(n[2] - 6, n[1] - 6, n[0] - 6, A.N)))  # compact support
    I = I.reshape(-1, A.N)
    vmax, _ = P.max_speed()
    dt = 0.3 * min(dx) / vmax
    out = P.transport(I, dt)
    out_full = np.zeros_like(I)
    P.interior(out_full)[...] = P.interior(out)
    E0 = (w * I * A.domega).sum(); E1 = (w * out_full * A.domega).sum()
    assert abs(E1 - E0) < 1e-13 * abs(E0)
    if kind == 1:  # angular fluxes did something
        cm = P.cell_index(6, 6, 6)
        assert np.abs(P.edge_coeffs(cm)[0]).max() > 1e-4


def test_stationary_solution_in_kerr_schild(oracle):
    """Pins sign and size of the angular flux against the spatial flux.  In a stationary spacetime k_0 is
    conserved along rays and I/nu^4 is invariant, so Ihat(x, n) = (-n_0(x, n))^-4 is an exact
    stationary solution of Eq.2.  The discrete rate of change must be a truncation error: small compared
    with the spatial term alone, and decreasing with resolution."""
    res = []
    for lev, n in ((2, 6), (4, 12)):
        A = oracle.Angles("geodesic", lev)
        L = 1.2
        dx = (L / n,) * 3
        P = oracle.Problem(A, (n, n, n), (3.0, 2.0, 1.0), dx, metric_kind=1, M=1.0, a=0.9, recon_space=1, couple=0)
        cell, _, _ = P.geometry()
        n4 = np.concatenate([np.ones((A.N, 1)), A.nhat], 1)
        n0 = cell[:, 17:21] @ n4.T
        I = (-n0) ** -4.0
        dt = 1e-3
        out = P.transport(I, dt)
        rate = np.abs(P.interior(out) / P.interior(I) - 1.0) / dt
        # size of the spatial term alone: |n^i d_i ln I| = 4 |n^i d_i ln(-n_0)|, estimated by differencing n_0
        n0g = n0.reshape(P.shape + (A.N,))
        dln = np.abs(np.log(-n0g[2:-2, 2:-2, 3:-1]) - np.log(-n0g[2:-2, 2:-2, 1:-3])).max() / (2 * dx[0])
        res.append((rate.mean(), rate.max(), 4 * dln))
    assert res[0][2] > 0.05                      # gravity is strong enough for the check to bite
    assert res[1][0] < 0.1 * res[1][2]           # residual << spatial term (a wrong-signed angular term gives ~2x)
    assert res[1][0] < 0.6 * res[0][0]           # and it converges (first order in the angular spacing)


def test_hohlraum_1d(oracle):
    """P13 / section 3.4: radiation leaving an isotropic wall into vacuum; exact moments Eq.61."""
    errs = []
    for nz, npsi in ((4, 8), (8, 16)):
        A = oracle.Angles("latlon", nz, npsi)
        nx = 64
        P = oracle.Problem(A, (nx, 1, 1), (0.0, 0.0, 0.0), (1.0 / nx, 1.0, 1.0), metric_kind=0,
                           bc_lo=(0, 1, 1), bc_hi=(2, 1, 1), recon_space=1, couple=0)
        I = np.zeros(P.shape + (A.N,))
        I[:, :, :2, :] = 1.0 / (4 * np.pi)       # the wall: fixed isotropic field of unit energy density
        I = I.reshape(-1, A.N)
        t, dt = 0.0, 0.4 / nx
        while t < 0.75 - 1e-12:
            h = min(dt, 0.75 - t)
            P.fill_ghosts(I)
            new = P.transport(I, h)
            Ii = P.interior(I.reshape(P.shape + (A.N,)))
            Ii[...] = P.interior(new)
            t += h
        mom = P.moments(I, 0)
        x = (np.arange(nx) + 0.5) / nx
        R = {q: P.interior(mom[q])[0, 0] for q in (0, 1, 4)}
        s = np.clip(x / 0.75, 0, 1)
        ex = {0: 0.5 * (1 - s), 1: 0.25 * (1 - s**2), 4: (1 - s**3) / 6}
        eps = np.sqrt(sum((np.abs(R[q] - ex[q]).sum() / nx) ** 2 for q in (0, 1, 4)) / 3)  # Eq.62
        errs.append(eps)
    assert errs[1] < errs[0] and errs[1] < 0.02, errs
