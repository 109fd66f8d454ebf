"""Oracle pins for the small steps: ghost fill (a7), ergosphere mask (a6), excision, moments (O6), stage weights (R8)."""
import numpy as np
import pytest


def test_ghost_fill_periodic_and_outflow(oracle):
    A = oracle.Angles("latlon", 1, 4)
    n = (4, 3, 1)
    P = oracle.Problem(A, n, (0, 0, 0), (1, 1, 1), bc_lo=(1, 2, 1), bc_hi=(1, 2, 1))
    rng = np.random.default_rng(0)
    core = rng.uniform(size=(n[2], n[1], n[0], A.N))
    I = np.full(P.shape + (A.N,), np.nan)
    I[2:-2, 2:-2, 2:-2] = core
    I = I.reshape(-1, A.N)
    P.fill_ghosts(I)
    # numpy's own padding modes are the textbook definitions: x periodic, y copy-of-edge, z periodic
    ref = np.pad(core, ((0, 0), (0, 0), (2, 2), (0, 0)), mode="wrap")
    ref = np.pad(ref, ((0, 0), (2, 2), (0, 0), (0, 0)), mode="edge")
    ref = np.pad(ref, ((2, 2), (0, 0), (0, 0), (0, 0)), mode="wrap")
    assert np.array_equal(I.reshape(ref.shape), ref)


def test_caller_filled_ghosts_are_left_alone(oracle):
    A = oracle.Angles("latlon", 1, 4)
    P = oracle.Problem(A, (2, 2, 2), (0, 0, 0), (1, 1, 1))
    I = np.arange(P.ncell * A.N, dtype=float).reshape(-1, A.N)
    J = I.copy()
    P.fill_ghosts(J)
    assert np.array_equal(I, J)


def test_ergosphere_mask(oracle):
    """a6: every step, I is zeroed wherever |n_0| < n_0^crit (~0.1); inside the ergosphere some
    directions have n_0 > 0 (negative-energy orbits), so the band |n_0| < 0.1 is non-empty there."""
    A = oracle.Angles("geodesic", 4)
    x = np.array([1.55, 0.0, 0.05])   # equatorial, between the horizon (r_h = 1.436) and the ergosphere (r = 2), a = 0.9
    dx = 0.02
    P = oracle.Problem(A, (1, 1, 1), tuple(x - dx / 2), (dx,) * 3, metric_kind=1, M=1.0, a=0.9, couple=0, n0_crit=0.1)
    g = oracle.geometry_point(1, 1.0, 0.9, x)
    assert g["g"][0, 0] > 0   # inside the ergosphere
    n0 = np.array([g["g"][0] @ g["e"] @ np.array([1.0, *nh]) for nh in A.nhat])
    assert (n0 > 0).any() and (n0 < 0).any()
    band = np.abs(n0) < 0.1
    assert 0 < band.sum() < 0.11 * A.N    # "less than 11% of the phase-space volume"
    I = np.ones((P.ncell, A.N))
    nc = P.ncell
    fluid = np.stack([np.ones(nc), np.ones(nc), np.zeros(nc), np.zeros(nc), np.zeros(nc)])
    opac = np.zeros((3, nc))
    T, dT0, nf = P.coupling(I, fluid, opac, 0.1)
    c = P.cell_index(2, 2, 2)
    assert np.array_equal(I[c] == 0.0, band) and (I[c][~band] == 1.0).all()


def test_excision(oracle):
    A = oracle.Angles("latlon", 2, 4)
    n = (8, 8, 8)
    P = oracle.Problem(A, n, (-2, -2, -2), (0.5, 0.5, 0.5), metric_kind=1, M=1.0, a=0.9, excise_r=1.8, couple=0)
    _, _, ex = P.geometry()
    k, j, i = np.meshgrid(*(np.arange(12),) * 3, indexing="ij")
    X = np.stack([-2 + (i - 1.5) * 0.5, -2 + (j - 1.5) * 0.5, -2 + (k - 1.5) * 0.5], -1).reshape(-1, 3)
    R2 = (X**2).sum(1); a = 0.9
    r = np.sqrt(0.5 * (R2 - a * a + np.sqrt((R2 - a * a) ** 2 + 4 * a * a * X[:, 2] ** 2)))
    assert np.array_equal(ex.astype(bool), r < 1.8) and ex.sum() > 8
    I = np.ones((P.ncell, A.N))
    out = P.transport(I, 0.01)
    exi = P.interior(ex.astype(bool))
    assert (P.interior(out)[exi] == 0).all() and np.isfinite(P.interior(out)).all()


@pytest.mark.parametrize("kind,a", [(0, 0.0), (1, 0.9)])
def test_moments(oracle, kind, a):
    """O6, Eq.45 / Eq.71d against numpy contractions of the point geometry"""
    A = oracle.Angles("geodesic", 2)
    P = oracle.Problem(A, (1, 1, 1), (3.0, 2.0, 1.0), (0.2, 0.2, 0.2), metric_kind=kind, M=1.0, a=a)
    c = P.cell_index(2, 2, 2)
    g = oracle.geometry_point(kind, 1.0, a, (3.1, 2.1, 1.1))
    rng = np.random.default_rng(1)
    I = rng.uniform(0.5, 1.5, (P.ncell, A.N))
    n4 = np.concatenate([np.ones((A.N, 1)), A.nhat], 1)
    ncon = n4 @ g["e"].T                       # n^mu = e^mu_ahat n^ahat  (Eq.8a)
    ncov = ncon @ g["g"]                       # n_mu
    iu = np.triu_indices(4)
    R = np.einsum("n,na,nb->ab", I[c] * A.domega, ncon, ncon)
    assert np.allclose(P.moments(I, 0)[:, c], R[iu], rtol=1e-14, atol=1e-15)
    Rm = np.einsum("n,n,na->a", I[c] * A.domega, ncon[:, 0], ncov)
    assert np.allclose(P.moments(I, 1)[:, c], Rm, rtol=1e-14, atol=1e-15)
    Rt = np.einsum("n,na,nb->ab", I[c] * A.domega, n4, n4)
    assert np.allclose(P.moments(I, 2)[:, c], Rt[iu], rtol=1e-14, atol=1e-15)
    # tensor transformation: R^{mu nu} = e e R^{ahat bhat}
    assert np.allclose(R, g["e"] @ Rt @ g["e"].T, atol=1e-13)
    # fluid frame (Eq.13-14 with G2, Eq.38): boost matrix Lambda applied to the tetrad-frame tensor
    unorm = np.array([0.3, -0.5, 0.4])
    W = np.sqrt(1 + unorm @ g["g"][1:, 1:] @ unorm)
    ucon = np.concatenate([[W / g["alpha"]], unorm - g["beta"] * W / g["alpha"]])
    uh = g["elow"] @ ucon
    Lam = np.zeros((4, 4))
    Lam[0, 0] = uh[0]; Lam[0, 1:] = -uh[1:]; Lam[1:, 0] = -uh[1:]
    Lam[1:, 1:] = np.outer(uh[1:], uh[1:]) / (1 + uh[0]) + np.eye(3)
    assert np.abs(Lam.T @ np.diag([-1.0, 1, 1, 1]) @ Lam - np.diag([-1.0, 1, 1, 1])).max() < 1e-14  # a Lorentz boost
    Rb = Lam @ Rt @ Lam.T
    nc = P.ncell
    fluid = np.stack([np.ones(nc), np.ones(nc)] + [np.full(nc, v) for v in unorm])
    assert np.allclose(P.moments(I, 3, fluid)[:, c], Rb[0], rtol=1e-13, atol=1e-15)


def test_stage_weights(oracle):
    """R8: C* = gam0 C0 + gam1 C - beta dt div.  With (0,1) it is forward Euler; with (1/2,1/2) and I0 it is
    the second stage of Heun's method: the average of I0 and a forward-Euler step from I."""
    A = oracle.Angles("geodesic", 1)
    P = oracle.Problem(A, (4, 4, 4), (3, 2, 1), (0.3, 0.3, 0.3), metric_kind=1, M=1.0, a=0.5, couple=0)
    rng = np.random.default_rng(2)
    I = rng.uniform(0.5, 1.5, (P.ncell, A.N)); I0 = rng.uniform(0.5, 1.5, (P.ncell, A.N))
    dt = 0.05
    fe = P.transport(I, 0.5 * dt)                        # I - (dt/2) div
    heun = P.transport(I, 0.5 * dt, I0=I0, gam0=0.5, gam1=0.5)
    expect = 0.5 * I0 + 0.5 * I + (fe - I)
    assert np.abs(P.interior(heun) - P.interior(expect)).max() < 1e-14


# ------------------------------------------------------------------------------------------------ signal speed and upwind tables
def face_geometry(oracle, P, kind, M, a, x0, dx):
    """alpha and the tetrad e[mu][ahat] at the centre of every cell's LOWER x, y, z face, straight from geometry_point (pinned in
    test_oracle_geometry.py), independent of the problem's own face table: arrays [ncell][3] and [ncell][3][4][4]"""
    ng = P.ng
    al = np.zeros((P.ncell, 3)); e = np.zeros((P.ncell, 3, 4, 4))
    for k in range(P.NK):
        for j in range(P.NJ):
            for i in range(P.NI):
                c = P.cell_index(k, j, i)
                ctr = np.array([x0[0] + (i - ng + 0.5) * dx[0], x0[1] + (j - ng + 0.5) * dx[1], x0[2] + (k - ng + 0.5) * dx[2]])
                for ax in range(3):
                    x = ctr.copy(); x[ax] -= 0.5 * dx[ax]
                    g = oracle.geometry_point(kind, M, a, x)
                    al[c, ax] = g["alpha"]; e[c, ax] = g["e"]
    return al, e


def test_max_speed_minkowski_is_the_largest_direction_cosine(oracle):
    """flat space, Cartesian tetrad: n^a / n^0 = nhat^a, so the bound per axis is max_n |nhat^a| exactly (R9)"""
    for angles in (("geodesic", 2), ("latlon", 3, 8)):
        A = oracle.Angles(*angles)
        P = oracle.Problem(A, (3, 2, 2), (0.0, 0.0, 0.0), (0.5, 0.4, 0.3), metric_kind=0)
        v, vax = P.max_speed()
        assert tuple(vax) == tuple(np.abs(A.nhat).max(0))
        assert v == max(vax)


def test_max_speed_and_face_signs_kerr_schild_against_geometry_point(oracle):
    """Kerr-Schild: |n^a / n^0| with n^a = e^a_0hat + e^a_bhat nhat^b and n^0 = e^0_0hat = 1 / alpha (Eq.11, R2) evaluated by numpy from
    geometry_point at every lower face centre (ghost cells included) reproduces orc_max_speed; the signs of the same n^a reproduce
    orc_upwind_tables' face table (Eq.24).  A shared misreading of the face record (n^0 taken for alpha, a transposed tetrad row, the
    cell centre instead of the face centre) fails here."""
    kind, M, a = 1, 1.0, 0.9
    x0, dx = (2.5, -1.0, 0.5), (0.4, 0.5, 0.3)
    A = oracle.Angles("geodesic", 2)
    P = oracle.Problem(A, (3, 4, 2), x0, dx, metric_kind=kind, M=M, a=a)
    al, e = face_geometry(oracle, P, kind, M, a, x0, dx)
    n4 = np.concatenate([np.ones((A.N, 1)), A.nhat], 1)
    assert np.abs(e[:, :, 0, 1:]).max() == 0.0 and np.abs(e[:, :, 0, 0] * al - 1).max() < 1e-14   # e^0_ahat = (1/alpha, 0, 0, 0)
    na = np.stack([e[:, ax, ax + 1, :] @ n4.T for ax in range(3)], 1)        # [ncell][3][N]: n^a through the lower face along a
    speed = np.abs(na) * al[:, :, None]
    v, vax = P.max_speed()
    assert np.abs(np.array(vax) - speed.max((0, 2))).max() < 1e-13
    assert v == max(vax) and 0.5 < v < 3.0          # light in Kerr-Schild coordinates near the hole: of order one, not alpha^2 or 1/alpha^2 off
    far = oracle.Problem(A, (2, 2, 2), (400.0, 300.0, 200.0), dx, metric_kind=kind, M=M, a=a)
    assert abs(far.max_speed()[0] - np.abs(A.nhat).max()) < 2e-2      # far from the hole the flat-space value comes back
    fs, es = P.upwind_tables()
    sure = np.abs(na) > 1e-12
    assert np.array_equal(fs[sure], np.sign(na[sure]).astype(np.int8))
    assert set(np.unique(fs)) <= {-1, 0, 1} and (fs == 1).any() and (fs == -1).any()


def test_edge_sign_table_is_the_sign_of_the_edge_coefficient(oracle):
    """orc_upwind_tables' edge table = sgn c_e cell by cell, with c_e from orc_edge_coeffs (pinned against Eq.16b,c in
    test_oracle_geometry.py) and, independently, as the numpy contraction -S[c][k] N^c (n^a n^b)_k of the cell record with the edge's
    midpoint direction and in-sphere normal (Eq.16-17, Eq.25)"""
    A = oracle.Angles("geodesic", 3)
    P = oracle.Problem(A, (3, 2, 2), (3.0, 2.0, 1.0), (0.3, 0.25, 0.2), metric_kind=1, M=1.0, a=0.9)
    _, es = P.upwind_tables(faces=False)
    cell = P.geometry()[0]
    n4 = np.concatenate([np.ones((A.E, 1)), A.edge_mid], 1)
    iu = [(p, q) for p in range(4) for q in range(p, 4)]
    quad = np.stack([n4[:, p] * n4[:, q] for p, q in iu], 1)                 # [E][10], the order 00,01,02,03,11,12,13,22,23,33
    for c in range(P.ncell):
        ce, _ = P.edge_coeffs(c)
        assert np.array_equal(es[c], np.sign(ce).astype(np.int8))
        S = cell[c, 33:63].reshape(3, 10)
        ce_np = -np.einsum("ck,ec,ek->e", S, A.edge_nrm, quad)
        sure = np.abs(ce_np) > 1e-12 * np.abs(S).max()
        assert np.abs(ce_np - ce).max() < 1e-13 * max(1.0, np.abs(S).max())
        assert np.array_equal(es[c][sure], np.sign(ce_np[sure]).astype(np.int8))
    assert (es == 1).any() and (es == -1).any()
