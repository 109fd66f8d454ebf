"""Pins P3-P6 of the oracle's geometry: 3+1 split, tetrad, Ricci rotation coefficients and the
angular "velocities" (paper section 2.1-2.2)."""
import numpy as np
import pytest

ETA = np.diag([-1.0, 1, 1, 1])
PTS = [(3.0, 2.0, 1.5), (-4.0, 1.0, 0.3), (2.6, 2.7, 2.9), (10.0, -7.0, 5.0)]


def ks_metric(x, M, a):
    """test-local Cartesian Kerr-Schild metric (textbook form g = eta + f l l), independent of the oracle"""
    X, Y, Z = x
    R2 = X * X + Y * Y + Z * Z
    r2 = 0.5 * (R2 - a * a + np.sqrt((R2 - a * a) ** 2 + 4 * a * a * Z * Z))
    r = np.sqrt(r2)
    f = 2 * M * r**3 / (r**4 + a * a * Z * Z)
    l = np.array([1.0, (r * X + a * Y) / (r2 + a * a), (r * Y - a * X) / (r2 + a * a), Z / r])
    return ETA + f * np.outer(l, l)


def christoffel_fd(x, M, a, h=1e-4):
    """Gamma^e_{ds} by 4th-order central differences of the test-local metric"""
    dg = np.zeros((4, 4, 4))  # dg[d][m][n] = d_d g_mn
    for i in range(3):
        def gs(s):
            y = np.array(x, float); y[i] += s * h
            return ks_metric(y, M, a)
        dg[i + 1] = (8 * (gs(1) - gs(-1)) - (gs(2) - gs(-2))) / (12 * h)
    gi = np.linalg.inv(ks_metric(x, M, a))
    G = np.zeros((4, 4, 4))
    for e in range(4):
        for d in range(4):
            for s in range(4):
                G[e, d, s] = 0.5 * sum(gi[e, l] * (dg[d, l, s] + dg[s, l, d] - dg[l, d, s]) for l in range(4))
    return G


@pytest.mark.parametrize("a", [0.0, 0.5, 0.9])
@pytest.mark.parametrize("x", PTS)
def test_metric_split_and_tetrad(oracle, x, a):
    g = oracle.geometry_point(1, 1.0, a, x)
    G = ks_metric(x, 1.0, a)
    assert np.abs(g["g"] - G).max() < 1e-14
    assert np.abs(g["ginv"] @ G - np.eye(4)).max() < 1e-14
    # Eq.5a,c
    gi = np.linalg.inv(G)
    assert abs(g["alpha"] - (-gi[0, 0]) ** -0.5) < 1e-14
    assert np.abs(g["beta"] - g["alpha"] ** 2 * gi[0, 1:]).max() < 1e-14
    # Kerr-Schild: unit determinant => alpha^2 det(gamma) = 1
    assert abs(g["alpha"] ** 2 * np.linalg.det(G[1:, 1:]) - 1) < 1e-13
    e = g["e"]  # e[mu][ahat]
    # Eq.10 orthonormality
    assert np.abs(e.T @ G @ e - ETA).max() < 1e-14
    # Eq.11
    assert np.abs(e[:, 0] + g["alpha"] * gi[0, :]).max() < 1e-15
    # R2: Gram-Schmidt of d_x, d_y, d_z => e^0_ahat = 0 and the spatial block is upper triangular, positive diagonal
    assert (e[0, 1:] == 0).all() and e[2, 1] == 0 and e[3, 1] == 0 and e[3, 2] == 0
    assert (np.diag(e)[1:] > 0).all()
    # Eq.9: elow is the inverse tetrad
    assert np.abs(g["elow"] @ e - np.eye(4)).max() < 1e-14
    # n^alpha = e^alpha_ahat n^ahat is null and future directed with n^0 = 1/alpha
    for nh in ([1, 0, 0], [0, -1, 0], [0.6, 0, 0.8], [-0.48, 0.6, 0.64]):
        n = e @ np.array([1.0, *nh])
        assert abs(n @ G @ n) < 1e-14 and abs(n[0] - 1 / g["alpha"]) < 1e-15


def test_minkowski_omega_vanishes(oracle):
    """P4: Cartesian tetrad in flat space => all Ricci rotation coefficients vanish"""
    g = oracle.geometry_point(0, 1.0, 0.0, (0.3, -2.0, 5.0))
    assert (g["omega"] == 0).all() and np.array_equal(g["e"], np.eye(4)) and g["alpha"] == 1.0


@pytest.mark.parametrize("a", [0.0, 0.9])
@pytest.mark.parametrize("x", PTS[:3])
def test_omega_antisymmetry_and_definition(oracle, x, a):
    """Eq.17 against an independent evaluation: finite-difference covariant derivative of the
    oracle's tetrad FIELD with finite-difference Christoffels of the test-local metric."""
    g = oracle.geometry_point(1, 1.0, a, x)
    om = g["omega"]  # om[c][a][b] = omega^chat_{ahat bhat}
    # lowering the first index with eta gives omega_{c a b} antisymmetric in (c, a): metric compatibility
    low = np.einsum("cd,dab->cab", ETA, om)
    assert np.abs(low + low.transpose(1, 0, 2)).max() < 1e-13
    h = 1e-4
    de = np.zeros((4, 4, 4))  # de[d][mu][ahat]
    for i in range(3):
        def es(s):
            y = np.array(x, float); y[i] += s * h
            return oracle.geometry_point(1, 1.0, a, y)["e"]
        de[i + 1] = (8 * (es(1) - es(-1)) - (es(2) - es(-2))) / (12 * h)
    Gam = christoffel_fd(x, 1.0, a)
    e, elow = g["e"], g["elow"]
    cov = de + np.einsum("eds,sa->dea", Gam, e)  # cov[d][eps][ahat] = nabla_d e^eps_ahat
    ref = np.einsum("ce,db,dea->cab", elow, e, cov)
    assert np.abs(ref - om).max() < 1e-9


def accel(om, nh):
    """R5: a^c = -omega^c_{ab} n^a n^b + n^c omega^0_{ab} n^a n^b, rate of change of the unit direction"""
    n4 = np.array([1.0, *nh])
    w = np.einsum("cab,a,b->c", om, n4, n4)
    return -w[1:] + np.asarray(nh) * w[0]


@pytest.mark.parametrize("a", [0.0, 0.9])
def test_direction_rate_matches_geodesic(oracle, a):
    """P6: a^c(n) equals d n^chat / d lambda along a null geodesic integrated independently (RK4 on the
    coordinate geodesic equation with finite-difference Christoffels of the test-local metric)."""
    M = 1.0
    x0 = np.array([3.0, 2.0, 1.5])
    g0 = oracle.geometry_point(1, M, a, x0)
    for nh in ([0.6, 0.0, 0.8], [-0.48, 0.6, 0.64], [0.0, 1.0, 0.0], [2 / 3, -2 / 3, 1 / 3]):
        nh = np.array(nh)
        k0 = g0["e"] @ np.array([1.0, *nh])  # k^mu with tetrad-frame frequency 1

        def rhs(s):
            x, k = s[:4], s[4:]
            G = christoffel_fd(x[1:], M, a)
            return np.concatenate([k, -np.einsum("eds,d,s->e", G, k, k)])

        def run(ds, nstep=4):
            s = np.concatenate([[0.0], x0, k0])
            for _ in range(nstep):
                k1 = rhs(s); k2 = rhs(s + 0.5 * ds * k1); k3 = rhs(s + 0.5 * ds * k2); k4 = rhs(s + ds * k3)
                s = s + ds / 6 * (k1 + 2 * k2 + 2 * k3 + k4)
            gq = oracle.geometry_point(1, M, a, s[1:4])
            kh = gq["elow"] @ s[4:]
            return kh[1:] / kh[0]

        d = 2e-3
        # d lambda = k^0hat ds and k^0hat = 1 at the centre point: central difference in the affine parameter
        rate = (run(d / 4) - run(-d / 4)) / (2 * d)
        ac = accel(g0["omega"], nh)
        assert abs(ac @ nh) < 1e-14          # stays a unit vector
        assert np.abs(rate - ac).max() < 2e-7, (rate, ac)
        assert np.linalg.norm(ac) > 1e-3      # the check is not vacuous


def _one_cell(oracle, A, x, a, kind=1):
    dx = 0.2
    P = oracle.Problem(A, (1, 1, 1), tuple(np.array(x) - 0.5 * dx), (dx, dx, dx), metric_kind=kind, M=1.0, a=a)
    return P, P.cell_index(2, 2, 2)


@pytest.mark.parametrize("a", [0.0, 0.9])
def test_latlon_coefficients_are_eq16(oracle, a):
    """P5: on the lat-lon grid the oracle's edge coefficients c_e (pinned 30-term chain) equal the paper's
    n^zeta (Eq.16b) on zeta-faces and n^psi (Eq.16c) on psi-faces, evaluated literally."""
    x = (3.0, 2.0, 1.5)
    A = oracle.Angles("latlon", 6, 12)
    P, c = _one_cell(oracle, A, x, a)
    ce, n0e = P.edge_coeffs(c)
    g = oracle.geometry_point(1, 1.0, a, x)
    om = g["omega"]
    for e in range(A.E):
        nh = A.edge_mid[e]
        n4 = np.array([1.0, *nh])
        w = np.einsum("cab,a,b->c", om, n4, n4)  # n^a n^b omega^c_ab
        s = np.sqrt(1 - nh[2] ** 2)
        lo, hi = A.edge_lo[e], A.edge_hi[e]
        if lo // 12 != hi // 12:
            lit = (n4[0] * w[3] - n4[3] * w[0]) / s          # Eq.16b: s^-1 n n n^[0 omega^3]
        else:
            lit = (n4[2] * w[1] - n4[1] * w[2]) / s**2       # Eq.16c: s^-2 n n n^[2 omega^1]
            # orientation lo -> hi is increasing psi except across the psi = 2 pi wrap
            if hi - lo != 1:
                lit = -lit
        assert abs(ce[e] - lit) < 1e-14, (e, ce[e], lit)
        # n_0 at the edge direction = g_{0 mu} e^mu_ahat n^ahat
        assert abs(n0e[e] - (g["g"][0] @ g["e"] @ n4)) < 1e-15
    assert np.abs(ce).max() > 1e-3


@pytest.mark.parametrize("a", [0.5])
def test_geodesic_coefficients(oracle, a):
    """c_e = a(n_e) . N_e on the geodesic grid; exactly zero in Minkowski (P4)."""
    x = (2.6, 2.7, 2.9)
    A = oracle.Angles("geodesic", 3)
    P, c = _one_cell(oracle, A, x, a)
    ce, _ = P.edge_coeffs(c)
    om = oracle.geometry_point(1, 1.0, a, x)["omega"]
    ref = np.array([accel(om, A.edge_mid[e]) @ A.edge_nrm[e] for e in range(A.E)])
    assert np.abs(ce - ref).max() < 1e-15
    P0, c0 = _one_cell(oracle, A, x, 0.0, kind=0)
    ce0, n0e0 = P0.edge_coeffs(c0)
    assert (ce0 == 0).all() and (n0e0 == -1).all()


def test_cell_and_face_tables(oracle):
    """the packed tables the stage uses are the point geometry at cell centres (R6: and at face centres)"""
    A = oracle.Angles("latlon", 2, 4)
    P = oracle.Problem(A, (2, 3, 2), (3.0, 2.0, 1.0), (0.5, 0.25, 0.5), metric_kind=1, M=1.0, a=0.9)
    cell, face, ex = P.geometry()
    k, j, i = 3, 4, 2
    c = P.cell_index(k, j, i)
    xc = (3.0 + (i - 2 + 0.5) * 0.5, 2.0 + (j - 2 + 0.5) * 0.25, 1.0 + (k - 2 + 0.5) * 0.5)
    g = oracle.geometry_point(1, 1.0, 0.9, xc)
    assert cell[c, 0] == g["alpha"] and np.array_equal(cell[c, 1:17].reshape(4, 4), g["e"])
    assert np.allclose(cell[c, 17:33].reshape(4, 4), g["g"] @ g["e"], atol=1e-15)
    S = cell[c, 33:63].reshape(3, 10)
    pairs = [(p, q) for p in range(4) for q in range(p, 4)]
    for ch in range(3):
        for kk, (p, q) in enumerate(pairs):
            w = g["omega"][ch + 1, p, q] + (g["omega"][ch + 1, q, p] if p != q else 0.0)
            assert S[ch, kk] == w
    assert np.array_equal(cell[c, 63:66], g["beta"])
    assert np.array_equal(cell[c, 66:72], g["g"][1:, 1:][np.triu_indices(3)])
    for ax in range(3):
        xf = list(xc); xf[ax] -= 0.5 * (0.5, 0.25, 0.5)[ax]
        gf = oracle.geometry_point(1, 1.0, 0.9, xf)
        assert np.allclose(face[c, ax, :4], gf["e"][ax + 1], atol=1e-15)
        assert np.allclose(face[c, ax, 4:], gf["g"][0] @ gf["e"], atol=1e-15)
        assert abs(face[c, ax, 4] + gf["alpha"]) < 1e-15   # E_0hat = -alpha
