"""Pins P1, P2 of the oracle's angle grids (paper section 2.6)."""
import numpy as np
import pytest


@pytest.mark.parametrize("nlev", [1, 2, 3, 4, 6])
def test_geodesic_counts_and_topology(oracle, nlev):
    A = oracle.Angles("geodesic", nlev)
    # N = 10 N_lev^2 + 2 cells, 12 of which are pentagons, the rest hexagons
    assert A.N == 10 * nlev * nlev + 2
    assert (A.nnbr == 5).sum() == 12 and (A.nnbr == 6).sum() == A.N - 12
    # Euler: a closed polyhedral sphere with N faces of degree 5/6 has E = (5*12 + 6*(N-12))/2 = 3N - 6 edges
    assert A.E == 3 * A.N - 6
    # index 0 is the north pole, "centered on a pentagonal cell"
    assert np.allclose(A.nhat[0], [0, 0, 1]) and A.nnbr[0] == 5
    # every unique edge sits in exactly two neighbour lists, once from each side
    cnt = np.zeros(A.E, int)
    for n in range(A.N):
        for s in range(A.nnbr[n]):
            e, m = A.nbr_edge[n, s], A.nbr[n, s]
            cnt[e] += 1
            assert {n, m} == {A.edge_lo[e], A.edge_hi[e]} and A.edge_lo[e] < A.edge_hi[e]
            assert n in A.nbr[m, : A.nnbr[m]]
        assert (A.nbr[n, A.nnbr[n]:] == -1).all()
        assert A.nbr[n, 0] == A.nbr[n, : A.nnbr[n]].min()  # R3: list starts at the smallest-index neighbour
    assert (cnt == 2).all()


@pytest.mark.parametrize("nlev", [1, 2, 3, 4])
def test_geodesic_geometry(oracle, nlev):
    A = oracle.Angles("geodesic", nlev)
    assert np.allclose(np.linalg.norm(A.nhat, axis=1), 1, atol=1e-15)
    # cells tile the sphere
    assert abs(A.domega.sum() - 4 * np.pi) < 1e-13
    # P2: icosahedral symmetry => the quadrature integrates l=1 and l=2 exactly
    assert np.abs((A.domega[:, None] * A.nhat).sum(0)).max() < 1e-14
    assert np.abs(np.einsum("n,ni,nj->ij", A.domega, A.nhat, A.nhat) - 4 * np.pi / 3 * np.eye(3)).max() < 1e-13
    # edges: midpoint and normal are unit, orthogonal, and the normal points lo -> hi
    assert np.allclose(np.linalg.norm(A.edge_mid, axis=1), 1, atol=1e-15)
    assert np.allclose(np.linalg.norm(A.edge_nrm, axis=1), 1, atol=1e-15)
    assert np.abs((A.edge_mid * A.edge_nrm).sum(1)).max() < 1e-15
    d = A.nhat[A.edge_hi] - A.nhat[A.edge_lo]
    assert ((A.edge_nrm * d).sum(1) > 0).all()
    # closure of each cell's perimeter.  Exact identity on the unit sphere for a region S with outward
    # in-sphere boundary normal N:  oint N dl = -2 int_S n dOmega  (|int_S n dOmega| -> dOmega for small cells).
    # It ties edge lengths, normals' outward orientation and the cell's solid angle and centre together.
    for n in range(0, A.N, 5):
        acc = np.zeros(3)
        for s in range(A.nnbr[n]):
            e = A.nbr_edge[n, s]
            sg = 1.0 if A.edge_lo[e] == n else -1.0
            acc += sg * A.edge_len[e] * A.edge_nrm[e]
        assert np.linalg.norm(acc + 2.0 * A.domega[n] * A.nhat[n]) < (0.1 / nlev) * 2.0 * A.domega[n]
    # icosahedron (level 1): 12 equal pentagons of 4 pi / 12, edges of equal length
    if nlev == 1:
        assert np.allclose(A.domega, 4 * np.pi / 12, atol=1e-14)
        # a face of the spherical dodecahedron has edge length acos(sqrt(5)/3)
        assert np.allclose(A.edge_len, np.arccos(np.sqrt(5) / 3), atol=1e-14)


def test_geodesic_first_occurrence_order(oracle):
    """R3: canonical index = first occurrence looping faces, i, j; face 0 = (V0, U_0, U_1)."""
    L = 4
    A = oracle.Angles("geodesic", L)
    c, s = 2 / np.sqrt(5), 1 / np.sqrt(5)
    V0 = np.array([0, 0, 1.0]); U0 = np.array([c, 0, s]); U1 = np.array([c * np.cos(2 * np.pi / 5), c * np.sin(2 * np.pi / 5), s])
    n = 0
    for i in range(L + 1):
        for j in range(L + 1 - i):
            p = V0 + (U0 - V0) * i / L + (U1 - V0) * j / L
            assert np.allclose(A.nhat[n], p / np.linalg.norm(p), atol=1e-15)
            n += 1


@pytest.mark.parametrize("nz,npsi", [(5, 16), (4, 8), (1, 4), (2, 4), (3, 1), (8, 16)])
def test_latlon(oracle, nz, npsi):
    A = oracle.Angles("latlon", nz, npsi)
    N = nz * npsi
    assert A.N == N
    # equal solid angles
    assert np.allclose(A.domega, 4 * np.pi / N, rtol=0, atol=1e-15)
    assert A.E == (nz - 1) * npsi + (nz * npsi if npsi > 1 else 0)  # 2N - N_psi for npsi>1
    mu = A.nhat[:, 2].reshape(nz, npsi)
    # equally spaced in cos(zeta) from +1 to -1 (faces) => centres at 1 - (2l+1)/nz
    assert np.allclose(mu, (1 - (2 * np.arange(nz) + 1) / nz)[:, None], atol=1e-15)
    psi = np.arctan2(A.nhat[:, 1], A.nhat[:, 0]) % (2 * np.pi)
    assert np.allclose(psi.reshape(nz, npsi), ((np.arange(npsi) + 0.5) * 2 * np.pi / npsi)[None, :], atol=1e-14)
    # slots: zeta-, zeta+, psi-, psi+; no neighbour across the poles
    nbr = A.nbr.reshape(nz, npsi, 6)
    assert (nbr[0, :, 0] == -1).all() and (nbr[-1, :, 1] == -1).all()
    for l in range(nz):
        for m in range(npsi):
            if l > 0: assert nbr[l, m, 0] == (l - 1) * npsi + m
            if l < nz - 1: assert nbr[l, m, 1] == (l + 1) * npsi + m
            if npsi > 1:
                assert nbr[l, m, 2] == l * npsi + (m - 1) % npsi and nbr[l, m, 3] == l * npsi + (m + 1) % npsi
    # Eq.20f weights: total zeta-face length on a parallel = its circumference 2 pi sin(zeta_f);
    # psi-face weights Delta(cos zeta) sum to 2 along a meridian
    for e in range(A.E):
        lo, hi = A.edge_lo[e], A.edge_hi[e]
        if lo // npsi != hi // npsi:  # zeta-face
            sf = np.sqrt(1 - A.edge_mid[e, 2] ** 2)
            assert abs(A.edge_len[e] - sf * 2 * np.pi / npsi) < 1e-15
            # normal = unit vector of increasing zeta: orthogonal to n_e, z-component -sin(zeta)
            assert abs(A.edge_nrm[e] @ A.edge_mid[e]) < 1e-15 and abs(A.edge_nrm[e, 2] + sf) < 1e-15
        else:
            assert abs(A.edge_len[e] - 2.0 / nz) < 1e-15
            s = np.sqrt(1 - A.edge_mid[e, 2] ** 2)
            # normal = e_psi / sin(zeta): horizontal, length 1/s, orthogonal to n_e
            assert abs(A.edge_nrm[e, 2]) == 0 and abs(np.linalg.norm(A.edge_nrm[e]) - 1 / s) < 1e-14
            assert abs(A.edge_nrm[e] @ A.edge_mid[e]) < 1e-15
    # P2 (midpoint-rule quadrature): second moment diag (1 - 1/nz^2)/3 x2 ... closed form for this grid:
    # sum_l mu_l^2 / nz = (1 - 1/nz^2)/3
    M2 = np.einsum("n,ni,nj->ij", A.domega, A.nhat, A.nhat) / (4 * np.pi)
    assert abs(M2[2, 2] - (1 - 1 / nz**2) / 3) < 1e-15
    if npsi >= 3:
        assert abs(M2[0, 0] - (1 - M2[2, 2]) / 2) < 1e-15 and abs(M2[0, 1]) < 1e-15


def test_pinned_edge_products(oracle):
    """edge_T[e][c][k] = N^c * (n^alpha n^beta), two roundings, in the order the sign chain uses."""
    A = oracle.Angles("geodesic", 3)
    n4 = np.concatenate([np.ones((A.E, 1)), A.edge_mid], axis=1)
    q = np.stack([n4[:, a] * n4[:, b] for a in range(4) for b in range(a, 4)], axis=1)
    T = (A.edge_nrm[:, :, None] * q[:, None, :]).reshape(A.E, 30)
    assert np.array_equal(T, A.edge_T)
