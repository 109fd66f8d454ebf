"""Oracle pins for the stretched Cartesian grid (first item: the Delta A_a / Delta V arrays of Eq.20b,c).
With sqrt(-g) = 1 (Cartesian Kerr-Schild and Minkowski) a tensor-product grid with unequal cell widths has Delta V = dx dy dz and
Delta A_x = dy dz, so Delta A_a / Delta V = 1 / Delta x^a of the cell; geometry is evaluated at the true cell and face centres; reading
R22: reconstruction in index space, as on the uniform grid."""
import numpy as np
import pytest


def stretched_faces(n, ng, x0, dx, ratio, seed):
    """faces of n + 2 ng cells starting at x0 - ng dx (like the uniform grid) whose widths vary smoothly and randomly within [1/ratio, ratio] dx"""
    rng = np.random.default_rng(seed)
    m = n + 2 * ng
    w = dx * ratio ** np.clip(np.cumsum(rng.normal(0, 0.25, m)), -1, 1)
    return np.concatenate([[x0 - ng * dx], x0 - ng * dx + np.cumsum(w)])


def uniform_faces(n, ng, x0, dx):
    return np.array([x0 + (i - ng) * dx for i in range(n + 2 * ng + 1)])


def weights(P, A):
    cell, _, _ = P.geometry()
    n4 = np.concatenate([np.ones((A.N, 1)), A.nhat], 1)
    return (cell[:, 1:5] @ n4.T) * (cell[:, 17:21] @ n4.T)     # n^0 n_0 per (cell, angle)


@pytest.mark.parametrize("kind,a", [(0, 0.0), (1, 0.9)])
def test_uniform_faces_reproduce_the_uniform_grid_bit_for_bit(oracle, kind, a):
    A = oracle.Angles("geodesic", 2)
    n, x0, dx = (6, 5, 4), (3.0, 2.0, 1.0), (0.25, 0.5, 0.125)   # binary fractions: x0 + i dx is exact
    xf = [uniform_faces(n[d], 2, x0[d], dx[d]) for d in range(3)]
    Pu = oracle.Problem(A, n, x0, dx, metric_kind=kind, M=1.0, a=a, couple=0)
    Ps = oracle.Problem(A, n, x0, dx, metric_kind=kind, M=1.0, a=a, couple=0, xf=xf)
    for u, s in zip(Pu.geometry(), Ps.geometry()):
        assert np.array_equal(u, s)
    I = np.exp(np.random.default_rng(1).normal(size=(Pu.ncell, A.N)))
    assert np.array_equal(Pu.transport(I, 0.03), Ps.transport(I, 0.03))


def test_geometry_is_taken_at_the_true_cell_and_face_centres(oracle):
    A = oracle.Angles("latlon", 2, 4)
    n, x0, dx = (5, 4, 3), (3.0, 2.0, 1.5), (0.3, 0.25, 0.2)
    xf = [stretched_faces(n[d], 2, x0[d], dx[d], 1.6, 10 + d) for d in range(3)]
    P = oracle.Problem(A, n, x0, dx, metric_kind=1, M=1.0, a=0.7, couple=0, xf=xf)
    cell, face, _ = P.geometry()
    xc = [0.5 * (f[:-1] + f[1:]) for f in xf]
    for (k, j, i) in [(0, 0, 0), (3, 4, 6), (6, 7, 8), (2, 5, 1)]:
        c = P.cell_index(k, j, i)
        g = oracle.geometry_point(1, 1.0, 0.7, (xc[0][i], xc[1][j], xc[2][k]))
        assert abs(cell[c, 0] - g["alpha"]) < 1e-15 and np.allclose(cell[c, 1:5], g["e"][0], rtol=0, atol=1e-15)   # lapse, e^0_ahat
        for ax in range(3):   # the lower face along ax: face coordinate along ax, centre coordinates across (R6)
            x = [xc[0][i], xc[1][j], xc[2][k]]
            x[ax] = xf[ax][(i, j, k)[ax]]
            gf = oracle.geometry_point(1, 1.0, 0.7, x)
            assert np.allclose(face[c, ax, 0:4], gf["e"][1 + ax], rtol=0, atol=1e-15)       # e^a_ahat at the face
            assert np.allclose(face[c, ax, 4:8], gf["g"][0] @ gf["e"], rtol=0, atol=1e-14)        # E_ahat = g_{0 mu} e^mu_ahat


@pytest.mark.parametrize("recon", [0, 1])
def test_isotropic_uniform_field_is_a_fixed_point_in_minkowski(oracle, recon):
    """every face flux equals its neighbour's whatever the cell widths: the divergence vanishes bit for bit"""
    A = oracle.Angles("geodesic", 2)
    n, x0, dx = (7, 6, 5), (0.0, 0.0, 0.0), (0.1, 0.1, 0.1)
    xf = [stretched_faces(n[d], 2, x0[d], dx[d], 2.0, 20 + d) for d in range(3)]
    P = oracle.Problem(A, n, x0, dx, metric_kind=0, recon_space=recon, couple=0, xf=xf)
    I = np.full((P.ncell, A.N), 0.37)
    assert np.array_equal(P.interior(P.transport(I, 0.02)), P.interior(I))


@pytest.mark.parametrize("kind,a", [(0, 0.0), (1, 0.9)])
@pytest.mark.parametrize("recon", [0, 1])
def test_energy_conservation_with_cell_volumes(oracle, kind, a, recon):
    """P8 on the stretched grid: sum n^0 n_0 I dOmega dV with dV = dx_i dy_j dz_k is conserved (fluxes telescope only with the volume weights)"""
    A = oracle.Angles("geodesic", 2)
    n, x0, dx = (10, 9, 8), (3.0, 2.5, 2.0), (0.3, 0.3, 0.3)
    xf = [stretched_faces(n[d], 2, x0[d], dx[d], 1.8, 30 + d) for d in range(3)]
    P = oracle.Problem(A, n, x0, dx, metric_kind=kind, M=1.0, a=a, recon_space=recon, couple=0, xf=xf)
    w = weights(P, A)
    wd = [np.diff(f) for f in xf]
    dV = (wd[2][:, None, None] * wd[1][None, :, None] * wd[0][None, None, :]).reshape(-1, 1)
    rng = np.random.default_rng(11)
    I = np.zeros(P.shape + (A.N,))
    I[5:-5, 5:-5, 5:-5] = np.exp(rng.normal(size=(n[2] - 6, n[1] - 6, n[0] - 6, A.N)))  # compact support
    I = I.reshape(-1, A.N)
    dt = 0.3 * min(v.min() for v in wd) / P.max_speed()[0]
    out = P.transport(I, dt)
    full = np.zeros_like(I)
    P.interior(full)[...] = P.interior(out)
    E0 = (w * I * A.domega * dV).sum(); E1 = (w * full * A.domega * dV).sum()
    assert abs(E1 - E0) < 1e-13 * abs(E0)
    # ... and NOT without them: the widths matter
    E0u = (w * I * A.domega).sum(); E1u = (w * full * A.domega).sum()
    assert abs(E1u - E0u) > 1e-6 * abs(E0u)


def test_single_angle_pulse_moves_at_the_coordinate_speed(oracle):
    """donor cell on a stretched grid, one direction along +x in Minkowski: the first moment of C dV about the FACE positions advances by
    exactly n^x dt per unit of conserved energy (summation by parts with dV_i / dx_i = dy dz and x_{i+1/2} - x_{i-1/2} = dx_i)"""
    A = oracle.Angles("latlon", 2, 4)
    n, x0, dx = (24, 3, 3), (0.0, 0.0, 0.0), (0.1, 0.1, 0.1)
    xf = [stretched_faces(n[0], 2, 0.0, 0.1, 1.7, 41), None, None]
    P = oracle.Problem(A, n, x0, dx, metric_kind=0, recon_space=0, couple=0, xf=xf)
    m = int(np.argmax(A.nhat[:, 0]))                      # the angle with the largest n^x
    I = np.zeros(P.shape + (A.N,))
    I[:, :, 8:14, m] = np.random.default_rng(3).uniform(1, 2, (P.NK, P.NJ, 6))
    I[...] = I[3:4, 3:4, :, :]                            # uniform in y and z: only x fluxes act
    I = I.reshape(-1, A.N)
    dt = 0.02
    out = P.transport(I, dt).reshape(P.shape + (A.N,))
    w = np.diff(xf[0]); xup = xf[0][1:]                   # upper face of each cell
    row0, row1 = I.reshape(P.shape + (A.N,))[3, 3, :, m], out[3, 3, :, m]
    row1 = np.where(np.arange(P.NI) >= 2, row1, 0.0)       # ghosts of the output are not written
    E = (row0 * w).sum()
    assert abs((row1 * w).sum() - E) < 1e-14 * E
    # with donor cell and n^x > 0 a cell's content leaves through its upper face: the sum of C dV x_(upper face of the cell it
    # sits in, taken one cell behind) telescopes; the clean statement is for S = sum_i C_i w_i X_i with X_i = x_{i+1/2}:
    # S1 - S0 = n^x dt sum_i C_i (x_{i+3/2} - x_{i+1/2}) = n^x dt sum_i C_i w_{i+1}
    S0, S1 = (row0 * w * xup).sum(), (row1 * w * xup).sum()
    assert abs((S1 - S0) - A.nhat[m, 0] * dt * (row0[:-1] * w[1:]).sum()) < 1e-13 * abs(S0)
