"""Pins of the oracle's optical-depth-aware spatial flux (NEXT-1: paper Eq.26-29; readings R15-R18, G1 in
DESIGN.md).  What the paper and the mathematics fix:
  * "a value of 0 reduces to the free-streaming case": tau_factor = 0 is Eq.24 bit for bit, and the flux tends to
    it continuously -- quadratically in tau, because the interpolating factor is 1 - exp(-tau^2) (this is what decides the
    garbled Eq.27: the printed -exp(-tau^2) would NOT reduce to free streaming at tau = 0);
  * the correction only acts on velocity DIFFERENCES between the two cells of a face: g_L = g_R = g when the fluid
    moves uniformly, so Eq.28 is Eq.24 for any optical depth;
  * the face flux stays single valued, so the scheme stays conservative;
  * the factor saturates for tau >> 1 (f -> 1).
The sign and form of g_L/R (Eq.29) have no anchor of this kind: "parity unpinned" for them."""
import numpy as np
import pytest


def setup(oracle, tau, kind=0, a=0.0, n=(7, 6, 5), uniform_v=None, seed=5):
    A = oracle.Angles("geodesic", 2)
    P = oracle.Problem(A, n, (3.0, 2.5, 2.0), (0.3, 0.3, 0.3), metric_kind=kind, M=1.0, a=a, recon_space=1, couple=0, tau_factor=tau)
    rng = np.random.default_rng(seed)
    I = np.exp(rng.normal(size=(P.ncell, A.N)))
    fluid = np.stack([rng.uniform(0.5, 2, P.ncell), rng.uniform(0.3, 1.5, P.ncell)] + [rng.uniform(-0.4, 0.4, P.ncell) for _ in range(3)])
    if uniform_v is not None:
        for q in range(3):
            fluid[2 + q] = uniform_v[q]
    opac = np.stack([rng.uniform(0.1, 30, P.ncell)] * 2 + [rng.uniform(0.1, 30, P.ncell)])
    return A, P, I, fluid, opac


def test_tau_zero_is_free_streaming(oracle):
    A, P, I, fluid, opac = setup(oracle, 0.0, kind=1, a=0.9)
    assert np.array_equal(P.transport_tau(I, 0.02, fluid, opac), P.transport(I, 0.02))


def test_small_tau_tends_to_free_streaming_quadratically(oracle):
    """P:L304 and Eq.27 with G1: the deviation from Eq.24 is O(tau^2) as tau -> 0 (f = 1 - exp(-tau^2) ~ tau^2)"""
    dev = []
    for tau in (1e-3, 2e-3):
        A, P, I, fluid, opac = setup(oracle, tau)
        free = P.interior(P.transport(I, 0.02))
        dev.append(np.abs(P.interior(P.transport_tau(I, 0.02, fluid, opac)) - free).max())
    assert 0 < dev[0] < 1e-6
    assert abs(dev[1] / dev[0] - 4.0) < 0.01


@pytest.mark.parametrize("tau", [0.3, 5.0])
def test_uniform_flow_is_free_streaming(oracle, tau):
    """Eq.28-29: with the same velocity in both cells of every face g_L = g_R = g, so the factor is 1 at any optical depth"""
    A, P, I, fluid, opac = setup(oracle, tau, uniform_v=(0.3, -0.2, 0.1))
    got, free = P.interior(P.transport_tau(I, 0.02, fluid, opac)), P.interior(P.transport(I, 0.02))
    assert np.abs(got - free).max() < 1e-13 * np.abs(free).max()
    # ... and it is not trivially inactive: with velocity differences the flux does change
    A, P, I, fluid, opac = setup(oracle, tau)
    assert np.abs(P.interior(P.transport_tau(I, 0.02, fluid, opac)) - P.interior(P.transport(I, 0.02))).max() > 1e-4


@pytest.mark.parametrize("kind,a", [(0, 0.0), (1, 0.9)])
def test_conservation_with_optical_depth_flux(oracle, kind, a):
    """every face flux is single valued also with Eq.28, so sum n^0 n_0 I dOmega dV is conserved"""
    A, P, I, fluid, opac = setup(oracle, 3.0, kind=kind, a=a, n=(10, 9, 8))
    cell, _, _ = P.geometry()
    n4 = np.concatenate([np.ones((A.N, 1)), A.nhat], 1)
    w = (cell[:, 1:5] @ n4.T) * (cell[:, 17:21] @ n4.T)     # n^0 n_0 per (cell, angle)
    Ic = np.zeros(P.shape + (A.N,))
    Ic[5:-5, 5:-5, 5:-5] = I.reshape(P.shape + (A.N,))[5:-5, 5:-5, 5:-5]  # compact support
    Ic = Ic.reshape(-1, A.N)
    vmax, _ = P.max_speed()
    out = P.transport_tau(Ic, 0.3 * 0.3 / vmax, fluid, opac)
    out_full = np.zeros_like(Ic)
    P.interior(out_full)[...] = P.interior(out)
    E0 = (w * Ic * A.domega).sum(); E1 = (w * out_full * A.domega).sum()
    assert abs(E1 - E0) < 1e-13 * abs(E0)


def test_factor_saturates_at_large_optical_depth(oracle):
    """f = 1 - exp(-tau^2) -> 1: for tau >> 1 the flux no longer depends on the constant of Eq.26"""
    outs = []
    for tau in (1e4, 1e5):   # tau >= 1e4 * 0.2 * 0.02 = 40 at every face
        A, P, I, fluid, opac = setup(oracle, tau)
        outs.append(P.interior(P.transport_tau(I, 0.02, fluid, opac)))
    assert np.array_equal(outs[0], outs[1])


def test_stage_uses_the_flux(oracle):
    """orc_stage = fill, transport with Eq.28, coupling: same as calling the pieces"""
    A, P, I, fluid, opac = setup(oracle, 2.0, kind=1, a=0.5)
    P2 = oracle.Problem(A, P.n, (3.0, 2.5, 2.0), (0.3, 0.3, 0.3), metric_kind=1, M=1.0, a=0.5, recon_space=1, couple=1, tau_factor=2.0)
    out, T, dT0, nf = P2.stage(I.copy(), fluid, opac, 0.02)
    ref = P2.transport_tau(I, 0.02, fluid, opac)
    P2.coupling(ref, fluid, opac, 0.02)
    assert np.array_equal(P2.interior(out), P2.interior(ref))
