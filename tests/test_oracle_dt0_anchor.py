"""The oracle's fluid increment dT^0_alpha against its long-double evaluation (tests/dt0_exact.py): how many eps |R^0_0| each of the
oracle's two forms (sum of differences; difference of two sums, P:L472 literally) sits from the exact-arithmetic result.
This anchors parity_util.dt0_floor to something other than a failed run ("What's weak" 1)."""
import numpy as np
import pytest

import dt0_exact as X
from parity_util import TOL_FLUID, dt0_floor

EPS = 2.0 ** -53


def problem(oracle, angles, n=(6, 5, 4), seed=5, **kw):
    A = oracle.Angles(*angles)
    P = oracle.Problem(A, n, (3.0, 2.0, 1.0), (0.3, 0.25, 0.2), metric_kind=1, M=1.0, a=0.9, n0_crit=0.0, **kw)
    rng = np.random.default_rng(seed)
    nc = P.ncell
    I = np.exp(rng.normal(size=(nc, A.N)))
    fluid = np.stack([rng.uniform(0.5, 2, nc), rng.uniform(0.3, 1.5, nc)] + [rng.uniform(-0.4, 0.4, nc) for _ in range(3)])
    opac = np.stack([rng.uniform(0.1, 30, nc), rng.uniform(0.1, 30, nc), rng.uniform(0.1, 30, nc)])
    return A, P, I, fluid, opac


def near_equilibrium(A, P, I, fluid, opac, a_rad=1.0, amp=1e-9, seed=6):
    """the floor's regime: radiation isotropic in the fluid frame at the gas temperature (Ibar = a_rad T^4 / 4 pi, Planck mean = energy
    mean), perturbed by `amp` relative noise -- the exact increment is ~amp |R^0_0|, far below the floor, while every term of its sum
    still carries a rounding of eps |I| dOmega"""
    n0bar = np.asarray(X.doppler_factors(P.geometry()[0], A.nhat, fluid), dtype=np.float64)
    rng = np.random.default_rng(seed)
    Ieq = (a_rad * fluid[1] ** 4 / (4 * np.pi))[:, None] / n0bar ** 4 * (1 + amp * rng.normal(size=I.shape))
    op = opac.copy(); op[1] = op[0]
    return Ieq, op


def k_of(dT0_impl, dT0_exact, R00, P):
    """per interior cell: max over alpha of |impl - exact| / (eps |R^0_0|)"""
    err = np.abs(dT0_impl.astype(X.LD) - dT0_exact)
    k = (err / (X.LD(EPS) * R00[None, :])).max(0)
    return P.interior(np.asarray(k, dtype=np.float64))


@pytest.mark.parametrize("angles", [("geodesic", 3), ("geodesic", 4), ("latlon", 5, 16)])
@pytest.mark.parametrize("literal", [0, 1])
@pytest.mark.parametrize("regime", ["far", "near"])
def test_oracle_increment_against_the_long_double_sum(oracle, angles, literal, regime):
    """each form of the oracle's increment sits within HALF the parity bar of the exact-arithmetic value: 0.5e-10 |dT^0_alpha| or
    2 sqrt(N) eps |R^0_0|, whichever is larger -- so that two implementations that both do are within the whole bar of each other.
    `far`: random intensities (increment ~ |R^0_0|); `near`: equilibrium + 1e-9 noise (every cell below the floor)"""
    X.assert_long_double_is_extended()
    A, P, I, fluid, opac = problem(oracle, angles, dt0_literal=literal)
    if regime == "near":
        I, opac = near_equilibrium(A, P, I, fluid, opac)
    cell = P.geometry()[0]
    dt = 0.03
    exact, Tex, ok, R00 = X.coupling_increment(cell, A.nhat, A.domega, fluid, opac, I, dt, 5.0 / 3.0, 1.0)
    Ic = I.copy()
    T_o, dT0_o, nf = P.coupling(Ic, fluid, opac, dt)
    assert nf == 0 and P.interior(ok).all()
    # the long-double temperature agrees with the oracle's to FP64 rounding (the two solve the same quartic)
    assert np.abs(P.interior(T_o) / P.interior(np.asarray(Tex, dtype=np.float64)) - 1).max() < 1e-14
    k = k_of(dT0_o, exact, R00, P)
    bound = 2.0 * np.sqrt(A.N)
    R = np.asarray(R00, dtype=np.float64); ex = np.asarray(exact, dtype=np.float64)
    size = P.interior(np.abs(ex).max(0) / R)      # |increment| / |R^0_0| per cell
    print(f"{angles} literal={literal} {regime}: k max {k.max():.2f}, median {np.median(k):.2f} (2 sqrt(N) = {bound:.1f}); |dT0|/|R00| median {np.median(size):.1e}")
    err = np.abs(dT0_o - ex)
    bar = np.maximum(0.5 * TOL_FLUID * np.abs(ex), bound * EPS * R[None, :])
    assert (P.interior((err <= bar).all(0))).all()
    # the floor is exactly twice that bound: TOL_FLUID * dt0_floor(N) = 4 sqrt(N) eps
    assert abs(TOL_FLUID * dt0_floor(A.N) / (2 * bound * EPS) - 1) < 1e-12
    if regime == "near":   # every cell is in the floor's regime, and there the k bound alone must hold
        assert size.max() < dt0_floor(A.N) and k.max() <= bound
    else:                  # the anchor is not vacuous: increments of the size of R^0_0 itself are reproduced to 1e-13
        assert np.median(size) > 1e-3
        assert (P.interior((err <= 1e-13 * np.abs(ex).max(0) + bound * EPS * R).all(0))).all()
