"""The CUDA coupling's fluid increment dT^0_alpha against the long-double evaluation of tests/dt0_exact.py, next to the oracle's
("What's weak" 1): both must sit within half the parity bar of the exact-arithmetic value, in the regime where the
increment is of the size of R^0_0 and in the floor's regime (equilibrium + 1e-9 noise).  Both sides get the same geometry numbers (the
oracle's records through the tabulated metric), so the exact value is one number.  Also: parity against the oracle's LITERAL form
(difference of two sums) at the same floor."""
import numpy as np
import pytest
import torch

import dt0_exact as X
from parity_util import TOL_FLUID, dt0_floor, err_dT0, oracle_tables_to_rad, rel_err
from test_gpu_parity import B, dev  # noqa: F401
from test_oracle_dt0_anchor import EPS, k_of, near_equilibrium, problem

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("angles", [("geodesic", 3), ("geodesic", 4), ("latlon", 5, 16), ("latlon", 7, 9)])
@pytest.mark.parametrize("regime", ["far", "near"])
def test_cuda_increment_against_the_long_double_sum(oracle, B, angles, regime):
    """("latlon", 7, 9): odd N, the generic coupling kernel; the others the streaming kernel"""
    X.assert_long_double_is_extended()
    n = (9, 6, 5)
    A, P, I, fluid, opac = problem(oracle, angles, n=n)
    _, Plit, _, _, _ = problem(oracle, angles, n=n, dt0_literal=1)
    if regime == "near":
        I, opac = near_equilibrium(A, P, I, fluid, opac)
    cell, face, ex = P.geometry()
    dt = 0.03
    exact, Tex, ok, R00 = X.coupling_increment(cell, A.nhat, A.domega, fluid, opac, I, dt, 5.0 / 3.0, 1.0)
    rc, rf = oracle_tables_to_rad(cell, face, ex)
    dop = dev(opac)
    h = B.rad_create(dict(kind=2, cell_tab=dev(rc), face_tab=dev(rf)), dict(n=n, x0=(3.0, 2.0, 1.0), dx=(0.3, 0.25, 0.2)), angles,
                     (dop[0], dop[1], dop[2]), dict(n0_crit=0.0))
    try:
        dI = dev(I); dT = torch.zeros(P.ncell, dtype=torch.float64, device="cuda"); ddT0 = torch.zeros(4, P.ncell, dtype=torch.float64, device="cuda")
        nf = B.rad_couple(h, dI, dev(fluid), dt, dT, ddT0, count_noroot=True)
        torch.cuda.synchronize()
        got, T_g, I_g = ddT0.cpu().numpy(), dT.cpu().numpy(), dI.cpu().numpy()
    finally:
        B.rad_destroy(h)
    assert nf == 0 and P.interior(ok).all()
    Io = I.copy(); T_o, dT0_o, _ = P.coupling(Io, fluid, opac, dt)
    Il = I.copy(); _, dT0_l, _ = Plit.coupling(Il, fluid, opac, dt)
    bound = 2.0 * np.sqrt(A.N)
    R = np.asarray(R00, dtype=np.float64); exd = np.asarray(exact, dtype=np.float64)
    kg, ko = k_of(got, exact, R00, P), k_of(dT0_o, exact, R00, P)
    print(f"{angles} {regime}: k (units of eps |R00|) CUDA max {kg.max():.2f} median {np.median(kg):.2f}; oracle max {ko.max():.2f} median {np.median(ko):.2f}; 2 sqrt(N) = {bound:.1f}")
    bar = np.maximum(0.5 * TOL_FLUID * np.abs(exd), bound * EPS * R[None, :])
    assert P.interior((np.abs(got - exd) <= bar).all(0)).all()
    assert P.interior((np.abs(dT0_o - exd) <= bar).all(0)).all()
    if regime == "near":
        size = P.interior(np.abs(exd).max(0) / R)
        assert size.max() < dt0_floor(A.N) and kg.max() <= bound and ko.max() <= bound
    # temperature: all three agree to rounding
    assert rel_err(P.interior(T_g), P.interior(np.asarray(Tex, dtype=np.float64)), 0.0) <= 1e-13
    # parity with both forms of the oracle at the suite's bar and floor
    for ref, out in ((dT0_o, Io), (dT0_l, Il)):
        eD, _ = err_dT0(P, got, ref, out)
        assert eD <= TOL_FLUID
