"""rad_stage_static: the stage for callers that cannot allocate device memory while they run.

Who needs it: a step loop that has already given the rest of the card to its own memory pool, or that keeps several streams busy
and would lose them all to the device-wide wait inside cudaMalloc / cudaFree.  rad_stage's optical-depth-aware flux (tau_factor > 0)
takes a per-cell table from cudaMalloc on its first call; rad_stage_static keeps that table in a 4 MiB array built into librad.so
(at most RAD_STATIC_MAX_CELLS = 65 536 cells per block, ghost layers included) and never calls the allocator.

What is checked here, against the existing rad_stage on the same inputs: two calls in a row (the second on a smaller block with other
inputs, so that the shared array still holds the first call's table beyond the second block's cells), on the tile-kernel route and on
the generic-kernel route; the size limit's error; and that the card's free memory does not move across calls.

This file sorts after every other test file on purpose: `pytest -x` stops at the first failure, and a failure here must not hide the
parity tests.  It makes no assumption about what ran before it: the first call in a process does the array's address look-up, later
ones reuse it, and both orders pass.
"""
import numpy as np
import pytest
import torch

from parity_util import TOL_FLUID, TOL_I, err_dT0, rel_err, rel_err_I
from test_gpu_parity import B, dev, small_problem  # noqa: F401  (B is the module fixture)

pytestmark = pytest.mark.gpu


def run(stage, P, h, I, fluid, dt, I0=None, weights=(0.0, 1.0)):
    """one stage through `stage` (B.rad_stage or B.rad_stage_static) on fresh device buffers; host copies of every output"""
    dI = dev(I); dO = torch.zeros_like(dI); dfl = dev(fluid)
    dT = torch.zeros(P.ncell, dtype=torch.float64, device="cuda"); ddT0 = torch.full((4, P.ncell), 9.0, dtype=torch.float64, device="cuda")
    nf = stage(h, dI, dO, None if I0 is None else dev(I0), dfl, weights[0], weights[1], dt, dT, ddT0, count_noroot=True)
    torch.cuda.synchronize()
    return dict(I_in=dI.cpu().numpy(), I=dO.cpu().numpy(), T=dT.cpu().numpy(), dT0=ddT0.cpu().numpy(), noroot=nf)


def same(P, got, want):
    """the new entry point against the existing path: within the parity tolerances of the suite (they run the same kernels on the
    same numbers, so the arrays are in fact identical, which is asserted too)"""
    assert got["noroot"] == want["noroot"]
    assert np.array_equal(got["I_in"], want["I_in"])  # ghost fill
    assert rel_err_I(P.interior(got["I"]), P.interior(want["I"])) <= TOL_I
    assert rel_err(P.interior(got["T"]), P.interior(want["T"]), 0.0) <= TOL_FLUID
    eD, _ = err_dT0(P, got["dT0"], want["dT0"], want["I"])
    assert eD <= TOL_FLUID
    for k in ("I", "T", "dT0"):
        assert np.array_equal(got[k], want[k]), k


@pytest.mark.parametrize("route", ["tile", "generic"])
def test_two_calls_in_a_row_match_rad_stage(oracle, B, route):
    """call 1 on a 9 x 6 x 5 block, call 2 straight after it on a 5 x 4 x 3 block with other inputs and another tau_factor: each equals
    rad_stage on its own context.  `tile`: the k_tau_table + k_stage5<TAU> route; `generic`: k_cell_velocity + k_fluxdiv<TAU>
    (no stored coefficients), which lays the shared array out differently (5 doubles per cell instead of 8)."""
    extra = dict(recompute_edge_coeffs=1) if route == "generic" else {}
    big = small_problem(oracle, B, (9, 6, 5), ("geodesic", 3), bc=(1, 2, 0, 1, 2, 0), tau_factor=2.0, seed=7, **extra)
    small = small_problem(oracle, B, (5, 4, 3), ("geodesic", 3), bc=(2, 1, 1, 2, 1, 1), tau_factor=0.7, seed=8, **extra)
    try:
        (A1, P1, h1, I1, f1, o1, _), (A2, P2, h2, I2, f2, o2, _) = big, small
        names = B.rad_stage_kernels(h1)
        assert names[0].startswith("k_stage5") == (route == "tile")
        I0 = np.exp(np.random.default_rng(9).normal(size=I2.shape))
        got1 = run(B.rad_stage_static, P1, h1, I1, f1, 0.03)
        got2 = run(B.rad_stage_static, P2, h2, I2, f2, 0.02, I0=I0, weights=(0.25, 0.75))   # an RK-style second stage
        want1 = run(B.rad_stage, P1, h1, I1, f1, 0.03)
        want2 = run(B.rad_stage, P2, h2, I2, f2, 0.02, I0=I0, weights=(0.25, 0.75))
        same(P1, got1, want1)
        same(P2, got2, want2)
        # and once more after rad_stage has run on the same contexts (its own table now exists next to the built-in one)
        same(P1, run(B.rad_stage_static, P1, h1, I1, f1, 0.03), want1)
        # the oracle agrees as well (tile route, first call)
        if route == "tile":
            out_o, T_o, dT0_o, nf_o = P1.stage(I1.copy(), f1, o1, 0.03)
            assert nf_o == got1["noroot"]
            assert rel_err_I(P1.interior(got1["I"]), P1.interior(out_o)) <= TOL_I
            assert rel_err(P1.interior(got1["T"]), P1.interior(T_o), 0.0) <= TOL_FLUID
    finally:
        B.rad_destroy(big[2]); B.rad_destroy(small[2])


def test_free_device_memory_does_not_move(oracle, B):
    """a 32^3 block (36^3 = 46 656 cells with ghosts, the paper's small block P:L1014; its table is 2.8 MiB of the array's 4): once
    the kernels are loaded, the card's free memory is the same before and after two more calls"""
    A, P, h, I, fluid, opac, _ = small_problem(oracle, B, (32, 32, 32), ("latlon", 2, 4), tau_factor=1.0)
    try:
        dI = dev(I); dO = torch.zeros_like(dI); dfl = dev(fluid)
        dT = torch.zeros(P.ncell, dtype=torch.float64, device="cuda"); ddT0 = torch.zeros(4, P.ncell, dtype=torch.float64, device="cuda")
        B.rad_stage_static(h, dI, dO, None, dfl, 0.0, 1.0, 0.02, dT, ddT0)   # loads the kernels' code (the driver loads lazily)
        torch.cuda.synchronize()
        first = dO.clone()
        free0 = torch.cuda.mem_get_info()[0]
        for _ in range(2):
            dO.zero_()
            B.rad_stage_static(h, dI, dO, None, dfl, 0.0, 1.0, 0.02, dT, ddT0)
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] == free0
        assert torch.equal(dO, first)
        assert float(dO.abs().max()) > 0.0 and bool(torch.isfinite(dO).all())
    finally:
        B.rad_destroy(h)


def test_block_beyond_the_built_in_table_is_refused(oracle, B):
    """41^3 interior cells = 45^3 = 91 125 cells with ghosts > RAD_STATIC_MAX_CELLS: RAD_EUNSUPPORTED with both numbers in the text,
    I_out untouched; rad_stage serves the same context"""
    n = (41, 41, 41)
    nc = 45 ** 3
    assert nc > B.STATIC_MAX_CELLS
    opac = torch.ones(3, nc, dtype=torch.float64, device="cuda")
    h = B.rad_create(dict(kind=0), dict(n=n, x0=(0, 0, 0), dx=(1, 1, 1)), ("latlon", 2, 4), (opac[0], opac[1], opac[2]), dict(tau_factor=1.0))
    try:
        dI = torch.rand(nc, 8, dtype=torch.float64, device="cuda") + 0.5
        dO = torch.full_like(dI, -3.0)
        fluid = torch.zeros(5, nc, dtype=torch.float64, device="cuda"); fluid[:2] = 1.0
        with pytest.raises(B.RadError) as e:
            B.rad_stage_static(h, dI, dO, None, fluid, 0.0, 1.0, 0.1)
        assert e.value.status == 4
        assert str(nc) in str(e.value) and str(B.STATIC_MAX_CELLS) in str(e.value)
        torch.cuda.synchronize()
        assert bool((dO == -3.0).all())
        B.rad_stage(h, dI, dO, None, fluid, 0.0, 1.0, 0.1)
        torch.cuda.synchronize()
        assert bool(torch.isfinite(dO).all())
    finally:
        B.rad_destroy(h)
