"""GPU parity tests: the CUDA path (through the C ABI) against the oracle, element by element, on the same
seeded inputs.  Bars (north_star): intensities <= 1e-11 relative, fluid energy / four-momentum <= 1e-10,
integer tables (angle neighbours, upwind signs) bit-exact."""
import numpy as np
import pytest
import torch

from paper_2302_04283_b200 import workloads as W
from parity_util import TOL_FLUID, TOL_I, err_dT0, make_oracle, make_rad, oracle_tables_to_rad, rel_err, rel_err_I

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    from paper_2302_04283_b200 import binding, build
    build.build()
    binding.lib()
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return binding


def dev(a):
    return torch.as_tensor(np.ascontiguousarray(a)).cuda()


# ------------------------------------------------------------------------------------------------ tables
@pytest.mark.parametrize("angles", [("latlon", 5, 16), ("latlon", 1, 4), ("latlon", 2, 1), ("geodesic", 1), ("geodesic", 3), ("geodesic", 4), ("geodesic", 7)])
def test_angle_tables_bit_exact(oracle, B, angles):
    A = oracle.Angles(*angles)
    h = B.rad_create(dict(kind=0), dict(n=(1, 1, 1), x0=(0, 0, 0), dx=(1, 1, 1)), angles, None, dict(couple=0))
    try:
        assert B.rad_get_table(h, B.TAB_NANG) == A.N and B.rad_get_table(h, B.TAB_NEDGE) == A.E
        for tab, ref in ((B.TAB_NNBR, A.nnbr), (B.TAB_NBR, A.nbr), (B.TAB_NBR_EDGE, A.nbr_edge), (B.TAB_EDGE_LO, A.edge_lo), (B.TAB_EDGE_HI, A.edge_hi)):
            assert np.array_equal(B.rad_get_table(h, tab), ref)
        assert np.array_equal(B.rad_get_table(h, B.TAB_NHAT), A.nhat)     # same operation order => same bits
        for tab, ref in ((B.TAB_DOMEGA, A.domega), (B.TAB_EDGE_LEN, A.edge_len), (B.TAB_EDGE_MID, A.edge_mid), (B.TAB_EDGE_NRM, A.edge_nrm)):
            assert np.abs(B.rad_get_table(h, tab) - ref).max() < 1e-15
    finally:
        B.rad_destroy(h)


@pytest.mark.parametrize("cfg,n", [("C1", 6), ("C2", 10), ("C3", 9), ("C4", 8), ("C5", 10)])
def test_geometry_tables(oracle, B, cfg, n):
    """level 1: geometry built by the CUDA kernel vs the oracle's, <= 1e-13; upwind sign mismatches counted (expected 0)"""
    A, P = make_oracle(oracle, cfg, n)
    cell, face, ex = P.geometry()
    rc, rf = oracle_tables_to_rad(cell, face, ex)
    h = make_rad(B, cfg, None, n, couple=0)
    try:
        gc, gf = B.rad_get_table(h, B.TAB_CELL), B.rad_get_table(h, B.TAB_FACE)
        assert np.abs(gc - rc).max() < 1e-13, np.abs(gc - rc).max(0)
        assert np.abs(gf - rf).max() < 1e-13
        fs, es = P.upwind_tables()
        assert (B.rad_get_table(h, B.TAB_FACE_SIGN) != fs).sum() == 0
        assert (B.rad_get_table(h, B.TAB_EDGE_SIGN) != es).sum() == 0
        vmax, vax = P.max_speed()
        assert np.abs(B.rad_get_table(h, B.TAB_MAXSPEED) - np.array(vax)).max() < 1e-13
    finally:
        B.rad_destroy(h)


@pytest.mark.parametrize("cfg,n", [("C2", 10), ("C3", 9)])
def test_upwind_tables_bit_exact_on_shared_geometry(oracle, B, cfg, n):
    """level 2: fed the oracle's geometry tables, the upwind index tables are identical bit for bit"""
    A, P = make_oracle(oracle, cfg, n)
    cell, face, ex = P.geometry()
    rc, rf = oracle_tables_to_rad(cell, face, ex)
    h = make_rad(B, cfg, None, n, tabulated=(dev(rc), dev(rf)), couple=0)
    try:
        fs, es = P.upwind_tables()
        assert np.array_equal(B.rad_get_table(h, B.TAB_FACE_SIGN), fs)
        assert np.array_equal(B.rad_get_table(h, B.TAB_EDGE_SIGN), es)
        assert (es != 0).any() and (fs != 0).all()
    finally:
        B.rad_destroy(h)


# ------------------------------------------------------------------------------------------------ the stage
def run_both(oracle, B, cfg, n, level, I0w=None, **kw):
    okw = {{"renorm_fluid_weights": "renorm"}.get(k, k): v for k, v in kw.items()}
    A, P = make_oracle(oracle, cfg, n, **okw)
    inp = W.make_inputs(cfg, A.nhat, n=n)
    I = inp["I"].numpy().reshape(-1, A.N).copy()
    fluid = inp["fluid"].numpy().reshape(5, -1).copy(); opac = inp["opac"].numpy().reshape(3, -1).copy()
    vmax, _ = P.max_speed()
    nn, ng, x0, dx = W.grid(cfg, n)
    dt = W.CFL * min(dx) / vmax
    I0 = None
    gam0, gam1, bdt = 0.0, 1.0, dt
    if I0w is not None:
        I0 = I * (1.0 + 0.05 * np.sin(np.arange(I.size).reshape(I.shape)))
        gam0, gam1, bdt = I0w
        bdt *= dt
    d_opac = dev(opac)
    tab = None
    if level == 2:
        rc, rf = oracle_tables_to_rad(*P.geometry())
        tab = (dev(rc), dev(rf))
    h = make_rad(B, cfg, d_opac, n, tabulated=tab, **kw)
    try:
        dI = dev(I); dO = torch.full_like(dI, -7.0); dfl = dev(fluid)
        dT = torch.zeros(P.ncell, dtype=torch.float64, device="cuda"); ddT0 = torch.zeros(4, P.ncell, dtype=torch.float64, device="cuda")
        nf_g = B.rad_stage(h, dI, dO, None if I0 is None else dev(I0), dfl, gam0, gam1, bdt, dT, ddT0, count_noroot=True)
        torch.cuda.synchronize()
        Iin_after = dI.cpu().numpy()
        out_g, T_g, dT0_g = dO.cpu().numpy(), dT.cpu().numpy(), ddT0.cpu().numpy()
    finally:
        B.rad_destroy(h)
    Iorc = I.copy()
    out_o, T_o, dT0_o, nf_o = P.stage(Iorc, fluid, opac, bdt, I0=I0, gam0=gam0, gam1=gam1)
    # ghost fill of I_in agrees bit for bit; ghosts of I_out are not touched
    assert np.array_equal(Iin_after, Iorc)
    full = out_g.reshape(P.shape + (A.N,)).copy()
    P.interior(full)[...] = -7.0
    assert (full == -7.0).all()
    eD, on_floor = err_dT0(P, dT0_g, dT0_o, out_o)
    print(f"{cfg} n={n} level={level}: cells with every |dT0| below the floor: {100 * on_floor:.1f} %")
    res = dict(I=rel_err_I(P.interior(out_g), P.interior(out_o)), T=rel_err(P.interior(T_g), P.interior(T_o), 0.0), dT0=eD, on_floor=on_floor,
               nf=(nf_g, nf_o), Tchange=float(np.abs(P.interior(T_o) / P.interior(fluid[1]) - 1).max()))
    return res


@pytest.mark.parametrize("level", [1, 2])
@pytest.mark.parametrize("cfg,n", [("C1", 16), ("C2", 21), ("C3", 19), ("C4", 13), ("C5", 18)])
def test_stage_parity(oracle, B, cfg, n, level):
    r = run_both(oracle, B, cfg, n, level)
    assert r["nf"][0] == r["nf"][1] == 0
    assert r["I"] <= TOL_I, r
    assert r["T"] <= TOL_FLUID and r["dT0"] <= TOL_FLUID, r
    assert r["Tchange"] > 1e-8  # the coupling did something (C2, C5 are gas-dominated: ~5e-7)
    # the dT0 floor is a noise allowance, not a hiding place: no cell of C1-C4 sits under it.  C5's recipe is gas dominated and close to
    # equilibrium (increments ~1e-6 |R^0_0|: most of its cells ARE in the floor's regime, where a relative bar of 1e-10 is not
    # reachable in FP64); that regime is anchored by test_gpu_dt0_anchor.py against a long-double evaluation instead
    if cfg != "C5":
        assert r["on_floor"] <= 0.01, r


@pytest.mark.parametrize("kw", [dict(recon_space=0), dict(couple=0), dict(renorm_fluid_weights=0), dict(n0_crit=0.0)])
def test_stage_parity_options(oracle, B, kw):
    r = run_both(oracle, B, "C2", 11, 1, **kw)
    assert r["I"] <= TOL_I and r["T"] <= TOL_FLUID and r["dT0"] <= TOL_FLUID, r


def test_stage_parity_rk_weights(oracle, B):
    """R8: second Heun stage, C* = (C0 + C)/2 - (dt/2) div"""
    r = run_both(oracle, B, "C2", 9, 1, I0w=(0.5, 0.5, 0.5))
    assert r["I"] <= TOL_I and r["T"] <= TOL_FLUID and r["dT0"] <= TOL_FLUID, r


# ------------------------------------------------------------------------------------------------ edge cases
def small_problem(oracle, B, n, angles, kind=1, a=0.9, bc=(0, 0, 0, 0, 0, 0), x0=(3.0, 2.0, 1.0), dx=(0.3, 0.25, 0.2), excise_r=0.0, ng=2, seed=42,
                  explicit=None, **params):
    """the same small problem on both sides; params = rad_params fields (the oracle gets the matching options);
    explicit = dict of host angle tables handed to the library instead of the grid's name (rad_angles kind 2)"""
    A = oracle.Angles(*angles)
    bl, bh = bc[:3], bc[3:]
    okw = dict(recon_space=params.get("recon_space", 1), renorm=params.get("renorm_fluid_weights", 1), couple=params.get("couple", 1),
               n0_crit=params.get("n0_crit", 0.1), tau_factor=params.get("tau_factor", 0.0), recon_angle=params.get("recon_angle", 0),
               vel_estimate=params.get("vel_estimate", 0))
    P = oracle.Problem(A, n, x0, dx, metric_kind=kind, M=1.0, a=a, excise_r=excise_r, ng=ng, bc_lo=bl, bc_hi=bh, **okw)
    rng = np.random.default_rng(seed)
    nc = P.ncell
    I = np.exp(rng.normal(size=(nc, A.N)))
    fluid = np.stack([rng.uniform(0.5, 2, nc), rng.uniform(0.3, 1.5, nc)] + [rng.uniform(-0.4, 0.4, nc) for _ in range(3)])
    opac = np.stack([rng.uniform(0.1, 30, nc), rng.uniform(0.1, 30, nc), rng.uniform(0.1, 30, nc)])   # Planck mean != energy mean != scattering
    d_opac = dev(opac)
    h = B.rad_create(dict(kind=kind, M=1.0, a=a, excise_r=excise_r), dict(n=n, ng=ng, x0=x0, dx=dx, bc_lo=bl, bc_hi=bh),
                     angles if explicit is None else ("explicit", explicit), (d_opac[0], d_opac[1], d_opac[2]), dict(params))
    return A, P, h, I, fluid, opac, d_opac


def compare_stage(B, A, P, h, I, fluid, opac, dt):
    dI = dev(I); dO = torch.zeros_like(dI); dfl = dev(fluid)
    dT = torch.zeros(P.ncell, dtype=torch.float64, device="cuda"); ddT0 = torch.full((4, P.ncell), 9.0, dtype=torch.float64, device="cuda")
    nf = B.rad_stage(h, dI, dO, None, dfl, 0.0, 1.0, dt, dT, ddT0, count_noroot=True)
    Io = I.copy()
    out_o, T_o, dT0_o, nf_o = P.stage(Io, fluid, opac, dt)
    assert nf == nf_o
    assert np.array_equal(dI.cpu().numpy(), Io)
    eI = rel_err_I(P.interior(dO.cpu().numpy()), P.interior(out_o))
    eT = rel_err(P.interior(dT.cpu().numpy()), P.interior(T_o), 0.0)
    eD, _ = err_dT0(P, ddT0.cpu().numpy(), dT0_o, out_o)     # includes excised and no-root cells (increment 0 on both sides)
    assert eI <= TOL_I and eT <= TOL_FLUID and eD <= TOL_FLUID, (eI, eT, eD)
    return dO.cpu().numpy(), out_o


@pytest.mark.parametrize("n", [(1, 1, 1), (3, 5, 9), (17, 2, 3), (8, 8, 8)])
@pytest.mark.parametrize("bc", [(0, 0, 0, 0, 0, 0), (1, 1, 1, 1, 1, 1), (2, 1, 0, 2, 1, 2)])
def test_ragged_grids_and_boundaries(oracle, B, n, bc):
    A, P, h, I, fluid, opac, _ = small_problem(oracle, B, n, ("geodesic", 2), bc=bc)
    try:
        compare_stage(B, A, P, h, I, fluid, opac, 0.05)
    finally:
        B.rad_destroy(h)


@pytest.mark.parametrize("angles", [("latlon", 1, 4), ("latlon", 3, 1), ("latlon", 4, 8), ("geodesic", 1), ("geodesic", 5)])
def test_angle_grids(oracle, B, angles):
    A, P, h, I, fluid, opac, _ = small_problem(oracle, B, (5, 4, 3), angles)
    try:
        compare_stage(B, A, P, h, I, fluid, opac, 0.05)
    finally:
        B.rad_destroy(h)


def test_ergosphere_mask_and_excision(oracle, B):
    A, P, h, I, fluid, opac, _ = small_problem(oracle, B, (8, 8, 4), ("geodesic", 3), x0=(-2.0, -2.0, -0.2), dx=(0.5, 0.5, 0.1), excise_r=1.5)
    try:
        got, ref = compare_stage(B, A, P, h, I, fluid, opac, 0.01)
        gi, ri = P.interior(got), P.interior(ref)
        assert np.array_equal(gi == 0.0, ri == 0.0)          # same cells/angles masked or excised
        ex = P.interior(P.geometry()[2].astype(bool))
        assert ex.any() and (ri[ex] == 0).all() and (ri[~ex] == 0).any() and (ri[~ex] != 0).any()
    finally:
        B.rad_destroy(h)


def test_no_root_is_counted(oracle, B):
    A, P, h, I, fluid, opac, _ = small_problem(oracle, B, (4, 3, 2), ("latlon", 2, 4), kind=0, a=0.0)
    try:
        fluid[1, ::2] = -3.0   # unphysical negative gas temperature in every other cell => no positive root there
        I[:] = 0.0
        dI = dev(I); dO = torch.zeros_like(dI); dfl = dev(fluid); dT = torch.zeros(P.ncell, dtype=torch.float64, device="cuda")
        nf = B.rad_stage(h, dI, dO, None, dfl, 0.0, 1.0, 0.1, dT, None, count_noroot=True)
        out_o, T_o, _, nf_o = P.stage(I.copy(), fluid, opac, 0.1)
        assert nf == nf_o and nf > 0
        assert np.array_equal(P.interior(dT.cpu().numpy())[P.interior(fluid[1]) < 0], P.interior(fluid[1])[P.interior(fluid[1]) < 0])
    finally:
        B.rad_destroy(h)


def test_error_codes(oracle, B):
    A, P, h, I, fluid, opac, _ = small_problem(oracle, B, (2, 2, 2), ("latlon", 2, 4))
    try:
        dI = dev(I); dfl = dev(fluid)
        with pytest.raises(B.RadError) as e:
            B.rad_stage(h, dI, dI, None, dfl, 0.0, 1.0, 0.1)
        assert e.value.status == 1 and "alias" in str(e.value)
        with pytest.raises(B.RadError) as e:
            B.rad_stage(h, dI, torch.zeros_like(dI), None, dfl, 0.0, 1.0, float("nan"))
        assert e.value.status == 1
        with pytest.raises(B.RadError):
            B.rad_moments(h, dI, 7, None, torch.zeros(10, P.ncell, dtype=torch.float64, device="cuda"))
    finally:
        B.rad_destroy(h)


@pytest.mark.parametrize("frame", [0, 1, 2, 3])
def test_moments_parity(oracle, B, frame):
    A, P, h, I, fluid, opac, _ = small_problem(oracle, B, (5, 4, 3), ("geodesic", 3))
    try:
        ncomp = 10 if frame in (0, 2) else 4
        out = torch.zeros(ncomp, P.ncell, dtype=torch.float64, device="cuda")
        B.rad_moments(h, dev(I), frame, dev(fluid), out)
        ref = P.moments(I, frame, fluid)
        for q in range(ncomp):
            assert rel_err(P.interior(out[q].cpu().numpy()), P.interior(ref[q]), 1e-13 * np.abs(ref).max()) < 1e-12
    finally:
        B.rad_destroy(h)


def test_stage_host_equals_stage(oracle, B):
    A, P, h, I, fluid, opac, _ = small_problem(oracle, B, (6, 5, 4), ("geodesic", 2), bc=(1, 1, 1, 1, 1, 1))
    try:
        out_h = np.zeros_like(I); T_h = np.zeros(P.ncell); dT0_h = np.zeros((4, P.ncell))
        nf = B.rad_stage_host(h, I, out_h, fluid, opac, 0.0, 1.0, 0.05, T_h, dT0_h, count_noroot=True)
        out_o, T_o, dT0_o, nf_o = P.stage(I.copy(), fluid, opac, 0.05)
        assert nf == nf_o
        assert rel_err_I(P.interior(out_h), P.interior(out_o)) <= TOL_I
        assert rel_err(P.interior(T_h), P.interior(T_o), 0.0) <= TOL_FLUID
    finally:
        B.rad_destroy(h)


@pytest.mark.parametrize("n,angles", [((6, 5, 20), ("geodesic", 2)), ((5, 9, 37), ("geodesic", 4)), ((4, 4, 9), ("latlon", 4, 8))])
def test_stage_host_pipelined(oracle, B, n, angles):
    """rad_stage_host with caller-filled boundaries runs slab by slab along z with overlapped copies: same values as the oracle,
    ghost cells of the returned array = those of the input, every slab boundary inside the block"""
    A, P, h, I, fluid, opac, _ = small_problem(oracle, B, n, angles)
    try:
        out_h = np.full_like(I, -3.0); T_h = np.zeros(P.ncell); dT0_h = np.zeros((4, P.ncell))
        nf = B.rad_stage_host(h, I, out_h, fluid, opac, 0.0, 1.0, 0.03, T_h, dT0_h, count_noroot=True)
        out_o, T_o, dT0_o, nf_o = P.stage(I.copy(), fluid, opac, 0.03)
        assert nf == nf_o
        assert rel_err_I(P.interior(out_h), P.interior(out_o)) <= TOL_I
        assert rel_err(P.interior(T_h), P.interior(T_o), 0.0) <= TOL_FLUID
        assert err_dT0(P, dT0_h, dT0_o, out_o)[0] <= TOL_FLUID
        full = out_h.reshape(P.shape + (A.N,)).copy(); ref = I.reshape(P.shape + (A.N,)).copy()
        P.interior(full)[...] = 0.0; P.interior(ref)[...] = 0.0
        assert np.array_equal(full, ref)
    finally:
        B.rad_destroy(h)


def test_invariants_on_gpu(oracle, B):
    """properties that hold at any size, checked on the CUDA path itself: isotropic fixed point in Minkowski (bit for bit)
    and conservation of sum n^0 n_0 I dOmega with sources off in Kerr-Schild"""
    n = (24, 20, 16)
    h = B.rad_create(dict(kind=0), dict(n=n, x0=(0, 0, 0), dx=(0.1, 0.1, 0.1), bc_lo=(1, 1, 1), bc_hi=(1, 1, 1)), ("geodesic", 3), None, dict(couple=0))
    try:
        nc = B.rad_ncells_total(h)
        I = torch.full((nc, 92), 0.731, dtype=torch.float64, device="cuda"); O = torch.zeros_like(I)
        B.rad_transport(h, I, O, None, 0.0, 1.0, 0.03)
        Oi = O.reshape(n[2] + 4, n[1] + 4, n[0] + 4, 92)[2:-2, 2:-2, 2:-2]
        assert (Oi == 0.731).all()
    finally:
        B.rad_destroy(h)
    h = B.rad_create(dict(kind=1, M=1.0, a=0.9), dict(n=n, x0=(3, 2, 1), dx=(0.2, 0.2, 0.2)), ("geodesic", 3), None, dict(couple=0, n0_crit=0.0))
    try:
        shp = (n[2] + 4, n[1] + 4, n[0] + 4, 92)
        I = torch.zeros(shp, dtype=torch.float64, device="cuda")
        g = torch.Generator(device="cuda").manual_seed(1)
        I[6:-6, 6:-6, 6:-6] = torch.exp(torch.randn((n[2] - 8, n[1] - 8, n[0] - 8, 92), generator=g, device="cuda", dtype=torch.float64))
        O = torch.zeros_like(I)
        vmax = B.rad_get_table(h, B.TAB_MAXSPEED).max()
        B.rad_transport(h, I, O, None, 0.0, 1.0, 0.3 * 0.2 / vmax)
        R0 = torch.zeros(4, nc, dtype=torch.float64, device="cuda"); R1 = torch.zeros_like(R0)
        B.rad_moments(h, I, 1, None, R0); B.rad_moments(h, O, 1, None, R1)
        e0, e1 = R0[0].sum().item(), R1[0].sum().item()   # R^0_0 = sum n^0 n_0 I dOmega per cell
        assert abs(e1 - e0) < 1e-12 * abs(e0) and e0 != 0
    finally:
        B.rad_destroy(h)


# ------------------------------------------------------------------------------------------------ full size, sampled
@pytest.mark.parametrize("cfg,m,corners", [("C3", 6, [(0, 0, 0), (61, 62, 63), (122, 122, 122), (3, 120, 50)]),
                                           ("C5", 5, [(0, 0, 0), (126, 127, 128), (251, 251, 251)]),
                                           ("C4", 6, [(0, 0, 0), (45, 46, 47), (90, 90, 90), (2, 88, 31)]),
                                           ("C2", 7, [(0, 0, 0), (29, 30, 31), (57, 57, 57)])])
def test_full_size_sampled(oracle, B, cfg, m, corners):
    """BASELINE.json's full-size blocks in the launch configuration bench.py times (one rad_stage on the whole block), checked on
    sampled sub-blocks: a cell's update reads at most 2 cells away, so the oracle run on m^3 cells whose 2-deep shell is cut
    out of the full input must reproduce the GPU's values there.  Corners of the block, its middle and a tile-straddling
    position are sampled (tiles are 4 x 2 / 4 x 3 cells in y-z)."""
    c = W.CONFIGS[cfg]
    nn, ng, x0, dx = W.grid(cfg)
    N = W.n_angles(cfg)
    h0 = B.rad_create(dict(kind=0), dict(n=(1, 1, 1), x0=(0, 0, 0), dx=(1, 1, 1)), c["angles"], None, dict(couple=0))
    nhat = B.rad_get_table(h0, B.TAB_NHAT)
    B.rad_destroy(h0)
    inp = W.make_inputs(cfg, nhat, device="cuda")
    shape = (nn[2] + 2 * ng, nn[1] + 2 * ng, nn[0] + 2 * ng)
    I = inp["I"].reshape(-1, N).contiguous(); fluid = inp["fluid"].reshape(5, -1).contiguous(); opac = inp["opac"].reshape(3, -1).contiguous()
    del inp
    h = make_rad(B, cfg, opac)
    try:
        vmax = float(B.rad_get_table(h, B.TAB_MAXSPEED).max())
        dt = W.CFL * min(dx) / vmax
        O = torch.full_like(I, -7.0)
        T = torch.zeros(I.shape[0], dtype=torch.float64, device="cuda"); dT0 = torch.zeros(4, I.shape[0], dtype=torch.float64, device="cuda")
        nf = B.rad_stage(h, I, O, None, fluid, 0.0, 1.0, dt, T, dT0, count_noroot=True)
        torch.cuda.synchronize()
        assert nf == 0
        A = oracle.Angles(*c["angles"])
        I5 = I.reshape(shape + (N,)); O5 = O.reshape(shape + (N,))
        f4 = fluid.reshape((5,) + shape); o4 = opac.reshape((3,) + shape); T3 = T.reshape(shape); d4 = dT0.reshape((4,) + shape)
        for (ai, aj, ak) in corners:
            sl = (slice(ak, ak + m + 2 * ng), slice(aj, aj + m + 2 * ng), slice(ai, ai + m + 2 * ng))
            P = oracle.Problem(A, (m, m, m), (x0[0] + ai * dx[0], x0[1] + aj * dx[1], x0[2] + ak * dx[2]), dx, metric_kind=c["metric"], M=c["M"], a=c["a"],
                               excise_r=W.excise_radius(cfg), bc_lo=(0, 0, 0), bc_hi=(0, 0, 0), gamma_gas=W.GAMMA_GAS, a_rad=W.A_RAD,
                               n0_crit=W.N0_CRIT, recon_space=1, renorm=1, couple=1)
            Is = I5[sl].cpu().numpy().reshape(-1, N).copy()
            fs = f4[(slice(None),) + sl].cpu().numpy().reshape(5, -1).copy(); os_ = o4[(slice(None),) + sl].cpu().numpy().reshape(3, -1).copy()
            out_o, T_o, dT0_o, nf_o = P.stage(Is, fs, os_, dt)
            got = O5[sl].cpu().numpy().reshape(-1, N)
            eI = rel_err_I(P.interior(got), P.interior(out_o))
            eT = rel_err(P.interior(T3[sl].cpu().numpy().reshape(-1)), P.interior(T_o), 0.0)
            eD, on_floor = err_dT0(P, np.stack([d4[(q,) + sl].cpu().numpy().reshape(-1) for q in range(4)]), dT0_o, out_o)
            assert eI <= TOL_I and eT <= TOL_FLUID and eD <= TOL_FLUID, (cfg, (ai, aj, ak), eI, eT, eD)
            assert cfg == "C5" or on_floor <= 0.01, (cfg, (ai, aj, ak), on_floor)   # (C5: see test_stage_parity)
        # ghost cells of I_out are never written
        assert float(O5[:ng].max()) == -7.0 and float(O5[:, :ng].max()) == -7.0 and float(O5[:, :, -ng:].max()) == -7.0
        if cfg == "C3":
            # rad_stage_host at the size bench.py's e2e figure is taken on (128 planes x 162 angles through the three-stream slab
            # pipeline): interior intensities, temperature and fluid increment equal rad_stage's bit for bit; ghosts of I_out carry I_in
            itr = (slice(ng, -ng),) * 3
            hI = I.cpu(); hO = torch.full_like(hI, -5.0); hfl = fluid.cpu(); hop = opac.cpu()
            hT = torch.zeros(I.shape[0], dtype=torch.float64); hd = torch.zeros(4, I.shape[0], dtype=torch.float64)
            nfh = B.rad_stage_host(h, hI, hO, hfl, hop, 0.0, 1.0, dt, hT, hd, count_noroot=True)
            assert nfh == 0
            hO5 = hO.reshape(shape + (N,)); want = O5.cpu()
            assert torch.equal(hO5[itr], want[itr])
            assert torch.equal(hT.reshape(shape)[itr], T3.cpu()[itr])
            assert torch.equal(hd.reshape((4,) + shape)[(slice(None),) + itr], d4.cpu()[(slice(None),) + itr])
            hI5 = hI.reshape(shape + (N,))
            assert torch.equal(hO5[:ng], hI5[:ng]) and torch.equal(hO5[:, :, -ng:], hI5[:, :, -ng:])
    finally:
        B.rad_destroy(h)


def test_three_stages_ping_pong(oracle, B):
    """three consecutive stages with periodic boundaries, the two intensity buffers swapped after each (the caller's time loop):
    the ghost fill of every stage works on the previous stage's output, the fluid temperature is carried along"""
    A, P, h, I, fluid, opac, _ = small_problem(oracle, B, (9, 6, 5), ("geodesic", 3), bc=(1, 1, 1, 1, 1, 1))
    try:
        dA = dev(I); dB_ = torch.zeros_like(dA); dfl = dev(fluid)
        dT = torch.zeros(P.ncell, dtype=torch.float64, device="cuda")
        Io, fo = I.copy(), fluid.copy()
        for step in range(3):
            nf = B.rad_stage(h, dA, dB_, None, dfl, 0.0, 1.0, 0.04, dT, None, count_noroot=True)
            out_o, T_o, _, nf_o = P.stage(Io, fo, opac, 0.04)
            assert nf == nf_o == 0
            assert rel_err_I(P.interior(dB_.cpu().numpy()), P.interior(out_o)) <= 3 * TOL_I, step
            assert rel_err(P.interior(dT.cpu().numpy()), P.interior(T_o), 0.0) <= 3 * TOL_FLUID, step
            dA, dB_ = dB_, dA
            Io = out_o.copy()
            Tin = P.interior(fo[1]); Tin[...] = P.interior(T_o)          # interior temperatures advance, ghosts keep theirs
            P.interior(dfl[1].reshape(P.shape))[...] = torch.as_tensor(P.interior(T_o)).cuda()
    finally:
        B.rad_destroy(h)


# ------------------------------------------------------------------------------------------------ NEXT-1: Eq.26-29
@pytest.mark.parametrize("n,angles,kind,tau", [((7, 6, 5), ("geodesic", 2), 1, 2.0), ((9, 4, 6), ("geodesic", 4), 1, 0.5), ((5, 5, 5), ("latlon", 4, 8), 0, 10.0)])
def test_optical_depth_flux_parity(oracle, B, n, angles, kind, tau):
    """stage with the optical-depth-aware spatial flux (tau_factor != 0): CUDA path against the oracle, same tolerances"""
    A = oracle.Angles(*angles)
    P = oracle.Problem(A, n, (3.0, 2.0, 1.0), (0.3, 0.25, 0.2), metric_kind=kind, M=1.0, a=0.9 if kind else 0.0, tau_factor=tau)
    rng = np.random.default_rng(7)
    nc = P.ncell
    I = np.exp(rng.normal(size=(nc, A.N)))
    fluid = np.stack([rng.uniform(0.5, 2, nc), rng.uniform(0.3, 1.5, nc)] + [rng.uniform(-0.4, 0.4, nc) for _ in range(3)])
    opac = np.stack([rng.uniform(0.1, 30, nc), rng.uniform(0.1, 30, nc), rng.uniform(0.1, 30, nc)])   # Planck mean != energy mean != scattering
    d_opac = dev(opac)
    h = B.rad_create(dict(kind=kind, M=1.0, a=0.9 if kind else 0.0), dict(n=n, x0=(3.0, 2.0, 1.0), dx=(0.3, 0.25, 0.2)), angles,
                     (d_opac[0], d_opac[1], d_opac[2]), dict(tau_factor=tau))
    try:
        got, ref = compare_stage(B, A, P, h, I, fluid, opac, 0.02)
        free = oracle.Problem(A, n, (3.0, 2.0, 1.0), (0.3, 0.25, 0.2), metric_kind=kind, M=1.0, a=0.9 if kind else 0.0).stage(I.copy(), fluid, opac, 0.02)[0]
        assert np.abs(P.interior(ref) - P.interior(free)).max() > 1e-6   # the flux factor did something
        with pytest.raises(B.RadError) as e:   # the transport half alone has no fluid state
            B.rad_transport(h, dev(I), torch.zeros_like(dev(I)), None, 0.0, 1.0, 0.02)
        assert e.value.status == 5
    finally:
        B.rad_destroy(h)


def test_optical_depth_flux_host_path_and_periodic(oracle, B):
    """tau_factor != 0 through rad_stage_host (not pipelined: the flux needs the neighbours' fluid state) with periodic ghosts of I"""
    A = oracle.Angles("geodesic", 3)
    n, x0, dx = (6, 5, 9), (0.0, 0.0, 0.0), (0.2, 0.2, 0.2)
    P = oracle.Problem(A, n, x0, dx, metric_kind=0, bc_lo=(1, 1, 1), bc_hi=(1, 1, 1), tau_factor=4.0)
    rng = np.random.default_rng(3)
    nc = P.ncell
    I = np.exp(rng.normal(size=(nc, A.N)))
    fluid = np.stack([rng.uniform(0.5, 2, nc), rng.uniform(0.3, 1.5, nc)] + [rng.uniform(-0.4, 0.4, nc) for _ in range(3)])
    opac = np.stack([rng.uniform(0.1, 30, nc), rng.uniform(0.1, 30, nc), rng.uniform(0.1, 30, nc)])   # Planck mean != energy mean != scattering
    d_opac = dev(opac)
    h = B.rad_create(dict(kind=0), dict(n=n, x0=x0, dx=dx, bc_lo=(1, 1, 1), bc_hi=(1, 1, 1)), ("geodesic", 3), (d_opac[0], d_opac[1], d_opac[2]), dict(tau_factor=4.0))
    try:
        out_h = np.zeros_like(I); T_h = np.zeros(nc); dT0_h = np.zeros((4, nc))
        nf = B.rad_stage_host(h, I, out_h, fluid, opac, 0.0, 1.0, 0.03, T_h, dT0_h, count_noroot=True)
        out_o, T_o, dT0_o, nf_o = P.stage(I.copy(), fluid, opac, 0.03)
        assert nf == nf_o
        assert rel_err_I(P.interior(out_h), P.interior(out_o)) <= TOL_I
        assert rel_err(P.interior(T_h), P.interior(T_o), 0.0) <= TOL_FLUID
    finally:
        B.rad_destroy(h)


@pytest.mark.parametrize("seed", [1, 2, 3])
def test_random_configurations(oracle, B, seed):
    """randomised sweep: angle grid, block shape (long x runs, partial tiles), metric, boundary codes, reconstruction, fluid-frame
    weight flag, mask, optical-depth factor -- every case within the stage tolerances"""
    import random
    rnd = random.Random(seed)
    angs = [("geodesic", 1), ("geodesic", 2), ("geodesic", 3), ("geodesic", 4), ("geodesic", 5), ("latlon", 4, 8), ("latlon", 5, 16), ("latlon", 2, 4), ("latlon", 6, 10)]
    for case in range(25):
        ang = rnd.choice(angs); n = (rnd.randint(1, 40 if seed == 3 else 14), rnd.randint(1, 11), rnd.randint(1, 11))
        kind = rnd.choice([0, 1, 1]); a = rnd.choice([0.0, 0.5, 0.9]) if kind else 0.0
        bc = tuple(rnd.choice([0, 1, 2]) for _ in range(6)); tau = rnd.choice([0.0, 0.0, 0.7, 5.0])
        params = dict(recon_space=rnd.choice([0, 1, 1]), renorm_fluid_weights=rnd.choice([0, 1]), n0_crit=rnd.choice([0.0, 0.1]), couple=1)
        dx = (rnd.uniform(0.15, 0.4), rnd.uniform(0.15, 0.4), rnd.uniform(0.15, 0.4))
        A = oracle.Angles(*ang)
        P = oracle.Problem(A, n, (3.0, 2.0, 1.0), dx, metric_kind=kind, M=1.0, a=a, bc_lo=bc[:3], bc_hi=bc[3:], recon_space=params["recon_space"],
                           renorm=params["renorm_fluid_weights"], couple=1, n0_crit=params["n0_crit"], tau_factor=tau)
        rng = np.random.default_rng(1000 * seed + case); nc = P.ncell
        I = np.exp(rng.normal(size=(nc, A.N)))
        fluid = np.stack([rng.uniform(0.5, 2, nc), rng.uniform(0.3, 1.5, nc)] + [rng.uniform(-0.4, 0.4, nc) for _ in range(3)])
        opac = np.stack([rng.uniform(0.1, 30, nc), rng.uniform(0.1, 30, nc), rng.uniform(0.1, 30, nc)])   # Planck mean != energy mean != scattering
        d_opac = dev(opac)
        h = B.rad_create(dict(kind=kind, M=1.0, a=a), dict(n=n, x0=(3.0, 2.0, 1.0), dx=dx, bc_lo=bc[:3], bc_hi=bc[3:]), ang,
                         (d_opac[0], d_opac[1], d_opac[2]), dict(params, tau_factor=tau))
        try:
            compare_stage(B, A, P, h, I, fluid, opac, rnd.uniform(0.01, 0.05))
        except AssertionError as e:
            raise AssertionError((case, ang, n, kind, a, bc, tau, params, str(e)))
        finally:
            B.rad_destroy(h)
