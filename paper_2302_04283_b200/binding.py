"""Thin Python binding of librad.so (include/rad.h): argument marshalling only.

Same names as the C ABI: rad_create, rad_stage, rad_stage_host, rad_transport, rad_couple,
rad_fill_ghosts, rad_moments, rad_get_table, rad_destroy.  Device buffers are torch CUDA
tensors (PyTorch is used for device memory and streams only); every step of the path runs in
the library's kernels.  There is no fallback: if librad.so is missing or no GPU is usable the
calls raise.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "librad.so")
NCELL, NFACE, MAXNBR = 52, 8, 6

(TAB_NANG, TAB_NEDGE, TAB_NHAT, TAB_DOMEGA, TAB_NNBR, TAB_NBR, TAB_NBR_EDGE, TAB_EDGE_LO, TAB_EDGE_HI, TAB_EDGE_LEN,
 TAB_EDGE_MID, TAB_EDGE_NRM, TAB_CELL, TAB_FACE, TAB_FACE_SIGN, TAB_EDGE_SIGN, TAB_MAXSPEED, TAB_OWN_EDGE, TAB_KE,
 TAB_STAGE_FACE_SIGN) = range(20)

EXPORTS = ["rad_create", "rad_stage", "rad_stage_static", "rad_stage_host", "rad_fill_ghosts", "rad_transport", "rad_couple", "rad_moments",
           "rad_get_table", "rad_edge_ownership", "rad_exchange_halo", "rad_stage_kernels", "rad_probe_fp64", "rad_ncells_total", "rad_launch_count", "rad_last_error", "rad_destroy"]


class RadError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"librad status {status}: {msg}")
        self.status = status


class _Metric(C.Structure):
    _fields_ = [("kind", C.c_int), ("M", C.c_double), ("a", C.c_double), ("excise_r", C.c_double),
                ("cell_tab", C.c_void_p), ("face_tab", C.c_void_p)]


class _Grid(C.Structure):
    _fields_ = [("n", C.c_int * 3), ("ng", C.c_int), ("x0", C.c_double * 3), ("dx", C.c_double * 3),
                ("bc_lo", C.c_int * 3), ("bc_hi", C.c_int * 3), ("xf", C.c_void_p * 3)]


class _Angles(C.Structure):
    _fields_ = [("kind", C.c_int), ("nzeta", C.c_int), ("npsi", C.c_int), ("nlev", C.c_int), ("nang", C.c_int),
                ("nhat", C.c_void_p), ("domega", C.c_void_p), ("edge_len", C.c_void_p), ("edge_mid", C.c_void_p), ("edge_nrm", C.c_void_p),
                ("nnbr", C.c_void_p), ("nbr", C.c_void_p)]


class _Opac(C.Structure):
    _fields_ = [("alpha_a_planck", C.c_void_p), ("alpha_a_energy", C.c_void_p), ("alpha_s", C.c_void_p)]


class _Params(C.Structure):
    _fields_ = [("gamma_gas", C.c_double), ("a_rad", C.c_double), ("n0_crit", C.c_double), ("recon_space", C.c_int),
                ("recon_angle", C.c_int), ("renorm_fluid_weights", C.c_int), ("couple", C.c_int), ("tau_factor", C.c_double),
                ("recompute_edge_coeffs", C.c_int), ("vel_estimate", C.c_int)]


_lib = None


def lib():
    """load librad.so (fails loudly if it has not been built: python -m paper_2302_04283_b200.build)"""
    global _lib
    if _lib is None:
        if not os.path.exists(_SO):
            raise RuntimeError(f"{_SO} is missing: build it with `python -m paper_2302_04283_b200.build` (no CPU fallback exists)")
        L = C.CDLL(_SO)
        vp, d, ll = C.c_void_p, C.c_double, C.POINTER(C.c_longlong)
        L.rad_create.argtypes = [C.POINTER(_Metric), C.POINTER(_Grid), C.POINTER(_Angles), C.POINTER(_Opac), C.POINTER(_Params), C.c_int, C.POINTER(vp)]
        L.rad_stage.argtypes = [vp, vp, vp, vp, vp, d, d, d, vp, vp, ll, vp]
        L.rad_stage_static.argtypes = [vp, vp, vp, vp, vp, d, d, d, vp, vp, ll, vp]
        L.rad_stage_host.argtypes = [vp, vp, vp, vp, vp, d, d, d, vp, vp, ll]
        L.rad_fill_ghosts.argtypes = [vp, vp, vp]
        L.rad_transport.argtypes = [vp, vp, vp, vp, d, d, d, vp]
        L.rad_couple.argtypes = [vp, vp, vp, d, vp, vp, ll, vp]
        L.rad_moments.argtypes = [vp, vp, C.c_int, vp, vp, vp]
        L.rad_get_table.argtypes = [vp, C.c_int, vp, C.c_size_t]
        L.rad_probe_fp64.argtypes = [vp, C.POINTER(C.c_double)]
        L.rad_edge_ownership.argtypes = [C.POINTER(_Angles), C.POINTER(C.c_int), C.POINTER(C.c_int), vp, vp, vp, vp, vp, C.c_size_t]
        L.rad_exchange_halo.argtypes = [vp, vp, vp, vp, C.c_int, vp]
        L.rad_stage_kernels.argtypes = [vp, C.c_char_p, C.c_size_t]
        L.rad_ncells_total.argtypes = [vp]; L.rad_ncells_total.restype = C.c_longlong
        L.rad_launch_count.argtypes = [vp]; L.rad_launch_count.restype = C.c_longlong
        L.rad_last_error.argtypes = [vp]; L.rad_last_error.restype = C.c_char_p
        L.rad_destroy.argtypes = [vp]; L.rad_destroy.restype = None
        for f in EXPORTS:
            if f not in ("rad_ncells_total", "rad_launch_count", "rad_last_error", "rad_destroy"):
                getattr(L, f).restype = C.c_int
        _lib = L
    return _lib


def _dp(t):
    """device pointer of a contiguous float64 CUDA tensor (or None)"""
    if t is None:
        return None
    if not (t.is_cuda and t.is_contiguous() and t.dtype.is_floating_point and t.element_size() == 8):
        raise ValueError("expected a contiguous float64 CUDA tensor")
    return C.c_void_p(t.data_ptr())


def _hp(a):
    """host pointer of a contiguous float64 numpy array or CPU tensor (or None)"""
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        if a.dtype != np.float64 or not a.flags.c_contiguous:
            raise ValueError("expected a contiguous float64 host array")
        return C.c_void_p(a.ctypes.data)
    if a.is_cuda or not a.is_contiguous() or a.element_size() != 8:
        raise ValueError("expected a contiguous float64 host tensor")
    return C.c_void_p(a.data_ptr())


def _stream(s):
    if s is None:
        import torch
        s = torch.cuda.current_stream()
    return C.c_void_p(s.cuda_stream if hasattr(s, "cuda_stream") else int(s))


def _check(ctx, st):
    if st != 0:
        raise RadError(st, lib().rad_last_error(ctx).decode())


def _angles(angles):
    """rad_angles from ("latlon", nzeta, npsi), ("geodesic", nlev) or ("explicit", dict of host tables: rad_angles kind 2 in rad.h);
    returns the struct and the host arrays it points into (to be kept alive across the call)"""
    if angles[0] == "latlon":
        return _Angles(0, int(angles[1]), int(angles[2]), 0), []
    if angles[0] == "geodesic":
        return _Angles(1, 0, 0, int(angles[1])), []
    if angles[0] != "explicit":
        raise ValueError("angle grid: ('latlon', nzeta, npsi), ('geodesic', nlev) or ('explicit', tables)")
    tb = angles[1]
    f64 = lambda k: np.ascontiguousarray(tb[k], dtype=np.float64)
    i32 = lambda k: np.ascontiguousarray(tb[k], dtype=np.int32)
    keep = [f64("nhat"), f64("domega"), f64("edge_len"), f64("edge_mid"), f64("edge_nrm"), i32("nnbr"), i32("nbr")]
    return _Angles(2, 0, 0, 0, int(keep[1].shape[0]), *[C.c_void_p(x.ctypes.data) for x in keep]), keep


def rad_create(metric, grid, angles, opac, params, device=0):
    """metric: dict(kind, M, a, excise_r, cell_tab, face_tab); grid: dict(n, x0, dx, bc_lo, bc_hi[, ng][, xf = per axis None or face coordinates]);
    angles: ("latlon", nzeta, npsi), ("geodesic", nlev) or ("explicit", dict(nhat, domega, nnbr, nbr, edge_len, edge_mid, edge_nrm)); opac: (alpha_a_planck, alpha_a_energy, alpha_s) CUDA
    tensors or None; params: dict of rad_params fields.  Returns an opaque handle."""
    m = _Metric(int(metric.get("kind", 0)), float(metric.get("M", 1.0)), float(metric.get("a", 0.0)), float(metric.get("excise_r", 0.0)),
                _dp(metric.get("cell_tab")), _dp(metric.get("face_tab")))
    i3, d3 = C.c_int * 3, C.c_double * 3
    xfa = [None if (grid.get("xf") is None or grid["xf"][d] is None) else np.ascontiguousarray(grid["xf"][d], dtype=np.float64) for d in range(3)]
    for d in range(3):
        if xfa[d] is not None and xfa[d].shape != (int(grid["n"][d]) + 2 * int(grid.get("ng", 2)) + 1,):
            raise ValueError("grid xf[%d] needs n + 2 ng + 1 face coordinates" % d)
    g = _Grid(i3(*grid["n"]), int(grid.get("ng", 2)), d3(*grid["x0"]), d3(*grid["dx"]), i3(*grid.get("bc_lo", (0, 0, 0))), i3(*grid.get("bc_hi", (0, 0, 0))),
              (C.c_void_p * 3)(*[None if v is None else v.ctypes.data for v in xfa]))
    a, keep = _angles(angles)
    o = _Opac(*(_dp(x) for x in opac)) if opac is not None else None
    p = _Params(float(params.get("gamma_gas", 5.0 / 3.0)), float(params.get("a_rad", 1.0)), float(params.get("n0_crit", 0.1)),
                int(params.get("recon_space", 1)), int(params.get("recon_angle", 0)), int(params.get("renorm_fluid_weights", 1)),
                int(params.get("couple", 1)), float(params.get("tau_factor", 0.0)), int(params.get("recompute_edge_coeffs", 0)), int(params.get("vel_estimate", 0)))
    h = C.c_void_p()
    st = lib().rad_create(C.byref(m), C.byref(g), C.byref(a), C.byref(o) if o is not None else None, C.byref(p), int(device), C.byref(h))
    _check(None, st)
    return h


def rad_destroy(ctx):
    lib().rad_destroy(ctx)


def rad_stage(ctx, I_in, I_out, I0, fluid, gam0, gam1, beta_dt, T_out=None, dT0=None, count_noroot=False, stream=None):
    n = C.c_longlong(0)
    st = lib().rad_stage(ctx, _dp(I_in), _dp(I_out), _dp(I0), _dp(fluid), gam0, gam1, beta_dt, _dp(T_out), _dp(dT0),
                         C.byref(n) if count_noroot else None, _stream(stream))
    _check(ctx, st)
    return n.value if count_noroot else None


STATIC_MAX_CELLS = 65536  # RAD_STATIC_MAX_CELLS


def rad_stage_static(ctx, I_in, I_out, I0, fluid, gam0, gam1, beta_dt, T_out=None, dT0=None, count_noroot=False, stream=None):
    """rad_stage without any device allocation, for step loops that run after the application has given the rest of the card to its own
    memory pool or that cannot afford the device-wide stall of a cudaMalloc: the optical-depth-aware flux's per-cell table sits in a
    4 MiB array inside librad.so instead.  Blocks of at most STATIC_MAX_CELLS cells (ghosts included), else RadError status 4;
    calls that may overlap on the GPU share that array and must be ordered by the caller (see rad.h)."""
    n = C.c_longlong(0)
    st = lib().rad_stage_static(ctx, _dp(I_in), _dp(I_out), _dp(I0), _dp(fluid), gam0, gam1, beta_dt, _dp(T_out), _dp(dT0),
                                C.byref(n) if count_noroot else None, _stream(stream))
    _check(ctx, st)
    return n.value if count_noroot else None


def rad_stage_host(ctx, I_in, I_out, fluid, opac, gam0, gam1, beta_dt, T_out=None, dT0=None, count_noroot=False):
    n = C.c_longlong(0)
    st = lib().rad_stage_host(ctx, _hp(I_in), _hp(I_out), _hp(fluid), _hp(opac), gam0, gam1, beta_dt, _hp(T_out), _hp(dT0),
                              C.byref(n) if count_noroot else None)
    _check(ctx, st)
    return n.value if count_noroot else None


def rad_fill_ghosts(ctx, I, stream=None):
    _check(ctx, lib().rad_fill_ghosts(ctx, _dp(I), _stream(stream)))


def rad_edge_ownership(angles):
    """host only (no device needed): dict(N, E, edge_lo, edge_hi, own_edge[N][3], own_partner[N][3], pull_pos[N][3]) of an angle grid
    given as ("latlon", nzeta, npsi), ("geodesic", nlev) or ("explicit", tables)"""
    a, keep = _angles(angles)  # noqa: F841  (keep: the host tables stay alive until the calls below return)
    n, e = C.c_int(0), C.c_int(0)
    L = lib()
    st = L.rad_edge_ownership(C.byref(a), C.byref(n), C.byref(e), None, None, None, None, None, 0)
    if st != 0:
        raise RadError(st, L.rad_last_error(None).decode())
    N, E = n.value, e.value
    cap = max(E, 3 * N)
    arr = [np.full(cap, -9, np.int32) for _ in range(5)]
    st = L.rad_edge_ownership(C.byref(a), C.byref(n), C.byref(e), *[C.c_void_p(x.ctypes.data) for x in arr], cap)
    if st != 0:
        raise RadError(st, L.rad_last_error(None).decode())
    return dict(N=N, E=E, edge_lo=arr[0][:E].copy(), edge_hi=arr[1][:E].copy(), own_edge=arr[2][:3 * N].reshape(N, 3).copy(),
                own_partner=arr[3][:3 * N].reshape(N, 3).copy(), pull_pos=arr[4][:3 * N].reshape(N, 3).copy())


def rad_exchange_halo(ctx_lo, I_lo, ctx_hi, I_hi, axis, stream=None):
    """halo exchange between block lo and its neighbour hi above it along `axis` (same device)"""
    _check(ctx_lo, lib().rad_exchange_halo(ctx_lo, _dp(I_lo), ctx_hi, _dp(I_hi), int(axis), _stream(stream)))


def rad_transport(ctx, I_in, I_out, I0, gam0, gam1, beta_dt, stream=None):
    _check(ctx, lib().rad_transport(ctx, _dp(I_in), _dp(I_out), _dp(I0), gam0, gam1, beta_dt, _stream(stream)))


def rad_couple(ctx, I, fluid, dt, T_out=None, dT0=None, count_noroot=False, stream=None):
    n = C.c_longlong(0)
    st = lib().rad_couple(ctx, _dp(I), _dp(fluid), dt, _dp(T_out), _dp(dT0), C.byref(n) if count_noroot else None, _stream(stream))
    _check(ctx, st)
    return n.value if count_noroot else None


def rad_moments(ctx, I, frame, fluid, out, stream=None):
    _check(ctx, lib().rad_moments(ctx, _dp(I), int(frame), _dp(fluid), _dp(out), _stream(stream)))


def rad_probe_fp64(ctx):
    """measured FP64 FMA rate of the context's device, lane-level DFMA operations per second"""
    v = C.c_double(0.0)
    _check(ctx, lib().rad_probe_fp64(ctx, C.byref(v)))
    return v.value


def rad_stage_kernels(ctx):
    """(flux-divergence kernel, coupling kernel) instance names of one rad_stage on this context"""
    buf = C.create_string_buffer(256)
    _check(ctx, lib().rad_stage_kernels(ctx, buf, 256))
    return tuple(buf.value.decode().split(";"))


def rad_ncells_total(ctx):
    return lib().rad_ncells_total(ctx)


def rad_launch_count(ctx):
    return lib().rad_launch_count(ctx)


def rad_get_table(ctx, which, n_interior=None):
    """host numpy copy of one of the library's tables (see rad_table in rad.h); TAB_KE needs n_interior = number of interior cells"""
    L = lib()

    def get(w, shape, dtype):
        a = np.zeros(shape, dtype)
        _check(ctx, L.rad_get_table(ctx, w, C.c_void_p(a.ctypes.data), a.nbytes))
        return a

    if which in (TAB_NANG, TAB_NEDGE):
        return int(get(which, (1,), np.int32)[0])
    N, E, nc = int(get(TAB_NANG, (1,), np.int32)[0]), int(get(TAB_NEDGE, (1,), np.int32)[0]), L.rad_ncells_total(ctx)
    spec = {TAB_NHAT: ((N, 3), np.float64), TAB_DOMEGA: ((N,), np.float64), TAB_NNBR: ((N,), np.int32), TAB_NBR: ((N, MAXNBR), np.int32),
            TAB_NBR_EDGE: ((N, MAXNBR), np.int32), TAB_EDGE_LO: ((E,), np.int32), TAB_EDGE_HI: ((E,), np.int32),
            TAB_EDGE_LEN: ((E,), np.float64), TAB_EDGE_MID: ((E, 3), np.float64), TAB_EDGE_NRM: ((E, 3), np.float64),
            TAB_CELL: ((nc, NCELL), np.float64), TAB_FACE: ((nc, 3, NFACE), np.float64), TAB_FACE_SIGN: ((nc, 3, N), np.int8),
            TAB_EDGE_SIGN: ((nc, E), np.int8), TAB_MAXSPEED: ((3,), np.float64), TAB_OWN_EDGE: ((N, 3), np.int32),
            TAB_KE: ((n_interior or 0, 3, N), np.float64), TAB_STAGE_FACE_SIGN: ((nc, 3, N), np.int8)}
    return get(which, *spec[which])
