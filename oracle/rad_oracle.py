"""oracle/rad_oracle.py -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

ctypes/numpy front end of the plain FP64 CPU oracle in ``rad_oracle.c`` (White et al.,
arXiv 2302.04283, section 2.2-2.6; see the C file for per-function citations).  Only
``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this module.  It imports nothing from the CUDA
package and the CUDA package imports nothing from here.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "librad_oracle.so")
_SRC = os.path.join(_HERE, "rad_oracle.c")
NPOINT, NCELL, NFACE, MAXNBR = 132, 72, 8, 6


def build(force=False):
    """Compile the oracle (gcc, -ffp-contract=off so only the explicit fma() chains fuse)."""
    hdr = os.path.join(_HERE, "rad_oracle.h")
    if not force and os.path.exists(_SO) and os.path.getmtime(_SO) >= max(os.path.getmtime(_SRC), os.path.getmtime(hdr)):
        return _SO
    cmd = ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared", "-Wall", "-o", _SO, _SRC, "-lm"]
    subprocess.check_call(cmd, cwd=_HERE)
    return _SO


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_SO)
        vp, dp, ip = C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int)
        L.orc_angles_latlon.restype = vp
        L.orc_angles_latlon.argtypes = [C.c_int, C.c_int]
        L.orc_angles_geodesic.restype = vp
        L.orc_angles_geodesic.argtypes = [C.c_int]
        L.orc_angles_free.argtypes = [vp]
        L.orc_angles_nang.argtypes = [vp]
        L.orc_angles_nedge.argtypes = [vp]
        L.orc_angles_tables.argtypes = [vp] + [vp] * 11
        L.orc_geometry_point.argtypes = [C.c_int, C.c_double, C.c_double, dp, dp]
        L.orc_create.restype = vp
        L.orc_create.argtypes = [C.c_int, C.c_double, C.c_double, C.c_double, ip, C.c_int, dp, dp, ip, ip, vp,
                                 C.c_double, C.c_double, C.c_double, C.c_int, C.c_int, C.c_int]
        L.orc_create_stretched.restype = vp
        L.orc_create_stretched.argtypes = L.orc_create.argtypes + [vp, vp, vp]
        L.orc_destroy.argtypes = [vp]
        L.orc_ncells_total.restype = C.c_longlong
        L.orc_ncells_total.argtypes = [vp]
        L.orc_get_geometry.argtypes = [vp, vp, vp, vp]
        L.orc_fill_ghosts.argtypes = [vp, vp]
        L.orc_transport.argtypes = [vp, vp, vp, C.c_double, C.c_double, C.c_double, vp]
        L.orc_coupling.restype = C.c_longlong
        L.orc_coupling.argtypes = [vp, vp, vp, vp, C.c_double, vp, vp]
        L.orc_stage.restype = C.c_longlong
        L.orc_stage.argtypes = [vp, vp, vp, vp, vp, vp, C.c_double, C.c_double, C.c_double, vp, vp]
        L.orc_set_tau_factor.argtypes = [vp, C.c_double]
        L.orc_cell_velocity.argtypes = [vp, vp, vp, vp]
        L.orc_transport_tau.argtypes = [vp, vp, vp, C.c_double, C.c_double, C.c_double, vp, vp, vp]
        L.orc_moments.argtypes = [vp, vp, C.c_int, vp, vp]
        L.orc_set_option.argtypes = [vp, C.c_int, C.c_int]
        L.orc_has_mirror.argtypes = [vp, C.c_int]
        L.orc_latlon_face_value.restype = C.c_double
        L.orc_latlon_face_value.argtypes = [vp, vp, C.c_int, C.c_int]
        L.orc_velocity_estimate_cell.argtypes = [vp, vp, vp] + [C.c_double] * 6 + [vp, vp, vp]
        L.orc_upwind_tables.argtypes = [vp, vp, vp]
        L.orc_edge_coeffs.argtypes = [vp, C.c_longlong, vp, vp]
        L.orc_max_speed.restype = C.c_double
        L.orc_max_speed.argtypes = [vp, dp]
        _lib = L
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _f64(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a


class Angles:
    """Angle grid tables.  kind 'latlon' (nzeta, npsi) or 'geodesic' (nlev)."""

    def __init__(self, kind, *args):
        L = lib()
        self.h = L.orc_angles_latlon(*args) if kind == "latlon" else L.orc_angles_geodesic(*args)
        if not self.h:
            raise ValueError("bad angle grid")
        N, E = L.orc_angles_nang(self.h), L.orc_angles_nedge(self.h)
        self.N, self.E = N, E
        self.nhat = np.zeros((N, 3)); self.domega = np.zeros(N)
        self.nnbr = np.zeros(N, np.int32); self.nbr = np.zeros((N, MAXNBR), np.int32)
        self.nbr_edge = np.zeros((N, MAXNBR), np.int32)
        self.edge_lo = np.zeros(E, np.int32); self.edge_hi = np.zeros(E, np.int32)
        self.edge_len = np.zeros(E); self.edge_mid = np.zeros((E, 3)); self.edge_nrm = np.zeros((E, 3))
        self.edge_T = np.zeros((E, 30))
        L.orc_angles_tables(self.h, _p(self.nhat), _p(self.domega), _p(self.nnbr), _p(self.nbr), _p(self.nbr_edge),
                            _p(self.edge_lo), _p(self.edge_hi), _p(self.edge_len), _p(self.edge_mid),
                            _p(self.edge_nrm), _p(self.edge_T))

    def latlon_face_value(self, Icell, u, slot):
        """R21: PLM value of angle cell u at its face in slot (0 zeta-, 1 zeta+, 2 psi-, 3 psi+) from one spatial cell's row"""
        Icell = _f64(Icell)
        return lib().orc_latlon_face_value(self.h, _p(Icell), int(u), int(slot))

    def __del__(self):
        try:
            lib().orc_angles_free(self.h)
        except Exception:
            pass


def geometry_point(kind, M, a, x):
    """dict of alpha, beta (3), g, ginv, e[mu][ahat], elow[ahat][mu], omega[c][a][b] at point x."""
    out = np.zeros(NPOINT)
    xx = _f64(x)
    lib().orc_geometry_point(kind, M, a, xx.ctypes.data_as(C.POINTER(C.c_double)), out.ctypes.data_as(C.POINTER(C.c_double)))
    return dict(alpha=out[0], beta=out[1:4].copy(), g=out[4:20].reshape(4, 4).copy(), ginv=out[20:36].reshape(4, 4).copy(),
                e=out[36:52].reshape(4, 4).copy(), elow=out[52:68].reshape(4, 4).copy(), omega=out[68:132].reshape(4, 4, 4).copy())


class Problem:
    """Grid + metric + angles + parameters; the oracle's stage, moments and tables."""

    def __init__(self, angles, n, x0, dx, metric_kind=0, M=1.0, a=0.0, excise_r=0.0, ng=2, bc_lo=(0, 0, 0), bc_hi=(0, 0, 0),
                 gamma_gas=5.0 / 3.0, a_rad=1.0, n0_crit=0.1, recon_space=1, renorm=1, couple=1, tau_factor=0.0, recon_angle=0,
                 vel_estimate=0, dt0_literal=0, xf=None):
        L = lib()
        self.angles = angles
        self.n = tuple(int(v) for v in n); self.ng = ng
        self.NI, self.NJ, self.NK = (self.n[0] + 2 * ng, self.n[1] + 2 * ng, self.n[2] + 2 * ng)
        self.shape = (self.NK, self.NJ, self.NI)
        self.N = angles.N
        i3 = (C.c_int * 3); d3 = (C.c_double * 3)
        # xf: face coordinates of a stretched Cartesian grid, per axis an array of n + 2 ng + 1 values or None (uniform spacing dx from x0)
        self.xf = [None if (xf is None or xf[d] is None) else np.ascontiguousarray(xf[d], dtype=np.float64) for d in range(3)]
        for d in range(3):
            if self.xf[d] is not None and self.xf[d].shape != (self.n[d] + 2 * ng + 1,):
                raise ValueError("xf[%d] needs n + 2 ng + 1 entries" % d)
        fp = [None if v is None else C.c_void_p(v.ctypes.data) for v in self.xf]
        self.h = L.orc_create_stretched(metric_kind, M, a, excise_r, i3(*self.n), ng, d3(*x0), d3(*dx), i3(*bc_lo), i3(*bc_hi), angles.h,
                                        gamma_gas, a_rad, n0_crit, recon_space, renorm, couple, *fp)
        self.ncell = L.orc_ncells_total(self.h)
        self.tau_factor = float(tau_factor)
        L.orc_set_tau_factor(self.h, self.tau_factor)   # constant of Eq.26; 0 = free-streaming flux Eq.24
        if recon_space == 2 and ng < 3:
            raise ValueError("PPM needs ng = 3")
        for which, val in ((0, recon_angle), (1, vel_estimate), (2, dt0_literal)):
            if L.orc_set_option(self.h, which, int(val)) != 0:
                raise ValueError("option %d = %d is not available on this angle grid" % (which, val))
        for d in range(3):
            if (bc_lo[d] == 3 or bc_hi[d] == 3) and not L.orc_has_mirror(self.h, d):
                raise ValueError("reflecting boundary along axis %d: the angle grid is not symmetric under that reflection" % d)

    def __del__(self):
        try:
            lib().orc_destroy(self.h)
        except Exception:
            pass

    def geometry(self):
        cell = np.zeros((self.ncell, NCELL)); face = np.zeros((self.ncell, 3, NFACE)); ex = np.zeros(self.ncell, np.int32)
        lib().orc_get_geometry(self.h, _p(cell), _p(face), _p(ex))
        return cell, face, ex

    def fill_ghosts(self, I):
        assert I.dtype == np.float64 and I.flags.c_contiguous
        lib().orc_fill_ghosts(self.h, _p(I))

    def transport(self, I_in, beta_dt, I0=None, gam0=0.0, gam1=1.0):
        I_in = _f64(I_in); out = np.zeros_like(I_in)
        lib().orc_transport(self.h, _p(I_in), _p(None if I0 is None else _f64(I0)), gam0, gam1, beta_dt, _p(out))
        return out

    def transport_tau(self, I_in, beta_dt, fluid, opac, I0=None, gam0=0.0, gam1=1.0):
        """transport with the optical-depth-aware flux of Eq.26-29 (tau_factor != 0); fluid/opac valid in ghosts too"""
        I_in = _f64(I_in); out = np.zeros_like(I_in)
        lib().orc_transport_tau(self.h, _p(I_in), _p(None if I0 is None else _f64(I0)), gam0, gam1, beta_dt, _p(_f64(fluid)), _p(_f64(opac)), _p(out))
        return out

    def cell_velocity(self, fluid, opac):
        """[ncell][5]: tetrad-frame u^alphahat and alpha_E of every cell"""
        vel = np.zeros((self.ncell, 5))
        lib().orc_cell_velocity(self.h, _p(_f64(fluid)), _p(_f64(opac)), _p(vel))
        return vel

    def coupling(self, I, fluid, opac, dt):
        """in place on I.  returns (T_out, dT0, n_noroot)."""
        assert I.dtype == np.float64 and I.flags.c_contiguous
        fluid = _f64(fluid); opac = _f64(opac)
        T = np.zeros(self.ncell); dT0 = np.zeros((4, self.ncell))
        nf = lib().orc_coupling(self.h, _p(I), _p(fluid), _p(opac), dt, _p(T), _p(dT0))
        return T, dT0, nf

    def stage(self, I_in, fluid, opac, beta_dt, I0=None, gam0=0.0, gam1=1.0):
        """returns (I_out, T_out, dT0, n_noroot); I_in's ghosts are filled in place per bc."""
        assert I_in.dtype == np.float64 and I_in.flags.c_contiguous
        fluid = _f64(fluid); opac = _f64(opac)
        out = np.zeros_like(I_in); T = np.zeros(self.ncell); dT0 = np.zeros((4, self.ncell))
        nf = lib().orc_stage(self.h, _p(I_in), _p(out), _p(None if I0 is None else _f64(I0)), _p(fluid), _p(opac),
                             gam0, gam1, beta_dt, _p(T), _p(dT0))
        return out, T, dT0, nf

    def velocity_estimate_cell(self, Icell, uh, rho, Tm, aP, aEa, aS, dt):
        """Eq.51-55 for one cell: returns (applied, u_estimate[4], G[4], f[3], R[10])"""
        Icell = _f64(Icell); u = _f64(np.array(uh, dtype=np.float64).copy())
        G = np.zeros(4); fr = np.zeros(3); R = np.zeros(10)
        ap = lib().orc_velocity_estimate_cell(self.h, _p(Icell), _p(u), rho, Tm, aP, aEa, aS, dt, _p(G), _p(fr), _p(R))
        return bool(ap), u, G, fr, R

    def moments(self, I, frame, fluid=None):
        ncomp = 10 if frame in (0, 2) else 4
        out = np.zeros((ncomp, self.ncell))
        lib().orc_moments(self.h, _p(_f64(I)), frame, _p(None if fluid is None else _f64(fluid)), _p(out))
        return out

    def upwind_tables(self, faces=True, edges=True):
        fs = np.zeros((self.ncell, 3, self.N), np.int8) if faces else None
        es = np.zeros((self.ncell, self.angles.E), np.int8) if edges else None
        lib().orc_upwind_tables(self.h, _p(fs), _p(es))
        return fs, es

    def edge_coeffs(self, cell):
        ce = np.zeros(self.angles.E); n0e = np.zeros(self.angles.E)
        lib().orc_edge_coeffs(self.h, int(cell), _p(ce), _p(n0e))
        return ce, n0e

    def cell_index(self, k, j, i):
        """flat index of ghosted cell (k,j,i)"""
        return (k * self.NJ + j) * self.NI + i

    def max_speed(self):
        ax = (C.c_double * 3)()
        v = lib().orc_max_speed(self.h, ax)
        return v, tuple(ax)

    def mirror(self, axis):
        """angle permutation of the reflection that flips tetrad component `axis` (R20), -1 where the grid has no image"""
        out = np.zeros(self.N, np.int32)
        for n in range(self.N):
            want = self.angles.nhat[n].copy(); want[axis] = -want[axis]
            d = np.abs(self.angles.nhat - want).max(1)
            out[n] = int(d.argmin()) if d.min() < 1e-12 else -1
        return out

    def interior(self, a):
        """view of the interior of an array whose leading dims are (NK,NJ,NI) flattened or not."""
        ng = self.ng
        a = a.reshape(self.shape + a.shape[1:]) if a.shape[0] == self.ncell else a
        return a[ng:-ng, ng:-ng, ng:-ng]
