"""ctypes binding of the oracle library (TEST INFRASTRUCTURE, NOT PRODUCT).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this module. It never imports the CUDA package and the CUDA package never imports it.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

_f64p = C.POINTER(C.c_double)
_i32p = C.POINTER(C.c_int32)


class _Mesh(C.Structure):
    _fields_ = [("n_nodes", C.c_int64), ("n_cells", C.c_int64), ("n_edges", C.c_int64),
                ("node_xy", _f64p), ("tri", _i32p), ("edge_cell", _i32p), ("cell_edge", _i32p),
                ("zb", _f64p), ("kst", _f64p)]


class _Params(C.Structure):
    _fields_ = [("g", C.c_double), ("h_dry", C.c_double), ("dt_max", C.c_double)]


class Info(C.Structure):
    _fields_ = [("t", C.c_double), ("dt_last", C.c_double), ("steps_done", C.c_int64), ("n_wet", C.c_int64),
                ("vol", C.c_double), ("vol_clipped", C.c_double), ("vol_in", C.c_double),
                ("vol_out", C.c_double), ("flags", C.c_int)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


_libs = {}


def lib(omp=False, single=False):
    """The oracle library: the single-threaded fp64 build (the default), the same source built for single precision
    (single=True: -DSWE_REF_REAL=float), or -- omp=True, bench.py's cpu_baseline_omp line only --
    the fp64 source built with OpenMP."""
    omp = (bool(omp), bool(single))
    if omp not in _libs:
        path = _build.build_f32() if single else (_build.build_omp() if omp[0] else _build.build())
        L = C.CDLL(path)
        L.swe_ref_create.argtypes = [C.POINTER(_Mesh), C.POINTER(_Params), C.POINTER(C.c_void_p)]
        L.swe_ref_create.restype = C.c_int
        L.swe_ref_set_boundary.argtypes = [C.c_void_p, C.c_int, C.c_int, _f64p, C.c_int]
        L.swe_ref_set_state.argtypes = [C.c_void_p, _f64p, _f64p, _f64p, C.c_double]
        L.swe_ref_step.argtypes = [C.c_void_p, C.c_int64, C.c_double, C.c_double, C.POINTER(Info)]
        L.swe_ref_get_state.argtypes = [C.c_void_p, _f64p, _f64p, _f64p]
        L.swe_ref_set_scalars.argtypes = [C.c_void_p, C.c_int, _f64p]
        L.swe_ref_get_scalars.argtypes = [C.c_void_p, _f64p]
        L.swe_ref_set_boundary_scalar.argtypes = [C.c_void_p, C.c_int, _f64p, C.c_int]
        L.swe_ref_set_morphology.argtypes = [C.c_void_p, C.c_int] + [C.c_double] * 5
        L.swe_ref_get_bed.argtypes = [C.c_void_p, _f64p]
        L.swe_ref_get_sediment_flux.argtypes = [C.c_void_p, _f64p]
        L.swe_ref_sediment_state.argtypes = [C.c_int] + [C.c_double] * 11 + [_f64p] * 4
        L.swe_ref_sediment_state.restype = None
        L.swe_ref_sediment_flux.argtypes = [C.c_double] * 8
        L.swe_ref_sediment_flux.restype = C.c_double
        L.swe_ref_destroy.argtypes = [C.c_void_p]
        L.swe_ref_destroy.restype = None
        L.swe_ref_last_error.argtypes = [C.c_void_p]
        L.swe_ref_last_error.restype = C.c_char_p
        L.swe_ref_edge_flux.argtypes = [C.c_double] * 11 + [_f64p] * 4
        L.swe_ref_edge_flux.restype = None
        L.swe_ref_wall_flux_via_ghost.argtypes = [C.c_double] * 4 + [_f64p] * 3
        L.swe_ref_wall_flux_via_ghost.restype = None
        L.swe_ref_get_geometry.argtypes = [C.c_void_p, _f64p, _f64p, _f64p, _f64p]
        L.swe_ref_get_edge_flux.argtypes = [C.c_void_p, _f64p, _f64p, _f64p, _f64p]
        L.swe_ref_peek_dt.argtypes = [C.c_void_p, C.c_double, C.c_double]
        L.swe_ref_peek_dt.restype = C.c_double
        L.swe_ref_cbrt.argtypes = [C.c_double]
        L.swe_ref_cbrt.restype = C.c_double
        _libs[omp] = L
    return _libs[omp]


def _p(a, typ):
    return a.ctypes.data_as(typ)


def edge_flux(g, heL, uL, vL, zL, heR, uR, vR, zR, nx, ny):
    """(F1, F3, GL, GR) of one interior edge."""
    o = [C.c_double() for _ in range(4)]
    lib().swe_ref_edge_flux(g, heL, uL, vL, zL, heR, uR, vR, zR, nx, ny, *[C.byref(x) for x in o])
    return tuple(x.value for x in o)


def cbrt(x):
    """Cube root rounded to nearest (R-14)."""
    return lib().swe_ref_cbrt(float(x))


GRASS, MPM = 1, 2


def sediment_state(formula, alpha, theta_cr, s, dm, g, h, u, v, gn2, nx, ny):
    """(q_B.n, psi = d q_Bn / d q_n, lambda_1, lambda_2) of one cell seen from one interface (Table 2, Eq. 16)."""
    o = [C.c_double() for _ in range(4)]
    lib().swe_ref_sediment_state(int(formula), alpha, theta_cr, s, dm, g, h, u, v, gn2, nx, ny, *[C.byref(x) for x in o])
    return tuple(x.value for x in o)


def sediment_flux(qBi, l1i, l2i, zi, qBj, l1j, l2j, zj):
    """q_Bij of Eq. 14-15."""
    return lib().swe_ref_sediment_flux(qBi, l1i, l2i, zi, qBj, l1j, l2j, zj)


def wall_flux_via_ghost(g, he, un, ut):
    o = [C.c_double() for _ in range(3)]
    lib().swe_ref_wall_flux_via_ghost(g, he, un, ut, *[C.byref(x) for x in o])
    return tuple(x.value for x in o)


class RefSolver:
    """Oracle context built from a workloads.configs.Workload (or the same arrays)."""

    def __init__(self, w, g=None, h_dry=None, dt_max=None, omp=False, precision="double"):
        assert precision in ("double", "single")
        L = self._L = lib(omp, precision == "single")
        self._keep = dict(
            node_xy=np.ascontiguousarray(w.node_xy, np.float64), tri=np.ascontiguousarray(w.tri, np.int32),
            edge_cell=np.ascontiguousarray(w.edge_cell, np.int32), cell_edge=np.ascontiguousarray(w.cell_edge, np.int32),
            zb=np.ascontiguousarray(w.zb, np.float64), kst=np.ascontiguousarray(w.kst, np.float64))
        k = self._keep
        self.n_cells, self.n_edges = k["tri"].shape[0], k["edge_cell"].shape[0]
        m = _Mesh(k["node_xy"].shape[0], self.n_cells, self.n_edges, _p(k["node_xy"], _f64p), _p(k["tri"], _i32p),
                  _p(k["edge_cell"], _i32p), _p(k["cell_edge"], _i32p), _p(k["zb"], _f64p), _p(k["kst"], _f64p))
        p = _Params(w.g if g is None else g, w.h_dry if h_dry is None else h_dry,
                    w.dt_max if dt_max is None else dt_max)
        h = C.c_void_p()
        rc = L.swe_ref_create(C.byref(m), C.byref(p), C.byref(h))
        if rc != 0:
            raise RuntimeError(f"swe_ref_create failed ({rc}): {L.swe_ref_last_error(None).decode()}")
        self._h = h
        for sid, typ, params in getattr(w, "strings", []):
            self.set_boundary(sid, typ, params)
        self.set_state(w.h, w.hu, w.hv, 0.0)

    def set_boundary(self, string_id, typ, params):
        a = np.ascontiguousarray(params, np.float64)
        rc = self._L.swe_ref_set_boundary(self._h, int(string_id), int(typ), _p(a, _f64p), int(a.size))
        assert rc == 0

    def set_state(self, h, hu, hv, t0=0.0):
        a = [np.ascontiguousarray(x, np.float64) for x in (h, hu, hv)]
        assert all(x.shape == (self.n_cells,) for x in a)
        rc = self._L.swe_ref_set_state(self._h, _p(a[0], _f64p), _p(a[1], _f64p), _p(a[2], _f64p), float(t0))
        assert rc == 0

    def set_scalars(self, qc):
        """qc: [n_species, n_cells] specific masses q_c = h * phi_c."""
        a = np.ascontiguousarray(qc, np.float64).reshape(-1, self.n_cells)
        self.n_species = a.shape[0]
        assert self._L.swe_ref_set_scalars(self._h, int(a.shape[0]), _p(a, _f64p)) == 0

    def get_scalars(self):
        out = np.empty((getattr(self, "n_species", 0), self.n_cells))
        assert self._L.swe_ref_get_scalars(self._h, _p(out, _f64p)) == 0
        return out

    def set_boundary_scalar(self, string_id, phi):
        a = np.ascontiguousarray(phi, np.float64)
        assert self._L.swe_ref_set_boundary_scalar(self._h, int(string_id), _p(a, _f64p), int(a.size)) == 0

    def set_morphology(self, formula, alpha, theta_cr=0.047, s=2.65, dm=1e-3, porosity=0.4):
        """Eq. 3 / Eq. 13-16: 0 fixed bed, 1 Grass-like, 2 MPM-like (R-20)."""
        rc = self._L.swe_ref_set_morphology(self._h, int(formula), float(alpha), float(theta_cr), float(s), float(dm),
                                          float(porosity))
        if rc != 0:
            raise ValueError(self._L.swe_ref_last_error(self._h).decode())

    def get_bed(self):
        out = np.empty(self.n_cells)
        assert self._L.swe_ref_get_bed(self._h, _p(out, _f64p)) == 0
        return out

    def sediment_fluxes(self):
        out = np.empty(self.n_edges)
        assert self._L.swe_ref_get_sediment_flux(self._h, _p(out, _f64p)) == 0
        return out

    def step(self, n_steps=-1, t_end=float("inf"), cfl=0.9):
        info = Info()
        rc = self._L.swe_ref_step(self._h, int(n_steps), float(t_end), float(cfl), C.byref(info))
        if rc != 0:
            raise RuntimeError(f"swe_ref_step failed ({rc})")
        return info.as_dict()

    def get_state(self):
        out = [np.empty(self.n_cells) for _ in range(3)]
        rc = self._L.swe_ref_get_state(self._h, *[_p(x, _f64p) for x in out])
        assert rc == 0
        return tuple(out)

    def geometry(self):
        area = np.empty(self.n_cells)
        nx, ny, ln = (np.empty(self.n_edges) for _ in range(3))
        self._L.swe_ref_get_geometry(self._h, _p(area, _f64p), _p(nx, _f64p), _p(ny, _f64p), _p(ln, _f64p))
        return area, nx, ny, ln

    def edge_fluxes(self):
        out = [np.empty(self.n_edges) for _ in range(4)]
        self._L.swe_ref_get_edge_flux(self._h, *[_p(x, _f64p) for x in out])
        return tuple(out)

    def peek_dt(self, cfl=0.9, t_end=float("inf")):
        return self._L.swe_ref_peek_dt(self._h, float(cfl), float(t_end))

    def close(self):
        if self._h:
            self._L.swe_ref_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
