"""Thin Python binding of the C-ABI in include/swe.h (libswe_b200.so, CUDA sm_100a).

Argument marshalling only: every step of the shallow-water path runs in the library's kernels.  PyTorch is
used for device memory (the workspace tensor lent to the library, optional device-resident state tensors)
and for the stream.  There is no CPU fallback: a missing library or a missing GPU raises.

    from paper_2102_12862_b200 import Solver
    s = Solver(node_xy, tri, edge_cell, cell_edge, zb, kst)      # swe_create
    s.set_boundary(0, BC_INFLOW_Q, [0, 100, 3600, 2000])         # swe_set_boundary
    s.set_state(h, hu, hv)                                       # swe_set_state
    info = s.step(n_steps=100, cfl=0.9)                          # swe_step
    h, hu, hv = s.get_state()                                    # swe_get_state
    s.close()                                                    # swe_destroy
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libswe_b200.so")

OK, EINVAL, EMESH, ENOMEM, ECUDA, ENONFINITE = 0, -1, -2, -3, -4, -5
EDGE_WALL, EDGE_TRANSMISSIVE = -1, -2
BC_NONE, BC_INFLOW_Q, BC_OUTFLOW_UNIFORM = 0, 1, 2
RENUMBER_NONE, RENUMBER_MORTON, RENUMBER_RCM = 0, 1, 2
FLAG_NONFINITE, FLAG_DT_UNBOUNDED, FLAG_STALLED = 1, 2, 4
VARIANT_AUTO, VARIANT_THREE_PASS, VARIANT_PATCH = 0, 1, 2
PRECISION_DOUBLE, PRECISION_SINGLE = 0, 1

_f64p = C.POINTER(C.c_double)
_i32p = C.POINTER(C.c_int32)

EXPORTS = (
    "swe_params_default", "swe_workspace_bytes", "swe_create", "swe_set_boundary", "swe_set_state", "swe_step",
    "swe_get_state", "swe_destroy", "swe_last_error", "swe_get_geometry", "swe_get_edge_flux", "swe_peek_dt",
    "swe_get_permutation", "swe_get_tables", "swe_device_cbrt", "swe_kernel_launches", "swe_profile_step",
    "swe_step_kernel_count", "swe_step_kernel_name", "swe_algorithmic_bytes", "swe_survey_bytes", "swe_get_patch_stats",
    "swe_set_scalars", "swe_get_scalars", "swe_set_boundary_scalar", "swe_host_preprocess",
    "swe_set_morphology", "swe_get_bed", "swe_get_sediment_flux", "swe_state_summary_static",
)


class SweMesh(C.Structure):
    _fields_ = [("n_nodes", C.c_int64), ("n_cells", C.c_int64), ("n_edges", C.c_int64),
                ("node_xy", _f64p), ("tri", _i32p), ("edge_cell", _i32p), ("cell_edge", _i32p),
                ("zb", _f64p), ("kst", _f64p)]


class SweParams(C.Structure):
    _fields_ = [("g", C.c_double), ("h_dry", C.c_double), ("dt_max", C.c_double), ("renumber", C.c_int),
                ("state_on_device", C.c_int), ("steps_per_graph", C.c_int), ("variant", C.c_int), ("patch_cells", C.c_int),
                ("n_species", C.c_int), ("morphology", C.c_int), ("precision", C.c_int), ("cuda_stream", C.c_void_p),
                ("workspace", C.c_void_p), ("workspace_bytes", C.c_size_t)]


class SweStepInfo(C.Structure):
    _fields_ = [("t", C.c_double), ("dt_last", C.c_double), ("steps_done", C.c_int64), ("n_wet", C.c_int64),
                ("vol", C.c_double), ("vol_clipped", C.c_double), ("vol_in", C.c_double), ("vol_out", C.c_double),
                ("flags", C.c_int)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


class SweError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"swe error {code}: {msg}")
        self.code = code


_lib = None


def lib():
    """Loads libswe_b200.so (built by `python -m paper_2102_12862_b200.build`); raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2102_12862_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        L.swe_params_default.argtypes = [C.POINTER(SweParams)]
        L.swe_params_default.restype = None
        L.swe_workspace_bytes.argtypes = [C.POINTER(SweMesh), C.POINTER(SweParams)]
        L.swe_workspace_bytes.restype = C.c_size_t
        L.swe_create.argtypes = [C.POINTER(SweMesh), C.POINTER(SweParams), C.POINTER(C.c_void_p)]
        L.swe_set_boundary.argtypes = [C.c_void_p, C.c_int, C.c_int, _f64p, C.c_int]
        L.swe_set_state.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_double]
        L.swe_step.argtypes = [C.c_void_p, C.c_int64, C.c_double, C.c_double, C.POINTER(SweStepInfo)]
        L.swe_get_state.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.swe_destroy.argtypes = [C.c_void_p]
        L.swe_destroy.restype = None
        L.swe_last_error.argtypes = [C.c_void_p]
        L.swe_last_error.restype = C.c_char_p
        L.swe_get_geometry.argtypes = [C.c_void_p, _f64p, _f64p, _f64p, _f64p]
        L.swe_get_edge_flux.argtypes = [C.c_void_p, _f64p, _f64p, _f64p, _f64p, _f64p]
        L.swe_peek_dt.argtypes = [C.c_void_p, C.c_double, C.c_double, _f64p]
        L.swe_get_permutation.argtypes = [C.c_void_p, _i32p, _i32p]
        L.swe_get_tables.argtypes = [C.c_void_p, C.POINTER(C.c_int64), _i32p, _i32p]
        L.swe_device_cbrt.argtypes = [_f64p, _f64p, C.c_int64]
        L.swe_kernel_launches.argtypes = [C.c_void_p]
        L.swe_kernel_launches.restype = C.c_int64
        L.swe_profile_step.argtypes = [C.c_void_p, C.c_int64, C.c_double, _f64p, C.c_int]
        L.swe_step_kernel_count.argtypes = [C.c_void_p]
        L.swe_step_kernel_name.argtypes = [C.c_void_p, C.c_int]
        L.swe_step_kernel_name.restype = C.c_char_p
        L.swe_algorithmic_bytes.argtypes = [C.c_void_p, C.c_int]
        L.swe_algorithmic_bytes.restype = C.c_int64
        L.swe_survey_bytes.argtypes = [C.c_void_p, C.c_int]
        L.swe_survey_bytes.restype = C.c_int64
        L.swe_get_patch_stats.argtypes = [C.c_void_p, C.POINTER(C.c_int64), C.c_int]
        L.swe_host_preprocess.argtypes = [C.POINTER(SweMesh), C.c_int, C.c_int, C.POINTER(C.c_int64), C.c_int, _i32p, _i32p]
        L.swe_set_scalars.argtypes = [C.c_void_p, C.c_void_p]
        L.swe_get_scalars.argtypes = [C.c_void_p, C.c_void_p]
        L.swe_set_boundary_scalar.argtypes = [C.c_void_p, C.c_int, _f64p, C.c_int]
        L.swe_set_morphology.argtypes = [C.c_void_p, C.c_int] + [C.c_double] * 5
        L.swe_get_bed.argtypes = [C.c_void_p, C.c_void_p]
        L.swe_get_sediment_flux.argtypes = [C.c_void_p, C.c_void_p]
        L.swe_state_summary_static.argtypes = [C.c_void_p] * 4 + [C.c_int64, C.c_double, C.c_void_p, C.c_void_p]
        _lib = L
    return _lib


def _p(a, typ):
    return a.ctypes.data_as(typ) if a is not None else None


class Solver:
    """One swe_ctx.  Mesh arrays are numpy (host); state arrays are numpy (host pointers) or, with
    state_on_device=True, torch CUDA float64 tensors (device pointers)."""

    def __init__(self, node_xy, tri, edge_cell=None, cell_edge=None, zb=None, kst=None, *, g=9.81, h_dry=1e-3,
                 dt_max=float("inf"), renumber=RENUMBER_MORTON, state_on_device=False, steps_per_graph=32,
                 device="cuda:0", own_workspace=False, variant=VARIANT_AUTO, patch_cells=0, n_species=0,
                 morphology=False, workspace_bytes=None, precision=PRECISION_DOUBLE):
        import torch  # device memory + stream only

        if not torch.cuda.is_available():
            raise RuntimeError("paper_2102_12862_b200 needs a CUDA device (sm_100a); there is no CPU fallback")
        L = lib()
        self._torch = torch
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        node_xy = np.ascontiguousarray(node_xy, np.float64)
        tri = np.ascontiguousarray(tri, np.int32)
        ec = None if edge_cell is None else np.ascontiguousarray(edge_cell, np.int32)
        ce = None if cell_edge is None else np.ascontiguousarray(cell_edge, np.int32)
        self.n_cells = int(tri.shape[0])
        zb = np.ascontiguousarray(zb if zb is not None else np.zeros(self.n_cells), np.float64)
        kst = np.ascontiguousarray(kst if kst is not None else np.full(self.n_cells, np.inf), np.float64)
        assert zb.shape == (self.n_cells,) and kst.shape == (self.n_cells,)
        n_edges = 0 if ec is None else int(ec.shape[0])
        mesh = SweMesh(int(node_xy.shape[0]), self.n_cells, n_edges, _p(node_xy, _f64p), _p(tri, _i32p),
                       _p(ec, _i32p), _p(ce, _i32p), _p(zb, _f64p), _p(kst, _f64p))
        prm = SweParams()
        L.swe_params_default(C.byref(prm))
        prm.g, prm.h_dry, prm.dt_max = float(g), float(h_dry), float(dt_max)
        prm.renumber, prm.state_on_device, prm.steps_per_graph = int(renumber), int(bool(state_on_device)), int(steps_per_graph)
        prm.variant, prm.patch_cells, prm.n_species = int(variant), int(patch_cells), int(n_species)
        prm.morphology = int(bool(morphology))
        prm.precision = int(precision)
        self.n_species = int(n_species)
        self.stream = torch.cuda.current_stream(self.device)
        prm.cuda_stream = self.stream.cuda_stream
        self.workspace = None
        if not own_workspace:
            # every device array of the context lives in this torch tensor (workspace_bytes: tests lend too little)
            nbytes = int(L.swe_workspace_bytes(C.byref(mesh), C.byref(prm))) if workspace_bytes is None else int(workspace_bytes)
            if nbytes > 0:       # 0: the arguments are invalid -- swe_create below reports why, with its error code
                self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
                prm.workspace, prm.workspace_bytes = self.workspace.data_ptr(), nbytes
        self.workspace_nbytes = 0 if self.workspace is None else int(self.workspace.numel())
        self.state_on_device = bool(state_on_device)
        h = C.c_void_p()
        rc = L.swe_create(C.byref(mesh), C.byref(prm), C.byref(h))
        if rc != OK:
            raise SweError(rc, L.swe_last_error(None).decode())
        self._h = h
        ne = C.c_int64()
        L.swe_get_tables(self._h, C.byref(ne), None, None)
        self.n_edges = int(ne.value)

    # ---- the five calls + boundary strings
    def _check(self, rc):
        if rc != OK:
            raise SweError(rc, lib().swe_last_error(self._h).decode())

    def set_boundary(self, string_id, typ, params):
        a = np.ascontiguousarray(params, np.float64)
        self._check(lib().swe_set_boundary(self._h, int(string_id), int(typ), _p(a, _f64p), int(a.size)))

    def _ptrs(self, arrs):
        if self.state_on_device:
            for x in arrs:
                assert x.is_cuda and x.dtype == self._torch.float64 and x.is_contiguous() and x.numel() == self.n_cells
            return [C.c_void_p(x.data_ptr()) for x in arrs]
        for x in arrs:
            assert x.dtype == np.float64 and x.flags.c_contiguous and x.shape == (self.n_cells,)
        return [C.c_void_p(x.ctypes.data) for x in arrs]

    def set_state(self, h, hu, hv, t0=0.0):
        if not self.state_on_device:
            h, hu, hv = (np.ascontiguousarray(x, np.float64) for x in (h, hu, hv))
        self._check(lib().swe_set_state(self._h, *self._ptrs((h, hu, hv)), float(t0)))

    def step(self, n_steps=-1, t_end=float("inf"), cfl=0.9, info=True):
        inf = SweStepInfo() if info else None
        rc = lib().swe_step(self._h, int(n_steps), float(t_end), float(cfl), C.byref(inf) if info else None)
        self._check(rc)
        return inf.as_dict() if info else None

    def get_state(self, out=None):
        if out is None:
            if self.state_on_device:
                out = tuple(self._torch.empty(self.n_cells, dtype=self._torch.float64, device=self.device) for _ in range(3))
            else:
                out = tuple(np.empty(self.n_cells) for _ in range(3))
        self._check(lib().swe_get_state(self._h, *self._ptrs(out)))
        return out

    def set_scalars(self, qc):
        """qc: [n_species, n_cells] specific masses q_c = h * phi_c (numpy, or a torch CUDA tensor with
        state_on_device=True)."""
        if self.state_on_device:
            assert qc.is_cuda and qc.dtype == self._torch.float64 and qc.is_contiguous()
            assert qc.numel() == self.n_species * self.n_cells
            ptr = C.c_void_p(qc.data_ptr())
        else:
            qc = np.ascontiguousarray(qc, np.float64).reshape(self.n_species, self.n_cells)
            ptr = C.c_void_p(qc.ctypes.data)
        self._check(lib().swe_set_scalars(self._h, ptr))

    def get_scalars(self):
        if self.state_on_device:
            out = self._torch.empty((self.n_species, self.n_cells), dtype=self._torch.float64, device=self.device)
            ptr = C.c_void_p(out.data_ptr())
        else:
            out = np.empty((self.n_species, self.n_cells))
            ptr = C.c_void_p(out.ctypes.data)
        self._check(lib().swe_get_scalars(self._h, ptr))
        return out

    def set_morphology(self, formula, alpha, theta_cr=0.047, s=2.65, dm=1e-3, porosity=0.4):
        """swe_set_morphology: 0 fixed bed, 1 Grass-like, 2 MPM-like (Eq. 3, Eq. 13-16, Table 2; R-20)."""
        self._check(lib().swe_set_morphology(self._h, int(formula), float(alpha), float(theta_cr), float(s), float(dm),
                                             float(porosity)))

    def _get_vector(self, fn, n):
        if self.state_on_device:
            out = self._torch.empty(n, dtype=self._torch.float64, device=self.device)
            ptr = C.c_void_p(out.data_ptr())
        else:
            out = np.empty(n)
            ptr = C.c_void_p(out.ctypes.data)
        self._check(fn(self._h, ptr))
        return out

    def get_bed(self):
        """z_B per cell, caller numbering."""
        return self._get_vector(lib().swe_get_bed, self.n_cells)

    def sediment_fluxes(self):
        """q_Bij per edge of the most recent step (inspection)."""
        return self._get_vector(lib().swe_get_sediment_flux, self.n_edges)

    def set_boundary_scalar(self, string_id, phi):
        a = np.ascontiguousarray(phi, np.float64)
        self._check(lib().swe_set_boundary_scalar(self._h, int(string_id), _p(a, _f64p), int(a.size)))

    def close(self):
        if getattr(self, "_h", None):
            lib().swe_destroy(self._h)
            self._h = None
            self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- inspection
    def geometry(self):
        area = np.empty(self.n_cells)
        nx, ny, ln = (np.empty(self.n_edges) for _ in range(3))
        self._check(lib().swe_get_geometry(self._h, _p(area, _f64p), _p(nx, _f64p), _p(ny, _f64p), _p(ln, _f64p)))
        return area, nx, ny, ln

    def edge_fluxes(self):
        out = [np.empty(self.n_edges) for _ in range(4)]
        theta = np.empty(self.n_cells)
        self._check(lib().swe_get_edge_flux(self._h, *[_p(x, _f64p) for x in out], _p(theta, _f64p)))
        return tuple(out) + (theta,)

    def peek_dt(self, cfl=0.9, t_end=float("inf")):
        dt = C.c_double()
        self._check(lib().swe_peek_dt(self._h, float(cfl), float(t_end), C.byref(dt)))
        return dt.value

    def permutation(self):
        cp = np.empty(self.n_cells, np.int32)
        ep = np.empty(self.n_edges, np.int32)
        self._check(lib().swe_get_permutation(self._h, _p(cp, _i32p), _p(ep, _i32p)))
        return cp, ep

    def tables(self):
        ec = np.empty((self.n_edges, 2), np.int32)
        ce = np.empty((self.n_cells, 3), np.int32)
        self._check(lib().swe_get_tables(self._h, None, _p(ec, _i32p), _p(ce, _i32p)))
        return ec, ce

    def step_kernels(self):
        """Names of the kernels of one time step of this context's variant, in launch order."""
        n = int(lib().swe_step_kernel_count(self._h))
        return [lib().swe_step_kernel_name(self._h, k).decode() for k in range(n)]

    def profile_step(self, n_steps, cfl=0.9):
        """{kernel name: mean device ms per step} over n_steps event-bracketed plain-launch steps (swe_profile_step)."""
        names = self.step_kernels()
        ms = np.zeros(len(names))
        self._check(lib().swe_profile_step(self._h, int(n_steps), float(cfl), _p(ms, _f64p), len(names)))
        return {nm: float(ms[k]) for k, nm in enumerate(names)}

    def algorithmic_bytes(self):
        """{kernel name: algorithmic DRAM bytes per launch} (swe_algorithmic_bytes)."""
        return {nm: int(lib().swe_algorithmic_bytes(self._h, k)) for k, nm in enumerate(self.step_kernels())}

    def survey_bytes(self):
        """{kernel name: bytes per launch on SURVEY.md section 8(d)'s per-cell figures} (swe_survey_bytes)."""
        return {nm: int(lib().swe_survey_bytes(self._h, k)) for k, nm in enumerate(self.step_kernels())}

    def patch_stats(self):
        out = (C.c_int64 * 12)()
        self._check(lib().swe_get_patch_stats(self._h, out, 12))
        keys = ("variant", "patches", "patch_cells", "smem_bytes", "sum_local_cells", "sum_local_edges",
                "max_local_cells", "max_local_edges", "patch_steps_skipped", "min_blocks_per_sm", "blob_stride",
                "blob_staged_bytes")
        return dict(zip(keys, (int(v) for v in out)))

    @property
    def kernel_launches(self):
        return int(lib().swe_kernel_launches(self._h))


def host_preprocess(node_xy, tri, edge_cell=None, cell_edge=None, zb=None, kst=None, renumber=RENUMBER_MORTON,
                    patch_cells=384):
    """swe_host_preprocess: the host part of swe_create (validation, tables, geometry, renumbering, patch tables).
    Needs no GPU.  Returns (stats dict, cell_perm, edge_perm); raises SweError for an invalid mesh."""
    node_xy = np.ascontiguousarray(node_xy, np.float64)
    tri = np.ascontiguousarray(tri, np.int32)
    n = int(tri.shape[0])
    ec = None if edge_cell is None else np.ascontiguousarray(edge_cell, np.int32)
    ce = None if cell_edge is None else np.ascontiguousarray(cell_edge, np.int32)
    zb = np.ascontiguousarray(zb if zb is not None else np.zeros(n), np.float64)
    kst = np.ascontiguousarray(kst if kst is not None else np.full(n, np.inf), np.float64)
    mesh = SweMesh(int(node_xy.shape[0]), n, 0 if ec is None else int(ec.shape[0]), _p(node_xy, _f64p), _p(tri, _i32p),
                   _p(ec, _i32p), _p(ce, _i32p), _p(zb, _f64p), _p(kst, _f64p))
    out = (C.c_int64 * 10)()
    cp = np.empty(n, np.int32)
    ep = np.empty(3 * n, np.int32)
    rc = lib().swe_host_preprocess(C.byref(mesh), int(renumber), int(patch_cells), out, 10, _p(cp, _i32p), _p(ep, _i32p))
    if rc != OK:
        raise SweError(rc, lib().swe_last_error(None).decode())
    keys = ("n_edges", "patches", "sum_local_cells", "sum_local_edges", "max_local_cells", "max_local_edges",
            "smem_bytes", "sum_own_cells", "distinct_own_cells", "patch_neighbour_entries")
    st = dict(zip(keys, (int(v) for v in out)))
    return st, cp, ep[:st["n_edges"]]


def workspace_bytes(node_xy, tri, edge_cell=None, cell_edge=None, zb=None, kst=None, **params):
    """swe_workspace_bytes: device bytes of a context for this mesh and these swe_params fields (renumber, variant,
    patch_cells, n_species, morphology); 0 if swe_create would reject them.  Needs no GPU."""
    node_xy = np.ascontiguousarray(node_xy, np.float64)
    tri = np.ascontiguousarray(tri, np.int32)
    n = int(tri.shape[0])
    ec = None if edge_cell is None else np.ascontiguousarray(edge_cell, np.int32)
    ce = None if cell_edge is None else np.ascontiguousarray(cell_edge, np.int32)
    zb = np.ascontiguousarray(zb if zb is not None else np.zeros(n), np.float64)
    kst = np.ascontiguousarray(kst if kst is not None else np.full(n, np.inf), np.float64)
    mesh = SweMesh(int(node_xy.shape[0]), n, 0 if ec is None else int(ec.shape[0]), _p(node_xy, _f64p), _p(tri, _i32p),
                   _p(ec, _i32p), _p(ce, _i32p), _p(zb, _f64p), _p(kst, _f64p))
    prm = SweParams()
    lib().swe_params_default(C.byref(prm))
    for k, v in params.items():
        setattr(prm, k, int(v))
    return int(lib().swe_workspace_bytes(C.byref(mesh), C.byref(prm)))


def device_cbrt(x):
    """Cube root rounded to nearest as the kernels evaluate it (swe_device_cbrt; R-14)."""
    x = np.ascontiguousarray(x, np.float64)
    y = np.empty_like(x)
    rc = lib().swe_device_cbrt(_p(x, _f64p), _p(y, _f64p), int(x.size))
    if rc != OK:
        raise SweError(rc, lib().swe_last_error(None).decode())
    return y


SUMMARY_STATIC_MAX_CELLS = 1 << 24   # include/swe.h SWE_SUMMARY_STATIC_MAX_CELLS


def state_summary_static(h, hu, hv, area, h_dry, out, n_cells=None, stream=None):
    """swe_state_summary_static: volume, wet-cell count and non-finite check of a state, with no allocation (the scratch
    is a static device array inside the library; calls must not overlap on the GPU).  h, hu, hv, area: CUDA float64
    tensors (or integer device addresses, then n_cells is required); out: a CUDA tensor of 24 bytes that receives
    (vol: f64, n_wet: i64, nonfinite: i32, pad: i32); stream: cudaStream_t as an integer (None: torch's current one).
    Nothing is copied or synchronised here: read `out` after the stream has run."""
    def ptr(x):
        return int(x.data_ptr()) if hasattr(x, "data_ptr") else int(x)
    if n_cells is None:
        n_cells = int(h.numel())
    if stream is None:
        import torch  # stream handle only
        stream = torch.cuda.current_stream().cuda_stream
    rc = lib().swe_state_summary_static(ptr(h), ptr(hu), ptr(hv), ptr(area), int(n_cells), float(h_dry), int(stream) or None,
                                        ptr(out))
    if rc != OK:
        raise SweError(rc, lib().swe_last_error(None).decode())


def from_workload(w, **kw):
    """Solver for a workloads.configs.Workload (mesh, parameters, boundary strings, initial state)."""
    kw.setdefault("g", w.g)
    kw.setdefault("h_dry", w.h_dry)
    kw.setdefault("dt_max", w.dt_max)
    s = Solver(w.node_xy, w.tri, w.edge_cell, w.cell_edge, w.zb, w.kst, **kw)
    for sid, typ, params in getattr(w, "strings", []):
        s.set_boundary(sid, typ, params)
    if s.state_on_device:
        import torch
        s.set_state(*(torch.from_numpy(np.ascontiguousarray(x)).to(s.device) for x in (w.h, w.hu, w.hv)), 0.0)
    else:
        s.set_state(w.h, w.hu, w.hv, 0.0)
    return s
