"""Seeded synthetic workloads: the five configurations of BASELINE.json plus the small cases the
oracle pins use. Inputs only -- no part of the scheme is evaluated here.

Every generator returns a `Workload` whose arrays go unchanged to the oracle (`oracle/`) and to the
CUDA library (`paper_2102_12862_b200`). Seeds follow SURVEY 8(d): seed = 12862*10 + config id.

The paper's own workloads (Malpasset T1 etc.) are not available; configs 3-5 stand
in for T1's shape: 1e5..1e7 irregular triangles, a shock running over friction-bearing terrain, CFL
0.9. Recipe details and the choices the paper leaves open are listed in DESIGN.md.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

from . import mesh as M

BC_INFLOW_Q = 1          # include/swe.h SWE_BC_INFLOW_Q
BC_OUTFLOW_UNIFORM = 2   # include/swe.h SWE_BC_OUTFLOW_UNIFORM


@dataclass
class Workload:
    name: str
    node_xy: np.ndarray          # [V,2] float64
    tri: np.ndarray              # [N,3] int32, CCW
    edge_cell: np.ndarray        # [E,2] int32
    cell_edge: np.ndarray        # [N,3] int32
    zb: np.ndarray               # [N] float64
    kst: np.ndarray              # [N] float64 (+inf = frictionless)
    h: np.ndarray                # [N]
    hu: np.ndarray               # [N]
    hv: np.ndarray               # [N]
    cfl: float = 0.9
    t_end: float = float("inf")
    n_steps: int = -1
    h_dry: float = 1e-3
    g: float = 9.81
    dt_max: float = float("inf")
    strings: list = field(default_factory=list)   # [(string_id, type, params ndarray)]
    meta: dict = field(default_factory=dict)

    @property
    def n_cells(self):
        return int(self.tri.shape[0])

    @property
    def n_edges(self):
        return int(self.edge_cell.shape[0])

    @property
    def n_nodes(self):
        return int(self.node_xy.shape[0])

    def permuted(self, seed: int):
        """The same problem with cells and edges randomly renumbered (SURVEY O-9 / R-15).
        Returns (workload, cell_perm) with new cell c = old cell cell_perm[c]."""
        rng = np.random.default_rng(seed)
        cp = rng.permutation(self.n_cells)
        ep = rng.permutation(self.n_edges)
        # members of a boundary string keep their relative order: "string order" = ascending caller edge id
        # is part of the definition of the string sums (R-11), so it is not a renumbering freedom
        is_member = self.edge_cell[ep, 1] <= -3
        ep[is_member] = np.sort(ep[is_member])
        tri, ec, ce = M.permute_mesh(self.tri, self.edge_cell, self.cell_edge, cp, ep)
        w = Workload(self.name + "-perm", self.node_xy, tri, ec, ce, self.zb[cp].copy(),
                     self.kst[cp].copy(), self.h[cp].copy(), self.hu[cp].copy(), self.hv[cp].copy(),
                     self.cfl, self.t_end, self.n_steps, self.h_dry, self.g, self.dt_max,
                     list(self.strings), dict(self.meta))
        return w, cp


def _seed(config_id: int) -> int:
    return 12862 * 10 + config_id


def _finish(name, node_xy, tri, zb, kst, h, **kw) -> Workload:
    edge_cell, cell_edge = M.build_edge_tables(tri, node_xy.shape[0])
    n = tri.shape[0]
    return Workload(name, np.ascontiguousarray(node_xy, dtype=np.float64),
                    np.ascontiguousarray(tri, dtype=np.int32), edge_cell, cell_edge,
                    np.ascontiguousarray(zb, dtype=np.float64), np.ascontiguousarray(kst, dtype=np.float64),
                    np.ascontiguousarray(h, dtype=np.float64), np.zeros(n), np.zeros(n), **kw)


def _set_boundary_codes(w: Workload, code_of_midpoint):
    """code_of_midpoint(mx, my) -> int array of boundary codes, applied to boundary edges only."""
    mid = M.edge_midpoints(w.node_xy, w.tri, w.edge_cell, w.cell_edge)
    b = w.edge_cell[:, 1] < 0
    w.edge_cell[b, 1] = code_of_midpoint(mid[b, 0], mid[b, 1]).astype(np.int32)


# ----------------------------------------------------------------------------- config 1 (+ twins)
def dam_break_channel(nx=500, ny=4, lx=100.0, ly=2.0, h_left=1.0, h_right=0.0, x_dam=50.0,
                      kst=float("inf"), t_end=4.0, cfl=0.9, transmissive_ends=False,
                      q_left=0.0, q_right=0.0) -> Workload:
    """BASELINE.json configs[0]: 100 m x 2 m channel, 500x4 quads split in two (4,000 cells), flat
    frictionless bed, h = h_left for x < x_dam else h_right, walls, CFL 0.9, run to t = 4 s.
    h_right = 0 -> Ritter; h_right > 0 -> Stoker twin. q_left/q_right != 0 with transmissive ends
    gives the hydrodynamic half of the paper's T5 (Eq. 22)."""
    node_xy, tri = M.structured_tri_mesh(nx, ny, lx, ly)
    cx = M.centroids(node_xy, tri)[:, 0]
    n = tri.shape[0]
    h = np.where(cx < x_dam, h_left, h_right).astype(np.float64)
    w = _finish(f"dam-break-channel-{nx}x{ny}", node_xy, tri, np.zeros(n), np.full(n, kst), h,
                cfl=cfl, t_end=t_end)
    w.hu = np.where(cx < x_dam, q_left, q_right).astype(np.float64)
    if transmissive_ends:
        _set_boundary_codes(w, lambda mx, my: np.where((mx < 1e-9) | (mx > lx - 1e-9),
                                                       M.BC_TRANSMISSIVE, M.BC_WALL))
    w.meta.update(dict(lx=lx, ly=ly, nx=nx, ny=ny, x_dam=x_dam, h_left=h_left, h_right=h_right))
    return w


def config1(refine: float = 1.0) -> Workload:
    nx = int(round(500 * refine))
    ny = max(1, int(round(4 * refine)))
    w = dam_break_channel(nx, ny)
    w.name = f"config1-ritter-{nx}x{ny}"
    return w


# ----------------------------------------------------------------------------- config 2
def gaussian_bumps(rng, n_bumps, lx, ly, amp=(0.5, 3.0), width=(20.0, 100.0)):
    c = np.stack([rng.uniform(0.0, lx, n_bumps), rng.uniform(0.0, ly, n_bumps)], axis=1)
    a = rng.uniform(*amp, n_bumps)
    wd = rng.uniform(*width, n_bumps)
    return c, a, wd


def eval_bumps(xy, c, a, wd):
    z = np.zeros(xy.shape[0])
    for m in range(c.shape[0]):
        d2 = (xy[:, 0] - c[m, 0]) ** 2 + (xy[:, 1] - c[m, 1]) ** 2
        z += a[m] * np.exp(-d2 / (2.0 * wd[m] ** 2))
    return z


def config2(n=200, n_steps=1000, eta=2.0) -> Workload:
    """BASELINE.json configs[1]: lake at rest over 8 Gaussian bumps, 1000 m x 1000 m, n x n quads
    split with alternating diagonal, interior nodes jittered by +-20 % of the spacing, eta = 2 m so
    the bump tops are dry, Strickler 30, walls."""
    rng = np.random.default_rng(_seed(2))
    lx = ly = 1000.0
    node_xy, tri = M.structured_tri_mesh(n, n, lx, ly, alternate=True, jitter=0.2, rng=rng)
    # seeded bumps; re-draw amplitudes until at least one bump top is dry
    c, a, wd = gaussian_bumps(rng, 8, lx, ly)
    zn = eval_bumps(node_xy, c, a, wd)
    zb = zn[tri].mean(axis=1)
    while not np.any(zb > eta):
        a = rng.uniform(0.5, 3.0, 8) + 0.5
        zn = eval_bumps(node_xy, c, a, wd)
        zb = zn[tri].mean(axis=1)
    h = np.maximum(0.0, eta - zb)
    w = _finish(f"config2-lake-at-rest-{n}x{n}", node_xy, tri, zb, np.full(tri.shape[0], 30.0), h,
                n_steps=n_steps)
    w.meta.update(dict(eta=eta))
    return w


# ----------------------------------------------------------------------------- config 3 / 5
def config3(target_cells=1_000_000, n_steps=2000, lx=2000.0, config_id=3) -> Workload:
    """BASELINE.json configs[2] (and configs[4] at 8M / 16M): circular dam break on an unstructured
    Delaunay mesh of blue-noise-like points. h = 10 m inside r = 0.1*lx of the centre, 1 m outside;
    bed = lognormal roughness 0.02*exp(0.5 N(0,1)) m per cell, k ~ U(20,40) per cell; transmissive
    boundaries; CFL 0.9.  The domain is lx x lx (2000 m at full size; tests shrink lx together with
    target_cells so that the spacing, hence the time step, stays that of the full-size problem)."""
    rng = np.random.default_rng(_seed(3))        # same field seeds for config 5
    ly = lx
    area_per_point = lx * ly / (0.5 * target_cells)
    a = np.sqrt(area_per_point / (np.sqrt(3.0) / 2.0))
    pts_in = M.jittered_hex_points(0.55 * a, lx - 0.55 * a, 0.55 * a, ly - 0.55 * a, a, 0.3, rng)
    pts_b = M.rectangle_boundary_points(0.0, lx, 0.0, ly, a)
    node_xy, tri = M.delaunay_tri_mesh(np.concatenate([pts_b, pts_in]), 1e-3 * a * a)
    n = tri.shape[0]
    ctr = M.centroids(node_xy, tri)
    zb = 0.02 * np.exp(0.5 * rng.standard_normal(n))
    kst = rng.uniform(20.0, 40.0, n)
    r = np.hypot(ctr[:, 0] - 0.5 * lx, ctr[:, 1] - 0.5 * ly)
    h = np.where(r < 0.1 * lx, 10.0, 1.0)
    w = _finish(f"config{config_id}-circular-dam-break-{n}", node_xy, tri, zb, kst, h, n_steps=n_steps)
    w.edge_cell[w.edge_cell[:, 1] < 0, 1] = M.BC_TRANSMISSIVE
    w.meta.update(dict(spacing=a, lx=lx))
    return w


def config5(target_cells=8_000_000, n_steps=1000) -> Workload:
    return config3(target_cells=target_cells, n_steps=n_steps, config_id=5)


# ----------------------------------------------------------------------------- config 4
def value_noise(xy, rng, base_cell, octaves=4, sigma=0.1):
    """4-octave bilinear value noise, rescaled to standard deviation sigma."""
    out = np.zeros(xy.shape[0])
    x = xy[:, 0] - xy[:, 0].min()
    y = xy[:, 1] - xy[:, 1].min()
    amp = 1.0
    cell = base_cell
    for _ in range(octaves):
        gx = int(np.ceil(x.max() / cell)) + 2
        gy = int(np.ceil(y.max() / cell)) + 2
        grid = rng.standard_normal((gx, gy))
        fx = x / cell
        fy = y / cell
        ix = np.floor(fx).astype(np.int64)
        iy = np.floor(fy).astype(np.int64)
        tx = fx - ix
        ty = fy - iy
        v = ((1 - tx) * (1 - ty) * grid[ix, iy] + tx * (1 - ty) * grid[ix + 1, iy]
             + (1 - tx) * ty * grid[ix, iy + 1] + tx * ty * grid[ix + 1, iy + 1])
        out += amp * v
        amp *= 0.5
        cell *= 0.5
    out *= sigma / out.std()
    return out


def river_section(d):
    """Trapezoid + floodplain, relative to the sloped datum: bottom 40 m wide
    at -3 m (d < 20), banks 2H:1V up to 0 at d = 26, floodplain rising 2 m from d = 26 to d = 350."""
    return np.where(d < 20.0, -3.0,
                    np.where(d < 26.0, -3.0 + (d - 20.0) / 2.0, 2.0 * (d - 26.0) / (350.0 - 26.0)))


def config4(target_cells=4_000_000, n_steps=5000, length=10000.0, stage=-2.0) -> Workload:
    """BASELINE.json configs[3]: river reach flood wave with wetting/drying. length x 500 m,
    centreline y = 100 sin(2 pi x / 1500), mesh 3x finer for d < 40 m (20 m graded transition),
    slope 0.001, fractal bed noise sigma 0.1 m, k = 25 (channel) / 15 (floodplain), channel 1 m deep
    initially, floodplain dry; west = inflow hydrograph 100 -> 2000 m3/s over 3600 s (string 0),
    east = normal-depth outflow S0 = 0.001 (string 1), north/south walls.  Tests shrink `length`
    with `target_cells` so the spacing (hence dt and the wet/dry behaviour) is that of the full size."""
    rng = np.random.default_rng(_seed(4))
    y0, y1 = -250.0, 250.0

    def yc(x):
        return 100.0 * np.sin(2.0 * np.pi * x / 1500.0)

    # spacing levels: fine s_f for d<40, 3 s_f beyond d>60, two intermediate bands in between
    ratios = np.array([1.0, 3.0 ** (1 / 3), 3.0 ** (2 / 3), 3.0])
    band_lo = np.array([0.0, 40.0, 50.0, 60.0])
    band_hi = np.array([40.0, 50.0, 60.0, 1e9])
    # points per unit s_f^-2: area_band / (ratio^2 * sqrt(3)/2)
    widths = np.array([80.0, 20.0, 20.0, (y1 - y0) - 120.0])
    pts_per_sf2 = (length * widths / (ratios ** 2 * np.sqrt(3.0) / 2.0)).sum()
    s_f = np.sqrt(pts_per_sf2 / (0.5 * target_cells))
    clouds = []
    for r, lo, hi in zip(ratios, band_lo, band_hi):
        s = s_f * r
        p = M.jittered_hex_points(0.55 * s, length - 0.55 * s, y0 + 0.55 * s, y1 - 0.55 * s, s, 0.3, rng)
        d = np.abs(p[:, 1] - yc(p[:, 0]))
        clouds.append(p[(d >= lo) & (d < hi)])

    def spacing_of(x, y):
        d = abs(y - yc(x))
        return s_f * ratios[int(np.searchsorted(band_hi, d, side="right"))]

    pts_b = M.rectangle_boundary_points(0.0, length, y0, y1, spacing_of)
    pts = np.concatenate([pts_b] + clouds)
    # drop the coarser point of any pair that sits too close across a band interface
    from scipy.spatial import cKDTree
    d_all = np.abs(pts[:, 1] - yc(pts[:, 0]))
    loc = s_f * ratios[np.minimum(np.searchsorted(band_hi, d_all, side="right"), 3)]
    pairs = cKDTree(pts).query_pairs(0.55 * s_f * ratios[-1], output_type="ndarray")
    if pairs.shape[0]:
        dist = np.hypot(*(pts[pairs[:, 0]] - pts[pairs[:, 1]]).T)
        too_close = dist < 0.5 * np.minimum(loc[pairs[:, 0]], loc[pairs[:, 1]])
        pr = pairs[too_close]
        nb = pts_b.shape[0]
        # never drop perimeter points; otherwise drop the one with the larger local spacing
        drop_second = (loc[pr[:, 1]] >= loc[pr[:, 0]]) & (pr[:, 1] >= nb) | (pr[:, 0] < nb)
        victims = np.where(drop_second, pr[:, 1], pr[:, 0])
        victims = victims[victims >= nb]
        keep = np.ones(pts.shape[0], dtype=bool)
        keep[victims] = False
        pts = pts[keep]
    node_xy, tri = M.delaunay_tri_mesh(pts, 1e-3 * s_f * s_f)
    n = tri.shape[0]
    dn = np.abs(node_xy[:, 1] - yc(node_xy[:, 0]))
    zn = -0.001 * node_xy[:, 0] + river_section(dn) + value_noise(node_xy, rng, base_cell=64.0)
    zb = zn[tri].mean(axis=1)
    ctr = M.centroids(node_xy, tri)
    dc = np.abs(ctr[:, 1] - yc(ctr[:, 0]))
    kst = np.where(dc < 26.0, 25.0, 15.0)
    h = np.maximum(0.0, (-0.001 * ctr[:, 0] + stage) - zb)     # stage = -2: 1 m over the channel bottom (the config)
    w = _finish(f"config4-river-reach-{n}", node_xy, tri, zb, kst, h, n_steps=n_steps, dt_max=10.0)
    _set_boundary_codes(w, lambda mx, my: np.where(mx < 1e-9, M.bc_string(0),
                                                   np.where(mx > length - 1e-9, M.bc_string(1), M.BC_WALL)))
    w.strings = [
        (0, BC_INFLOW_Q, np.array([0.0, 100.0, 3600.0, 2000.0])),
        (1, BC_OUTFLOW_UNIFORM, np.array([0.001])),
    ]
    w.meta.update(dict(s_f=s_f, length=length))
    return w


# ----------------------------------------------------------------------------- oracle-pin cases
def uniform_flow_channel(nx=200, ny=4, lx=1000.0, ly=20.0, slope=0.001, kst=30.0, q=2.0,
                         h0=1.0, t_end=3000.0) -> Workload:
    """SURVEY O-8: prismatic sloped channel, unit discharge q in (INFLOW_Q string 0, Q = q*ly),
    OUTFLOW_UNIFORM out (string 1); steady state is the normal depth (q/(k sqrt(S0)))^(3/5)."""
    node_xy, tri = M.structured_tri_mesh(nx, ny, lx, ly)
    ctr = M.centroids(node_xy, tri)
    n = tri.shape[0]
    zb = -slope * ctr[:, 0]
    w = _finish("uniform-flow-channel", node_xy, tri, zb, np.full(n, kst), np.full(n, h0),
                t_end=t_end, dt_max=10.0)
    w.hu = np.full(n, q)
    _set_boundary_codes(w, lambda mx, my: np.where(mx < 1e-9, M.bc_string(0),
                                                   np.where(mx > lx - 1e-9, M.bc_string(1), M.BC_WALL)))
    w.strings = [(0, BC_INFLOW_Q, np.array([0.0, q * ly, 1.0, q * ly])),
                 (1, BC_OUTFLOW_UNIFORM, np.array([slope]))]
    w.meta.update(dict(q=q, slope=slope, kst=kst, lx=lx, ly=ly))
    return w


def t6_cones(spacing=0.5) -> Workload:
    """Hydrodynamic half of the paper's T6 (Eq. 23-24): [0,75]x[-15,15] m, three
    cones, dam at x = 16 m, Manning 0.01, closed walls.  Eq. 24's 'h' is read as water-surface
    elevation over the flat bed (SURVEY R-18), which reproduces the printed rest depth 0.364 m."""
    nx = int(round(75.0 / spacing))
    ny = int(round(30.0 / spacing))
    node_xy, tri = M.structured_tri_mesh(nx, ny, 75.0, 30.0, y0=-15.0, alternate=True)

    def eta(x, y):
        e1 = 1.0 - np.hypot(x - 30.0, y + 9.0) / 8.0
        e2 = 1.0 - np.hypot(x - 30.0, y - 9.0) / 8.0
        e3 = 3.0 - 0.3 * np.hypot(x - 47.5, y)
        return np.maximum(0.0, np.maximum(e1, np.maximum(e2, e3)))

    zn = eta(node_xy[:, 0], node_xy[:, 1])
    zb = zn[tri].mean(axis=1)
    ctr = M.centroids(node_xy, tri)
    level = np.where(ctr[:, 0] < 16.0, 1.0, 0.125)
    h = np.maximum(0.0, level - zb)
    w = _finish("t6-three-cones", node_xy, tri, zb, np.full(tri.shape[0], 1.0 / 0.01), h, cfl=0.95)
    w.meta.update(dict(eta=eta))
    return w


def tiny_mesh(kind: str) -> Workload:
    """2-4 cell meshes for hand-computed fluxes (SURVEY O-1)."""
    if kind == "two-cells":       # unit square split by the diagonal (0,0)-(1,1)
        node_xy = np.array([[0.0, 0.0], [1.0, 0.0], [1.0, 1.0], [0.0, 1.0]])
        tri = np.array([[0, 1, 2], [0, 2, 3]], dtype=np.int32)
    elif kind == "two-cells-x":   # two triangles sharing the vertical edge x = 1 (normal (1,0))
        node_xy = np.array([[0.0, 0.5], [1.0, 0.0], [1.0, 1.0], [2.0, 0.5]])
        tri = np.array([[0, 1, 2], [1, 3, 2]], dtype=np.int32)
    elif kind == "four-cells":    # square with its centre node
        node_xy = np.array([[0.0, 0.0], [2.0, 0.0], [2.0, 2.0], [0.0, 2.0], [1.0, 1.0]])
        tri = np.array([[0, 1, 4], [1, 2, 4], [2, 3, 4], [3, 0, 4]], dtype=np.int32)
    else:
        raise ValueError(kind)
    n = tri.shape[0]
    return _finish("tiny-" + kind, node_xy, tri, np.zeros(n), np.full(n, np.inf), np.ones(n))


def by_id(config_id: int, scale: float = 1.0) -> Workload:
    """BASELINE.json configs[config_id-1]; scale < 1 shrinks the cell count (and, for the
    unstructured configs, the domain) for tests."""
    if config_id == 1:
        return config1(refine=scale)
    if config_id == 2:
        return config2(n=max(4, int(round(200 * np.sqrt(scale)))))
    if config_id == 3:
        return config3(target_cells=int(1_000_000 * scale), lx=2000.0 * np.sqrt(scale))
    if config_id == 4:
        return config4(target_cells=int(4_000_000 * scale), length=10000.0 * scale)
    if config_id == 5:
        return config5(target_cells=int(8_000_000 * scale))
    raise ValueError(config_id)
