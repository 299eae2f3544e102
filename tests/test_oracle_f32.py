"""Pins of the single-precision oracle ("single or double"): the same
oracle source built with -DSWE_REF_REAL=float (R-21: state, geometry and every flux / update operation in
fp32; time, dt, the hydrograph lookup and the volume bookkeeping in fp64; cube root = correctly rounded fp64 cube root
rounded to fp32).  The fp64 build is pinned by the other test_oracle_* modules; here the fp32 build is pinned to
  * the hand-computed values of tests/golden/ (to fp32 round-off),
  * invariants with their fp32 bounds: mass to fp32 round-off, lake at rest, every stored value an fp32 number,
  * the analytic dam-break solutions, with errors within a stated factor of the fp64 build's,
so that a wrong cast, a double-rounded constant or an operation left in fp64 shows up."""
import os

import numpy as np
import pytest

from workloads import configs as C, mesh as M

G = 9.81
EPS32 = 2.0 ** -24


@pytest.fixture(scope="module")
def ref():
    from oracle import swe_ref
    swe_ref.lib(single=True)
    return swe_ref


def golden(name):
    out = {}
    for line in open(os.path.join(os.path.dirname(__file__), "golden", name)):
        if line.strip() and not line.startswith("#"):
            parts = line.split()
            out[" ".join(parts[:-1])] = float(parts[-1])
    return out


def f32(x):
    return np.asarray(x, np.float64).astype(np.float32).astype(np.float64)


def test_hand_fluxes_to_fp32_roundoff(ref):
    """The worked interior / dry-right values of tests/golden/hand_fluxes.txt through the fp32 edge flux: a handful of
    fp32 operations, so a few units of 2^-24 relative to the largest term (F2 = 12.45)."""
    g = golden("hand_fluxes.txt")
    L = ref.lib(single=True)
    import ctypes
    out = [ctypes.c_double() for _ in range(4)]
    L.swe_ref_edge_flux(G, 2.0, 1.0, 0.5, 0.0, 1.0, 0.0, 0.0, 0.5, 1.0, 0.0, *[ctypes.byref(o) for o in out])
    F1, F3, GL, GR = (o.value for o in out)
    tol = 16 * EPS32 * g["interior F2"]
    assert abs(F1 - g["interior F1"]) <= tol and abs(F3 - g["interior F3"]) <= tol
    assert abs(GL - g["interior GL"]) <= tol and abs(GR - g["interior GR"]) <= tol
    assert (F1, F3, GL, GR) == tuple(f32([F1, F3, GL, GR]))          # results are fp32 numbers
    # ... and they are NOT the fp64 results (the build really computes in fp32)
    L64 = ref.lib()
    out64 = [ctypes.c_double() for _ in range(4)]
    L64.swe_ref_edge_flux(G, 2.0, 1.0, 0.5, 0.0, 1.0, 0.0, 0.0, 0.5, 1.0, 0.0, *[ctypes.byref(o) for o in out64])
    assert abs(out64[0].value - g["interior F1"]) <= 1e-12 and out64[0].value != F1
    # dry bed on the right: F1 = 2/3 c h, GL = -g h^2 / 6
    L.swe_ref_edge_flux(G, 1.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 1.0, 0.0, *[ctypes.byref(o) for o in out])
    assert abs(out[0].value - g["dryright F1"]) <= 8 * EPS32 * 5.0 and abs(out[2].value - g["dryright GL"]) <= 8 * EPS32 * 5.0
    # rest state over a step: both face depths equal -> F1 = 0 and G = 0 exactly, in fp32 as in fp64
    L.swe_ref_edge_flux(G, 2.0, 0.0, 0.0, 0.0, 1.5, 0.0, 0.0, 0.5, 0.6, 0.8, *[ctypes.byref(o) for o in out])
    assert out[0].value == 0.0 and out[2].value == 0.0 and out[3].value == 0.0


def test_limiter_moving_water_fp32(ref):
    """tests/golden/limiter_moving_water.txt (hand-computed, R-8b) through one fp32 step: dt from the fp32 rate in fp64,
    theta, the four limited components and the receiver's new state, all to fp32 round-off."""
    gold = golden("limiter_moving_water.txt")
    w = C.tiny_mesh("two-cells-x")
    e = int(np.nonzero((w.edge_cell[:, 0] == 0) & (w.edge_cell[:, 1] == 1))[0][0])
    w.h[:] = [0.01, 0.0]
    w.hu[:] = [0.04, 0.0]
    w.hv[:] = [0.01, 0.0]
    s = ref.RefSolver(w, precision="single")
    info = s.step(n_steps=1, cfl=0.9)
    assert abs(info["dt_last"] - gold["dt"]) <= 4 * EPS32 * gold["dt"]
    F1, F3, GL, GR = s.edge_fluxes()
    for name, got in (("F1", F1[e]), ("F3", F3[e]), ("GL", GL[e]), ("GR", GR[e])):
        assert abs(got - gold[name]) <= 16 * EPS32 * abs(gold[name]), (name, got, gold[name])
    h, hu, hv = s.get_state()
    assert abs(h[0]) <= 8 * EPS32 * 0.01 and hu[0] == 0.0 and hv[0] == 0.0
    assert abs(h[1] - gold["h1_new"]) <= 8 * EPS32 * 0.01
    assert abs(hu[1] - gold["qx1_new"]) <= 16 * EPS32 * 0.04 and abs(hv[1] - gold["qy1_new"]) <= 16 * EPS32 * 0.01


def test_state_and_geometry_are_fp32_numbers_dt_is_fp64(ref):
    w = C.by_id(3, 0.005)
    s, d = ref.RefSolver(w, precision="single"), ref.RefSolver(w)
    for a, b in zip(s.geometry(), d.geometry()):
        assert np.array_equal(a, f32(b))                  # the fp64 geometry rounded ONCE to fp32
    # dt = cfl / (fp32 rate) evaluated in fp64: close to the fp64 oracle's, and (generally) not an fp32 number
    dt32, dt64 = s.peek_dt(0.9), d.peek_dt(0.9)
    assert abs(dt32 - dt64) <= 8 * EPS32 * dt64 and dt32 != float(np.float32(dt32))
    i = s.step(25, float("inf"), 0.9)
    for x in s.get_state():
        assert np.array_equal(x, f32(x))
    assert abs(i["t"] - 25 * dt64) < 0.2 * i["t"] and i["t"] != float(np.float32(i["t"]))


def test_mass_conserved_to_fp32_roundoff_in_a_closed_box(ref):
    """PAPER.md:591 ("fully conservative") in fp32: the mass flux of an edge enters its two cells with opposite signs,
    so the volume only drifts by the rounding of h - a * dH: ~1200 steps of a sloshing dam break stay within 1e-6
    relative (measured 1.0e-7), nothing is created by clipping beyond that."""
    w = C.dam_break_channel(nx=250, ny=2, t_end=60.0, kst=30.0)
    s = ref.RefSolver(w, precision="single")
    area = s.geometry()[0]
    v0 = float(np.sum(f32(w.h) * area))
    i = s.step(-1, 60.0, 0.9)
    h = s.get_state()[0]
    assert i["steps_done"] > 1000 and h.min() >= 0.0
    assert abs(float(np.sum(h * area)) - v0) <= 1e-6 * v0
    assert i["vol_clipped"] <= 1e-6 * v0
    assert abs(i["vol"] - float(np.sum(h * area))) <= 1e-12 * v0        # the bookkeeping itself is fp64


def test_lake_at_rest_fp32_bound(ref):
    """B:configs[1] (shrunk) in fp32: with h = fl32(eta - z) the two face depths of an edge differ by at most one fp32
    ulp of the depth, which leaves velocity noise of order g * ulp32 * dt * l / A per step that does not grow:
    max |u| <= 1e-4 m/s after 300 steps (measured 1e-5; the fp64 build: 2e-14), wet mask and depths unchanged to 1e-6."""
    w = C.by_id(2, 0.05)
    s = ref.RefSolver(w, precision="single")
    s.step(300, float("inf"), w.cfl)
    h, hu, hv = s.get_state()
    wet = h > w.h_dry
    assert np.array_equal(wet, w.h > w.h_dry)
    assert np.max(np.abs(hu[wet] / h[wet])) <= 1e-4 and np.max(np.abs(hv[wet] / h[wet])) <= 1e-4
    assert np.max(np.abs(h - w.h)) <= 2e-6


def test_dam_break_errors_within_a_factor_of_the_fp64_build(ref):
    """Ritter (dry bed) on the 500 x 4 channel, t = 4 s: the L1 errors of h and hu against the analytic solution are those
    of the first-order scheme, not of the arithmetic -- the fp32 build's are within 2 % of the fp64 build's; Stoker
    (h_R = 0.1): plateau depth and velocity within 1 % of the analytic values (0.39617, 2.32136 in
    tests/golden/analytic_dam_break.txt) and within 1e-4 relative of the fp64 build's."""
    from test_oracle_analytic import ritter, stoker     # the closed forms the fp64 pins use
    w = C.dam_break_channel(h_right=0.0)
    x = M.centroids(w.node_xy, w.tri)[:, 0]
    he, ue = ritter(x, 4.0)
    errs = {}
    for prec in ("double", "single"):
        s = ref.RefSolver(w, precision=prec)
        area = s.geometry()[0]
        s.step(-1, 4.0, 0.9)
        h, hu, _ = s.get_state()
        errs[prec] = (float(np.sum(np.abs(h - he) * area)), float(np.sum(np.abs(hu - he * ue) * area)))
    for k in range(2):
        assert abs(errs["single"][k] - errs["double"][k]) <= 0.02 * errs["double"][k], errs
    hm, um, S = stoker(1.0, 0.1)
    w = C.dam_break_channel(h_right=0.1)
    cm = np.sqrt(G * hm)
    m = (x > 50 + (um - cm) * 4 + 2.0) & (x < 50 + S * 4 - 2.0)
    plateau = {}
    for prec in ("double", "single"):
        s = ref.RefSolver(w, precision=prec)
        s.step(-1, 4.0, 0.9)
        h, hu, _ = s.get_state()
        plateau[prec] = (h[m].mean(), (hu[m] / h[m]).mean())
    assert abs(plateau["single"][0] - hm) < 0.01 * hm and abs(plateau["single"][1] - um) < 0.01 * um
    assert abs(plateau["single"][0] - plateau["double"][0]) < 1e-4 * hm
    assert abs(plateau["single"][1] - plateau["double"][1]) < 1e-4 * um
