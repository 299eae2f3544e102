"""Pins for the oracle's geometry, time step (Eq. 21), friction source, limiter and bookkeeping.
CPU only; every expected value is a closed form or a brute-force numpy evaluation written here."""
import os

import numpy as np
import pytest

from workloads import configs as C
from workloads import mesh as M

G = 9.81


def random_delaunay(seed, n_pts=60):
    rng = np.random.default_rng(seed)
    pts = np.concatenate([M.rectangle_boundary_points(0, 10, 0, 7, 1.0), rng.uniform(0.3, 9.7, (n_pts, 2)) * [1, 0.7]])
    node_xy, tri = M.delaunay_tri_mesh(pts, 1e-6)
    return node_xy, tri


@pytest.mark.parametrize("seed", range(3))
def test_geometry_closed_forms(ref, seed):
    """SURVEY O-3. PAPER.md:226-228 (n_ij unit, towards j), PAPER.md:312 (rho = twice the centroid-edge distance)."""
    node_xy, tri = random_delaunay(seed)
    n = tri.shape[0]
    w = C._finish("geo", node_xy, tri, np.zeros(n), np.full(n, np.inf), np.ones(n))
    s = ref.RefSolver(w)
    area, nx, ny, ln = s.geometry()
    p = node_xy[tri]
    # shoelace area
    sh = 0.5 * np.abs(p[:, 0, 0] * (p[:, 1, 1] - p[:, 2, 1]) + p[:, 1, 0] * (p[:, 2, 1] - p[:, 0, 1])
                      + p[:, 2, 0] * (p[:, 0, 1] - p[:, 1, 1]))
    assert np.allclose(area, sh, rtol=1e-13, atol=0)
    assert np.allclose(nx * nx + ny * ny, 1.0, rtol=0, atol=1e-14)
    ctr = p.mean(axis=1)
    closure = np.zeros((n, 2))
    for k in range(3):
        e = w.cell_edge[:, k]
        sgn = np.where(w.edge_cell[e, 0] == np.arange(n), 1.0, -1.0)
        a, b = p[:, k], p[:, (k + 1) % 3]
        # length and outward normal against the node coordinates
        assert np.allclose(ln[e], np.hypot(*(b - a).T), rtol=1e-14)
        mid = 0.5 * (a + b)
        outward = (mid - ctr)
        assert np.all(sgn * (nx[e] * outward[:, 0] + ny[e] * outward[:, 1]) > 0)      # points away from i
        assert np.allclose(nx[e] * (b - a)[:, 0] + ny[e] * (b - a)[:, 1], 0.0, atol=1e-13)  # normal to the edge
        closure += (sgn * ln[e])[:, None] * np.stack([nx[e], ny[e]], axis=1)
        # rho_ij = 2 * dist(centroid, line(a,b)) must equal 4A/(3l)
        d = np.abs((b - a)[:, 0] * (a - ctr)[:, 1] - (b - a)[:, 1] * (a - ctr)[:, 0]) / np.hypot(*(b - a).T)
        assert np.allclose(2.0 * d, 4.0 * area / (3.0 * ln[e]), rtol=1e-12)
    assert np.all(np.abs(closure) < 1e-12)                                             # sum_j l_ij n_ij = 0
    # the interior normal points from L to R ("points toward the cell Omega_j")
    inter = w.edge_cell[:, 1] >= 0
    L, R = w.edge_cell[inter, 0], w.edge_cell[inter, 1]
    dvec = ctr[R] - ctr[L]
    assert np.all(nx[inter] * dvec[:, 0] + ny[inter] * dvec[:, 1] > 0)


def brute_dt(w, s, cfl, h_dry=1e-3):
    """Eq. 21 literally: CFL * min_i min_j rho_ij / lambda_ij with rho = 2 * dist(centroid, edge)."""
    h, hu, hv = s.get_state()
    p = w.node_xy[w.tri]
    ctr = p.mean(axis=1)
    best = np.inf
    for i in range(w.n_cells):
        if h[i] <= h_dry:
            continue
        u, v = hu[i] / h[i], hv[i] / h[i]
        for k in range(3):
            a, b = p[i, k], p[i, (k + 1) % 3]
            t = (b - a) / np.hypot(*(b - a))
            nrm = np.array([t[1], -t[0]])
            dist = abs((ctr[i] - a) @ nrm)
            lam = abs(u * nrm[0] + v * nrm[1]) + np.sqrt(G * h[i])
            best = min(best, 2.0 * dist / lam)
    return cfl * best


def test_dt_matches_eq21_brute_force(ref):
    """SURVEY R-7 pin: brute-force min over (i, j) on a small random mesh with random wet/dry state."""
    node_xy, tri = random_delaunay(11, 40)
    n = tri.shape[0]
    rng = np.random.default_rng(5)
    h = rng.uniform(0.0, 2.0, n)
    h[rng.uniform(size=n) < 0.3] = 0.0
    w = C._finish("dt", node_xy, tri, rng.uniform(-0.2, 0.2, n), np.full(n, 30.0), h)
    w.hu = h * rng.uniform(-2, 2, n)
    w.hv = h * rng.uniform(-2, 2, n)
    s = ref.RefSolver(w)
    for cfl in (0.9, 0.5):
        assert abs(s.peek_dt(cfl) - brute_dt(w, s, cfl)) < 1e-13 * s.peek_dt(cfl)
    # t_end clipping and dt_max
    assert s.peek_dt(0.9, t_end=1e-5) == 1e-5
    s2 = ref.RefSolver(w, dt_max=1e-4)
    assert s2.peek_dt(0.9) == 1e-4


def test_dt_config1_initial(ref):
    """dt at t = 0 of config 1 = 0.9 * rho_min / sqrt(g h0) (SURVEY R-7): legs 0.2 and 0.5, hypotenuse
    sqrt(0.29); area 0.05; rho_min = 4A/(3 l_max)."""
    w = C.config1()
    s = ref.RefSolver(w)
    rho_min = 4 * 0.05 / (3 * np.sqrt(0.2 ** 2 + 0.5 ** 2))
    assert abs(s.peek_dt(0.9) - 0.9 * rho_min / np.sqrt(G * 1.0)) < 1e-14


def test_friction_closed_form(ref):
    """SURVEY R-5/R-6: the source term is isolated by a state with no gradients, where the edge fluxes
    cancel in every cell sum: uniform (h, q) on a mesh whose boundary is transmissive.  Then dq/dt = -g |q| q / (k^2 h^(7/3)) exactly (Eq. 2 + Strickler row of
    Table 1), whose solution over dt is q / (1 + dt*gamma*|q|)."""
    node_xy, tri = M.structured_tri_mesh(6, 5, 6.0, 5.0, alternate=True)
    n = tri.shape[0]
    h0, k = 0.8, 28.0
    qx0, qy0 = 1.3, -0.6
    w = C._finish("fric", node_xy, tri, np.zeros(n), np.full(n, k), np.full(n, h0))
    w.edge_cell[w.edge_cell[:, 1] < 0, 1] = M.BC_TRANSMISSIVE
    w.hu[:] = qx0
    w.hv[:] = qy0
    s = ref.RefSolver(w)
    dt = 0.02      # well inside the stable range, so the draining limiter stays inactive
    info = s.step(n_steps=1, t_end=dt, cfl=1e9)
    assert info["dt_last"] == dt
    h, hu, hv = s.get_state()
    gamma = G / (k * k * h0 ** (7.0 / 3.0))
    D = 1.0 + dt * gamma * np.hypot(qx0, qy0)
    assert np.allclose(h, h0, rtol=1e-13)
    assert np.allclose(hu, qx0 / D, rtol=1e-12) and np.allclose(hv, qy0 / D, rtol=1e-12)
    # n steps of the exact integrator compose to the exact solution of the Riccati ODE at time n*dt
    q0 = np.hypot(qx0, qy0)
    s.set_state(np.full(n, h0), np.full(n, qx0), np.full(n, qy0))
    t = 0.0
    for _ in range(7):
        t += 0.01
        s.step(n_steps=1, t_end=t, cfl=1e9)
    h, hu, hv = s.get_state()
    assert np.allclose(np.hypot(hu, hv), q0 / (1.0 + t * gamma * q0), rtol=1e-12)
    # frictionless: k = +inf leaves q untouched
    w.kst[:] = np.inf
    s = ref.RefSolver(w)
    s.step(n_steps=1, t_end=dt, cfl=1e9)
    h, hu, hv = s.get_state()
    assert np.allclose(hu, qx0, rtol=1e-13) and np.allclose(hv, qy0, rtol=1e-13)


def test_thin_film_has_no_momentum(ref):
    """DESIGN R-8: cells with h <= h_dry keep their water, carry no momentum, do not constrain dt, but
    still take part in the hydrostatic reconstruction (so a shoreline film does not break lake-at-rest)."""
    w = C.tiny_mesh("four-cells")
    w.h[:] = 5e-4
    w.hu[:] = 1.0
    s = ref.RefSolver(w, dt_max=0.5)
    assert s.peek_dt(0.9) == 0.5                 # no wet cell -> dt_max
    info = s.step(n_steps=3)
    h, hu, hv = s.get_state()
    assert np.all(h == 5e-4) and np.all(hu == 0.0) and np.all(hv == 0.0)
    assert info["n_wet"] == 0 and info["steps_done"] == 3
    # a film next to a deep cell at the same surface level: exact rest (face depths are equal)
    w2 = C.tiny_mesh("two-cells")
    w2.zb[:] = [0.0, 1.0 - 4e-4]
    w2.h[:] = [1.0, 4e-4]
    s2 = ref.RefSolver(w2)
    s2.step(n_steps=5)
    h, hu, hv = s2.get_state()
    # (face depths 1.0 - 0.9996 and 4e-4 differ by an ulp, so 'rest' holds to round-off, not bitwise)
    assert np.abs(h - w2.h).max() < 1e-15 and np.abs(hu).max() < 1e-15 and np.abs(hv).max() < 1e-15
    # a film higher than its neighbour's surface drains into it (mass only), conserving volume
    w3 = C.tiny_mesh("two-cells")
    w3.zb[:] = [0.0, 2.0]
    w3.h[:] = [1.0, 8e-4]
    s3 = ref.RefSolver(w3)
    info = s3.step(n_steps=5)
    h, hu, hv = s3.get_state()
    assert h[1] < 8e-4 and h[0] > 1.0 and hu[1] == 0.0
    assert abs((h * s3.geometry()[0]).sum() - (w3.h * s3.geometry()[0]).sum()) < 1e-15


def test_draining_limiter_positivity_and_mass(ref):
    """DESIGN R-8b: an isolated wet cell surrounded by dry bed would lose 2.4x its content in one step at
    CFL 0.9 (Eq. 21 with rho = 4A/3l); the draining-time limiter scales its outgoing fluxes so that it
    ends exactly empty, and the total volume is conserved to round-off with nothing clipped."""
    node_xy, tri = M.structured_tri_mesh(5, 5, 5.0, 5.0, alternate=True)
    n = tri.shape[0]
    h = np.zeros(n)
    ctr = M.centroids(node_xy, tri)
    i0 = int(np.argmin(np.hypot(ctr[:, 0] - 2.5, ctr[:, 1] - 2.5)))
    h[i0] = 1.0
    w = C._finish("drain", node_xy, tri, np.zeros(n), np.full(n, np.inf), h)
    s = ref.RefSolver(w)
    area = s.geometry()[0]
    v0 = (h * area).sum()
    info = s.step(n_steps=1, cfl=0.9)
    h1, hu1, hv1 = s.get_state()
    assert h1.min() >= 0.0 and abs(h1[i0]) < 1e-15
    assert abs((h1 * area).sum() - v0) < 1e-14 and info["vol_clipped"] < 1e-15
    # with a small CFL the limiter is inactive: the loss is the unlimited dry-bed flux 2/3 c h per edge
    s.set_state(h, np.zeros(n), np.zeros(n))
    dt = s.peek_dt(0.1)
    s.step(n_steps=1, cfl=0.1)
    h2 = s.get_state()[0]
    ln = s.geometry()[3]
    per = ln[w.cell_edge[i0]].sum()
    assert abs((1.0 - h2[i0]) - dt * per * (2.0 / 3.0) * np.sqrt(G) / area[i0]) < 1e-14


def test_limiter_scales_every_flux_component_moving_water(ref):
    """DESIGN R-8b with moving water, against values computed by hand (tests/golden/limiter_moving_water.txt): a fast
    thin cell drains into a dry neighbour with theta = 0.8986; F1, F3, GL and GR of the edge are all scaled by theta,
    the donor ends empty and the receiver gets exactly (dt/A) theta = 1/4 of every component.  Leaving G or F3
    unscaled changes q_x by 11 % and q_y by 11 %."""
    gold = {}
    for line in open(os.path.join(os.path.dirname(__file__), "golden", "limiter_moving_water.txt")):
        if line.strip() and not line.startswith("#"):
            k, v = line.split()
            gold[k] = float(v)
    w = C.tiny_mesh("two-cells-x")
    e = int(np.nonzero((w.edge_cell[:, 0] == 0) & (w.edge_cell[:, 1] == 1))[0][0])      # the shared edge, L = cell 0
    w.h[:] = [0.01, 0.0]
    w.hu[:] = [0.04, 0.0]
    w.hv[:] = [0.01, 0.0]
    s = ref.RefSolver(w)
    area, nx, ny, ln = s.geometry()
    assert np.allclose(area, 0.5, rtol=0, atol=1e-16) and (nx[e], ny[e], ln[e]) == (1.0, 0.0, 1.0)
    assert abs(s.peek_dt(0.9) - gold["dt"]) <= 1e-15
    info = s.step(n_steps=1, cfl=0.9)
    assert abs(info["dt_last"] - gold["dt"]) <= 1e-15
    F1, F3, GL, GR = s.edge_fluxes()                                  # after the limiter
    for name, got in (("F1", F1[e]), ("F3", F3[e]), ("GL", GL[e]), ("GR", GR[e])):
        assert abs(got - gold[name]) <= 1e-15 * max(1.0, abs(gold[name])) * 4, (name, got, gold[name])
    walls = np.arange(w.n_edges) != e
    assert np.all(F1[walls] == 0.0) and np.all(F3[walls] == 0.0)     # reflective walls carry no mass
    h, hu, hv = s.get_state()
    assert abs(h[0] - gold["h0_new"]) <= 2e-18 and hu[0] == 0.0 and hv[0] == 0.0     # emptied: below h_dry, no momentum
    assert abs(h[1] - gold["h1_new"]) <= 1e-17
    assert abs(hu[1] - gold["qx1_new"]) <= 1e-16 and abs(hv[1] - gold["qy1_new"]) <= 1e-17
    assert info["vol_clipped"] <= 1e-18 and abs((h * area).sum() - 0.005) <= 1e-18     # mass conserved, nothing clipped


def test_restart_and_stop_conditions(ref):
    """SURVEY O-10 + boundary semantics: 100 steps == 50 + get/set + 50 bitwise; t_end is hit exactly."""
    w = C.dam_break_channel(nx=60, ny=2, lx=12.0, ly=0.4, x_dam=6.0, h_right=0.2, kst=30.0)
    a = ref.RefSolver(w)
    a.step(n_steps=100)
    b = ref.RefSolver(w)
    i50 = b.step(n_steps=50)
    st = b.get_state()
    c = ref.RefSolver(w)
    c.set_state(*st, t0=i50["t"])
    i100 = c.step(n_steps=50)
    for x, y in zip(a.get_state(), c.get_state()):
        assert np.array_equal(x, y)
    d = ref.RefSolver(w)
    info = d.step(t_end=0.7)
    assert info["t"] == 0.7 and info["steps_done"] > 3
    info2 = d.step(n_steps=5, t_end=0.7)          # already there: nothing happens
    assert info2["steps_done"] == info["steps_done"] and info2["t"] == 0.7


def test_hydrograph_inflow_bookkeeping(ref):
    """DESIGN R-11: vol_in = sum dt*Q(t^n) with Q piecewise linear; the domain gains exactly that volume."""
    w = C.uniform_flow_channel(nx=40, ny=2, lx=200.0, ly=10.0, t_end=50.0)
    w.strings[0] = (0, C.BC_INFLOW_Q, np.array([0.0, 5.0, 20.0, 25.0, 40.0, 25.0]))
    w.edge_cell[w.edge_cell[:, 1] == M.bc_string(1), 1] = M.BC_WALL       # close the outlet
    w.strings = w.strings[:1]
    s = ref.RefSolver(w)
    area = s.geometry()[0]
    v0 = (w.h * area).sum()
    tq, vin = 0.0, 0.0
    for _ in range(60):
        dt = s.peek_dt(0.9, 50.0)
        Q = np.interp(tq, [0.0, 20.0, 40.0], [5.0, 25.0, 25.0])
        info = s.step(n_steps=1, t_end=50.0)
        vin += dt * Q
        tq = info["t"]
        assert abs(info["vol_in"] - vin) < 1e-11 * max(1.0, vin)
        assert abs(info["vol"] - v0 - info["vol_in"]) < 1e-10 * v0
        assert info["vol_clipped"] < 1e-12


# ------------------------------------------------------------------------------------------------
# R-14: the oracle's cube root is the correctly rounded one.  Pin: exact integer arithmetic in Python
# (fractions of big integers), which shares nothing with the C++ limbs.
# ------------------------------------------------------------------------------------------------
def _cbrt_rn_exact(x: float) -> float:
    """Nearest double to x^(1/3), by exact comparison of cubes of big integers."""
    import math
    from fractions import Fraction
    if x == 0.0:
        return x
    if x < 0:
        return -_cbrt_rn_exact(-x)
    fx = Fraction(x)
    k = max(0, 70 - math.frexp(x)[1] // 3)    # estimate: integer cube root of floor(x * 8^k) (>= 64 bits), as a double
    n = int(fx * 8 ** k)
    t = 1 << (n.bit_length() // 3 + 1)
    while True:                               # integer Newton from above
        u = (2 * t + n // (t * t)) // 3
        if u >= t:
            break
        t = u
    y = float(Fraction(t, 2 ** k))
    for _ in range(8):                        # walk to the double whose rounding interval holds the root
        lo = Fraction(y) - (Fraction(y) - Fraction(math.nextafter(y, 0.0))) / 2
        hi = Fraction(y) + (Fraction(math.nextafter(y, math.inf)) - Fraction(y)) / 2
        if lo ** 3 > fx:
            y = math.nextafter(y, 0.0)
        elif hi ** 3 < fx:
            y = math.nextafter(y, math.inf)
        else:
            assert lo ** 3 != fx and hi ** 3 != fx     # no ties exist
            return y
    raise AssertionError("estimate too far off")


def test_cbrt_is_correctly_rounded(ref):
    import math
    rng = np.random.default_rng(128620)
    xs = [1.0, 8.0, 27.0, 0.125, 1e-3, 2.0, 3.0, 7.999999999999999, 1.0000000000000002, 5e-324, 2.2250738585072014e-308,
          1.7976931348623157e308, 0.001 + 1e-18, 10.0, 1e-300, 3.0 ** 30, -8.0, -2.5]
    xs += list(np.exp(rng.uniform(np.log(1e-6), np.log(1e4), 20000)))      # depths in metres
    xs += list(np.ldexp(rng.uniform(0.5, 1.0, 3000), rng.integers(-1070, 1023, 3000)))
    # hard cases: doubles right next to the cube of a half-way point m * 2^-53, m odd (54 bits)
    for _ in range(3000):
        m = int(rng.integers(2 ** 53, 2 ** 54)) | 1
        c = (m ** 3) >> (159 - 52)            # 53-56 significant bits of m^3, as an integer
        k = int(rng.integers(-30, 30))
        for d in (0, 1):
            xs.append(math.ldexp(float(c + d), 3 * k - 52) if c + d < 2 ** 53 else math.ldexp(float((c >> 3) + d), 3 * k - 49))
    n_hard = 0
    for x in xs:
        got = ref.cbrt(x)
        want = _cbrt_rn_exact(x)
        assert got == want, (x, got, want)
        n_hard += got != math.copysign(abs(x) ** (1.0 / 3.0), x)
    assert n_hard > 100                        # the pin does separate a 1-ulp cbrt from the rounded one
    assert ref.cbrt(0.0) == 0.0 and math.isinf(ref.cbrt(math.inf))
