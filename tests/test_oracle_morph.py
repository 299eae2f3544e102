"""Pins of the oracle's morphodynamic step (Eq. 3; Eq. 13-16; Table 2 PAPER.md:152-161;
DESIGN.md R-20) against what the paper and the mathematics fix: Table 2 evaluated by hand, the derivative in Eq. 16 by
finite differences, Eq. 16's two speeds through Vieta's relations of the quadratic they solve, the textbook special cases
of an HLL flux (consistency, one-sided upwinding, Rusanov), Eq. 13 re-assembled with numpy from the per-edge fluxes, the
porosity factor, conservation of sediment volume in a closed box, a fixed bed when the module is off, and the celerity
of a small bed hump under a Grass-like law (the bed-wave eigenvalue of the coupled shallow-water / Exner system).
CPU only."""
import numpy as np
import pytest

from workloads import configs as C
from workloads import mesh as M

G = 9.81


def _velocity(un, ut, nx, ny):
    return un * nx - ut * ny, un * ny + ut * nx


def test_grass_transport_by_hand(ref):
    """Table 2 Grass-like row, m = 3, u_cr = 0: |q_B| = alpha |u|^3 along u."""
    alpha, h, u, v, nx, ny = 0.01, 2.0, 1.5, -0.5, 0.6, 0.8
    q, psi, l1, l2 = ref.sediment_state(ref.GRASS, alpha, 0.0, 2.65, 1e-3, G, h, u, v, 0.0, nx, ny)
    speed = np.hypot(u, v)
    assert q == pytest.approx(alpha * speed ** 3 * ((u * nx + v * ny) / speed), rel=1e-14)
    # along the flow the whole magnitude passes, across it nothing
    q_al = ref.sediment_state(ref.GRASS, alpha, 0.0, 2.65, 1e-3, G, h, u, v, 0.0, u / speed, v / speed)[0]
    q_ac = ref.sediment_state(ref.GRASS, alpha, 0.0, 2.65, 1e-3, G, h, u, v, 0.0, -v / speed, u / speed)[0]
    assert q_al == pytest.approx(alpha * speed ** 3, rel=1e-14)
    assert abs(q_ac) < 1e-17
    # still water: no transport, psi = 0, speeds (-c, 0)
    q0, p0, a1, a2 = ref.sediment_state(ref.GRASS, alpha, 0.0, 2.65, 1e-3, G, h, 0.0, 0.0, 0.0, nx, ny)
    assert (q0, p0, a2) == (0.0, 0.0, 0.0) and a1 == pytest.approx(-np.sqrt(G * h), rel=1e-15)


def test_mpm_transport_by_hand(ref):
    """Table 2 MPM-like row with [55]'s alpha = 8, m = 1.5, theta_cr = 0.047; Shields parameter from the Strickler
    bed shear stress of Table 1: theta = |u|^2 / (k_st^2 h^(1/3) (s-1) d_m)."""
    kst, h, u, v, s, dm = 30.0, 1.3, 2.0, 0.0, 2.65, 0.005
    theta = (u * u + v * v) / (kst ** 2 * h ** (1.0 / 3.0) * (s - 1.0) * dm)
    want = 8.0 * (theta - 0.047) ** 1.5 * np.sqrt((s - 1.0) * G * dm ** 3)
    q = ref.sediment_state(ref.MPM, 8.0, 0.047, s, dm, G, h, u, v, G / kst ** 2, 1.0, 0.0)[0]
    assert theta > 0.3 and q == pytest.approx(want, rel=1e-13)
    # [56]'s parameter set differs in alpha only as far as this build goes (m stays 1.5): linear in alpha
    q2 = ref.sediment_state(ref.MPM, 4.0, 0.047, s, dm, G, h, u, v, G / kst ** 2, 1.0, 0.0)[0]
    assert q2 == pytest.approx(0.5 * want, rel=1e-13)
    # below the threshold of motion nothing moves: theta(u = 0.3) = 0.012 < 0.047
    q3, psi3, _, l2 = ref.sediment_state(ref.MPM, 8.0, 0.047, s, dm, G, h, 0.3, 0.0, G / kst ** 2, 1.0, 0.0)
    assert (q3, psi3, l2) == (0.0, 0.0, 0.0)
    # no friction law, no shear stress, no transport
    assert ref.sediment_state(ref.MPM, 8.0, 0.047, s, dm, G, h, u, v, 0.0, 1.0, 0.0)[0] == 0.0


@pytest.mark.parametrize("formula,alpha,gn2", [(1, 0.01, 0.0), (2, 8.0, G / 900.0)])
@pytest.mark.parametrize("un,ut", [(1.7, 0.0), (1.1, -0.9), (-0.8, 1.4), (0.0, 1.5)])
def test_psi_is_the_derivative_of_eq16(ref, formula, alpha, gn2, un, ut):
    """Eq. 16 needs d(q_B,n)/d(q_n); q_n = h u_n with h and the tangential velocity fixed: central differences of the
    oracle's own q_B,n(u_n) must reproduce psi * h."""
    h, nx, ny, dm = 0.9, 0.28, 0.96, 0.004
    def qn(a):
        u, v = _velocity(a, ut, nx, ny)
        return ref.sediment_state(formula, alpha, 0.047, 2.65, dm, G, h, u, v, gn2, nx, ny)[0]
    u, v = _velocity(un, ut, nx, ny)
    q, psi, l1, l2 = ref.sediment_state(formula, alpha, 0.047, 2.65, dm, G, h, u, v, gn2, nx, ny)
    d = 1e-5
    fd = (qn(un + d) - qn(un - d)) / (2 * d) / h
    assert psi == pytest.approx(fd, rel=1e-6, abs=1e-12)
    assert psi >= 0.0
    # Eq. 16: lambda_1,2 are the roots of lambda^2 - (u_n - c) lambda - psi c^2 = 0 (Vieta)
    c = np.sqrt(G * h)
    assert l1 + l2 == pytest.approx(un - c, rel=1e-13)
    assert l1 * l2 == pytest.approx(-psi * c * c, rel=1e-12, abs=1e-18)
    assert l1 <= 0.0 <= l2


def test_hll_sediment_flux_special_cases(ref):
    """Eq. 14-15 as an HLL flux ([18] ch. 10): consistency, one-sided upwinding, the Rusanov form, and the speeds of
    Eq. 15 (min of the left-going, max of the right-going ones)."""
    f = ref.sediment_flux
    assert f(0.3, -2.0, 0.5, 1.0, 0.3, -2.0, 0.5, 1.0) == pytest.approx(0.3, rel=1e-15)          # i == j
    assert f(0.3, 0.0, 0.5, 1.0, 0.9, 0.0, 0.7, 4.0) == pytest.approx(0.3, rel=1e-15)            # lambda- = 0: upwind = i
    assert f(0.3, -2.0, 0.0, 1.0, 0.9, -1.0, 0.0, 4.0) == pytest.approx(0.9, rel=1e-15)          # lambda+ = 0: upwind = j
    a = 1.25                                                                                       # lambda+- = +-a
    assert f(0.3, -a, a, 1.0, 0.9, -a, a, 4.0) == pytest.approx(0.5 * (0.3 + 0.9) - 0.5 * a * (4.0 - 1.0), rel=1e-15)
    # Eq. 15 picks min(l1i, l1j) and max(l2i, l2j): swapping which side holds the extreme changes nothing
    assert f(0.3, -3.0, 0.2, 1.0, 0.9, -1.0, 0.6, 4.0) == f(0.3, -1.0, 0.6, 1.0, 0.9, -3.0, 0.2, 4.0)
    want = (0.6 * 0.3 + 3.0 * 0.9 + 0.6 * -3.0 * (4.0 - 1.0)) / 3.6
    assert f(0.3, -3.0, 0.2, 1.0, 0.9, -1.0, 0.6, 4.0) == pytest.approx(want, rel=1e-15)
    assert f(0.3, 0.0, 0.0, 1.0, 0.9, 0.0, 0.0, 4.0) == 0.0                                      # nothing moves: no flux


def _mobile_dam_break():
    w = C.dam_break_channel(nx=60, ny=3, lx=30.0, ly=1.5, h_left=1.0, h_right=0.2, x_dam=15.0, t_end=float("inf"))
    return w


def test_module_off_is_the_fixed_bed_scheme(ref):
    w = _mobile_dam_break()
    a, b, c = ref.RefSolver(w), ref.RefSolver(w), ref.RefSolver(w)
    b.set_morphology(0, 0.05)
    c.set_morphology(ref.GRASS, 0.0)
    for s in (a, b, c):
        s.step(50, cfl=0.9)
    for x, y, z in zip(a.get_state(), b.get_state(), c.get_state()):
        assert np.array_equal(x, y) and np.array_equal(x, z)
    assert np.array_equal(b.get_bed(), w.zb) and np.array_equal(c.get_bed(), w.zb)


def test_exner_update_reassembled_and_porosity(ref):
    """Eq. 13 with S_b = 0: one step's bed change must equal -(dt/((1-p)|Omega_i|)) * sum_j (+-) l_ij q_Bij assembled with
    numpy from the oracle's per-edge q_Bij; walls and interfaces with a dry side carry nothing (R-20); p enters as
    1/(1-p) only."""
    w = _mobile_dam_break()
    x = M.centroids(w.node_xy, w.tri)[:, 0]
    w.h[x > 25.0] = 0.0                                   # a dry reach downstream
    w.hu = np.where(w.h > 0, 0.4, 0.0)
    dz = {}
    for p in (0.0, 0.5):
        s = ref.RefSolver(w)
        s.set_morphology(ref.GRASS, 0.05, porosity=p)
        info = s.step(1, cfl=0.9)
        qB = s.sediment_fluxes()
        area, nx, ny, ln = s.geometry()
        acc = np.zeros(w.n_cells)
        L, R = w.edge_cell[:, 0], w.edge_cell[:, 1]
        np.add.at(acc, L, ln * qB)
        inner = R >= 0
        np.add.at(acc, R[inner], -(ln * qB)[inner])
        dz[p] = s.get_bed() - w.zb
        assert np.allclose(dz[p], -info["dt_last"] / ((1.0 - p) * area) * acc, rtol=1e-12, atol=1e-18)
        assert np.all(qB[R == -1] == 0.0)
        dry = w.h <= w.h_dry
        assert np.all(qB[inner & (dry[L] | dry[np.where(inner, R, 0)])] == 0.0)
        assert np.any(qB != 0.0)
    assert np.allclose(dz[0.5], 2.0 * dz[0.0], rtol=1e-12, atol=1e-18)


@pytest.mark.parametrize("formula,alpha", [(1, 0.02), (2, 8.0)])
def test_sediment_volume_is_conserved_in_a_closed_box(ref, formula, alpha):
    """Eq. 3 in a box of walls: (1-p) * sum z_B |Omega| is constant to round-off while the bed moves, and the water
    volume stays conserved too."""
    w = _mobile_dam_break()
    w.kst[:] = 35.0
    s = ref.RefSolver(w)
    s.set_morphology(formula, alpha, theta_cr=0.047, s=2.65, dm=0.002, porosity=0.4)
    area = s.geometry()[0]
    v0 = (w.h * area).sum()
    info = s.step(400, cfl=0.9)
    zb = s.get_bed()
    assert np.abs(zb - w.zb).max() > 1e-4                       # the bed did move
    assert abs(((zb - w.zb) * area).sum()) < 1e-13 * area.sum()
    assert abs(info["vol"] - v0 - info["vol_clipped"]) < 1e-12 * v0
    assert np.all(np.isfinite(zb))


def test_uniform_stream_leaves_a_flat_bed_flat(ref):
    """A uniform stream over a flat bed carries a uniform q_B: div q_B = 0, and through the open ends as much leaves as
    enters (equilibrium boundary, R-20)."""
    w = C.dam_break_channel(nx=40, ny=3, lx=40.0, ly=3.0, h_left=2.0, h_right=2.0, transmissive_ends=True,
                            q_left=3.0, q_right=3.0, t_end=float("inf"))
    s = ref.RefSolver(w)
    s.set_morphology(ref.GRASS, 0.05)
    s.step(200, cfl=0.7)       # regular right-triangle mesh: the hydrodynamic scheme needs CFL <= 0.75 here (R-7)
    assert np.abs(s.get_bed()).max() < 1e-13
    assert np.abs(s.get_state()[0] - 2.0).max() < 1e-12


def bed_wave_celerity(u, h, alpha, p, g=G):
    """Exact speed of the bed wave of the coupled shallow-water / Exner system with q_B = alpha u^3 (linearised about a
    uniform stream): the smallest root in modulus of the characteristic polynomial
    lambda^3 - 2u lambda^2 + (u^2 - g(h + d)) lambda + g u d = 0,  d = 3 alpha u^2 / (1 - p)
    of the matrix [[u, h, 0], [g, u, g], [0, d, 0]] acting on (h, u, z_B).  For weak transport it tends to the
    quasi-steady value 3 alpha u^3 / ((1-p) h (1 - Fr^2))."""
    d = 3.0 * alpha * u * u / (1.0 - p)
    r = np.roots([1.0, -2.0 * u, u * u - g * (h + d), g * u * d])
    r = r[np.abs(r.imag) < 1e-12].real
    return r[np.argmin(np.abs(r))]


def test_bed_wave_celerity_limits():
    assert bed_wave_celerity(1.0, 10.0, 1e-6, 0.4) == pytest.approx(3e-6 / (0.6 * 10.0 * (1.0 - 1.0 / 98.1)), rel=1e-5)
    assert bed_wave_celerity(1.0, 10.0, 0.2, 0.4) == pytest.approx(0.09167, rel=1e-3)
    assert bed_wave_celerity(-1.0, 10.0, 0.2, 0.4) == pytest.approx(-0.09167, rel=1e-3)


@pytest.mark.parametrize("direction", [1.0, -1.0])
def test_bed_hump_travels_with_the_bed_wave_celerity(ref, direction):
    """A low hump on the bed of a slow deep stream (Fr = 0.1) under q_B = alpha u^3 moves downstream with the bed-wave
    speed of the coupled system (27.5 m in 300 s here; the scheme gives 28.5 m on this mesh, 28.3 m on finer ones: the
    crest, where the water is shallower, runs a little faster than the linearised speed).  Checked on the centroid of
    the hump, in both flow directions (Eq. 16 is not symmetric in u_n)."""
    lx, H, q, alpha, p = 400.0, 10.0, 10.0, 0.2, 0.4
    w = C.dam_break_channel(nx=200, ny=2, lx=lx, ly=4.0, h_left=H, h_right=H, transmissive_ends=True,
                            q_left=direction * q, q_right=direction * q, t_end=float("inf"))
    x = M.centroids(w.node_xy, w.tri)[:, 0]
    w.zb = 0.2 * np.exp(-((x - 200.0) / 20.0) ** 2)
    w.h = H - w.zb
    s = ref.RefSolver(w)
    s.set_morphology(ref.GRASS, alpha, porosity=p)
    area = s.geometry()[0]
    T = 300.0
    s.step(t_end=T, cfl=0.7)
    zb = s.get_bed()
    xc0 = (w.zb * x * area).sum() / (w.zb * area).sum()
    xc1 = (zb * x * area).sum() / (zb * area).sum()
    cb = bed_wave_celerity(direction * q / H, H, alpha, p)
    print("hump displacement", xc1 - xc0, "expected", cb * T, "crest", zb.max())
    assert abs(cb * T) > 25.0
    assert xc1 - xc0 == pytest.approx(cb * T, rel=0.05)
    assert (zb * area).sum() == pytest.approx((w.zb * area).sum(), rel=2e-3)     # what left through the ends is tiny
    assert zb.max() > 0.08                                                      # still a hump, not smeared away


def test_scalars_ride_on_a_moving_bed(ref):
    """Modules active together ("synchronous-decoupled ... same integration timestep"):
    scalars and the mobile bed in one run.  The scalar update of Eq. 20 uses the hydrodynamic mass flux only, so a uniform
    concentration stays uniform while the bed moves under it (q_c == phi0 * h bit for bit with phi0 = 1, to round-off for
    phi0 = 0.37), the hydrodynamic state and the bed are exactly those of the run without scalars, and scalar mass is
    conserved in the closed box."""
    w = C.dam_break_channel(nx=80, ny=4, lx=20.0, ly=1.0, h_left=1.0, h_right=0.2, x_dam=10.0, t_end=float("inf"))
    w.kst[:] = 35.0
    morph = (ref.GRASS, 0.02, 0.0, 2.65, 1e-3, 0.4)
    a = ref.RefSolver(w)                       # mobile bed, no scalars
    a.set_morphology(*morph)
    b = ref.RefSolver(w)                       # mobile bed + two species: phi = 1 and phi = 0.37
    b.set_scalars(np.stack([w.h.copy(), 0.37 * w.h]))
    b.set_morphology(*morph)
    area = a.geometry()[0]
    m0 = float(np.sum(0.37 * w.h * area))
    ia, ib = a.step(150, float("inf"), 0.7), b.step(150, float("inf"), 0.7)
    assert ia == ib
    for x, y in zip(a.get_state(), b.get_state()):
        assert np.array_equal(x, y)
    assert np.array_equal(a.get_bed(), b.get_bed()) and np.abs(a.get_bed() - w.zb).max() > 1e-5      # the bed did move
    h = b.get_state()[0]
    qc = b.get_scalars()
    assert np.array_equal(qc[0], h)                                     # phi = 1: q_c is h, bit for bit
    assert np.max(np.abs(qc[1] - 0.37 * h)) <= 1e-14                    # phi = 0.37 stays uniform to round-off
    assert abs(float(np.sum(qc[1] * area)) - m0) <= 1e-13 * m0          # scalar mass conserved in the closed box
