"""Pins of the oracle's passive-scalar advection (Eq. 8 advective part, Eq. 20 with
A_ij = F1 * phi of the upwind side, R-19) against what the paper and the mathematics fix:
the paper's T5 (a steady contact wave between two diverging rarefactions; "the exact solution for the
scalar advection is identical to the given initial conditions"), consistency with the continuity equation (a uniform
concentration stays uniform: q_c = phi h, bit for bit when phi = 1), conservation of scalar mass, the maximum principle
of donor-cell upwinding, the closed-form travelled mass in a uniform stream, linearity in the species, and the inflow
bookkeeping.  CPU only."""
import numpy as np
import pytest

from workloads import configs as C
from workloads import mesh as M


def phi_of(qc, h):
    return np.where(h > 0.0, qc / np.where(h > 0.0, h, 1.0), 0.0)


def test_t5_steady_contact_between_two_rarefactions(ref):
    """PAPER.md:544-553 (Eq. 22): 100 m x 0.1 m channel, 1362 cells, h = 1, q_x = -/+3, phi = 1 | 0, transparent ends,
    CFL 0.95, t = 2.5 s.  The scalar discontinuity must stay where it is while the depth drops to h* = 0.2715 m."""
    w = C.dam_break_channel(nx=681, ny=1, ly=0.1, h_left=1.0, h_right=1.0, cfl=0.95, transmissive_ends=True,
                            q_left=-3.0, q_right=3.0, t_end=2.5)
    assert w.n_cells == 1362
    x = M.centroids(w.node_xy, w.tri)[:, 0]
    phi0 = np.where(x < 50.0, 1.0, 0.0)
    s = ref.RefSolver(w)
    s.set_scalars(phi0 * w.h)
    info = s.step(t_end=2.5, cfl=0.95)
    assert info["t"] == 2.5
    h = s.get_state()[0]
    phi = phi_of(s.get_scalars()[0], h)
    assert np.max(np.abs(phi - phi0)) <= 1e-12
    mid = np.abs(x - 50.0) < 2.0
    assert np.all(np.abs(h[mid] - 0.2715) < 0.02)          # the water depression of the two rarefactions (Toro [18])


@pytest.mark.parametrize("phi_c", [1.0, 0.37])
def test_uniform_concentration_stays_uniform(ref, phi_c):
    """Consistency with continuity: with phi = const everywhere (and in the inflow) q_c = phi h for ever -- through
    wetting and drying, the limiter, friction and both boundary strings.  phi = 1: the scalar update is the depth
    update operation by operation, so q_c == h bit for bit."""
    w = C.by_id(4, 0.004)
    s = ref.RefSolver(w)
    s.set_scalars(phi_c * w.h)
    s.set_boundary_scalar(0, [phi_c])
    info = s.step(300, float("inf"), w.cfl)
    assert info["vol_clipped"] == 0.0 and info["n_wet"] != int(np.sum(w.h > w.h_dry))
    h = s.get_state()[0]
    qc = s.get_scalars()[0]
    if phi_c == 1.0:
        assert np.array_equal(qc, h)
    wet = h > 1e-9
    assert np.max(np.abs(qc[wet] / h[wet] - phi_c)) <= 1e-11
    assert np.max(np.abs(qc[~wet] - phi_c * h[~wet])) <= 1e-15


def test_scalar_mass_and_maximum_principle_closed_box(ref):
    """Closed domain (walls), Ritter dam break over a dry bed with phi = 1 in part of the reservoir: scalar mass is
    conserved to round-off and 0 <= phi <= 1 (donor-cell upwinding with the limited mass flux is monotone)."""
    w = C.config1()
    x = M.centroids(w.node_xy, w.tri)[:, 0]
    s = ref.RefSolver(w)
    area = s.geometry()[0]
    qc0 = np.where(x < 49.0, 1.0, 0.0) * w.h            # the last metre of the reservoir holds clear water
    s.set_scalars(qc0)
    for _ in range(4):
        s.step(t_end=s.step(0)["t"] + 1.0)
        h = s.get_state()[0]
        qc = s.get_scalars()[0]
        assert abs(np.sum(qc * area) - np.sum(qc0 * area)) <= 1e-13 * np.sum(qc0 * area)
        phi = phi_of(qc, h)
        assert phi.min() >= -1e-12 and phi.max() <= 1.0 + 1e-12
    # Ritter particle paths: water from x0 = 49 m has reached x = 58.9 m at t = 4 s, the clear water runs ahead of it
    assert phi[(x > 52.0) & (x < 56.0)].max() > 0.1
    front_cells = (x > 70.0) & (h > w.h_dry)
    assert front_cells.any() and phi[front_cells].max() < 0.05


def test_travelled_mass_in_a_uniform_stream(ref):
    """Uniform stream h = 1, u = 1 in a frictionless flat channel with transparent ends, phi = 1 for x < 20: the
    integral of phi over x is 20 + u t exactly (what enters at the left end carries phi = 1, nothing has reached the
    right end), and the smeared front is centred on x = 20 + u t."""
    w = C.dam_break_channel(nx=200, ny=2, lx=100.0, ly=1.0, h_left=1.0, h_right=1.0, transmissive_ends=True,
                            q_left=1.0, q_right=1.0, t_end=30.0)
    x = M.centroids(w.node_xy, w.tri)[:, 0]
    s = ref.RefSolver(w)
    area = s.geometry()[0]
    s.set_scalars(np.where(x < 20.0, 1.0, 0.0) * w.h)
    info = s.step(t_end=30.0, cfl=0.7)      # regular right-triangle mesh: Eq. 21's rho needs CFL <= 0.75 (R-7)
    h, hu, hv = s.get_state()
    assert np.max(np.abs(h - 1.0)) <= 1e-12 and np.max(np.abs(hu - 1.0)) <= 1e-12      # the stream stays uniform
    qc = s.get_scalars()[0]
    assert abs(np.sum(qc * area) / 1.0 - (20.0 + 1.0 * info["t"])) <= 1e-10
    phi = qc / h
    order = np.argsort(x)
    xs, ps = x[order], phi[order]
    front = xs[np.argmin(np.abs(ps - 0.5))]
    assert abs(front - 50.0) <= 1.0
    assert ps[xs < 40.0].min() > 0.999 and ps[xs > 60.0].max() < 1e-3


def test_species_are_independent_and_linear(ref):
    w = C.by_id(3, 0.004)
    rng = np.random.default_rng(7)
    phi = rng.random(w.n_cells)
    s = ref.RefSolver(w)
    s.set_scalars(np.stack([phi * w.h, 2.0 * phi * w.h, np.zeros(w.n_cells), 0.25 * w.h, 0.5 * phi * w.h]))
    s.step(80, float("inf"), w.cfl)
    q = s.get_scalars()
    assert np.array_equal(q[1], 2.0 * q[0]) and np.array_equal(q[4], 0.5 * q[0])       # exact: powers of two
    assert np.all(q[2] == 0.0)
    h = s.get_state()[0]
    assert np.max(np.abs(q[3] / h - 0.25)) <= 1e-13
    one = ref.RefSolver(w)                                                                # same as running it alone
    one.set_scalars(phi * w.h)
    one.step(80, float("inf"), w.cfl)
    assert np.array_equal(one.get_scalars()[0], q[0])


def test_inflow_string_carries_its_concentration(ref):
    """INFLOW_Q string with phi_in = 0.8 into clear water: scalar mass in the domain = 0.8 * vol_in until the marked
    water reaches the outlet."""
    w = C.uniform_flow_channel(nx=120, ny=3, lx=600.0, ly=15.0)
    s = ref.RefSolver(w)
    area = s.geometry()[0]
    s.set_scalars(np.zeros(w.n_cells))
    s.set_boundary_scalar(0, [0.8])
    info = s.step(t_end=60.0, cfl=0.7)
    qc = s.get_scalars()[0]
    assert info["vol_in"] > 0.0
    assert abs(np.sum(qc * area) - 0.8 * info["vol_in"]) <= 1e-11 * info["vol_in"]
    x = M.centroids(w.node_xy, w.tri)[:, 0]
    assert qc[x > 400.0].max() < 1e-30                       # numerical diffusion only
