"""GPU parity of the passive-scalar module (R-19; Eq. 8 advective part, PAPER.md:298-304
Eq. 20) against the oracle, through the C-ABI (swe_set_scalars / swe_get_scalars / swe_set_boundary_scalar), for both
step variants.  Bar: the hydrodynamic state as in test_gpu_parity.py; q_c <= 1e-10 relative (expected: bit-identical)."""
import numpy as np
import pytest

from workloads import configs as C
from workloads import mesh as M

from test_gpu_parity import assert_state_close, check_info

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu tests must run on the B200 box")
    import paper_2102_12862_b200 as P
    P.lib()
    return P


def assert_scalars_close(got, want, what):
    assert got.shape == want.shape
    for sp in range(want.shape[0]):
        scale = np.max(np.abs(want[sp])) if want[sp].size else 0.0
        tol = 1e-10 * np.abs(want[sp]) + 1e-14 * scale
        bad = np.nonzero(~(np.abs(got[sp] - want[sp]) <= tol))[0]
        assert bad.size == 0, f"{what}, species {sp}: {bad.size} cells out of tolerance, e.g. {bad[:5]}"


def both(gpu, ref, w, qc0, phi_in, variant, patch_cells, chunks):
    n_sp = qc0.shape[0]
    s = gpu.from_workload(w, variant=variant, patch_cells=patch_cells, n_species=n_sp)
    o = ref.RefSolver(w)
    s.set_scalars(qc0)
    o.set_scalars(qc0)
    for sid, phi in phi_in.items():
        s.set_boundary_scalar(sid, phi)
        o.set_boundary_scalar(sid, phi)
    identical = True
    for n in chunks:
        ig, io = s.step(n, float("inf"), w.cfl), o.step(n, float("inf"), w.cfl)
        sg, so = s.get_state(), o.get_state()
        assert np.array_equal(sg[0] > w.h_dry, so[0] > w.h_dry)
        assert_state_close(sg, so, f"{w.name} after {io['steps_done']} steps")
        check_info(ig, io)
        qg, qo = s.get_scalars(), o.get_scalars()
        assert_scalars_close(qg, qo, f"{w.name} after {io['steps_done']} steps")
        identical &= np.array_equal(qg, qo)
    s.close()
    o.close()
    return identical, qg, sg


VARIANTS = [(1, 0), (2, 96), (2, 0)]


@pytest.mark.parametrize("variant,pc", VARIANTS)
def test_river_reach_two_species(gpu, ref, variant, pc):
    """Wet/dry fronts, limiter, friction, hydrograph inflow carrying species 0, normal-depth outflow."""
    w = C.by_id(4, 0.01)
    rng = np.random.default_rng(11)
    qc0 = np.stack([rng.random(w.n_cells) * w.h, 0.5 * w.h])
    ident, qg, sg = both(gpu, ref, w, qc0, {0: [0.9, 0.5]}, variant, pc, (1, 9, 90))
    assert ident
    wet = sg[0] > 1e-9
    assert np.max(np.abs(qg[1][wet] / sg[0][wet] - 0.5)) <= 1e-11        # a uniform concentration stays uniform


@pytest.mark.parametrize("variant,pc", VARIANTS)
def test_five_species_all_wet(gpu, ref, variant, pc):
    w = C.by_id(3, 0.02)
    rng = np.random.default_rng(12)
    qc0 = np.stack([rng.random(w.n_cells) * w.h for _ in range(5)])
    qc0[3] = w.h                                                            # phi = 1: q_c stays equal to h bit for bit
    ident, qg, sg = both(gpu, ref, w, qc0, {}, variant, pc, (40, 60))
    assert ident
    assert np.array_equal(qg[3], sg[0])


@pytest.mark.parametrize("variant,pc", VARIANTS)
def test_t5_steady_contact(gpu, ref, variant, pc):
    """The paper's T5 through the CUDA path: the scalar step stays where it is."""
    w = C.dam_break_channel(nx=681, ny=1, ly=0.1, h_left=1.0, h_right=1.0, cfl=0.95, transmissive_ends=True,
                            q_left=-3.0, q_right=3.0, t_end=2.5)
    x = M.centroids(w.node_xy, w.tri)[:, 0]
    phi0 = np.where(x < 50.0, 1.0, 0.0)
    s = gpu.from_workload(w, variant=variant, patch_cells=pc, n_species=1)
    s.set_scalars(phi0 * w.h)
    info = s.step(-1, 2.5, 0.95)
    assert info["t"] == 2.5
    h = s.get_state()[0]
    phi = s.get_scalars()[0] / h
    assert np.max(np.abs(phi - phi0)) <= 1e-12
    o = ref.RefSolver(w)
    o.set_scalars(phi0 * w.h)
    o.step(-1, 2.5, 0.95)
    assert_scalars_close(s.get_scalars(), o.get_scalars(), "T5")
    s.close()


@pytest.mark.parametrize("variant,pc", [(2, 64), (1, 0)])
def test_ritter_marked_water_over_dry_bed(gpu, ref, variant, pc):
    """Dam break over a dry bed with marked water: dry patches are skipped and re-wetted while carrying no scalar;
    scalar mass is conserved to round-off in the closed box."""
    w = C.config1()
    x = M.centroids(w.node_xy, w.tri)[:, 0]
    qc0 = (np.where(x < 49.0, 1.0, 0.0) * w.h)[None, :]
    ident, qg, sg = both(gpu, ref, w, qc0, {}, variant, pc, (5, 60, 200))
    assert ident
    s = gpu.from_workload(w, variant=variant, patch_cells=pc, n_species=1)
    area = s.geometry()[0]
    s.close()
    assert abs(np.sum(qg[0] * area) - np.sum(qc0[0] * area)) <= 1e-13 * np.sum(qc0[0] * area)


def test_scalars_do_not_change_the_flow_and_api_errors(gpu):
    w = C.by_id(4, 0.01)
    a = gpu.from_workload(w)
    b = gpu.from_workload(w, n_species=2)
    b.set_scalars(np.stack([w.h, 0.3 * w.h]))
    ia, ib = a.step(50, float("inf"), w.cfl), b.step(50, float("inf"), w.cfl)
    assert ia == ib
    for x, y in zip(a.get_state(), b.get_state()):
        assert np.array_equal(x, y)
    with pytest.raises(gpu.SweError):
        a.get_scalars()                                  # created with n_species = 0
    with pytest.raises(gpu.SweError):
        gpu.from_workload(w, n_species=6)                # "up to a maximum of 5"
    # restart round trip with scalars: get -> new context -> set
    c = gpu.from_workload(w, n_species=2)
    c.set_state(*b.get_state(), t0=ib["t"])
    c.set_scalars(b.get_scalars())
    b.step(30, float("inf"), w.cfl)
    c.step(30, float("inf"), w.cfl)
    assert np.array_equal(b.get_scalars(), c.get_scalars())
    for s in (a, b, c):
        s.close()


def test_auto_switches_variant_with_scalars_on_board(gpu, ref):
    """AUTO moves from the patch step to the three-pass step while a dam break wets a short channel; the scalar
    masses travel with the state through the switch (buffer b -> buffer a) and stay equal to the oracle's."""
    w = C.dam_break_channel(nx=120, ny=4, lx=24.0, ly=0.8, x_dam=8.0, t_end=20.0)
    x = M.centroids(w.node_xy, w.tri)[:, 0]
    qc0 = np.stack([np.where(x < 4.0, 1.0, 0.0) * w.h, 0.25 * w.h])
    s = gpu.from_workload(w, variant=gpu.VARIANT_AUTO, n_species=2, patch_cells=384)   # fat patches: AUTO's wet-fraction rule applies
    o = ref.RefSolver(w)
    s.set_scalars(qc0)
    o.set_scalars(qc0)
    seen = [s.patch_stats()["variant"]]
    for _ in range(10):
        ig, io = s.step(35, float("inf"), w.cfl), o.step(35, float("inf"), w.cfl)
        assert_state_close(s.get_state(), o.get_state(), f"after {io['steps_done']} steps")
        assert_scalars_close(s.get_scalars(), o.get_scalars(), f"after {io['steps_done']} steps")
        check_info(ig, io)
        seen.append(s.patch_stats()["variant"])
    assert seen[0] == gpu.VARIANT_PATCH and seen[-1] == gpu.VARIANT_THREE_PASS, seen
    s.close()
