"""Randomised GPU parity: seeded random meshes, beds, roughness, states (with dry regions, thin films and fast flow),
boundary codes and boundary strings, both step variants with random patch sizes, against the oracle through the C-ABI.
Every case is bit-for-bit reproducible from its seed; the bar is the one of test_gpu_parity.py."""
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


def random_workload(seed):
    rng = np.random.default_rng(1286200 + seed)
    n_pts = int(rng.integers(200, 6000))
    lx, ly = rng.uniform(20.0, 400.0), rng.uniform(20.0, 400.0)
    spacing = np.sqrt(lx * ly / n_pts)
    pts_in = np.stack([rng.uniform(0.3 * spacing, lx - 0.3 * spacing, n_pts),
                       rng.uniform(0.3 * spacing, ly - 0.3 * spacing, n_pts)], axis=1)
    pts_b = M.rectangle_boundary_points(0.0, lx, 0.0, ly, spacing)
    node_xy, tri = M.delaunay_tri_mesh(np.concatenate([pts_b, pts_in]), 1e-4 * spacing * spacing)
    n = tri.shape[0]
    ctr = M.centroids(node_xy, tri)
    # bed: a few bumps + noise; water level so that a random share of the domain is dry
    zb = np.zeros(n)
    for _ in range(int(rng.integers(1, 5))):
        c = rng.uniform([0, 0], [lx, ly])
        zb += rng.uniform(0.2, 3.0) * np.exp(-np.sum((ctr - c) ** 2, axis=1) / (2 * rng.uniform(0.05, 0.3) ** 2 * lx * ly))
    zb += 0.02 * rng.standard_normal(n)
    level = np.quantile(zb, rng.uniform(0.3, 1.0)) + rng.uniform(0.0, 1.0)
    h = np.maximum(0.0, level - zb)
    h[rng.random(n) < 0.02] = 10.0 ** rng.uniform(-9, -3)                 # thin films below and around h_dry
    h *= (1.0 + 0.3 * rng.random(n))                                       # not at rest
    speed = rng.uniform(0.0, 3.0)
    hu = h * speed * rng.standard_normal(n)
    hv = h * speed * rng.standard_normal(n)
    kst = np.where(rng.random(n) < 0.2, np.inf, rng.uniform(10.0, 60.0, n))
    w = C._finish(f"fuzz-{seed}", node_xy, tri, zb, kst, h, cfl=float(rng.uniform(0.3, 0.9)), dt_max=5.0)
    w.hu, w.hv = hu, hv
    # boundary codes by side: walls, transmissive, and up to two strings (inflow on the west, outflow on the east)
    kinds = rng.integers(0, 3, size=4)
    def code(mx, my):
        out = np.full(mx.shape, M.BC_WALL)
        west, east, south, north = mx < 1e-9, mx > lx - 1e-9, my < 1e-9, my > ly - 1e-9
        out[west] = [M.BC_WALL, M.BC_TRANSMISSIVE, M.bc_string(0)][kinds[0]]
        out[east] = [M.BC_WALL, M.BC_TRANSMISSIVE, M.bc_string(1)][kinds[1]]
        out[south] = [M.BC_WALL, M.BC_TRANSMISSIVE, M.BC_WALL][kinds[2]]
        out[north] = [M.BC_WALL, M.BC_TRANSMISSIVE, M.BC_TRANSMISSIVE][kinds[3]]
        return out
    C._set_boundary_codes(w, code)
    if kinds[0] == 2:
        q = rng.uniform(0.1, 5.0) * ly
        w.strings.append((0, C.BC_INFLOW_Q, np.array([0.0, q, 3.0, 2.0 * q, 10.0, 0.5 * q])))
    if kinds[1] == 2:
        w.strings.append((1, C.BC_OUTFLOW_UNIFORM, np.array([rng.uniform(0.0, 0.01)])))
    return w, rng


@pytest.mark.parametrize("seed", range(24))
def test_random_case(gpu, ref, seed):
    w, rng = random_workload(seed)
    n_sp = int(rng.integers(0, 3))
    variant = [gpu.VARIANT_THREE_PASS, gpu.VARIANT_PATCH][seed % 2]
    pc = int(rng.choice([32, 64, 96, 160, 384])) if variant == gpu.VARIANT_PATCH else 0
    s = gpu.from_workload(w, variant=variant, patch_cells=pc, n_species=n_sp, steps_per_graph=int(rng.choice([0, 4, 32])))
    o = ref.RefSolver(w)
    if n_sp:
        qc0 = np.stack([rng.random(w.n_cells) * w.h for _ in range(n_sp)])
        s.set_scalars(qc0)
        o.set_scalars(qc0)
        for sid, typ, _ in w.strings:
            if typ == C.BC_INFLOW_Q:
                phi = list(rng.random(n_sp))
                s.set_boundary_scalar(sid, phi)
                o.set_boundary_scalar(sid, phi)
    for n in (1, int(rng.integers(2, 40)), int(rng.integers(2, 60))):
        ig, io = s.step(n, float("inf"), w.cfl), o.step(n, float("inf"), w.cfl)
        sg, so = s.get_state(), o.get_state()
        assert np.array_equal(sg[0] > w.h_dry, so[0] > w.h_dry), f"seed {seed}: wet/dry masks differ"
        assert_state_close(sg, so, f"seed {seed} after {io['steps_done']} steps")
        check_info(ig, io)
        if n_sp:
            qg, qo = s.get_scalars(), o.get_scalars()
            for sp in range(n_sp):
                scale = np.max(np.abs(qo[sp]))
                assert np.all(np.abs(qg[sp] - qo[sp]) <= 1e-10 * np.abs(qo[sp]) + 1e-14 * scale), f"seed {seed}, species {sp}"
    s.close()
    o.close()


@pytest.mark.parametrize("seed", range(100, 110))
def test_random_case_single_precision(gpu, ref, seed):
    """The same random cases in single precision (R-21), both step variants with random patch sizes, against the
    fp32 build of the oracle: bit-identical states (thin films, dry regions, fast flow, strings), fp64 clock."""
    ref.lib(single=True)
    w, rng = random_workload(seed)
    variant = [gpu.VARIANT_THREE_PASS, gpu.VARIANT_PATCH][seed % 2]
    pc = int(rng.choice([32, 64, 96, 160, 240])) if variant == gpu.VARIANT_PATCH else 0
    s = gpu.from_workload(w, variant=variant, patch_cells=pc, precision=gpu.PRECISION_SINGLE,
                          steps_per_graph=int(rng.choice([0, 4, 32])))
    o = ref.RefSolver(w, precision="single")
    for n in (1, int(rng.integers(2, 40)), int(rng.integers(2, 60))):
        ig, io = s.step(n, float("inf"), w.cfl), o.step(n, float("inf"), w.cfl)
        for nm, a, b in zip(("h", "hu", "hv"), s.get_state(), o.get_state()):
            assert np.array_equal(a, b), (seed, nm, float(np.max(np.abs(a - b))))
        assert ig["steps_done"] == io["steps_done"] and ig["n_wet"] == io["n_wet"] and ig["flags"] == io["flags"]
        assert abs(ig["t"] - io["t"]) <= 1e-12 * abs(io["t"]) and abs(ig["dt_last"] - io["dt_last"]) <= 1e-12 * io["dt_last"]
        assert abs(ig["vol"] - io["vol"]) <= 1e-12 * abs(io["vol"])
    s.close()
    o.close()
