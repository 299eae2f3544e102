"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times (default renumbering,
default CUDA-graph step loop, one swe_step call per window): configs[3] (river reach, ~4M cells, wetting/drying,
hydrograph inflow, normal-depth outflow) and configs[2] (circular dam break, ~1M cells).  The oracle steps the
whole mesh too (about 0.6 s per step at 4M cells); the configs[3] windows follow SURVEY section 8(d): 100 steps from
the initial state and from the GPU's own states at steps 1000 and 4000 (get_state -> oracle set_state), where the
flood wave has wetted part of the floodplain; configs[4] is checked at 8M and at 16M cells.  All cells are compared;
mass balance and wet counts are checked as well."""
import numpy as np
import pytest

from workloads import configs as C

from test_gpu_parity import assert_state_close, check_info, DT_RTOL


def make(gpu, w, **kw):
    return gpu.from_workload(w, **kw)     # defaults = the launch configuration bench.py times

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu tests must run on the B200 box")
    import paper_2102_12862_b200 as P
    P.lib()
    return P


_CONFIG4 = []


def config4_full():
    """configs[3] at full size, generated once for the three tests that step it (50 s each time; nobody writes to it)."""
    if not _CONFIG4:
        _CONFIG4.append(C.config4())
    return _CONFIG4[0]


def window(s, o, w, n, what):
    ig = s.step(n, float("inf"), w.cfl)
    io = o.step(n, float("inf"), w.cfl)
    sg, so = s.get_state(), o.get_state()
    assert np.array_equal(sg[0] > w.h_dry, so[0] > w.h_dry), f"{what}: wet/dry masks differ"
    assert_state_close(sg, so, what)
    assert ig["n_wet"] == io["n_wet"] and ig["steps_done"] == io["steps_done"]
    assert abs(ig["dt_last"] - io["dt_last"]) <= DT_RTOL * io["dt_last"]
    assert abs(ig["t"] - io["t"]) <= DT_RTOL * abs(io["t"])
    assert abs(ig["vol"] - io["vol"]) <= 1e-12 * io["vol"]
    return ig, io, sg


def test_config4_full_size_windows(gpu, ref):
    """SURVEY section 8(d) parity windows on configs[3] at full size, all cells: 100 steps from the initial state, and
    100-step windows started from the GPU's own states at steps 1000 and 4000 (get_state -> oracle set_state), where
    the flood wave has wetted part of the floodplain."""
    w = config4_full()
    assert 3.8e6 < w.n_cells < 4.2e6
    s = make(gpu, w)
    o = ref.RefSolver(w)
    area = s.geometry()[0]
    vol0 = float(np.sum(w.h * area))
    ig, io, _ = window(s, o, w, 100, "config4 full size, steps 0-100")
    check_info(ig, io)
    wet0 = int(np.sum(w.h > w.h_dry))
    for start in (1000, 4000):
        # GPU only up to `start` steps, then both sides continue from the GPU's state
        ig = s.step(start - ig["steps_done"], float("inf"), w.cfl)
        assert ig["flags"] == 0 and ig["steps_done"] == start
        # mass balance over the whole run so far (property that holds at any size)
        bal = ig["vol"] - vol0 - ig["vol_in"] + ig["vol_out"] - ig["vol_clipped"]
        assert abs(bal) <= 1e-11 * vol0, bal
        assert ig["vol_in"] > 0.0 and ig["vol_out"] > 0.0
        st = s.get_state()
        assert ig["n_wet"] == int(np.sum(st[0] > w.h_dry)) and ig["n_wet"] != wet0
        o.set_state(*st, t0=ig["t"])
        # (the GPU keeps stepping from its own state: no swe_set_state, so steps_done and the volume counters run on)
        io = o.step(100, float("inf"), w.cfl)
        ig = s.step(100, float("inf"), w.cfl)
        sg, so = s.get_state(), o.get_state()
        what = f"config4 full size, 100 steps from the GPU state at step {start}"
        assert np.array_equal(sg[0] > w.h_dry, so[0] > w.h_dry), f"{what}: wet/dry masks differ"
        assert_state_close(sg, so, what)
        assert ig["n_wet"] == io["n_wet"] and ig["steps_done"] == start + 100
        assert abs(ig["dt_last"] - io["dt_last"]) <= DT_RTOL * io["dt_last"]
        assert abs(ig["t"] - io["t"]) <= DT_RTOL * abs(io["t"])
        assert abs(ig["vol"] - io["vol"]) <= 1e-12 * io["vol"]
    s.close()
    o.close()


def test_config5_16m_window(gpu, ref):
    """BASELINE.json configs[4], second size (16M triangles): every cell against the oracle over the first 6 steps, in
    the launch configuration bench.py times, then the three-pass step against the fused patch step (AUTO's choice) over 40 more."""
    w = C.by_id(5, 2.0)
    assert 15.5e6 < w.n_cells < 16.5e6
    s = make(gpu, w)
    o = ref.RefSolver(w)
    ig, io, _ = window(s, o, w, 6, "config5 16M, steps 0-6")
    check_info(ig, io)
    o.close()
    t = gpu.from_workload(w, variant=gpu.VARIANT_THREE_PASS)
    t.step(6, float("inf"), w.cfl, info=False)
    i1, i2 = s.step(40, float("inf"), w.cfl), t.step(40, float("inf"), w.cfl)
    assert i1 == i2 and i1["flags"] == 0 and i1["n_wet"] == w.n_cells
    for x, y in zip(s.get_state(), t.get_state()):
        assert np.array_equal(x, y)
    s.close()
    t.close()


def test_config3_full_size_window(gpu, ref):
    """configs[2] at full size, with two passive scalar species riding along (R-19)."""
    w = C.config3()
    assert 0.95e6 < w.n_cells < 1.05e6
    rng = np.random.default_rng(3)
    qc0 = np.stack([rng.random(w.n_cells) * w.h, w.h])
    s = make(gpu, w, n_species=2)
    o = ref.RefSolver(w)
    s.set_scalars(qc0)
    o.set_scalars(qc0)
    ig, io, sg = window(s, o, w, 40, "config3 full size, steps 0-40")
    check_info(ig, io)
    assert ig["vol_clipped"] == 0.0
    qg, qo = s.get_scalars(), o.get_scalars()
    for sp in range(2):
        assert np.all(np.abs(qg[sp] - qo[sp]) <= 1e-10 * np.abs(qo[sp]) + 1e-14 * np.max(np.abs(qo[sp])))
    assert np.array_equal(qg[1], sg[0])                  # phi = 1: q_c == h bit for bit
    s.close()
    o.close()


def test_config5_8m_window_and_variants(gpu, ref):
    """BASELINE.json configs[4] at 8M cells: a 10-step window against the oracle on all cells, then a property that
    holds at any size -- the two step variants (fused patch = AUTO's choice, and three-pass, which share no kernel on the flux /
    update path) stay bit-identical over 300 steps -- and the volume balance of the transmissive domain."""
    w = C.config5()
    assert 7.8e6 < w.n_cells < 8.2e6
    s = gpu.from_workload(w)                                           # AUTO, as bench.py runs it: the fused patch step
    assert s.patch_stats()["variant"] == gpu.VARIANT_PATCH and s.patch_stats()["min_blocks_per_sm"] == 4
    o = ref.RefSolver(w)
    ig, io, _ = window(s, o, w, 10, "config5 8M, steps 0-10")
    check_info(ig, io)
    o.close()
    t = gpu.from_workload(w, variant=gpu.VARIANT_THREE_PASS)
    t.step(10, float("inf"), w.cfl, info=False)
    i1, i2 = s.step(300, float("inf"), w.cfl), t.step(300, float("inf"), w.cfl)
    assert i1 == i2 and i1["flags"] == 0 and i1["steps_done"] == 310
    for x, y in zip(s.get_state(), t.get_state()):
        assert np.array_equal(x, y)
    assert i1["n_wet"] == w.n_cells and i1["vol_clipped"] == 0.0
    s.close()
    t.close()


def test_config4_full_size_mobile_bed(gpu, ref):
    """configs[3] at full size with the morphodynamic module on (R-20; MPM-like law, d_m = 5 mm): every cell's state and
    bed elevation and every edge's q_Bij against the oracle over a short window; a cell no water ever reached keeps its
    bed (property that holds at any size)."""
    w = config4_full()
    s = make(gpu, w, morphology=True)
    o = ref.RefSolver(w)
    morph = (2, 8.0, 0.047, 2.65, 0.005, 0.4)
    s.set_morphology(*morph)
    o.set_morphology(*morph)
    assert s.step_kernels()[-1] == "k_patch_step"          # AUTO stays on the fused patch step with the mobile bed
    window(s, o, w, 12, "config4 full size, mobile bed, steps 0-12")
    zg, zo = s.get_bed(), o.get_bed()
    assert np.array_equal(zg, zo)
    assert np.array_equal(s.sediment_fluxes(), o.sediment_fluxes())
    moved = zg != w.zb
    assert moved.any() and not moved[(w.h <= w.h_dry) & (s.get_state()[0] == 0.0)].any()
    ig = s.step(500, float("inf"), w.cfl)
    assert ig["flags"] == 0 and np.all(np.isfinite(s.get_bed()))
    s.close()
    o.close()


def test_config4_full_size_single_precision(gpu, ref):
    """configs[3] at full size in single precision (R-21), both step variants against the fp32 build of the oracle: all
    cells bit-identical over a short window from the initial state and over a window started from the GPU's own state
    after 600 more steps (AUTO: the fused fp32 patch step, 32 % of the cells wet)."""
    ref.lib(single=True)
    w = config4_full()
    a = gpu.from_workload(w, precision=gpu.PRECISION_SINGLE)
    b = gpu.from_workload(w, precision=gpu.PRECISION_SINGLE, variant=gpu.VARIANT_THREE_PASS)
    o = ref.RefSolver(w, precision="single")
    assert a.step_kernels() == ["k_step_control", "k_patch_step"] and len(b.step_kernels()) == 4
    ia, ib, io = a.step(15, float("inf"), w.cfl), b.step(15, float("inf"), w.cfl), o.step(15, float("inf"), w.cfl)
    for x, y, z in zip(a.get_state(), b.get_state(), o.get_state()):
        assert np.array_equal(x, z) and np.array_equal(y, z)
    assert ia["t"] == ib["t"] == io["t"] and ia["n_wet"] == ib["n_wet"] == io["n_wet"]
    b.close()
    ia = a.step(600, float("inf"), w.cfl)
    assert ia["flags"] == 0 and a.patch_stats()["patch_steps_skipped"] > 0
    o.set_state(*a.get_state(), ia["t"])
    a.step(10, float("inf"), w.cfl)
    o.step(10, float("inf"), w.cfl)
    for x, z in zip(a.get_state(), o.get_state()):
        assert np.array_equal(x, z)
    a.close()
    o.close()
