"""Single-precision variant (R-21) through the C-ABI, against
the single-precision build of the oracle on the same seeded inputs.  Both sides evaluate the same parenthesisation with
IEEE fp32 operations (no FMA contraction, correctly rounded division / square root, cube root = correctly rounded fp64
root rounded to fp32), so the expected result is bit-identical states; the test states the tolerance the arithmetic
allows if it were not (1e-5 relative after 100 steps) and additionally reports the distance to the fp64 oracle."""
import numpy as np
import pytest

from workloads import configs as C

pytestmark = pytest.mark.gpu

CASES = {
    "config1-ritter": lambda: C.config1(),
    "config2-lake-small": lambda: C.by_id(2, 0.05),
    "config3-small": lambda: C.by_id(3, 0.02),
    "config4-small": lambda: C.by_id(4, 0.01),
    "uniform-flow": lambda: C.uniform_flow_channel(nx=60, ny=3),
}


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu tests must run on the B200 box")
    import paper_2102_12862_b200 as P
    P.lib()
    return P


@pytest.fixture(scope="module")
def ref():
    from oracle import swe_ref
    swe_ref.lib(single=True)
    return swe_ref


def f32(x):
    return np.asarray(x, np.float64).astype(np.float32).astype(np.float64)


@pytest.mark.parametrize("variant", [1, 2], ids=["three-pass", "patch"])
@pytest.mark.parametrize("name", list(CASES))
def test_parity_with_the_fp32_oracle(gpu, ref, name, variant):
    """Both step variants in fp32 (16-byte records; the fused patch step with 4-byte staged geometry) against the fp32
    build of the oracle: bit-identical."""
    w = CASES[name]()
    s = gpu.from_workload(w, precision=gpu.PRECISION_SINGLE, variant=variant, patch_cells=96 if variant == 2 else 0)
    o = ref.RefSolver(w, precision="single")
    assert s.step_kernels() == (["k_step_control", "k_edge_flux", "k_theta_lazy", "k_cell_update"] if variant == 1
                                else ["k_step_control", "k_patch_step"])
    for a, b in zip(s.geometry(), o.geometry()):
        assert np.array_equal(a, b)                                     # fp64 geometry rounded once to fp32, both sides
    assert s.peek_dt(w.cfl) == o.peek_dt(w.cfl)                         # fp32 rate, dt = cfl / rate in fp64
    for n in (1, 9, 90):
        ig, io = s.step(n, float("inf"), w.cfl), o.step(n, float("inf"), w.cfl)
        sg, so = s.get_state(), o.get_state()
        assert np.array_equal(sg[0] > w.h_dry, so[0] > w.h_dry), f"{name}: wet/dry masks differ"
        for nm, a, b in zip(("h", "hu", "hv"), sg, so):
            assert np.array_equal(a, f32(a)), nm                        # what comes back are fp32 numbers
            tol = 1e-5 * np.abs(b) + 1e-6 * np.max(np.abs(b))
            assert np.all(np.abs(a - b) <= tol), (name, nm, float(np.max(np.abs(a - b))))
            assert np.array_equal(a, b), (name, nm, "not bit-identical", float(np.max(np.abs(a - b))))
        assert ig["steps_done"] == io["steps_done"] and ig["n_wet"] == io["n_wet"]
        assert abs(ig["dt_last"] - io["dt_last"]) <= 1e-12 * io["dt_last"] and abs(ig["t"] - io["t"]) <= 1e-12 * io["t"]
        assert abs(ig["vol"] - io["vol"]) <= 1e-12 * io["vol"]
        assert abs(ig["vol_in"] - io["vol_in"]) <= 1e-12 * max(1.0, io["vol_in"])
        assert abs(ig["vol_out"] - io["vol_out"]) <= 1e-9 * max(1.0, io["vol_out"])
    if variant == 1:                                                    # (the fp32 patch step does not export its fluxes)
        F, Fo = s.edge_fluxes(), o.edge_fluxes()
        for a, b in zip(F[:4], Fo):
            assert np.array_equal(a, b)
    else:
        with pytest.raises(RuntimeError, match="single-precision patch step"):
            s.edge_fluxes()
    s.close()
    o.close()


def test_fp32_variants_agree_and_auto_picks_the_patch_step(gpu, ref):
    """AUTO in single precision: the fused patch step (default patch size, four blocks per SM) -- bit-identical to the
    fp32 three-pass step and to the fp32 oracle over 150 steps of the river reach, dry patches skipped."""
    w = CASES["config4-small"]()
    a = gpu.from_workload(w, precision=gpu.PRECISION_SINGLE)
    b = gpu.from_workload(w, precision=gpu.PRECISION_SINGLE, variant=gpu.VARIANT_THREE_PASS)
    o = ref.RefSolver(w, precision="single")
    assert a.patch_stats()["variant"] == gpu.VARIANT_PATCH and a.step_kernels() == ["k_step_control", "k_patch_step"]
    for n in (33, 117):
        ia, ib, io = a.step(n, float("inf"), w.cfl), b.step(n, float("inf"), w.cfl), o.step(n, float("inf"), w.cfl)
        for x, y, z in zip(a.get_state(), b.get_state(), o.get_state()):
            assert np.array_equal(x, y) and np.array_equal(x, z)
        assert ia["t"] == ib["t"] == io["t"] and ia["n_wet"] == ib["n_wet"] == io["n_wet"]
        assert ia["vol_in"] == ib["vol_in"] and abs(ia["vol_out"] - ib["vol_out"]) <= 1e-12 * max(1.0, ib["vol_out"])
    assert a.patch_stats()["patch_steps_skipped"] > 0
    for s in (a, b):
        s.close()
    o.close()
    # an all-wet state: in fp32 the three-pass step moves half the bytes and is the faster one -- AUTO takes it
    w3 = CASES["config3-small"]()
    c3 = gpu.from_workload(w3, precision=gpu.PRECISION_SINGLE)
    o3 = ref.RefSolver(w3, precision="single")
    assert c3.patch_stats()["variant"] == gpu.VARIANT_THREE_PASS and len(c3.step_kernels()) == 4
    c3.step(40, float("inf"), w3.cfl)
    o3.step(40, float("inf"), w3.cfl)
    for x, z in zip(c3.get_state(), o3.get_state()):
        assert np.array_equal(x, z)
    c3.close()
    o3.close()


def test_distance_to_the_fp64_oracle_and_mass(gpu, ref):
    """Error report of the fp32 variant against the fp64 oracle (configs[3] shrunk, wetting/drying, strings): after 100
    steps the depth differs by fp32 round-off amplified by the step count, far below the scheme's own error; the mass
    balance closes to fp32 round-off."""
    w = CASES["config4-small"]()
    s = gpu.from_workload(w, precision=gpu.PRECISION_SINGLE)
    o = ref.RefSolver(w)                                             # fp64
    area = o.geometry()[0]
    ig, io = s.step(100, float("inf"), w.cfl), o.step(100, float("inf"), w.cfl)
    hg, ho = s.get_state()[0], o.get_state()[0]
    wet = ho > 0.05
    rel = np.abs(hg[wet] - ho[wet]) / ho[wet]
    assert np.median(rel) < 1e-5 and np.sum(np.abs(hg - ho) * area) / np.sum(ho * area) < 1e-4
    assert abs(ig["t"] - io["t"]) <= 1e-4 * io["t"]
    vol0 = float(np.sum(f32(w.h) * area))
    bal = ig["vol"] - vol0 - ig["vol_in"] + ig["vol_out"] - ig["vol_clipped"]
    assert abs(bal) <= 2e-6 * vol0, bal
    s.close()
    o.close()


def test_single_precision_is_hydrodynamics_only(gpu):
    w = CASES["config3-small"]()
    for kw in (dict(n_species=1), dict(morphology=True)):
        with pytest.raises(RuntimeError, match="single precision"):
            gpu.from_workload(w, precision=gpu.PRECISION_SINGLE, **kw)
    s = gpu.from_workload(w, precision=gpu.PRECISION_SINGLE, variant=gpu.VARIANT_THREE_PASS)
    assert s.patch_stats()["variant"] == gpu.VARIANT_THREE_PASS
    d = gpu.from_workload(w, variant=gpu.VARIANT_THREE_PASS)
    assert s.workspace_nbytes < 0.66 * d.workspace_nbytes              # 16-byte records, 4-byte reals; the int32 tables stay
    s.close()
    d.close()
