"""GPU parity: the CUDA path (through the C-ABI of include/swe.h) against the oracle, element by element,
on the same seeded inputs.  Run on the B200 box with `-m gpu`.

Bar (BASELINE.json north_star, R-14): after 100 steps per-cell relative error of h, hu, hv <= 1e-10,
dt agrees to <= 1e-12 relative, wet/dry masks identical.  Geometry, fluxes before any cbrt, theta and the dt of
the first step are expected bit-identical (only + - * / sqrt min max on both sides, no FMA contraction).
"""
import numpy as np
import pytest

from workloads import configs as C
from workloads import mesh as M

pytestmark = pytest.mark.gpu

RTOL, ATOL_SCALE, DT_RTOL = 1e-10, 1e-14, 1e-12


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu tests must run on the B200 box")
    import paper_2102_12862_b200 as P
    P.lib()
    return P


_VARIANT = {"v": 0}


@pytest.fixture(autouse=True, params=[1, 2], ids=["three-pass", "patch"])
def variant(request):
    """Every test of this module runs with both step variants (include/swe.h SWE_VARIANT_*): the edge-flux ->
    theta -> gather/update three-pass step and the fused shared-memory patch step."""
    _VARIANT["v"] = request.param
    yield request.param


def make(gpu, w, **kw):
    kw.setdefault("variant", _VARIANT["v"])
    if kw["variant"] == 2:
        kw.setdefault("patch_cells", 192)      # small patches: the small test meshes still span many patches
    return gpu.from_workload(w, **kw)


def mk(gpu, *a, **kw):
    kw.setdefault("variant", _VARIANT["v"])
    return gpu.Solver(*a, **kw)


def assert_state_close(got, want, what=""):
    """abs(d) <= 1e-10 abs(ref) + 1e-14 max abs(ref) per field (R-14), and report the strict relative error
    on cells that are not pure round-off."""
    for name, a, b in zip(("h", "hu", "hv"), got, want):
        scale = np.max(np.abs(b)) if b.size else 0.0
        err = np.abs(a - b)
        tol = RTOL * np.abs(b) + ATOL_SCALE * scale
        bad = np.nonzero(~(err <= tol))[0]
        assert bad.size == 0, (f"{what} {name}: {bad.size} cells out of tolerance, worst at {bad[:5]}: "
                               f"got {a[bad[:5]]}, want {b[bad[:5]]}")
        sig = np.abs(b) > 1e-8 * scale
        if np.any(sig):
            assert np.max(err[sig] / np.abs(b[sig])) <= RTOL, f"{what} {name}: strict relative error too large"


def run_both(gpu, ref, w, n_steps, t_end=float("inf"), chunks=(None,), **kw):
    """Steps oracle and GPU side by side in the given chunks; returns the two solvers and info dicts."""
    o = ref.RefSolver(w)
    s = make(gpu, w, **kw)
    io = o.step(n_steps, t_end, w.cfl)
    ig = s.step(n_steps, t_end, w.cfl)
    return o, s, io, ig


def check_info(ig, io):
    assert ig["steps_done"] == io["steps_done"]
    assert ig["n_wet"] == io["n_wet"]
    assert ig["flags"] == io["flags"]
    assert abs(ig["t"] - io["t"]) <= DT_RTOL * abs(io["t"])
    assert abs(ig["dt_last"] - io["dt_last"]) <= DT_RTOL * abs(io["dt_last"])
    assert abs(ig["vol"] - io["vol"]) <= 1e-12 * abs(io["vol"])
    for k in ("vol_in", "vol_out"):
        assert abs(ig[k] - io[k]) <= 1e-11 * max(abs(io[k]), 1e-300) + 0.0, (k, ig[k], io[k])
    assert abs(ig["vol_clipped"] - io["vol_clipped"]) <= 1e-9 * abs(io["vol_clipped"]) + 1e-13 * abs(io["vol"])


CASES = {
    "config1-ritter": lambda: C.config1(),
    "config1-stoker": lambda: C.dam_break_channel(h_right=0.1),
    "config2-lake-small": lambda: C.by_id(2, 0.1),
    "config3-small": lambda: C.by_id(3, 0.02),
    "config4-small": lambda: C.by_id(4, 0.01),
    "uniform-flow": lambda: C.uniform_flow_channel(nx=60, ny=3, lx=300.0, ly=15.0),
    "t5-rarefactions": lambda: C.dam_break_channel(nx=681, ny=1, ly=0.1, h_left=1.0, h_right=1.0, cfl=0.95,
                                                   transmissive_ends=True, q_left=-3.0, q_right=3.0, t_end=2.5),
}


@pytest.mark.parametrize("name", ["config2-lake-small", "config3-small", "config4-small"])
def test_geometry_bit_identical(gpu, ref, name):
    """Section 4.1 geometry: areas, lengths, normals as the kernels use them == the oracle's."""
    w = CASES[name]()
    o = ref.RefSolver(w)
    s = make(gpu, w)
    for a, b in zip(s.geometry(), o.geometry()):
        assert np.array_equal(a, b)
    s.close()


@pytest.mark.parametrize("name", list(CASES))
def test_first_step_edge_by_edge(gpu, ref, name):
    """S0 + S1 + S1c of the first step, per edge: fluxes after the limiter, theta, dt."""
    w = CASES[name]()
    o = ref.RefSolver(w)
    s = make(gpu, w)
    assert s.peek_dt(w.cfl) == o.peek_dt(w.cfl)                      # Eq. 21: exact max, one division
    io = o.step(1, float("inf"), w.cfl)
    ig = s.step(1, float("inf"), w.cfl)
    assert ig["dt_last"] == io["dt_last"]
    F = s.edge_fluxes()
    Fo = o.edge_fluxes()
    inflow = np.zeros(w.n_edges, bool)
    for sid, typ, _ in w.strings:
        if typ == C.BC_INFLOW_Q:
            inflow |= w.edge_cell[:, 1] == -3 - sid
    for nm, a, b in zip(("F1", "F3", "GL", "GR"), F[:4], Fo):
        # bit-identical except where cbrt enters (conveyance-weighted inflow / normal-depth outflow edges)
        plain = np.ones(w.n_edges, bool)
        for sid, typ, _ in w.strings:
            plain &= w.edge_cell[:, 1] != -3 - sid
        assert np.array_equal(a[plain], b[plain]), nm
        assert np.allclose(a[~plain], b[~plain], rtol=1e-14, atol=0), nm
    assert_state_close(s.get_state(), o.get_state(), name)
    check_info(ig, io)
    s.close()


@pytest.mark.parametrize("name", list(CASES))
def test_parity_100_steps(gpu, ref, name):
    """The north_star bar: 100 steps, state <= 1e-10 relative, dt <= 1e-12 relative, identical wet/dry masks.
    Stepped in chunks of 1, 9 and 90 so that graph launches, tails and repeated calls are all exercised."""
    w = CASES[name]()
    o = ref.RefSolver(w)
    s = make(gpu, w)
    for n in (1, 9, 90):
        io = o.step(n, float("inf"), w.cfl)
        ig = s.step(n, float("inf"), w.cfl)
        so, sg = o.get_state(), s.get_state()
        assert np.array_equal(sg[0] > w.h_dry, so[0] > w.h_dry), "wet/dry masks differ"
        assert_state_close(sg, so, f"{name} after {io['steps_done']} steps")
        check_info(ig, io)
        assert abs(s.peek_dt(w.cfl) - o.peek_dt(w.cfl)) <= DT_RTOL * o.peek_dt(w.cfl)
    assert io["steps_done"] == 100
    s.close()


def test_config1_to_t_end(gpu, ref):
    """BASELINE.json configs[0] in full: Ritter dam break to t = 4 s; the last step lands on t_end exactly."""
    w = C.config1()
    o, s, io, ig = run_both(gpu, ref, w, -1, w.t_end)
    assert ig["t"] == 4.0 and io["t"] == 4.0
    check_info(ig, io)
    assert_state_close(s.get_state(), o.get_state(), "config1 t=4")
    # calling again does nothing
    ig2 = s.step(-1, w.t_end, w.cfl)
    assert ig2["steps_done"] == ig["steps_done"] and ig2["t"] == 4.0
    s.close()


def test_config2_lake_at_rest_1000_steps(gpu, ref):
    """BASELINE.json configs[1] in full (80k cells, 1000 steps): |u|,|v| <= 1e-12, mass to round-off, and parity."""
    w = C.config2()
    s = make(gpu, w)
    ig = s.step(1000, float("inf"), w.cfl)
    h, hu, hv = s.get_state()
    wet = h > w.h_dry
    assert np.array_equal(wet, w.h > w.h_dry)
    assert np.max(np.abs(hu[wet] / h[wet])) <= 1e-12 and np.max(np.abs(hv[wet] / h[wet])) <= 1e-12
    area = s.geometry()[0]
    assert abs(np.sum(h * area) - np.sum(w.h * area)) <= 1e-13 * np.sum(w.h * area)
    assert ig["vol_clipped"] == 0.0
    o = ref.RefSolver(w)
    io = o.step(1000, float("inf"), w.cfl)
    check_info(ig, io)
    assert_state_close((h, hu, hv), o.get_state(), "config2 1000 steps")
    s.close()


@pytest.mark.parametrize("name", ["config3-small", "config4-small"])
def test_renumbering_does_not_change_results(gpu, name):
    """R-15: Morton numbering vs caller numbering vs a randomly permuted input: bit-identical states."""
    w = CASES[name]()
    # caller numbering is Qhull's (not spatially compact): AUTO must fall back to the three-pass step for it
    a = make(gpu, w, renumber=gpu.RENUMBER_NONE, variant=gpu.VARIANT_AUTO, patch_cells=0)
    b = make(gpu, w, renumber=gpu.RENUMBER_MORTON)
    wp, cp = w.permuted(7)
    c = make(gpu, wp, renumber=gpu.RENUMBER_MORTON)
    d = make(gpu, w, renumber=gpu.RENUMBER_RCM, variant=gpu.VARIANT_AUTO, patch_cells=0)   # reverse Cuthill-McKee
    for s in (a, b, c, d):
        s.step(60, float("inf"), w.cfl)
    sa, sb, sc, sd = a.get_state(), b.get_state(), c.get_state(), d.get_state()
    for x, y, z, r in zip(sa, sb, sc, sd):
        assert np.array_equal(x, y)
        assert np.array_equal(x[cp], z)
        assert np.array_equal(x, r)
    rp = d.permutation()[0]
    assert np.array_equal(np.sort(rp), np.arange(w.n_cells)) and not np.array_equal(rp, b.permutation()[0])
    d.close()
    perm = b.permutation()[0]
    assert np.array_equal(np.sort(perm), np.arange(w.n_cells)) and not np.array_equal(perm, np.arange(w.n_cells))
    for s in (a, b, c):
        s.close()


def test_graph_and_plain_launches_agree(gpu):
    """The CUDA-graph step loop and plain kernel launches give bit-identical states; launch counts add up."""
    w = CASES["config4-small"]()
    a = make(gpu, w, steps_per_graph=0)
    b = make(gpu, w, steps_per_graph=8)
    c = make(gpu, w, steps_per_graph=32)
    infos = [s.step(75, float("inf"), w.cfl) for s in (a, b, c)]
    for s in (b, c):
        for x, y in zip(a.get_state(), s.get_state()):
            assert np.array_equal(x, y)
    assert infos[0] == infos[1] == infos[2]
    assert a.kernel_launches >= 75 * len(a.step_kernels())
    for s in (a, b, c):
        s.close()


def test_restart_round_trip(gpu):
    """S9 / O-10: get_state at step 50 -> new context -> set_state -> 50 more == 100 straight steps, bitwise."""
    w = CASES["config3-small"]()
    a = make(gpu, w)
    a.step(100, float("inf"), w.cfl)
    b = make(gpu, w)
    i50 = b.step(50, float("inf"), w.cfl)
    st = b.get_state()
    c = make(gpu, w)
    c.set_state(*st, t0=i50["t"])
    ic = c.step(50, float("inf"), w.cfl)
    for x, y in zip(a.get_state(), c.get_state()):
        assert np.array_equal(x, y)
    assert ic["steps_done"] == 50
    for s in (a, b, c):
        s.close()


def test_state_on_device_and_own_workspace(gpu):
    """Device-pointer state (torch tensors) and a library-owned workspace give the same results as host pointers."""
    import torch
    w = CASES["config3-small"]()
    a = make(gpu, w)
    b = make(gpu, w, state_on_device=True)
    c = make(gpu, w, own_workspace=True)
    for s in (a, b, c):
        s.step(40, float("inf"), w.cfl, info=False)
    ref_state = a.get_state()
    dev = b.get_state()
    torch.cuda.synchronize()
    for x, y, z in zip(ref_state, dev, c.get_state()):
        assert np.array_equal(x, y.cpu().numpy())
        assert np.array_equal(x, z)
    for s in (a, b, c):
        s.close()


def test_tables_built_by_the_library(gpu):
    """edge_cell / cell_edge = NULL: the library builds both; all boundary edges are walls; same result as the
    harness tables up to the edge numbering."""
    w = CASES["config2-lake-small"]()
    a = make(gpu, w)
    b = mk(gpu, w.node_xy, w.tri, None, None, w.zb, w.kst, h_dry=w.h_dry)
    b.set_state(w.h, w.hu, w.hv)
    ec, ce = b.tables()
    assert b.n_edges == w.n_edges
    # slot k of cell i is the edge between tri[k] and tri[(k+1)%3], L/R consistent
    for k in range(3):
        e = ce[:, k]
        assert np.all((ec[e, 0] == np.arange(w.n_cells)) | (ec[e, 1] == np.arange(w.n_cells)))
    a.step(30, float("inf"), 0.9)
    b.step(30, float("inf"), 0.9)
    for x, y in zip(a.get_state(), b.get_state()):
        assert np.array_equal(x, y)
    a.close()
    b.close()


def test_degenerate_and_error_cases(gpu):
    w = C.tiny_mesh("two-cells")
    # all dry, dt_max = inf: dt unbounded -> flag, no step, no hang
    s = mk(gpu, w.node_xy, w.tri, w.edge_cell, w.cell_edge, w.zb, w.kst)
    s.set_state(np.zeros(2), np.zeros(2), np.zeros(2))
    info = s.step(5, float("inf"), 0.9)
    assert info["steps_done"] == 0 and info["flags"] & gpu.FLAG_DT_UNBOUNDED
    # all dry with a finite dt_max: steps of dt_max that change nothing
    s2 = mk(gpu, w.node_xy, w.tri, w.edge_cell, w.cell_edge, w.zb, w.kst, dt_max=2.0)
    s2.set_state(np.zeros(2), np.zeros(2), np.zeros(2))
    info = s2.step(3, float("inf"), 0.9)
    assert info["steps_done"] == 3 and info["t"] == 6.0 and info["vol"] == 0.0
    # n_steps = 0 is a no-op; unlimited steps without t_end is refused
    assert s2.step(0, float("inf"), 0.9)["steps_done"] == 3
    with pytest.raises(gpu.SweError) as ei:
        s2.step(-1, float("inf"), 0.9)
    assert ei.value.code == gpu.EINVAL
    # clockwise triangle -> SWE_EMESH
    bad = w.tri.copy()
    bad[0] = bad[0][::-1]
    with pytest.raises(gpu.SweError) as ei:
        mk(gpu, w.node_xy, bad, None, None, w.zb, w.kst)
    assert ei.value.code == gpu.EMESH
    # inconsistent tables -> SWE_EMESH
    ec = w.edge_cell.copy()
    ec[:, 0] = ec[::-1, 0]
    with pytest.raises(gpu.SweError) as ei:
        mk(gpu, w.node_xy, w.tri, ec, w.cell_edge, w.zb, w.kst)
    assert ei.value.code == gpu.EMESH
    # non-finite state is reported
    s3 = mk(gpu, w.node_xy, w.tri, w.edge_cell, w.cell_edge, w.zb, w.kst)
    s3.set_state(np.array([1.0, np.nan]), np.zeros(2), np.zeros(2))
    with pytest.raises(gpu.SweError) as ei:
        s3.step(1, float("inf"), 0.9)
    assert ei.value.code == gpu.ENONFINITE
    # boundary string that no edge belongs to
    with pytest.raises(gpu.SweError):
        s.set_boundary(3, gpu.BC_INFLOW_Q, [0.0, 1.0])
    for x in (s, s2, s3):
        x.close()


def test_hand_values_through_the_abi(gpu):
    """The worked interior-edge values of tests/golden/hand_fluxes.txt through the CUDA path:
    two cells sharing the edge x = 1 with normal (1, 0)."""
    import os
    gold = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "hand_fluxes.txt")) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                case, q, v = line.split()
                gold[(case, q)] = float(v)
    w = C.tiny_mesh("two-cells-x")
    w.zb = np.array([0.0, 0.5])
    s = mk(gpu, w.node_xy, w.tri, w.edge_cell, w.cell_edge, w.zb, w.kst)
    s.set_state(np.array([2.0, 1.0]), np.array([2.0, 0.0]), np.array([1.0, 0.0]))
    s.step(1, float("inf"), 1e-6)          # tiny CFL: theta = 1
    F1, F3, GL, GR, theta = s.edge_fluxes()
    e = int(np.nonzero(w.edge_cell[:, 1] >= 0)[0][0])
    sign = 1.0 if w.edge_cell[e, 0] == 0 else -1.0   # normal stored from L to R; the hand values are for L = cell 0
    assert sign == 1.0
    assert abs(F1[e] - gold[("interior", "F1")]) < 5e-13
    assert abs(F3[e] - gold[("interior", "F3")]) < 5e-13
    assert abs(GL[e] - gold[("interior", "GL")]) < 5e-12
    assert abs(GR[e] - gold[("interior", "GR")]) < 5e-12
    assert np.all(theta == 1.0)
    s.close()


def test_device_cbrt_matches(gpu, ref):
    """R-14: the kernels' cube root is the correctly rounded one, like the oracle's (pinned against exact integer
    arithmetic in test_oracle_scheme.py): random mantissas over 600 binades, neighbours of exact cubes and of
    powers of two, subnormals, the ends of the range."""
    rng = np.random.default_rng(128620)
    x = np.ldexp(1.0 + rng.random(400000), rng.integers(-300, 300, 400000))
    i = np.arange(1.0, 20001.0)
    cubes = i * i * i
    pw = np.ldexp(1.0, np.arange(-1070, 1020))
    near = np.concatenate([np.nextafter(c, d) for c in (cubes, pw) for d in (0.0, np.inf)] +
                          [np.nextafter(np.nextafter(pw, 0.0), 0.0), np.nextafter(np.nextafter(pw, np.inf), np.inf)])
    x = np.concatenate([x, cubes, pw, near, [5e-324, 1e-310, 1.7e308, 0.0, 1e-3, 1.0]])
    x = x[np.isfinite(x) & (x >= 0)]
    got = gpu.device_cbrt(x)
    want = np.array([ref.cbrt(float(v)) for v in x])
    assert np.array_equal(got, want)
    assert np.array_equal(gpu.device_cbrt(-x[:1000]), -want[:1000])


@pytest.mark.parametrize("name", ["config3-small", "config4-small", "uniform-flow", "config1-ritter"])
def test_variants_and_patch_sizes_bit_identical(gpu, name):
    """The fused patch step (any patch size, ragged last patch, patches larger than the mesh) and the three-pass
    step evaluate the same arithmetic: bit-identical states, dt and volume counters."""
    w = CASES[name]()
    ref_s = gpu.from_workload(w, variant=gpu.VARIANT_THREE_PASS)
    i0 = ref_s.step(70, float("inf"), w.cfl)
    s0 = ref_s.get_state()
    for pc in (32, 100, 512, 700):                   # 512 / 700 exceed the cell count of the smallest case; 700 cells: a 1024-thread block
        s = gpu.from_workload(w, variant=gpu.VARIANT_PATCH, patch_cells=pc)
        st = s.patch_stats()
        assert st["variant"] == gpu.VARIANT_PATCH and st["patches"] == -(-w.n_cells // pc)
        i1 = s.step(70, float("inf"), w.cfl)
        for x, y in zip(s0, s.get_state()):
            assert np.array_equal(x, y), (name, pc)
        assert i1 == i0, (name, pc)
        s.close()
    ref_s.close()


def test_dry_patches_are_skipped_and_rewetted(gpu, ref):
    """Fused patch step: blocks whose whole patch (own cells + both halo rings) is dry skip the flux work; the
    Ritter front then runs into such patches.  States stay equal to the oracle's; all-wet meshes skip nothing."""
    w = C.config1()
    s = gpu.from_workload(w, variant=gpu.VARIANT_PATCH, patch_cells=64)
    o = ref.RefSolver(w)
    skipped = []
    for n in (5, 60, 200):
        ig, io = s.step(n, float("inf"), w.cfl), o.step(n, float("inf"), w.cfl)
        assert_state_close(s.get_state(), o.get_state(), f"ritter after {io['steps_done']} steps")
        check_info(ig, io)
        skipped.append(s.patch_stats()["patch_steps_skipped"])
    st = s.patch_stats()
    assert skipped[0] > 0                                           # the dry half of the channel is skipped at first
    per_step = np.diff([0] + skipped) / np.array([5, 60, 200])
    assert per_step[2] < per_step[0]                                # ... and less and less as the front wets it
    assert ig["n_wet"] > int(np.sum(w.h > w.h_dry))
    s.close()
    w3 = CASES["config3-small"]()
    s3 = gpu.from_workload(w3, variant=gpu.VARIANT_PATCH, patch_cells=128)
    s3.step(20, float("inf"), w3.cfl)
    assert s3.patch_stats()["patch_steps_skipped"] == 0
    s3.close()


def test_skip_flags_are_exact(gpu):
    """The 32-byte flag test of the fused patch step is exact, not just safe: in every step the number of skipped
    patches equals the number of patches whose local cells (own cells and everything within two edges of them) are all
    exactly (0, 0, 0) in the state the step reads and that no boundary-string edge can feed -- counted here on the host
    from the state and the mesh alone.  First step: flags written after swe_set_state; later steps: flags the blocks
    publish to their neighbours (one byte per neighbour, from the per-cell reader masks)."""
    w = CASES["config4-small"]()
    P = 64
    s = gpu.from_workload(w, variant=gpu.VARIANT_PATCH, patch_cells=P)
    perm = s.permutation()[0]                               # perm[internal id] = caller id
    n = w.n_cells
    patch_of = np.empty(n, np.int64)
    patch_of[perm] = np.arange(n) // P
    n_patches = (n + P - 1) // P
    L, R = w.edge_cell[:, 0].astype(np.int64), w.edge_cell[:, 1].astype(np.int64)
    inner = R >= 0

    def dilate(mask):                                       # cells within one edge of a marked cell
        out = mask.copy()
        np.logical_or.at(out, L[inner], mask[R[inner]])     # (a cell is L or R of up to three edges: unbuffered)
        np.logical_or.at(out, R[inner], mask[L[inner]])
        return out

    fed = np.zeros(n, bool)
    fed[L[R <= -3]] = True                                  # cells with a boundary-string edge
    fed_patch = np.zeros(n_patches, bool)
    np.logical_or.at(fed_patch, patch_of, dilate(fed))      # ... among the own and ring-1 cells of the patch

    def expected_skips(state):
        nz = (state[0] != 0.0) | (state[1] != 0.0) | (state[2] != 0.0)
        near = np.zeros(n_patches, bool)
        np.logical_or.at(near, patch_of, dilate(dilate(nz)))
        return int(np.count_nonzero(~near & ~fed_patch))

    seen = []
    done = 0
    for before in (0, 1, 2, 37, 38, 120):
        if before > done:
            s.step(before - done, float("inf"), w.cfl)
            done = before
        want = expected_skips(s.get_state())
        k0 = s.patch_stats()["patch_steps_skipped"]
        s.step(1, float("inf"), w.cfl)
        done += 1
        assert s.patch_stats()["patch_steps_skipped"] - k0 == want, (before, want)
        seen.append(want)
    assert 0 < min(seen) and max(seen) < n_patches and len(set(seen)) > 1   # the flood moves the count
    s.close()


def test_auto_picks_the_variant_from_the_wet_fraction(gpu, ref):
    """AUTO keeps both step variants ready and picks one at every swe_set_state.  With the default patch size four blocks
    of the patch kernel fit an SM and it is the faster step at any wet fraction; with fatter blocks (here: 384-cell
    patches, two per SM) the fused patch step runs while part of the domain is dry and the three-pass step on (almost)
    all-wet states.  Switching is invisible in the results."""
    w4, w3 = CASES["config4-small"](), CASES["config3-small"]()
    d = gpu.from_workload(w3, variant=gpu.VARIANT_AUTO, patch_cells=0)
    assert d.patch_stats()["variant"] == gpu.VARIANT_PATCH and d.step_kernels() == ["k_patch_step"]   # all wet, default patches; self-controlled: one kernel per step
    assert d.patch_stats()["min_blocks_per_sm"] >= 4
    d.close()
    a = gpu.from_workload(w4, variant=gpu.VARIANT_AUTO, patch_cells=384)
    assert a.patch_stats()["variant"] == gpu.VARIANT_PATCH and a.step_kernels() == ["k_patch_step"]
    assert a.patch_stats()["min_blocks_per_sm"] < 4
    b = gpu.from_workload(w3, variant=gpu.VARIANT_AUTO, patch_cells=384)
    assert b.patch_stats()["variant"] == gpu.VARIANT_THREE_PASS and len(b.step_kernels()) == 4
    # odd number of steps (the patch step ping-pongs), then flood the river reach: AUTO switches to three-pass
    o = ref.RefSolver(w4)
    a.step(33, float("inf"), w4.cfl)
    o.step(33, float("inf"), w4.cfl)
    assert_state_close(a.get_state(), o.get_state(), "river, patch step")
    h, hu, hv = a.get_state()
    h2 = h + 0.5
    a.set_state(h2, hu, hv, t0=1.0)
    o.set_state(h2, hu, hv, t0=1.0)
    assert a.patch_stats()["variant"] == gpu.VARIANT_THREE_PASS
    ia, io = a.step(40, float("inf"), w4.cfl), o.step(40, float("inf"), w4.cfl)
    assert_state_close(a.get_state(), o.get_state(), "flooded river, three-pass step")
    check_info(ia, io)
    # and back: the original state again -> patch step
    a.set_state(w4.h, w4.hu, w4.hv, t0=0.0)
    o.set_state(w4.h, w4.hu, w4.hv, t0=0.0)
    assert a.patch_stats()["variant"] == gpu.VARIANT_PATCH
    ia, io = a.step(25, float("inf"), w4.cfl), o.step(25, float("inf"), w4.cfl)
    assert_state_close(a.get_state(), o.get_state(), "river again, patch step")
    check_info(ia, io)
    a.close()
    b.close()


def test_auto_follows_a_spreading_flood(gpu, ref):
    """AUTO re-evaluates its choice whenever swe_step returns info: a dam break that wets the whole (short) channel
    starts on the patch step and ends on the three-pass step, with the state equal to the oracle's throughout."""
    w = C.dam_break_channel(nx=120, ny=4, lx=24.0, ly=0.8, x_dam=8.0, t_end=20.0)
    s = gpu.from_workload(w, variant=gpu.VARIANT_AUTO, patch_cells=384)      # fat patches: the wet-fraction rule applies
    o = ref.RefSolver(w)
    seen = [s.patch_stats()["variant"]]
    for _ in range(16):
        ig, io = s.step(35, float("inf"), w.cfl), o.step(35, float("inf"), w.cfl)     # odd chunks: the patch step ping-pongs
        assert_state_close(s.get_state(), o.get_state(), f"after {io['steps_done']} steps")
        check_info(ig, io)
        seen.append(s.patch_stats()["variant"])
    assert seen[0] == gpu.VARIANT_PATCH and seen[-1] == gpu.VARIANT_THREE_PASS, seen
    assert ig["n_wet"] == w.n_cells
    s.close()


def _many_strings_workload(nx, ny, n_in, n_out):
    """A wide basin with the west side cut into n_in INFLOW_Q strings and the east side into n_out OUTFLOW_UNIFORM
    strings (string ids interleaved), walls north and south."""
    lx, ly = 4.0 * nx, 2.0 * ny
    node_xy, tri = M.structured_tri_mesh(nx, ny, lx, ly, alternate=True)
    n = tri.shape[0]
    ctr = M.centroids(node_xy, tri)
    rng = np.random.default_rng(77)
    zb = -0.002 * ctr[:, 0] + 0.01 * rng.standard_normal(n)
    w = C._finish(f"many-strings-{nx}x{ny}-{n_in}+{n_out}", node_xy, tri, zb, np.full(n, 30.0),
                  np.full(n, 0.8) + 0.05 * rng.random(n), cfl=0.7, dt_max=2.0)
    w.hu = 0.5 * w.h
    def code(mx, my):
        out = np.full(mx.shape, M.BC_WALL)
        west, east = mx < 1e-9, mx > lx - 1e-9
        seg_w = np.minimum((my / ly * n_in).astype(int), n_in - 1)
        seg_e = np.minimum((my / ly * n_out).astype(int), n_out - 1)
        out[west] = [M.bc_string(2 * k) for k in seg_w[west]]
        out[east] = [M.bc_string(2 * k + 1) for k in seg_e[east]]
        return out
    C._set_boundary_codes(w, code)
    for k in range(n_in):
        q = (0.4 + 0.1 * k) * ly / n_in
        w.strings.append((2 * k, C.BC_INFLOW_Q, np.array([0.0, q, 5.0, 2.0 * q])))
    for k in range(n_out):
        w.strings.append((2 * k + 1, C.BC_OUTFLOW_UNIFORM, np.array([0.002])))
    return w


@pytest.mark.parametrize("nx,ny,n_in,n_out", [(6, 40, 3, 3),        # six strings: general path of k_step_control
                                               (4, 1500, 1, 1),     # 1500 members: more than the control block's threads
                                               (3, 4500, 1, 1),     # 4500 members: pairwise tree in global scratch
                                               (8, 64, 2, 2),       # four short strings: the up-front path
                                               (4, 300, 1, 1)])     # 300 members: a 512-leaf tree, more leaves than threads
def test_boundary_string_sums_many_and_long_strings(gpu, ref, nx, ny, n_in, n_out):
    """R-11: the fixed-shape pairwise sums over boundary strings (conveyance weights, outflow volume) and the volume
    bookkeeping, for string counts and sizes on both sides of the limits of k_step_control's up-front path."""
    w = _many_strings_workload(nx, ny, n_in, n_out)
    s, o = make(gpu, w), ref.RefSolver(w)
    for n in (1, 7, 40):
        ig, io = s.step(n, float("inf"), w.cfl), o.step(n, float("inf"), w.cfl)
        assert_state_close(s.get_state(), o.get_state(), w.name)
        check_info(ig, io)
        assert ig["vol_in"] > 0.0 and ig["vol_out"] > 0.0
        assert abs(ig["vol_in"] - io["vol_in"]) <= 1e-13 * io["vol_in"]
        assert abs(ig["vol_out"] - io["vol_out"]) <= 1e-13 * io["vol_out"]
    s.close()
    o.close()
