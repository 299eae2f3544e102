"""swe_state_summary_static (include/swe.h): the entry point that allocates nothing -- the reductions of swe_step_info
(water volume, wet cells, non-finite check) with the scratch of the k_info kernel in a static __device__ array of the
library.  Checked against the existing path (swe_step's info: k_info with scratch in the context's workspace) on two
calls in a row that share the static array, plus the size limit.  This file is collected last on purpose (test_zz_*):
the suite runs with pytest -x."""
import struct

import numpy as np
import pytest

from workloads import configs as C

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu tests must run on the B200 box")
    import paper_2102_12862_b200 as P
    P.lib()
    return P


def summary(gpu, dev, state, area_d, h_dry, n=None):
    """One call of the new entry point on device copies of a host state; returns (vol, n_wet, nonfinite)."""
    import torch
    h, hu, hv = (torch.from_numpy(np.ascontiguousarray(a)).to(dev) for a in state)
    out = torch.full((24,), 0xAB, dtype=torch.uint8, device=dev)          # poisoned: the kernel must write all of it
    gpu.state_summary_static(h, hu, hv, area_d, h_dry, out, n_cells=n)
    torch.cuda.synchronize()
    vol, n_wet, bad, pad = struct.unpack("<dqii", bytes(out.cpu().numpy()))
    assert pad == 0
    return vol, n_wet, bad


def test_static_summary_matches_step_info_on_two_calls_in_a_row(gpu):
    """Two calls in a row (the second sees the scratch the first left behind, on a different state and then on a
    shorter array) against swe_step's info of the same states: n_wet and the non-finite flag exactly, vol to the 1e-12
    relative the other GPU tests use for it (the two paths sum in different cell orders)."""
    import torch
    dev = "cuda:0"
    w = C.by_id(4, 0.02)                                   # river reach, ~80k cells: 20 blocks of the static kernel
    s = gpu.from_workload(w, device=dev)
    area = s.geometry()[0]
    area_d = torch.from_numpy(area).to(dev)
    results = []
    for n_steps in (40, 60):
        info = s.step(n_steps, float("inf"), w.cfl)        # existing path: k_info, scratch in the context's workspace
        state = s.get_state()
        vol, n_wet, bad = summary(gpu, dev, state, area_d, w.h_dry)
        results.append((vol, n_wet))
        assert n_wet == info["n_wet"] and n_wet > 0
        assert bad == 0 and info["flags"] == 0
        assert abs(vol - info["vol"]) <= 1e-12 * abs(info["vol"]), (vol, info["vol"])
        # and against the plain definition on the host
        assert abs(vol - float(np.dot(state[0], area))) <= 1e-12 * abs(vol)
        assert n_wet == int(np.count_nonzero(state[0] > w.h_dry))
    assert results[0] != results[1]                        # the inflow hydrograph has added water in between
    # a shorter array right after a longer one: stale partials of the earlier calls must not be read
    state = s.get_state()
    m = 4096 + 17                                          # two blocks, a ragged tail
    vol, n_wet, bad = summary(gpu, dev, state, area_d, w.h_dry, n=m)
    assert abs(vol - float(np.dot(state[0][:m], area[:m]))) <= 1e-12 * max(abs(vol), 1e-300)
    assert n_wet == int(np.count_nonzero(state[0][:m] > w.h_dry)) and bad == 0
    # same inputs, same bits (fixed summation order), and a non-finite momentum is seen
    again = summary(gpu, dev, state, area_d, w.h_dry)
    assert again == summary(gpu, dev, state, area_d, w.h_dry)
    poisoned = (state[0], state[1].copy(), state[2])
    poisoned[1][w.n_cells // 2] = np.nan
    assert summary(gpu, dev, poisoned, area_d, w.h_dry)[2] == 1
    s.close()


def test_static_summary_allocates_nothing(gpu):
    """Free device memory is the same before and after a call (the first call on the device has been made above or
    is made here as warm-up: module load is not an allocation of the call)."""
    import torch
    dev = "cuda:0"
    n = 300_000
    rng = np.random.default_rng(128620)
    state = (rng.random(n), rng.standard_normal(n), rng.standard_normal(n))
    area_d = torch.from_numpy(rng.random(n) + 0.5).to(dev)
    h, hu, hv = (torch.from_numpy(a).to(dev) for a in state)
    out = torch.zeros(24, dtype=torch.uint8, device=dev)
    gpu.state_summary_static(h, hu, hv, area_d, 1e-3, out)             # warm-up
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for _ in range(3):
        gpu.state_summary_static(h, hu, hv, area_d, 1e-3, out)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0
    vol = struct.unpack("<dqii", bytes(out.cpu().numpy()))[0]
    assert abs(vol - float(np.dot(state[0], area_d.cpu().numpy()))) <= 1e-12 * vol


def test_static_summary_rejects_sizes_beyond_the_static_array(gpu):
    import torch
    dev = "cuda:0"
    x = torch.zeros(16, dtype=torch.float64, device=dev)
    out = torch.zeros(24, dtype=torch.uint8, device=dev)
    for n in (gpu.SUMMARY_STATIC_MAX_CELLS + 1, 0, -5):
        with pytest.raises(gpu.SweError) as e:
            gpu.state_summary_static(x, x, x, x, 1e-3, out, n_cells=n)     # rejected before anything is launched
        assert e.value.code == gpu.EINVAL and "SWE_SUMMARY_STATIC_MAX_CELLS" in str(e.value)
    with pytest.raises(gpu.SweError):
        gpu.state_summary_static(0, x, x, x, 1e-3, out, n_cells=16)       # null pointer
    # the largest admitted size runs (4096 partials: the whole static array)
    n = gpu.SUMMARY_STATIC_MAX_CELLS
    h = torch.full((n,), 0.5, dtype=torch.float64, device=dev)
    z = torch.zeros(n, dtype=torch.float64, device=dev)
    a = torch.full((n,), 2.0, dtype=torch.float64, device=dev)
    gpu.state_summary_static(h, z, z, a, 1e-3, out)
    torch.cuda.synchronize()
    vol, n_wet, bad, _ = struct.unpack("<dqii", bytes(out.cpu().numpy()))
    assert vol == float(n) and n_wet == n and bad == 0
