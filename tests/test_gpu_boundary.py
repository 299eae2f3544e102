"""The boundary's memory contract (include/swe.h; "PyTorch is used only for device memory and streams"):
every device array of a context is carved from the workspace the caller lends (sized by swe_workspace_bytes(mesh,
params)); a too-small workspace is refused with SWE_ENOMEM; a swe_create that fails half-way leaves nothing behind."""
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


def free_bytes():
    import torch
    torch.cuda.synchronize()
    return torch.cuda.mem_get_info()[0]


def test_every_device_array_lives_in_the_lent_workspace(gpu):
    """With a lent workspace the library allocates no device memory of its own (the driver's own bookkeeping for the
    captured CUDA graphs aside: < 16 MB), with scalars and the mobile bed reserved too; without one it makes ONE
    allocation of the size swe_workspace_bytes names."""
    import torch
    w = C.by_id(4, 0.05)                                   # ~200k cells: a workspace of ~75 MB
    args = (w.node_xy, w.tri, w.edge_cell, w.cell_edge, w.zb, w.kst)
    need = gpu.workspace_bytes(*args, n_species=2, morphology=1)
    warm = gpu.from_workload(w)                            # module load, context creation, kernel images: once
    warm.step(40, float("inf"), w.cfl)
    warm.close()
    torch.cuda.empty_cache()
    f0 = free_bytes()
    s = gpu.from_workload(w, n_species=2, morphology=True)
    assert s.workspace_nbytes == need
    s.set_scalars(np.stack([w.h, 0.5 * w.h]))
    s.set_morphology(1, 0.001)
    s.step(70, float("inf"), w.cfl)
    f1 = free_bytes()
    grew = f0 - f1
    assert need <= grew + (2 << 20) and grew - need < (32 << 20), (need, grew)     # the torch tensor, and little else
    s.close()
    torch.cuda.empty_cache()
    assert abs(free_bytes() - f0) < (8 << 20)
    t = gpu.from_workload(w, own_workspace=True)
    f2 = free_bytes()
    own = gpu.workspace_bytes(*args)
    assert own <= f0 - f2 < own + (32 << 20)
    t.close()
    assert abs(free_bytes() - f0) < (8 << 20)


def test_too_small_workspace_is_refused_and_nothing_leaks(gpu):
    import torch
    w = C.by_id(3, 0.02)
    need = gpu.workspace_bytes(w.node_xy, w.tri, w.edge_cell, w.cell_edge, w.zb, w.kst)
    gpu.from_workload(w).close()

    def refused(n):
        for _ in range(n):
            for short in (256, need // 2):
                with pytest.raises(gpu.SweError) as ei:
                    gpu.from_workload(w, workspace_bytes=need - short)
                assert ei.value.code == gpu.ENOMEM and "workspace too small" in str(ei.value)
        torch.cuda.empty_cache()
        return free_bytes()

    f1 = refused(1)
    f8 = refused(8)
    assert abs(f8 - f1) < (1 << 20)                           # eight more refusals: not a byte less free memory
    s = gpu.from_workload(w, workspace_bytes=need)            # exactly enough: fine
    s.step(10, float("inf"), w.cfl)
    s.close()


def test_create_that_fails_half_way_leaves_nothing_behind(gpu):
    """swe_create with its own allocation on a device that has too little memory left: the one cudaMalloc fails after
    the host planning is done -> SWE_ENOMEM, and repeating it does not eat memory (pinned control block, context).
    A mesh the host part refuses never reaches the device."""
    import torch
    w = C.by_id(3, 0.1)                                        # ~100k cells: ~40 MB
    need = gpu.workspace_bytes(w.node_xy, w.tri, w.edge_cell, w.cell_edge, w.zb, w.kst)
    gpu.from_workload(w).close()
    torch.cuda.empty_cache()
    hog = torch.empty(free_bytes() - need // 4, dtype=torch.uint8, device="cuda")     # leave a quarter of what is needed

    def refused(n):
        for _ in range(n):
            with pytest.raises(gpu.SweError) as ei:
                gpu.from_workload(w, own_workspace=True)
            assert ei.value.code == gpu.ENOMEM and "device memory" in str(ei.value)
        return free_bytes()

    f1 = refused(1)
    f6 = refused(6)
    assert abs(f6 - f1) < (1 << 20)
    del hog
    torch.cuda.empty_cache()
    s = gpu.from_workload(w, own_workspace=True)               # with the memory back the same call succeeds
    s.step(5, float("inf"), w.cfl)
    s.close()
    bad = w.tri.copy()
    bad[5] = bad[5][::-1]                                      # a clockwise cell: refused by the host part
    with pytest.raises(gpu.SweError) as ei:
        gpu.Solver(w.node_xy, bad, None, None, w.zb, w.kst)
    assert ei.value.code == gpu.EMESH
