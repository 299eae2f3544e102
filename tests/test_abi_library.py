"""The C-ABI library of include/swe.h: it builds here (nvcc cross-compiles sm_100a without a GPU), loads, and
exports every symbol the header declares.  No compute call is made: there is no GPU on this box and the library
has no CPU fallback."""
import ctypes
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "swe.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(swe_[a-z_0-9]+)\s*\(", src)))


def test_header_declares_the_five_calls():
    names = declared_symbols()
    for n in ("swe_create", "swe_set_state", "swe_step", "swe_get_state", "swe_destroy", "swe_set_boundary",
              "swe_workspace_bytes", "swe_last_error", "swe_params_default"):
        assert n in names


def test_library_builds_loads_and_exports_every_declared_symbol():
    from paper_2102_12862_b200 import build as B
    import paper_2102_12862_b200 as P
    path = B.build()
    assert os.path.exists(path)
    L = ctypes.CDLL(path)
    names = declared_symbols()
    for n in names:
        assert hasattr(L, n), f"{n} is declared in include/swe.h but not exported"
    assert sorted(P.EXPORTS) == names            # the binding binds exactly what the header declares
    # the device code is sm_100a
    out = subprocess.run(["cuobjdump", "-lelf", path], capture_output=True, text=True).stdout
    assert "sm_100a" in out


def test_host_only_entry_points():
    """Entry points that touch no device: defaults, workspace size (monotone, aligned, covers every array)."""
    import paper_2102_12862_b200 as P
    L = P.lib()
    prm = P.SweParams()
    L.swe_params_default(ctypes.byref(prm))
    assert prm.g == 9.81 and prm.h_dry == 1e-3 and prm.dt_max == float("inf")
    assert prm.renumber == P.RENUMBER_MORTON and prm.state_on_device == 0
    assert prm.morphology == 0 and prm.n_species == 0 and prm.patch_cells == 0


def test_workspace_bytes_sizes_every_array_on_the_host():
    """swe_workspace_bytes(mesh, params) runs the host part of swe_create (no CUDA call, works here): the size covers
    the base arrays, the patch blobs of the fused step, the scalar species and the mobile-bed arrays, and a mesh that
    swe_create would reject gives 0 with a message."""
    import numpy as np
    import paper_2102_12862_b200 as P
    from workloads import configs as C
    w = C.by_id(4, 0.01)
    N, E = w.n_cells, w.n_edges
    args = (w.node_xy, w.tri, w.edge_cell, w.cell_edge, w.zb, w.kst)
    three = P.workspace_bytes(*args, variant=P.VARIANT_THREE_PASS)
    auto = P.workspace_bytes(*args)
    assert three % 256 == 0 and three >= 64 * N + 64 * E          # both state buffers, edge geometry and edge fluxes
    assert three < 400 * N + (1 << 20)                             # a 4M-cell context stays well below 2 GB of the 180 GB
    st, _, _ = P.host_preprocess(*args, patch_cells=256)
    assert auto - three >= st["patches"] * 64                      # + patch blobs and flag words
    assert auto > three + 100 * N                                  # blobs: > 100 bytes per cell (edge records + slot words)
    assert P.workspace_bytes(*args, n_species=2) - auto >= 2 * (16 * N + 8 * E)
    assert P.workspace_bytes(*args, morphology=1) - auto >= 8 * E + 16 * N
    assert P.workspace_bytes(*args, patch_cells=128, variant=P.VARIANT_PATCH) != P.workspace_bytes(*args, patch_cells=512, variant=P.VARIANT_PATCH)
    # rejected arguments -> 0 and a reason
    bad = w.tri.copy()
    bad[0] = bad[0][::-1]                                          # a clockwise triangle
    assert P.workspace_bytes(w.node_xy, bad, None, None, w.zb, w.kst) == 0
    assert b"counter-clockwise" in P.lib().swe_last_error(None)
    assert P.workspace_bytes(*args, n_species=6) == 0
    assert P.workspace_bytes(*args, patch_cells=7) == 0


def test_product_fails_loudly_without_gpu():
    import torch
    import paper_2102_12862_b200 as P
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    import numpy as np
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        P.Solver(np.zeros((3, 2)), np.array([[0, 1, 2]], np.int32))


def test_product_never_touches_the_oracle():
    """The oracle is test infrastructure: nothing under the package imports, links or opens it."""
    pkg = os.path.join(ROOT, "paper_2102_12862_b200")
    for dp, _, fs in os.walk(pkg):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".hpp")):
                txt = open(os.path.join(dp, f)).read()
                assert "oracle" not in txt.replace("the oracle", "").replace("The oracle", "") or \
                    not re.search(r"(import\s+oracle|from\s+oracle|swe_ref|libswe_ref)", txt), f
