"""Host logic of swe_create, through swe_host_preprocess (no GPU needed): mesh validation and its error codes, edge
tables built by the library, Morton and reverse Cuthill-McKee renumbering, the patch tables of the fused step."""
import numpy as np
import pytest

from workloads import configs as C
from workloads import mesh as M


@pytest.fixture(scope="module")
def P():
    import paper_2102_12862_b200 as P
    P.lib()
    return P


def new_ids(perm):
    inv = np.empty(perm.size, np.int64)
    inv[perm] = np.arange(perm.size)
    return inv


def test_permutations_and_locality(P):
    w = C.by_id(3, 0.02)
    wp, _ = w.permuted(5)                                    # caller order is random
    ctr = M.centroids(wp.node_xy, wp.tri)
    interior = wp.edge_cell[:, 1] >= 0
    L, R = wp.edge_cell[interior, 0], wp.edge_cell[interior, 1]
    spans = {}
    for name, mode in (("none", P.RENUMBER_NONE), ("morton", P.RENUMBER_MORTON), ("rcm", P.RENUMBER_RCM)):
        st, cp, ep = P.host_preprocess(wp.node_xy, wp.tri, wp.edge_cell, wp.cell_edge, wp.zb, wp.kst, renumber=mode,
                                       patch_cells=0)
        assert st["n_edges"] == wp.n_edges
        assert np.array_equal(np.sort(cp), np.arange(wp.n_cells)) and np.array_equal(np.sort(ep), np.arange(wp.n_edges))
        nid = new_ids(cp)
        spans[name] = np.abs(nid[L] - nid[R])
        if name == "none":
            assert np.array_equal(cp, np.arange(wp.n_cells)) and np.array_equal(ep, np.arange(wp.n_edges))
        else:
            # edges are ordered by the lower new cell id they touch
            key = np.minimum(nid[wp.edge_cell[ep, 0]], np.where(wp.edge_cell[ep, 1] >= 0, nid[np.maximum(wp.edge_cell[ep, 1], 0)],
                                                               nid[wp.edge_cell[ep, 0]]))
            assert np.all(np.diff(key) >= 0)
        if name == "morton":                                 # consecutive cells are close in space
            step = np.linalg.norm(np.diff(ctr[cp], axis=0), axis=1)
            assert np.median(step) < 2.0 * w.meta["spacing"]
    n = wp.n_cells
    assert np.median(spans["none"]) > 0.1 * n                # random numbering: neighbours are far apart in memory
    assert np.median(spans["morton"]) < 0.002 * n + 64
    assert spans["rcm"].max() < 6.0 * np.sqrt(n)             # RCM: small bandwidth (a few BFS levels)
    assert spans["rcm"].max() < spans["morton"].max()        # ... smaller than the Z-curve's worst jumps


def test_tables_built_by_the_library_match_the_harness(P):
    w = C.by_id(2, 0.05)
    a, _, _ = P.host_preprocess(w.node_xy, w.tri, w.edge_cell, w.cell_edge, w.zb, w.kst, patch_cells=0)
    b, _, _ = P.host_preprocess(w.node_xy, w.tri, None, None, w.zb, w.kst, patch_cells=0)
    assert a["n_edges"] == b["n_edges"] == w.n_edges


@pytest.mark.parametrize("pc", [32, 256, 1000])
def test_patch_tables(P, pc):
    w = C.by_id(4, 0.01)
    st, _, _ = P.host_preprocess(w.node_xy, w.tri, w.edge_cell, w.cell_edge, w.zb, w.kst, patch_cells=pc)
    assert st["patches"] == -(-w.n_cells // pc)
    assert st["sum_own_cells"] == st["distinct_own_cells"] == w.n_cells      # the patches partition the cells
    assert st["sum_local_cells"] > w.n_cells and st["sum_local_edges"] > w.n_edges
    if pc == 256:       # two halo rings of a compact 256-cell blob: 30-70 % more cells, < 50 % more edges; 3 blocks/SM fit
        assert 1.3 < st["sum_local_cells"] / w.n_cells < 1.7
        assert st["sum_local_edges"] / w.n_edges < 1.5
        assert 3 * (st["smem_bytes"] + 1024) <= 228 * 1024
    # on a random numbering the "patches" are not compact: the halos explode (AUTO then takes the three-pass step)
    wp, _ = w.permuted(3)
    bad, _, _ = P.host_preprocess(wp.node_xy, wp.tri, wp.edge_cell, wp.cell_edge, wp.zb, wp.kst, renumber=P.RENUMBER_NONE,
                                  patch_cells=pc)
    assert bad["sum_local_cells"] > 3 * st["sum_local_cells"] or pc >= 1000


def test_invalid_meshes_are_refused(P):
    w = C.tiny_mesh("four-cells")
    ok, _, _ = P.host_preprocess(w.node_xy, w.tri, w.edge_cell, w.cell_edge, w.zb, w.kst)
    assert ok["n_edges"] == 8 and ok["patches"] == 1

    def code(**kw):
        a = dict(node_xy=w.node_xy, tri=w.tri, edge_cell=w.edge_cell, cell_edge=w.cell_edge, zb=w.zb, kst=w.kst)
        a.update(kw)
        with pytest.raises(P.SweError) as ei:
            P.host_preprocess(a["node_xy"], a["tri"], a["edge_cell"], a["cell_edge"], a["zb"], a["kst"])
        return ei.value.code

    cw = w.tri.copy(); cw[1] = cw[1][::-1]
    assert code(tri=cw, edge_cell=None, cell_edge=None) == P.EMESH                    # clockwise triangle
    flat = w.node_xy.copy(); flat[4] = [1.0, 0.0]
    assert code(node_xy=flat) == P.EMESH                                              # zero-area triangle
    oob = w.tri.copy(); oob[0, 0] = 99
    assert code(tri=oob, edge_cell=None, cell_edge=None) == P.EMESH                   # node id out of range
    ec = w.edge_cell.copy(); ec[:, 0] = ec[::-1, 0]
    assert code(edge_cell=ec) == P.EMESH                                              # tables inconsistent
    ce = w.cell_edge.copy(); ce[0, 0], ce[0, 1] = ce[0, 1], ce[0, 0]
    assert code(cell_edge=ce) == P.EMESH                                              # slot order violated
    dup = np.vstack([w.tri, w.tri[:1]])
    assert code(tri=dup, edge_cell=None, cell_edge=None, zb=np.zeros(5), kst=np.full(5, np.inf)) == P.EMESH   # non-manifold
    assert code(edge_cell=w.edge_cell, cell_edge=None) == P.EINVAL                    # only one table given
    k = w.kst.copy(); k[2] = 0.0
    assert code(kst=k) == P.EINVAL                                                    # Strickler k must be > 0
    z = w.zb.copy(); z[1] = np.nan
    assert code(zb=z) == P.EINVAL
