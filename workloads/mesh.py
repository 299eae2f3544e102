"""Seeded synthetic mesh construction shared by the oracle tests, the GPU tests and bench.py.

This module holds NONE of the method's arithmetic (no areas used by the scheme, no normals, no
fluxes): it only produces the *inputs* of `swe_create` -- node coordinates, CCW triangles and the
two topology tables -- in the conventions of include/swe.h:

  edge_cell[e] = (L, R)   L >= 0; R >= 0 for an interior edge, R < 0 = boundary code
  cell_edge[i][k]         = edge between tri[i][k] and tri[i][(k+1)%3]      (slot order)

Paper: the triangulation is conforming, each cell has three neighbours j=1..3 across the edges
Gamma_ij (section 4.1, Fig. 2).
"""
from __future__ import annotations

import numpy as np

BC_WALL = -1          # PAPER.md:332 (section 5.2): default for every external edge
BC_TRANSMISSIVE = -2  # PAPER.md:342 "zerogradient (i.e. Neumann BC)"


def bc_string(s: int) -> int:
    """Boundary code of boundary string s (include/swe.h): -3 - s."""
    return -3 - int(s)


def orient_ccw(node_xy: np.ndarray, tri: np.ndarray) -> np.ndarray:
    """Return tri with every triangle counter-clockwise (swap two nodes where it is not)."""
    p = node_xy[tri]
    cross = (p[:, 1, 0] - p[:, 0, 0]) * (p[:, 2, 1] - p[:, 0, 1]) - (p[:, 2, 0] - p[:, 0, 0]) * (
        p[:, 1, 1] - p[:, 0, 1]
    )
    tri = tri.copy()
    flip = cross < 0
    tri[flip, 1], tri[flip, 2] = tri[flip, 2].copy(), tri[flip, 1].copy()
    return tri


def signed_area2(node_xy: np.ndarray, tri: np.ndarray) -> np.ndarray:
    """Twice the signed triangle area (used only to filter degenerate Delaunay slivers)."""
    p = node_xy[tri]
    return (p[:, 1, 0] - p[:, 0, 0]) * (p[:, 2, 1] - p[:, 0, 1]) - (p[:, 2, 0] - p[:, 0, 0]) * (
        p[:, 1, 1] - p[:, 0, 1]
    )


def build_edge_tables(tri: np.ndarray, n_nodes: int | None = None):
    """edge_cell [E,2] int32 and cell_edge [N,3] int32 from CCW triangles.

    Edges are numbered by sorted (min node, max node); L is the lower-numbered cell of the pair
    (so the normal of an interior edge, taken from L's slot, points from L to R). Boundary edges get
    R = BC_WALL; callers overwrite R with other codes by edge midpoint.
    """
    tri = np.ascontiguousarray(tri, dtype=np.int64)
    n = tri.shape[0]
    if n_nodes is None:
        n_nodes = int(tri.max()) + 1 if n else 0
    a = tri.reshape(-1)                         # slot k of cell i sits at 3*i + k
    b = np.roll(tri, -1, axis=1).reshape(-1)
    key = np.minimum(a, b) * np.int64(n_nodes) + np.maximum(a, b)
    order = np.argsort(key, kind="stable")      # stable: lower cell id first inside a pair
    skey = key[order]
    first = np.ones(skey.shape[0], dtype=bool)
    first[1:] = skey[1:] != skey[:-1]
    edge_of_sorted = np.cumsum(first) - 1
    n_edges = int(edge_of_sorted[-1]) + 1 if n else 0
    counts = np.bincount(edge_of_sorted, minlength=n_edges)
    if counts.max(initial=0) > 2:
        raise ValueError("non-manifold mesh: an edge is shared by more than two cells")
    cell_of_sorted = order // 3
    edge_cell = np.full((n_edges, 2), BC_WALL, dtype=np.int32)
    idx_first = np.nonzero(first)[0]
    edge_cell[:, 0] = cell_of_sorted[idx_first]
    second = ~first
    edge_cell[edge_of_sorted[second], 1] = cell_of_sorted[second]
    cell_edge = np.empty(3 * n, dtype=np.int32)
    cell_edge[order] = edge_of_sorted
    return edge_cell, cell_edge.reshape(n, 3)


def edge_midpoints(node_xy, tri, edge_cell, cell_edge):
    """Midpoint of every edge (for assigning boundary codes by position)."""
    n_edges = edge_cell.shape[0]
    mid = np.empty((n_edges, 2))
    for k in range(3):
        e = cell_edge[:, k]
        mid[e] = 0.5 * (node_xy[tri[:, k]] + node_xy[tri[:, (k + 1) % 3]])
    return mid


def centroids(node_xy, tri):
    return node_xy[tri].mean(axis=1)


def structured_tri_mesh(nx: int, ny: int, lx: float, ly: float, x0=0.0, y0=0.0,
                        alternate: bool = False, jitter: float = 0.0, rng=None):
    """(nx x ny) quads on [x0,x0+lx] x [y0,y0+ly], each split into 2 CCW triangles.

    alternate=False: every quad is split along the same diagonal (config 1).
    alternate=True : the diagonal alternates with (i+j) parity (config 2).
    jitter: interior nodes are moved by U(-jitter, jitter) * spacing in x and y (seeded by rng).
    """
    xs = np.linspace(x0, x0 + lx, nx + 1)
    ys = np.linspace(y0, y0 + ly, ny + 1)
    X, Y = np.meshgrid(xs, ys, indexing="ij")      # node (i, j) -> id i*(ny+1)+j
    if jitter > 0.0:
        dx, dy = lx / nx, ly / ny
        jx = rng.uniform(-jitter, jitter, size=X.shape) * dx
        jy = rng.uniform(-jitter, jitter, size=Y.shape) * dy
        jx[0, :] = jx[-1, :] = 0.0
        jx[:, 0] = jx[:, -1] = 0.0
        jy[0, :] = jy[-1, :] = 0.0
        jy[:, 0] = jy[:, -1] = 0.0
        X = X + jx
        Y = Y + jy
    node_xy = np.stack([X.reshape(-1), Y.reshape(-1)], axis=1)
    i, j = np.meshgrid(np.arange(nx), np.arange(ny), indexing="ij")
    i = i.reshape(-1)
    j = j.reshape(-1)
    n00 = i * (ny + 1) + j
    n10 = (i + 1) * (ny + 1) + j
    n01 = i * (ny + 1) + (j + 1)
    n11 = (i + 1) * (ny + 1) + (j + 1)
    # diagonal n00-n11: (n00,n10,n11), (n00,n11,n01); diagonal n10-n01: (n00,n10,n01), (n10,n11,n01)
    t_a0 = np.stack([n00, n10, n11], axis=1)
    t_a1 = np.stack([n00, n11, n01], axis=1)
    t_b0 = np.stack([n00, n10, n01], axis=1)
    t_b1 = np.stack([n10, n11, n01], axis=1)
    if alternate:
        use_b = ((i + j) % 2 == 1)[:, None]
        t0 = np.where(use_b, t_b0, t_a0)
        t1 = np.where(use_b, t_b1, t_a1)
    else:
        t0, t1 = t_a0, t_a1
    tri = np.empty((2 * nx * ny, 3), dtype=np.int32)
    tri[0::2] = t0
    tri[1::2] = t1
    tri = orient_ccw(node_xy, tri).astype(np.int32)
    return node_xy, tri


def jittered_hex_points(x0, x1, y0, y1, spacing, jitter, rng):
    """Blue-noise-like points: hexagonal lattice of the given spacing, each point moved uniformly
    inside a disc of radius jitter*spacing (stand-in for Poisson-disk sampling)."""
    dy = spacing * np.sqrt(3.0) / 2.0
    ny = int(np.floor((y1 - y0) / dy)) + 1
    nx = int(np.floor((x1 - x0) / spacing)) + 2
    jj, ii = np.meshgrid(np.arange(ny), np.arange(nx), indexing="ij")
    x = x0 + (ii + 0.5 * (jj % 2)) * spacing - 0.25 * spacing
    y = y0 + jj * dy + 0.5 * ((y1 - y0) - (ny - 1) * dy)
    x = x.reshape(-1)
    y = y.reshape(-1)
    r = jitter * spacing * np.sqrt(rng.uniform(0.0, 1.0, size=x.shape))
    th = rng.uniform(0.0, 2.0 * np.pi, size=x.shape)
    x = x + r * np.cos(th)
    y = y + r * np.sin(th)
    keep = (x > x0) & (x < x1) & (y > y0) & (y < y1)
    return np.stack([x[keep], y[keep]], axis=1)


def rectangle_boundary_points(x0, x1, y0, y1, spacing_of):
    """Points on the rectangle's perimeter. spacing_of(x, y) -> local spacing (callable or float)."""
    def side(p0, p1):
        p0 = np.asarray(p0, float)
        p1 = np.asarray(p1, float)
        length = float(np.hypot(*(p1 - p0)))
        if callable(spacing_of):
            # march with the local spacing
            s = [0.0]
            while True:
                p = p0 + (p1 - p0) * (s[-1] / length)
                step = float(spacing_of(p[0], p[1]))
                if s[-1] + 1.5 * step >= length:
                    break
                s.append(s[-1] + step)
            s = np.asarray(s)
        else:
            n = max(1, int(round(length / float(spacing_of))))
            s = np.arange(n) * (length / n)
        return p0[None, :] + (p1 - p0)[None, :] * (s / length)[:, None]

    return np.concatenate([
        side((x0, y0), (x1, y0)), side((x1, y0), (x1, y1)),
        side((x1, y1), (x0, y1)), side((x0, y1), (x0, y0)),
    ])


def delaunay_tri_mesh(points: np.ndarray, min_area: float):
    """Delaunay triangulation (scipy/Qhull) -> (node_xy, tri CCW int32); slivers with area below
    min_area (collinear hull points) are dropped, unused nodes are removed."""
    from scipy.spatial import Delaunay

    dl = Delaunay(points)
    tri = dl.simplices.astype(np.int64)
    a2 = signed_area2(points, tri)
    tri = tri[np.abs(a2) > 2.0 * min_area]
    used = np.zeros(points.shape[0], dtype=bool)
    used[tri.reshape(-1)] = True
    new_id = np.cumsum(used) - 1
    node_xy = np.ascontiguousarray(points[used])
    tri = new_id[tri]
    tri = orient_ccw(node_xy, tri).astype(np.int32)
    return node_xy, tri


def permute_mesh(tri, edge_cell, cell_edge, cell_perm, edge_perm):
    """Renumber cells and edges: new cell c = old cell cell_perm[c]; new edge e = old edge edge_perm[e].
    Slot order inside each cell and the L/R orientation of each edge are kept (SURVEY R-15)."""
    n = tri.shape[0]
    ne = edge_cell.shape[0]
    inv_c = np.empty(n, dtype=np.int64)
    inv_c[cell_perm] = np.arange(n)
    inv_e = np.empty(ne, dtype=np.int64)
    inv_e[edge_perm] = np.arange(ne)
    tri2 = tri[cell_perm]
    ce2 = inv_e[cell_edge[cell_perm]].astype(np.int32)
    ec_old = edge_cell[edge_perm]
    ec2 = ec_old.copy()
    ec2[:, 0] = inv_c[ec_old[:, 0]]
    inter = ec_old[:, 1] >= 0
    ec2[inter, 1] = inv_c[ec_old[inter, 1]]
    return tri2, ec2.astype(np.int32), ce2
