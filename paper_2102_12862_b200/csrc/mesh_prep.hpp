// Host-side mesh preprocessing for swe_create (once per mesh, not on the timed path):
// validation, edge tables, geometry of section 4.1, Morton renumbering of cells and edges.
// Pure C++ (no CUDA).  Compiled with -ffp-contract=off: the geometry is part of the arithmetic contract (R-14).
#pragma once
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <limits>
#include <numeric>
#include <string>
#include <vector>

#include "swe_types.h"

namespace swe {

struct HostMesh {
  int64_t nc = 0, ne = 0, nn = 0;
  // caller numbering
  std::vector<int32_t> edge_cell;   // [ne][2]
  std::vector<int32_t> cell_edge;   // [nc][3]
  std::vector<double> area, nx, ny, len;
  // internal numbering
  std::vector<int32_t> cell_perm;   // [nc] new -> caller
  std::vector<int32_t> edge_perm;   // [ne] new -> caller
  std::vector<int32_t> cell_new;    // [nc] caller -> new
  std::vector<int32_t> edge_new;    // [ne] caller -> new
};

// Builds edge_cell / cell_edge from CCW triangles: edges numbered by sorted (min node, max node); L is the
// cell that comes first; every boundary edge is a wall.
inline bool build_tables(int64_t nc, int64_t nn, const int32_t *tri, HostMesh &m, std::string &err) {
  struct Half { uint64_t key; int32_t slot; };
  std::vector<Half> hs((size_t)3 * nc);
  for (int64_t i = 0; i < nc; ++i)
    for (int k = 0; k < 3; ++k) {
      const int64_t a = tri[3 * i + k], b = tri[3 * i + (k + 1) % 3];
      if (a < 0 || a >= nn || b < 0 || b >= nn || a == b) { err = "triangle " + std::to_string(i) + " has an invalid node id"; return false; }
      hs[3 * i + k] = {(uint64_t)std::min(a, b) * (uint64_t)nn + (uint64_t)std::max(a, b), (int32_t)(3 * i + k)};
    }
  std::stable_sort(hs.begin(), hs.end(), [](const Half &x, const Half &y) { return x.key < y.key; });
  m.cell_edge.assign((size_t)3 * nc, -1);
  m.edge_cell.clear();
  size_t p = 0;
  while (p < hs.size()) {
    size_t q = p + 1;
    while (q < hs.size() && hs[q].key == hs[p].key) ++q;
    if (q - p > 2) { err = "non-manifold mesh: an edge is shared by more than two cells"; return false; }
    const int32_t e = (int32_t)(m.edge_cell.size() / 2);
    m.edge_cell.push_back(hs[p].slot / 3);
    m.edge_cell.push_back(q - p == 2 ? hs[p + 1].slot / 3 : -1);
    for (size_t r = p; r < q; ++r) m.cell_edge[hs[r].slot] = e;
    p = q;
  }
  m.ne = (int64_t)m.edge_cell.size() / 2;
  return true;
}

// Validation + geometry.  Triangle (p0,p1,p2) CCW: |Omega| = 1/2 [(x1-x0)(y2-y0) - (x2-x0)(y1-y0)] > 0; slot k is
// the edge p_k -> p_{k+1}; with d = p_{k+1} - p_k: l = sqrt(dx^2+dy^2), outward unit normal (dy/l, -dx/l).  An
// edge stores the numbers of its L cell's slot, so that n points from L to R ("toward the cell Omega_j").
inline bool validate_and_measure(int64_t nc, int64_t nn, const double *xy, const int32_t *tri, HostMesh &m,
                                 std::string &err) {
  const int64_t ne = m.ne;
  m.area.assign(nc, 0.0);
  m.nx.assign(ne, 0.0); m.ny.assign(ne, 0.0); m.len.assign(ne, 0.0);
  std::vector<uint8_t> seenL(ne, 0), seenR(ne, 0);
  std::vector<int32_t> na(ne, -1), nb(ne, -1);   // node pair of the edge as seen from L
  for (int64_t e = 0; e < ne; ++e) {
    const int32_t L = m.edge_cell[2 * e], R = m.edge_cell[2 * e + 1];
    if (L < 0 || L >= nc || R >= nc || R == L) { err = "edge " + std::to_string(e) + ": edge_cell out of range"; return false; }
  }
  for (int pass = 0; pass < 2; ++pass)       // pass 0: L slots (geometry); pass 1: R slots (conformity)
    for (int64_t i = 0; i < nc; ++i) {
      const int32_t *t = tri + 3 * i;
      if (pass == 0) {
        for (int k = 0; k < 3; ++k)
          if (t[k] < 0 || t[k] >= nn) { err = "cell " + std::to_string(i) + ": node id out of range"; return false; }
        const double x0 = xy[2 * t[0]], y0 = xy[2 * t[0] + 1];
        const double x1 = xy[2 * t[1]], y1 = xy[2 * t[1] + 1];
        const double x2 = xy[2 * t[2]], y2 = xy[2 * t[2] + 1];
        const double A = 0.5 * ((x1 - x0) * (y2 - y0) - (x2 - x0) * (y1 - y0));
        if (!(A > 0.0) || !std::isfinite(A)) { err = "cell " + std::to_string(i) + " is not counter-clockwise / has no area"; return false; }
        m.area[i] = A;
      }
      for (int k = 0; k < 3; ++k) {
        const int32_t e = m.cell_edge[3 * i + k];
        if (e < 0 || e >= ne) { err = "cell " + std::to_string(i) + ": cell_edge out of range"; return false; }
        const int32_t a = t[k], b = t[(k + 1) % 3];
        const bool isL = (m.edge_cell[2 * e] == i);
        if (pass == 0 && isL) {
          if (seenL[e]) { err = "edge " + std::to_string(e) + " is referenced twice by its L cell"; return false; }
          seenL[e] = 1; na[e] = a; nb[e] = b;
          const double dx = xy[2 * b] - xy[2 * a], dy = xy[2 * b + 1] - xy[2 * a + 1];
          const double l = std::sqrt(dx * dx + dy * dy);
          m.len[e] = l; m.nx[e] = dy / l; m.ny[e] = -dx / l;
        } else if (pass == 1 && !isL) {
          if (m.edge_cell[2 * e + 1] != i) { err = "edge_cell / cell_edge tables are inconsistent at cell " + std::to_string(i); return false; }
          if (seenR[e]) { err = "edge " + std::to_string(e) + " is referenced twice by its R cell"; return false; }
          seenR[e] = 1;
          if (!(na[e] == b && nb[e] == a)) { err = "edge " + std::to_string(e) + ": L and R cells do not share its two nodes (non-conforming)"; return false; }
        }
      }
    }
  for (int64_t e = 0; e < ne; ++e) {
    if (!seenL[e]) { err = "edge " + std::to_string(e) + " is not a slot of its L cell"; return false; }
    if ((m.edge_cell[2 * e + 1] >= 0) != (seenR[e] != 0)) { err = "edge " + std::to_string(e) + " is not a slot of its R cell"; return false; }
  }
  return true;
}

inline uint64_t spread_bits_21(uint64_t v) {   // 21 bits -> every third... here every second bit (2-D Morton)
  v &= 0x1fffffull;
  v = (v | (v << 16)) & 0x0000ffff0000ffffull;
  v = (v | (v << 8)) & 0x00ff00ff00ff00ffull;
  v = (v | (v << 4)) & 0x0f0f0f0f0f0f0f0full;
  v = (v | (v << 2)) & 0x3333333333333333ull;
  v = (v | (v << 1)) & 0x5555555555555555ull;
  return v;
}

// mode 1: cells along the Morton (Z-order) curve of their centroids; mode 2: reverse Cuthill-McKee (below); edges in
// the order of the lower new cell id they touch (ties: the other cell).  Slot order inside a cell and L/R of an edge are untouched (R-15).
inline void renumber(int mode, int64_t nc, const double *xy, const int32_t *tri, HostMesh &m) {
  const int64_t ne = m.ne;
  m.cell_perm.resize(nc); m.cell_new.resize(nc); m.edge_perm.resize(ne); m.edge_new.resize(ne);
  std::iota(m.cell_perm.begin(), m.cell_perm.end(), 0);
  std::iota(m.edge_perm.begin(), m.edge_perm.end(), 0);
  if (mode != 0 && nc > 0) {
    double xmin = std::numeric_limits<double>::infinity(), xmax = -xmin, ymin = xmin, ymax = -xmin;
    std::vector<double> cx(nc), cy(nc);
    for (int64_t i = 0; i < nc; ++i) {
      const int32_t *t = tri + 3 * i;
      cx[i] = (xy[2 * t[0]] + xy[2 * t[1]] + xy[2 * t[2]]) / 3.0;
      cy[i] = (xy[2 * t[0] + 1] + xy[2 * t[1] + 1] + xy[2 * t[2] + 1]) / 3.0;
      xmin = std::min(xmin, cx[i]); xmax = std::max(xmax, cx[i]);
      ymin = std::min(ymin, cy[i]); ymax = std::max(ymax, cy[i]);
    }
    const double span = std::max(std::max(xmax - xmin, ymax - ymin), 1e-300);
    const double scale = 2097151.0 / span;      // one scale for both axes: square Z-curve cells
    std::vector<std::pair<uint64_t, int32_t>> keyed(nc);
    for (int64_t i = 0; i < nc; ++i) {
      const uint64_t ix = (uint64_t)((cx[i] - xmin) * scale), iy = (uint64_t)((cy[i] - ymin) * scale);
      keyed[i] = {spread_bits_21(ix) | (spread_bits_21(iy) << 1), (int32_t)i};
    }
    std::sort(keyed.begin(), keyed.end());
    for (int64_t i = 0; i < nc; ++i) m.cell_perm[i] = keyed[i].second;
  }
  if (mode == 2 && nc > 0) {
    // Reverse Cuthill-McKee on the cell adjacency graph (degree <= 3): breadth-first levels from the cell with the
    // lowest Morton key, neighbours visited in ascending (degree, Morton rank), the whole order reversed.
    std::vector<int32_t> rank(nc);                       // Morton rank of every caller cell (computed above)
    for (int64_t i = 0; i < nc; ++i) rank[m.cell_perm[i]] = (int32_t)i;
    std::vector<int32_t> morton = m.cell_perm, order;
    order.reserve(nc);
    std::vector<uint8_t> seen(nc, 0);
    auto degree = [&](int32_t c) {
      int d = 0;
      for (int k = 0; k < 3; ++k) d += m.edge_cell[2 * m.cell_edge[3 * c + k] + 1] >= 0;
      return d;
    };
    size_t next_seed = 0;
    while ((int64_t)order.size() < nc) {
      while (seen[morton[next_seed]]) ++next_seed;
      size_t head = order.size();
      order.push_back(morton[next_seed]); seen[morton[next_seed]] = 1;
      while (head < order.size()) {
        const int32_t c = order[head++];
        int32_t nb[3]; int n = 0;
        for (int k = 0; k < 3; ++k) {
          const int32_t e = m.cell_edge[3 * c + k];
          const int32_t L = m.edge_cell[2 * e], R = m.edge_cell[2 * e + 1];
          const int32_t o = (L == c) ? R : L;
          if (o >= 0 && !seen[o]) { seen[o] = 1; nb[n++] = o; }
        }
        std::sort(nb, nb + n, [&](int32_t a, int32_t b) {
          const int da = degree(a), db = degree(b);
          return da != db ? da < db : rank[a] < rank[b];
        });
        for (int k = 0; k < n; ++k) order.push_back(nb[k]);
      }
    }
    for (int64_t i = 0; i < nc; ++i) m.cell_perm[i] = order[nc - 1 - i];
  }
  for (int64_t i = 0; i < nc; ++i) m.cell_new[m.cell_perm[i]] = (int32_t)i;
  if (mode != 0 && ne > 0) {
    std::vector<std::pair<uint64_t, int32_t>> keyed(ne);
    for (int64_t e = 0; e < ne; ++e) {
      const uint64_t a = (uint64_t)m.cell_new[m.edge_cell[2 * e]];
      const int32_t R = m.edge_cell[2 * e + 1];
      const uint64_t b = R >= 0 ? (uint64_t)m.cell_new[R] : a;
      keyed[e] = {(std::min(a, b) << 32) | std::max(a, b), (int32_t)e};
    }
    std::sort(keyed.begin(), keyed.end());
    for (int64_t e = 0; e < ne; ++e) m.edge_perm[e] = keyed[e].second;
  }
  for (int64_t e = 0; e < ne; ++e) m.edge_new[m.edge_perm[e]] = (int32_t)e;
}

}  // namespace swe
