// Host-side construction of the patch tables of the fused step (once per mesh, inside swe_create).
// Pure C++ (no CUDA).  Input: the mesh in INTERNAL numbering (cells along the Morton curve, so that a range of
// consecutive cells is a compact blob), output: per patch the local cell / edge lists described in swe_types.h.
#pragma once
#include <algorithm>
#include <cstdint>
#include <string>
#include <vector>

#include "swe_types.h"

namespace swe {

struct PatchTables {
  int patch_cells = 0;
  std::vector<PatchHeader> hdr;
  std::vector<int32_t> halo_ids;    // global (internal) cell id of every ring-1 / ring-2 cell, patch after patch
  std::vector<double> halo_area;    // |Omega| of the same cells (used for ring 1 only)
  std::vector<PatchEdge> pedge;
  std::vector<uint32_t> pce;        // 4 words per record
  std::vector<int32_t> patch_nbr;   // ids of the patches owning each patch's halo cells (distinct, ascending)
  int max_loc = 0, max_c1 = 0, max_e = 0, max_eown = 0;   // maxima over patches: shared-memory carving
  int64_t sum_loc = 0, sum_e = 0;   // totals over patches: redundancy statistics
};

// geom: EdgeGeom per internal edge (L, R internal cell ids; R < 0 boundary code); cell_edge: 4 ints per cell
// (3 internal edge ids); string_pos[e] = position of boundary-string edge e in string_edges[], -1 otherwise.
inline bool build_patches(int64_t nc, int64_t ne, const std::vector<EdgeGeom> &geom, const std::vector<int32_t> &cell_edge4,
                          const std::vector<double> &area, const std::vector<int32_t> &string_pos, int patch_cells,
                          PatchTables &pt, std::string &err) {
  pt = PatchTables{};
  pt.patch_cells = patch_cells;
  const int64_t np = (nc + patch_cells - 1) / patch_cells;
  pt.hdr.reserve(np);
  std::vector<int32_t> cstamp(nc, -1), cloc(nc, 0), estamp(ne, -1), eloc(ne, 0);
  std::vector<int32_t> ring, edges;      // scratch: global ids in local order (halo cells; local edges)
  for (int64_t p = 0; p < np; ++p) {
    const int32_t c0 = (int32_t)(p * patch_cells);
    const int32_t n_own = (int32_t)std::min<int64_t>(patch_cells, nc - c0);
    ring.clear(); edges.clear();
    for (int32_t l = 0; l < n_own; ++l) { cstamp[c0 + l] = (int32_t)p; cloc[c0 + l] = l; }
    auto touch_edge = [&](int32_t e) {
      if (estamp[e] != (int32_t)p) { estamp[e] = (int32_t)p; eloc[e] = (int32_t)edges.size(); edges.push_back(e); }
    };
    auto touch_cell = [&](int32_t c) {
      if (c >= 0 && cstamp[c] != (int32_t)p) { cstamp[c] = (int32_t)p; cloc[c] = n_own + (int32_t)ring.size(); ring.push_back(c); }
    };
    for (int32_t l = 0; l < n_own; ++l)
      for (int k = 0; k < 3; ++k) touch_edge(cell_edge4[4 * (size_t)(c0 + l) + k]);
    const int32_t n_eown = (int32_t)edges.size();
    for (int32_t j = 0; j < n_eown; ++j) { touch_cell(geom[edges[j]].L); touch_cell(geom[edges[j]].R); }
    const int32_t n_r1 = (int32_t)ring.size();
    for (int32_t j = 0; j < n_r1; ++j)
      for (int k = 0; k < 3; ++k) touch_edge(cell_edge4[4 * (size_t)ring[j] + k]);
    const int32_t n_e = (int32_t)edges.size();
    for (int32_t j = n_eown; j < n_e; ++j) { touch_cell(geom[edges[j]].L); touch_cell(geom[edges[j]].R); }
    const int32_t n_r2 = (int32_t)ring.size() - n_r1;
    const int32_t n_loc = n_own + n_r1 + n_r2;
    if (n_loc >= 0xFFFF || n_e >= 0x8000) { err = "patch too large for 16-bit local indices"; return false; }

    PatchHeader h{};
    h.cell0 = c0; h.n_own = n_own; h.n_r1 = n_r1; h.n_r2 = n_r2; h.n_eown = n_eown; h.n_er1 = n_e - n_eown;
    h.halo_off = (int32_t)pt.halo_ids.size(); h.edge_off = (int32_t)pt.pedge.size(); h.pce_off = (int32_t)(pt.pce.size() / 4);
    if (pt.pedge.size() + (size_t)n_e > 0x7fffffffull) { err = "patch edge table exceeds 2^31 records"; return false; }
    pt.hdr.push_back(h);
    for (int32_t c : ring) { pt.halo_ids.push_back(c); pt.halo_area.push_back(area[c]); }
    {
      std::vector<int32_t> nb;
      for (int32_t c : ring) nb.push_back(c / patch_cells);
      std::sort(nb.begin(), nb.end());
      nb.erase(std::unique(nb.begin(), nb.end()), nb.end());
      pt.hdr.back().nbr_off = (int32_t)pt.patch_nbr.size();
      pt.hdr.back().n_nbr = (int32_t)nb.size();
      pt.patch_nbr.insert(pt.patch_nbr.end(), nb.begin(), nb.end());
    }
    int32_t n_string = 0;
    for (int32_t j = 0; j < n_e; ++j) n_string += geom[edges[j]].R <= -3;
    pt.hdr.back().n_string_edges = n_string;
    for (int32_t j = 0; j < n_e; ++j) {
      const EdgeGeom &g = geom[edges[j]];
      PatchEdge pe{};
      pe.nx = g.nx; pe.ny = g.ny; pe.len = g.len;
      pe.L = (uint16_t)cloc[g.L];
      if (g.R >= 0) { pe.R = (uint16_t)cloc[g.R]; pe.aux = 0; }
      else {
        pe.R = 0xFFFF;
        pe.aux = (g.R <= -3) ? -3 - string_pos[edges[j]] : g.R;
      }
      pt.pedge.push_back(pe);
    }
    for (int32_t l = 0; l < n_own + n_r1; ++l) {
      const int32_t c = l < n_own ? c0 + l : ring[l - n_own];
      for (int k = 0; k < 3; ++k) {
        const int32_t e = cell_edge4[4 * (size_t)c + k];
        const EdgeGeom &g = geom[e];
        const bool isL = (g.L == c);
        const int32_t other = isL ? g.R : g.L;
        const uint32_t nb = other >= 0 ? (uint32_t)cloc[other] : kPceNoNeighbour;
        pt.pce.push_back((uint32_t)eloc[e] | (isL ? 0x8000u : 0u) | (nb << 16));
      }
      pt.pce.push_back(0u);
    }
    pt.max_loc = std::max(pt.max_loc, n_loc); pt.max_c1 = std::max(pt.max_c1, n_own + n_r1);
    pt.max_e = std::max(pt.max_e, n_e); pt.max_eown = std::max(pt.max_eown, n_eown);
    pt.sum_loc += n_loc; pt.sum_e += n_e;
  }
  return true;
}

}  // namespace swe
