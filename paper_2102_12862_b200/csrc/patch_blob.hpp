// Host-side construction of the patch blobs of the fused step (once per mesh, inside swe_create; the sizing pass
// of swe_workspace_bytes runs the same code with `emit = false`).  Pure C++ (no CUDA call).
// Input: the mesh in INTERNAL numbering (cells along the Morton curve, so that a range of consecutive cells is a
// compact blob of the plane).  Output: one fixed-stride blob per patch as laid out by blob_layout() in swe_types.h.
//
// Local numbering inside a patch (section 5b of DESIGN.md):
//   cells : [0, n_own) own, then ring 1 (cells sharing an edge with an own cell), then ring 2 (cells sharing an
//           edge with a ring-1 cell; the limiter factor theta of a ring-1 donor depends on all three of its edges, R-8b)
//   edges : [0, n_eown) every edge of an own cell, then [n_eown, n_eown + n_er1) the other edges of ring-1 cells
#pragma once
#include <algorithm>
#include <cstdint>
#include <cstring>
#include <string>
#include <vector>

#include "swe_types.h"

namespace swe {

struct PatchBlobs {
  BlobLayout lay{};
  int64_t n_patches = 0;
  std::vector<unsigned char> bytes;      // n_patches * lay.stride (empty after a sizing pass)
  int max_loc = 0, max_e = 0, max_nbr = 0;
  int64_t sum_loc = 0, sum_e = 0, sum_nbr = 0;   // totals over patches: redundancy statistics
  int64_t n_unskippable = 0;             // patches with a boundary-string edge or more than kPflagSlots neighbours
};

struct PatchScratch {                    // what pass 1 finds for one patch (global ids in local order)
  std::vector<int32_t> ring, edges, nbr;
  int32_t n_own = 0, n_r1 = 0, n_r2 = 0, n_eown = 0;
};

// geom: EdgeGeom per internal edge (L, R internal cell ids; R < 0 boundary code); cell_edge4: 4 ints per cell
// (3 internal edge ids); string_pos[e] = position of boundary-string edge e in string_edges[], -1 otherwise.
inline bool build_blobs(int64_t nc, int64_t ne, const std::vector<EdgeGeom> &geom, const std::vector<int32_t> &cell_edge4,
                        const std::vector<double> &area, const std::vector<double> &inv_area, const std::vector<double> &gn2,
                        const std::vector<int32_t> &string_pos, int P, bool emit, PatchBlobs &pb, std::string &err, int rb = 8) {
  pb = PatchBlobs{};
  // rb: bytes of a real in the staged arrays; 4 = single precision: the fp64 values rounded once to fp32 (R-21)
  if (P < 32 || P > 1024) { err = "patch_cells must be in [32, 1024]"; return false; }
  const int64_t np = (nc + P - 1) / P;
  pb.n_patches = np;
  std::vector<int32_t> cstamp(nc, -1), cloc(nc, 0), estamp(ne, -1), eloc(ne, 0);

  // discovery of the rings / edges / neighbour patches of patch p
  // (stamp: a value no earlier call has used -- the two passes below visit every patch once each)
  auto discover = [&](int64_t p, int32_t stamp, PatchScratch &s) {
    const int32_t c0 = (int32_t)(p * P);
    s.n_own = (int32_t)std::min<int64_t>(P, nc - c0);
    s.ring.clear(); s.edges.clear(); s.nbr.clear();
    for (int32_t l = 0; l < s.n_own; ++l) { cstamp[c0 + l] = stamp; cloc[c0 + l] = l; }
    auto touch_edge = [&](int32_t e) {
      if (estamp[e] != stamp) { estamp[e] = stamp; eloc[e] = (int32_t)s.edges.size(); s.edges.push_back(e); }
    };
    auto touch_cell = [&](int32_t c) {
      if (c >= 0 && cstamp[c] != stamp) { cstamp[c] = stamp; cloc[c] = s.n_own + (int32_t)s.ring.size(); s.ring.push_back(c); }
    };
    for (int32_t l = 0; l < s.n_own; ++l)
      for (int k = 0; k < 3; ++k) touch_edge(cell_edge4[4 * (size_t)(c0 + l) + k]);
    s.n_eown = (int32_t)s.edges.size();
    for (int32_t j = 0; j < s.n_eown; ++j) { touch_cell(geom[s.edges[j]].L); touch_cell(geom[s.edges[j]].R); }
    s.n_r1 = (int32_t)s.ring.size();
    for (int32_t j = 0; j < s.n_r1; ++j)
      for (int k = 0; k < 3; ++k) touch_edge(cell_edge4[4 * (size_t)s.ring[j] + k]);
    const int32_t n_e = (int32_t)s.edges.size();
    for (int32_t j = s.n_eown; j < n_e; ++j) { touch_cell(geom[s.edges[j]].L); touch_cell(geom[s.edges[j]].R); }
    s.n_r2 = (int32_t)s.ring.size() - s.n_r1;
    for (int32_t c : s.ring) s.nbr.push_back(c / P);
    std::sort(s.nbr.begin(), s.nbr.end());
    s.nbr.erase(std::unique(s.nbr.begin(), s.nbr.end()), s.nbr.end());
  };

  // ---- pass 1: capacities (maxima over the patches) and the neighbour lists (kept: pass 2 needs the slot a patch
  // has in each neighbour's list, and "p is a neighbour of q" is symmetric: distance-2 adjacency of cells)
  int cap_halo = 1, cap_r1 = 1, cap_e = 1, cap_eown = 1, cap_nbr = 1;
  std::vector<int64_t> nbr_off(np + 1, 0);
  std::vector<int32_t> nbr_all;
  PatchScratch s;
  for (int64_t p = 0; p < np; ++p) {
    discover(p, (int32_t)p, s);
    const int32_t n_e = (int32_t)s.edges.size(), n_loc = s.n_own + s.n_r1 + s.n_r2;
    if (n_loc >= 0xFFFF || n_e >= 0x8000) { err = "patch too large for 16-bit local indices"; return false; }
    cap_halo = std::max(cap_halo, s.n_r1 + s.n_r2); cap_r1 = std::max(cap_r1, s.n_r1);
    cap_e = std::max(cap_e, n_e); cap_eown = std::max(cap_eown, s.n_eown);
    cap_nbr = std::max<int>(cap_nbr, (int)s.nbr.size());
    pb.max_loc = std::max(pb.max_loc, n_loc); pb.max_e = std::max(pb.max_e, n_e);
    pb.sum_loc += n_loc; pb.sum_e += n_e; pb.sum_nbr += (int64_t)s.nbr.size();
    nbr_all.insert(nbr_all.end(), s.nbr.begin(), s.nbr.end());
    nbr_off[p + 1] = (int64_t)nbr_all.size();
  }
  pb.max_nbr = cap_nbr;
  // round the capacities up a little so that the SoA arrays of the staged part stay 16-byte aligned
  cap_halo = blob_align(cap_halo, 4); cap_r1 = blob_align(cap_r1, 2); cap_e = blob_align(cap_e, 4); cap_eown = blob_align(cap_eown, 2);
  cap_nbr = blob_align(cap_nbr, 4);
  pb.lay = blob_layout(P, cap_nbr, cap_halo, cap_r1, cap_e, cap_eown, rb);
  if ((int64_t)pb.lay.stride * np > (int64_t)1 << 40) { err = "patch blobs exceed 1 TB"; return false; }
  if (!emit) return true;                       // sizing pass (swe_workspace_bytes)

  // ---- pass 2: the blobs
  const BlobLayout &L = pb.lay;
  pb.bytes.assign((size_t)L.stride * (size_t)np, 0);
  // own_mask[c]: bit j is set when cell c (owned by patch p = c / P) is a halo cell of the j-th neighbour patch of p
  // (j < 32): what p must look at to tell that neighbour "none of MY cells YOU read holds water" (the flag bytes)
  std::vector<uint32_t> own_mask(nc, 0u);
  for (int64_t p = 0; p < np; ++p) {
    discover(p, (int32_t)(np + p), s);
    unsigned char *B = pb.bytes.data() + (size_t)L.stride * (size_t)p;
    const int32_t c0 = (int32_t)(p * P);
    const int32_t n_e = (int32_t)s.edges.size();
    int32_t n_string = 0;
    for (int32_t j = 0; j < n_e; ++j) n_string += geom[s.edges[j]].R <= -3;
    BlobHeader h{};
    h.n_own = s.n_own; h.n_r1 = s.n_r1; h.n_r2 = s.n_r2; h.n_eown = s.n_eown; h.n_er1 = n_e - s.n_eown;
    h.n_string_edges = n_string; h.n_nbr = (int32_t)s.nbr.size();
    std::memcpy(B, &h, sizeof h);
    std::memcpy(B + L.off_stage + L.s_hdr, &h, sizeof h);
    if (n_string > 0 || h.n_nbr > kPflagSlots) ++pb.n_unskippable;
    int32_t *nbr = (int32_t *)(B + L.off_nbr), *nbr_slot = (int32_t *)(B + L.off_nbr_slot);
    for (int32_t j = 0; j < L.cap_nbr; ++j) { nbr[j] = -1; nbr_slot[j] = -1; }
    for (int32_t j = 0; j < h.n_nbr; ++j) {
      const int32_t q = s.nbr[j];
      nbr[j] = q;
      // my slot in q's (ascending) list; only the first kPflagSlots entries of a list have a flag byte
      const int32_t *qb = nbr_all.data() + nbr_off[q], *qe = nbr_all.data() + nbr_off[q + 1];
      const int32_t *it = std::lower_bound(qb, qe, (int32_t)p);
      const int32_t slot = (it != qe && *it == (int32_t)p) ? (int32_t)(it - qb) : -1;
      nbr_slot[j] = (slot >= 0 && slot < kPflagSlots) ? slot : -1;
    }
    std::memcpy(B + L.off_stage + L.s_nbr, nbr, 4 * (size_t)L.cap_nbr);
    std::memcpy(B + L.off_stage + L.s_nbr_slot, nbr_slot, 4 * (size_t)L.cap_nbr);
    int32_t *halo_ids = (int32_t *)(B + L.off_halo_ids);
    for (int32_t j = 0; j < L.cap_halo; ++j) halo_ids[j] = j < (int32_t)s.ring.size() ? s.ring[j] : -1;
    for (int32_t c : s.ring) {                    // this patch p reads cell c of patch o: bit (position of p in o's list)
      const int32_t o = c / P;
      const int32_t *ob = nbr_all.data() + nbr_off[o], *oe = nbr_all.data() + nbr_off[o + 1];
      const int32_t *it = std::lower_bound(ob, oe, (int32_t)p);
      if (it == oe || *it != (int32_t)p) { err = "patch neighbourhood is not symmetric"; return false; }
      const int32_t j = (int32_t)(it - ob);
      if (j < 32) own_mask[c] |= 1u << j;
    }
    unsigned char *S = B + L.off_stage;
    auto put = [&](int32_t off, int32_t idx, double v) {          // element idx of the staged real array at offset off
      if (rb == 4) ((float *)(S + off))[idx] = (float)v; else ((double *)(S + off))[idx] = v;
    };
    for (int32_t j = 0; j < s.n_r1; ++j) put(L.s_halo_area, j, area[s.ring[j]]);
    uint32_t *pce = (uint32_t *)(S + L.s_pce);
    for (int32_t l = 0; l < s.n_own + s.n_r1; ++l) {
      const int32_t c = l < s.n_own ? c0 + l : s.ring[l - s.n_own];
      for (int k = 0; k < 3; ++k) {
        const int32_t e = cell_edge4[4 * (size_t)c + k];
        const EdgeGeom &g = geom[e];
        const bool isL = (g.L == c);
        const int32_t other = isL ? g.R : g.L;
        const uint32_t nb = other >= 0 ? (uint32_t)cloc[other] : kPceNoNeighbour;
        pce[4 * l + k] = (uint32_t)eloc[e] | (isL ? 0x8000u : 0u) | (nb << 16);
      }
      pce[4 * l + 3] = 0u;
    }
    uint32_t *lr = (uint32_t *)(S + L.s_lr);
    int32_t *aux = (int32_t *)(S + L.s_aux);
    for (int32_t j = 0; j < n_e; ++j) {
      const EdgeGeom &g = geom[s.edges[j]];
      put(L.s_nx, j, g.nx); put(L.s_ny, j, g.ny); put(L.s_len, j, g.len);
      const uint32_t Ll = (uint32_t)cloc[g.L];
      if (g.R >= 0) { lr[j] = Ll | ((uint32_t)cloc[g.R] << 16); aux[j] = 0; }
      else { lr[j] = Ll | (0xFFFFu << 16); aux[j] = (g.R <= -3) ? -3 - string_pos[s.edges[j]] : g.R; }
    }
    for (int32_t l = 0; l < s.n_own; ++l) {
      put(L.s_area, l, area[c0 + l]); put(L.s_gn2, l, gn2[c0 + l]);
      if (rb == 4) put(L.s_inv_area, l, inv_area[c0 + l]);
    }
  }
  // the fourth word of an own cell's slot record: its mask (complete only now that every patch has been visited)
  for (int64_t p = 0; p < np; ++p) {
    uint32_t *pce = (uint32_t *)(pb.bytes.data() + (size_t)L.stride * (size_t)p + L.off_stage + L.s_pce);
    const int32_t c0 = (int32_t)(p * P), n_own = (int32_t)std::min<int64_t>(P, nc - c0);
    for (int32_t l = 0; l < n_own; ++l) pce[4 * l + 3] = own_mask[c0 + l];
  }
  return true;
}

}  // namespace swe
