// Device-resident data layout of the shallow-water step.
//
// Everything that is gathered through an index (cell state by edge->cell, edge geometry and edge fluxes by
// cell->edge) is a 32-byte, 32-byte-aligned record = exactly one DRAM/L2 sector, moved by one 256-bit
// LDG/STG.  Arrays that are only ever streamed by their own index (area, 1/area, g/k^2, theta) are plain SoA.
#pragma once
#include <cstdint>

namespace swe {

struct __align__(32) CellRec {   // state U = (h, q_x, q_y) + cell-mean bed z_B (R-13)
  double h, qx, qy, z;
};

struct __align__(32) EdgeGeom {  // section 4.1: unit normal from L to R, edge length, the two cells
  double nx, ny, len;
  int32_t L, R;                  // R < 0: boundary code (include/swe.h)
};

struct __align__(32) EdgeFlux {  // S1 outputs: F1 mass, F3 tangential momentum, G_K = F2 - 1/2 g hs_K^2
  double F1, F3, GL, GR;
};

// ---- fused patch step: the mesh is cut into patches of consecutive (Morton-ordered) cells;
// one thread block advances one patch by a whole time step out of shared memory.
//   local cells : [0, n_own) the patch's own cells, then ring 1 (cells sharing an edge with an own cell), then
//                 ring 2 (cells sharing an edge with a ring-1 cell; needed because the limiter factor theta of a
//                 ring-1 cell depends on all three of its edges)
//   local edges : [0, n_eown) every edge of an own cell, then [n_eown, n_eown + n_er1) the other edges of ring 1
struct __align__(16) PatchHeader {
  int32_t cell0, n_own, n_r1, n_r2;
  int32_t n_eown, n_er1;
  int32_t halo_off;              // first entry of this patch in halo_ids[] / halo_area[]  (n_r1 + n_r2 entries)
  int32_t edge_off;              // first record of this patch in pedge[]
  int32_t pce_off;               // first record of this patch in pce[]  (n_own + n_r1 records)
  int32_t n_string_edges;        // boundary-string edges among the local edges (such a patch is never skipped)
  int32_t nbr_off, n_nbr;        // the patches that own this patch's ring-1 / ring-2 cells: entries of patch_nbr[]
};

struct __align__(32) PatchEdge { // geometry of section 4.1 + the two cells in patch-local numbering
  double nx, ny, len;
  uint16_t L, R;                 // R == 0xFFFF: boundary edge
  int32_t aux;                   // boundary: -1 wall, -2 transmissive, <= -3: -3 - (position in string_edges[])
};

// pce[] record = uint4 {slot0, slot1, slot2, unused}; slot = edge (bits 0-14) | isL (bit 15) | neighbour cell (bits 16-31)
constexpr uint32_t kPceNoNeighbour = 0xFFFFu;

struct BoundaryString {          // one boundary string (R-11, R-12); lives in device memory
  int32_t type;                  // SWE_BC_*
  int32_t n_edges;               // members
  int32_t first;                 // offset of its members in string_edges[] (ascending caller edge id)
  int32_t pow2;                  // n_edges rounded up to a power of two (shape of the pairwise tree)
  int32_t scratch;               // offset of its pow2 doubles in string_scratch[]
  int32_t n_params;
  const double *params;          // INFLOW_Q: (t_k, Q_k) table; OUTFLOW_UNIFORM: (S_0)
  double sumL;                   // tree sum of the member lengths (constant)
  double Q, sumK;                // INFLOW_Q: values at t^n, written by k_step_control
  double S0;                     // OUTFLOW_UNIFORM
  double phi_in[5];              // INFLOW_Q: concentration of every scalar species in the entering water (R-19)
};

constexpr int kMaxSpecies = 5;   // "up to a maximum of 5"

struct Scalars {                 // passive scalars q_c = h phi_c (section 3.3, Eq. 8; R-19), SoA per species
  int n;                         // species in use (0: the module is off)
  double *qa[kMaxSpecies];       // [n_cells] state buffer a (the only one of the three-pass step)
  double *qb[kMaxSpecies];       // [n_cells] state buffer b (fused patch step)
  double *phi_up[kMaxSpecies];   // [n_edges] three-pass step: concentration on the upwind side of every edge
};

struct Morph {                   // morphodynamics (section 3.2 Eq. 3, section 4.3 Eq. 13-16; R-20); formula 0: fixed bed
  int formula;                   // 1 Grass-like alpha |u|^3, 2 MPM-like alpha (theta - theta_cr)^1.5 sqrt((s-1) g d_m^3)
  double alpha, theta_cr;
  double shields_den;            // g (s-1) d_m: theta = (g/k_st^2) |u|^2 / (h^(1/3) * shields_den)
  double Gm;                     // alpha sqrt((s-1) g d_m^3)
  double inv1mp;                 // 1 / (1 - p)
  double2 *cell;                 // [n_cells] MPM-like law: (g / k_st^2, cbrt(h)) of the CURRENT state -- the cube root
                                 // k_cell_update takes for the friction term anyway, kept for the next step's edges
                                 // (0 where the cell is dry or has no friction law: not used there)
  double *qB;                    // [n_edges] normal sediment flux q_Bij of the step in flight
};

struct Control {                 // device-side step-loop state: nothing of it is read by the host per step
  double t, dt, t_end, cfl, dt_max, g, h_dry;
  double dt_last, vol_in, vol_out, vol_clipped;
  unsigned long long rate_bits;  // bit pattern of max_i max_j lambda_ij/rho_ij of the CURRENT state (>= 0)
  long long steps_left;          // < 0: unlimited
  long long steps_done;
  int32_t active;                // 1: the kernels of this step do work; 0: they return at once
  int32_t pending;               // 1: volume bookkeeping of the previous step not yet done
  int32_t flags;                 // SWE_FLAG_*
  int32_t n_strings;
  int32_t cur;                   // index of the state buffer that holds (or will hold, once the enqueued steps have
                                 // run) the newest state; the fused patch step ping-pongs, the three-pass step stays 0
  int32_t src;                   // state buffer the step in flight reads (it writes src ^ ping_pong)
  int32_t ping_pong;             // 1: fused patch step (two state buffers); 0: in-place three-pass step
  int32_t pad2_;
  unsigned long long patches_skipped;   // fused patch step: blocks that found their whole patch dry, since swe_create
  // swe_step_info reductions (k_info)
  double vol;
  long long n_wet;
  int32_t nonfinite;
  int32_t pad_;
};

}  // namespace swe
