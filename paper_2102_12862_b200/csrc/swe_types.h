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
  // swe_step_info reductions (k_info)
  double vol;
  long long n_wet;
  int32_t nonfinite;
  int32_t pad_;
};

}  // namespace swe
