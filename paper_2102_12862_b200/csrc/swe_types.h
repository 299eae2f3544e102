// Device-resident data layout of the shallow-water step.
//
// Everything that is gathered through an index (cell state by edge->cell, edge geometry and edge fluxes by
// cell->edge) is a 32-byte, 32-byte-aligned record = exactly one DRAM/L2 sector, moved by one 256-bit
// LDG/STG.  Arrays that are only ever streamed by their own index (area, 1/area, g/k^2, theta) are plain SoA.
#pragma once
#include <cstddef>
#include <cstdint>

namespace swe {

// T = double (the default arithmetic) or float (single precision, swe_params.precision; R-21): a record
// is 32 bytes = one sector in fp64 and 16 bytes in fp32.
template <typename T> struct CellRecT;     // state U = (h, q_x, q_y) + cell-mean bed z_B (R-13)
template <> struct __align__(32) CellRecT<double> { double h, qx, qy, z; };
template <> struct __align__(16) CellRecT<float> { float h, qx, qy, z; };

template <typename T> struct EdgeGeomT;    // section 4.1: unit normal from L to R, edge length, the two cells
template <> struct __align__(32) EdgeGeomT<double> {
  double nx, ny, len;
  int32_t L, R;                  // R < 0: boundary code (include/swe.h)
};
template <> struct __align__(16) EdgeGeomT<float> {   // R lives in a separate int32 array (only the edge kernel reads it)
  float nx, ny, len;
  int32_t L;
};

template <typename T> struct EdgeFluxT;    // S1 outputs: F1 mass, F3 tangential momentum, G_K = F2 - 1/2 g hs_K^2
template <> struct __align__(32) EdgeFluxT<double> { double F1, F3, GL, GR; };
template <> struct __align__(16) EdgeFluxT<float> { float F1, F3, GL, GR; };

typedef CellRecT<double> CellRec;
typedef EdgeGeomT<double> EdgeGeom;
typedef EdgeFluxT<double> EdgeFlux;

// pce[] record = uint4 {slot0, slot1, slot2, unused}; slot = edge (bits 0-14) | isL (bit 15) | neighbour cell (bits 16-31)
constexpr uint32_t kPceNoNeighbour = 0xFFFFu;

// ---- patch blobs: everything a patch streams lives in ONE contiguous, fixed-stride block of
// device memory ("blob"), so that a thread block knows every address from blockIdx alone and pulls the part it
// computes from into shared memory with one bulk asynchronous copy (cp.async.bulk + mbarrier).  All offsets are in
// bytes from the start of the blob and are the same for every patch (capacities = maxima over the patches).
//   [0, off_stage)          "cold" part, read straight from global memory when needed:
//                             BlobHeader | nbr[cap_nbr] int32 | nbr_slot[cap_nbr] int32 | halo_ids[cap_halo] int32
//   [off_stage, off_stage + stage_bytes)   staged into shared memory by the bulk copy, SoA (bank-conflict-free):
//                             BlobHeader copy | nbr, nbr_slot copies | halo_area[cap_r1] | pce[cap_c1] uint4 | nx, ny, len [cap_e] double |
//                             lr[cap_e] uint32 (L | R << 16; R = 0xFFFF boundary) | aux[cap_e] int32 |
//                             area, gn2 [P] double  (1 / area is formed in the kernel: the same IEEE quotient)
struct BlobHeader {              // 32 bytes
  int32_t n_own, n_r1, n_r2, n_eown, n_er1, n_string_edges, n_nbr, pad_;
};

struct BlobLayout {
  int32_t P;                     // own cells per patch (= threads per block)
  int32_t cap_nbr, cap_halo, cap_r1, cap_c1, cap_loc, cap_e, cap_eown;
  int32_t off_nbr, off_nbr_slot, off_halo_ids, off_stage;
  // offsets RELATIVE TO off_stage (= offsets inside the staged copy in shared memory)
  int32_t s_hdr, s_nbr, s_nbr_slot, s_halo_area, s_pce, s_nx, s_ny, s_len, s_lr, s_aux, s_area, s_gn2, s_inv_area;
  int32_t rb;                    // bytes of a real in the staged arrays: 8, or 4 (single precision, R-21)
  int32_t stage_bytes;           // multiple of 16
  int32_t stride;                // bytes per blob, multiple of 128
};

// per patch and state buffer: 32 flag bytes {neighbour 0..29 | own | skippable}.  Own byte: 1 when every own cell of
// the patch is exactly (0, 0, 0) in that buffer.  Neighbour byte j: 1 when every cell of the j-th neighbour patch that
// is a halo cell of THIS patch is exactly (0, 0, 0) (the neighbour writes it: the fourth word of an own cell's slot
// record names the neighbours that read the cell).  Byte 31: 1 when the patch has no boundary-string edge and at most
// kPflagSlots neighbours -- constant.  All 32 bytes == 1  <=>  every local cell of the patch is dry and nothing can
// feed it: the block may skip the patch (section 5b).
constexpr int kPflagBytes = 32, kPflagSlots = 30, kPflagOwn = 30, kPflagSkippable = 31;

__host__ __device__ inline int32_t blob_align(int32_t x, int32_t a) { return (x + a - 1) / a * a; }

__host__ __device__ inline BlobLayout blob_layout(int P, int cap_nbr, int cap_halo, int cap_r1, int cap_e, int cap_eown, int rb = 8) {
  BlobLayout L;
  L.rb = rb;
  L.P = P; L.cap_nbr = cap_nbr; L.cap_halo = cap_halo; L.cap_r1 = cap_r1; L.cap_c1 = P + cap_r1; L.cap_loc = P + cap_halo;
  L.cap_e = cap_e; L.cap_eown = cap_eown;
  int32_t o = (int32_t)sizeof(BlobHeader);
  L.off_nbr = o; o += 4 * cap_nbr;
  L.off_nbr_slot = o; o += 4 * cap_nbr;
  L.off_halo_ids = o; o += 4 * cap_halo;
  L.off_stage = blob_align(o, 128);
  int32_t s = 0;
  L.s_hdr = s; s += (int32_t)sizeof(BlobHeader);
  L.s_nbr = s; s += 4 * cap_nbr;
  L.s_nbr_slot = s; s += 4 * cap_nbr;
  s = blob_align(s, 8);
  L.s_halo_area = s; s += rb * cap_r1;
  s = blob_align(s, 16);
  L.s_pce = s; s += 16 * L.cap_c1;
  L.s_nx = s; s += rb * cap_e;
  L.s_ny = s; s += rb * cap_e;
  L.s_len = s; s += rb * cap_e;
  L.s_lr = s; s += 4 * cap_e;
  L.s_aux = s; s += 4 * cap_e;
  s = blob_align(s, 8);
  L.s_area = s; s += rb * P;
  L.s_gn2 = s; s += rb * P;
  // single precision: 1 / abs(Omega) is the host's fp64 quotient rounded once (R-21), so it is staged; the fp64 kernel
  // forms the same IEEE quotient itself
  L.s_inv_area = s; s += rb == 4 ? 4 * P : 0;
  L.stage_bytes = blob_align(s, 16);
  L.stride = blob_align(L.off_stage + L.stage_bytes, 128);
  return L;
}

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

struct StepSlot {
  double t, dt_last, vol_in, vol_out;
  unsigned long long rate_bits;  // max rate of the state this slot describes
  long long steps_left, steps_done;
  int32_t src;                   // state buffer that holds this state
  int32_t flags;
  int32_t pending;               // 1: the step that produced this state wrote outflow terms not yet booked in vol_out
  int32_t pad_;
};

struct Control {                 // device-side step-loop state: nothing of it is read by the host per step
  // first 128-byte line: what the kernels of a step only read (every block of the fused patch step fetches active, src,
  // dt, g, h_dry from it when it starts)
  double t, dt, t_end, cfl, dt_max, g, h_dry;
  double dt_last, vol_in, vol_out;
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
  // second line: the words the blocks of a step update atomically -- kept off the line above, which every starting
  // block reads while the finishing ones send their atomics
  double vol_clipped;
  unsigned long long rate_bits;  // bit pattern of max_i max_j lambda_ij/rho_ij of the CURRENT state (>= 0)
  unsigned long long patches_skipped;   // fused patch step: blocks that found their whole patch dry, since swe_create
  unsigned long long pad_line_[13];
  // swe_step_info reductions (k_info)
  double vol;
  long long n_wet;
  int32_t nonfinite;
  int32_t pad_;
  // fused patch step without a control kernel: step number n reads slot[n % 4] -- every block
  // derives dt, t and the stop rules from it by itself --, block 0 writes slot[(n + 1) % 4], the rate of the new state
  // is collected in slot[(n + 1) % 4].rate_bits and slot[(n + 2) % 4].rate_bits is cleared for the step after.
  // swe_step copies the classic fields above into a slot when it starts and back when it ends.
  StepSlot slot[4];
};

static_assert(offsetof(Control, vol_clipped) == 128 && offsetof(Control, vol) == 256, "Control: one line read, one line of atomics");

}  // namespace swe
