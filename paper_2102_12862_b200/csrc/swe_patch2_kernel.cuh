// Fused patch step (sm_100a), second design: one thread block advances one patch of P consecutive (Morton-ordered)
// cells by a whole time step -- S1 edge fluxes, S1c limiter, S2 gather, S3 update + friction, and Eq. 21 of the new
// state for the next dt -- out of shared memory, one thread per own cell.  Edge fluxes never go to DRAM; the state
// ping-pongs between two buffers because neighbouring patches read the old state of this patch's cells.
// Arithmetic and parenthesisation are those of the three-pass kernels in swe_kernels.cuh (R-14), so
// both variants give bit-identical states.
//
// Data movement (what differs from the first design, profiles/r1j: long-scoreboard stalls 5.3 cycles per issue):
//   * everything a patch streams sits in ONE fixed-stride blob (patch_blob.hpp); the block knows every address from
//     blockIdx alone, there is no header -> table -> record chain of dependent loads;
//   * the blob's staged part and the patch's own cell records arrive in shared memory by two bulk asynchronous
//     copies (cp.async.bulk.shared.global + mbarrier complete_tx; SASS: UBLKCP) issued by one thread right after
//     the skip test; no thread holds a register for a load in flight, and phases 2-4 read shared memory only;
//   * the halo records (ring 1 / ring 2: a gather) are fetched by the other threads while the bulk copies fly, and
//     their velocities are formed at once;
//   * the skip test is ONE 32-byte load: every patch owns a word of flag bytes {neighbours..., own, skippable} per
//     state buffer, and a block that finishes publishes its flag into its neighbours' words (byte stores).
//
// Phases (separated by __syncthreads):
//   1  states of the local cells (own, ring 1, ring 2) -> shared memory as (h, u, v, z)
//   2  every local edge: hydrostatic reconstruction + HLLC, boundary edges
//   3  theta of own and ring-1 cells (R-8b)
//   4  own cells: limited fluxes in slot order (Eq. 12), update, friction (Eq. 2), Eq. 21 rate
#pragma once
#include "swe_kernels.cuh"

namespace swe {

struct Patch2Args {
  const unsigned char *blob;
  BlobLayout L;
  void *rec_a, *rec_b;            // CellRecT<T> of the kernel's arithmetic T
  const void *kst;                // T per cell
  const BoundaryString *strings;
  const int32_t *slot_string;     // string id of every position of string_edges[]
  double *string_M;               // l * (limited F1) of every boundary-string edge, by position in string_edges[]
  unsigned char *pflag_a, *pflag_b;   // [n_patches][kPflagBytes], one array per state buffer
  int32_t n_cells;
  // self-controlled step (kSelf): no control kernel runs between two steps
  int32_t step_k;                 // this launch reads Control::slot[step_k] and writes slot[(step_k + 1) % 4]
  int32_t n_strings, n_string_edges;
  const double *string_lk;        // l_e * k_weight(k_st of cell L) of every boundary-string edge (R-11), by position
  const int32_t *string_cell;     // cell L of every boundary-string edge, by position
  int32_t prefetch_dist;          // > 0: block b pulls the tables of patch b + prefetch_dist into L2 (about the blocks
                                  // resident at a time, so that it is the patch that takes over this block's slot)
  Scalars sc;                     // passive scalars (kScalars instantiation only)
  Morph mp;                       // mobile bed (kMorph instantiation only; mp.cell / mp.qB are not used here)
  const double *gn2;              // g / k_st^2 per cell (kMorph, MPM-like law: the halo cells' values)
};

// ---- shared-memory carving (bytes), the same for every block of a context
struct Patch2Smem {
  int32_t strs, stage, crec, h, u, v, z, theta, F1, F3, GL, GR, phi, qB, fcx, fcy, total;
};

// morph: 0 fixed bed, 1 Grass-like law (q_B per own edge), 2 MPM-like law (+ (g/k^2, cbrt h) of every local cell)
__host__ __device__ inline Patch2Smem patch2_smem_layout(const BlobLayout &L, int n_species, int morph = 0, bool self = true) {
  Patch2Smem s;
  const int32_t rb = L.rb;                         // bytes of a real (fp64: 8; single precision: 4)
  int32_t o = 128;                                  // [0, 8): the mbarrier
  s.strs = o; o += self ? blob_align(kCtlPre * (int32_t)sizeof(BoundaryString), 128) : 0;   // kSelf: the strings with Q, sumK of t^n
  s.stage = o; o += blob_align(L.stage_bytes, 128);
  s.h = o; o += rb * L.cap_loc; s.u = o; o += rb * L.cap_loc; s.v = o; o += rb * L.cap_loc; s.z = o; o += rb * L.cap_loc;
  s.theta = o; o += rb * L.cap_c1;
  s.F1 = o; o += rb * L.cap_e;
  o = blob_align(o, 32);
  // the own CellRec records as the bulk copy delivers them are consumed in phase 1 (the momenta stay in registers),
  // the fluxes F3 / GL / GR of the own edges are written from phase 2 on: the two share their shared memory
  s.crec = o;
  s.F3 = o; s.GL = o + rb * L.cap_eown; s.GR = o + 2 * rb * L.cap_eown;
  o += (3 * rb * L.cap_eown > 4 * rb * L.P) ? 3 * rb * L.cap_eown : 4 * rb * L.P;
  s.phi = o; o += 8 * n_species * L.cap_loc;        // concentrations of the local cells, species-major
  s.qB = o; o += morph ? 8 * L.cap_eown : 0;        // normal sediment flux of the own edges (R-20)
  s.fcx = o; o += morph == 2 ? 8 * L.cap_loc : 0; s.fcy = o; o += morph == 2 ? 8 * L.cap_loc : 0;
  s.total = o;
  return s;
}

// ---- mbarrier / bulk-copy primitives (PTX ISA: mbarrier, cp.async.bulk)
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}
__device__ __forceinline__ void bulk_prefetch_l2(const void *src, uint32_t bytes) {   // bytes: a multiple of 16
  asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred P1;\n"
      "LAB_WAIT:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
      "@P1 bra DONE;\n"
      "bra LAB_WAIT;\n"
      "DONE:\n"
      "}" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}

// own flag + the byte this patch has in each neighbour's flag word (nbr / nbr_slot: cap_nbr entries, -1 padded)
// dirty: bit j set = an own cell that the j-th neighbour reads is not (0, 0, 0) (j < 32; beyond: the own flag decides)
template <int kThreads>
__device__ __forceinline__ void publish_flag(unsigned char *pf_out_base, int b, const int32_t *nbr, const int32_t *nbr_slot,
                                             int cap_nbr, unsigned char flag, uint32_t dirty = 0u) {
  if (threadIdx.x == 0) pf_out_base[(size_t)b * kPflagBytes + kPflagOwn] = flag;
  for (int j = threadIdx.x; j < cap_nbr; j += kThreads) {
    const int q = nbr[j], sl = nbr_slot[j];
    if (q >= 0 && sl >= 0) pf_out_base[(size_t)q * kPflagBytes + sl] = j < 32 ? (unsigned char)(((dirty >> j) & 1u) ^ 1u) : flag;
  }
}

// S0 / S4 for a step that reads slot S (the arithmetic of k_step_control): dt from the rate of the state, the stop rules
struct StepChoice { int active, flags; double dt, t_new; };
__device__ __forceinline__ StepChoice choose_step(const StepSlot &S, double t_end, double cfl, double dt_max) {
  StepChoice c;
  c.active = 0; c.flags = S.flags; c.dt = 0.0; c.t_new = S.t;
  if (S.steps_left != 0 && S.t < t_end && !(S.flags & (kFlagUnbounded | kFlagStalled))) {
    const double r = __longlong_as_double((long long)S.rate_bits);
    double dt = (r > 0.0) ? cfl / r : dt_max;
    dt = fmin(dt, dt_max);
    const double rem = t_end - S.t;
    double t_new;
    if (dt >= rem) { dt = rem; t_new = t_end; } else { t_new = S.t + dt; }
    if (!isfinite(dt)) c.flags |= kFlagUnbounded;
    else if (!(dt > 0.0) || !(t_new > S.t)) c.flags |= kFlagStalled;
    else { c.active = 1; c.dt = dt; c.t_new = t_new; }
  }
  return c;
}

// outflow volume of the step that produced slot S: dt_last * tree sum of the string's l * (limited F1), by the whole
// block (v: scratch of pow2 doubles in shared memory).  Returns vol_out with it added (every thread gets the value).
template <int kThreads>
__device__ __forceinline__ double book_outflow(const StepSlot &S, const BoundaryString *__restrict__ strings, int n_strings,
                                               const double *__restrict__ M_prev, double *v) {
  double vol_out = S.vol_out;
  if (!S.pending) return vol_out;
  for (int s = 0; s < n_strings; ++s) {
    const int type = strings[s].type;
    if (type != kBcOutflowUniform) continue;
    const int n = strings[s].n_edges, first = strings[s].first, pow2 = strings[s].pow2;
    for (int j = threadIdx.x; j < pow2; j += kThreads) v[j] = j < n ? M_prev[first + j] : 0.0;
    const double sum = block_tree_sum(v, pow2);
    vol_out += S.dt_last * sum;
  }
  return vol_out;
}

// start of an swe_step call in self-controlled mode: the classic fields -> slot[k0]
static __global__ void k_self_begin(Control *ctl, long long n_steps, double t_end, double cfl, int k0) {
  ctl->steps_left = n_steps; ctl->t_end = t_end; ctl->cfl = cfl;
  ctl->flags &= ~(kFlagUnbounded | kFlagStalled);
  StepSlot S;
  S.t = ctl->t; S.dt_last = ctl->dt_last; S.vol_in = ctl->vol_in; S.vol_out = ctl->vol_out; S.rate_bits = ctl->rate_bits;
  S.steps_left = n_steps; S.steps_done = ctl->steps_done; S.src = ctl->cur; S.flags = ctl->flags; S.pending = 0; S.pad_ = 0;
  ctl->slot[k0 & 3] = S;
  ctl->slot[(k0 + 1) & 3].rate_bits = 0ull;
  ctl->slot[(k0 + 2) & 3].rate_bits = 0ull;
}

// slot[k] -> the classic fields (final: with the outflow bookkeeping of the last step; else a snapshot for polling t)
template <int kThreads>
__global__ void __launch_bounds__(kThreads)
k_self_finish(Control *ctl, const BoundaryString *__restrict__ strings, int n_strings, const double *__restrict__ string_M,
              int n_string_edges, int k, int final) {
  __shared__ double v[1024];
  const StepSlot S = ctl->slot[k & 3];
  double vol_out = S.vol_out;
  if (final) vol_out = book_outflow<kThreads>(S, strings, n_strings, string_M + (size_t)((k & 1) ^ 1) * n_string_edges, v);
  if (threadIdx.x != 0) return;
  ctl->t = S.t; ctl->dt_last = S.dt_last; ctl->dt = S.dt_last; ctl->vol_in = S.vol_in; ctl->vol_out = vol_out;
  ctl->rate_bits = S.rate_bits; ctl->steps_left = S.steps_left; ctl->steps_done = S.steps_done;
  ctl->flags = S.flags; ctl->cur = S.src; ctl->src = S.pending ? (S.src ^ 1) : S.src;
  ctl->active = 0; ctl->pending = 0;
  if (final) { ctl->slot[k & 3].vol_out = vol_out; ctl->slot[k & 3].pending = 0; ctl->vol = 0.0; ctl->n_wet = 0; ctl->nonfinite = 0; }
}

// kThreads >= BlobLayout::P (one thread per own cell; the host picks the smallest instance that covers P).  kScalars: the passive-scalar module (R-19) is on:
// concentrations of the local cells in shared memory, one more gather per species in phase 4.
// kSelf: no k_step_control between the steps -- every block derives dt / t / stop rules from Control::slot[step_k], block 0
// writes the next slot and books the volumes, the blocks that own boundary-string edges evaluate Q(t^n) and the
// conveyance sums themselves (same fixed-shape trees, R-11).
// kMorph: the mobile bed (R-20): q_Bij of every own edge in phase 2 (Table 2, Eq. 14-16), Eq. 13 in phase 4 -- the bed
// rides in the state record.  A skipped patch keeps its bed: no transport where a side is dry.
// T: the arithmetic of the step (double; float = single precision, R-21: plain hydrodynamics behind k_step_control only)
template <int kThreads, int kMinBlocks, bool kScalars = false, bool kSelf = false, bool kMorph = false, typename T = double>
__global__ void __launch_bounds__(kThreads, kMinBlocks)
k_patch2(Control *__restrict__ ctl, const Patch2Args A) {
  static_assert(sizeof(T) == 8 || (!kScalars && !kSelf && !kMorph), "single precision: hydrodynamics behind k_step_control only");
  typedef CellRecT<T> Rec;
  typedef EdgeFluxT<T> Flux;
  extern __shared__ __align__(128) unsigned char smraw[];
  const BlobLayout &L = A.L;
  const int tid = threadIdx.x, b = blockIdx.x;
  const int n_sp = kScalars ? A.sc.n : 0;
  const unsigned char *blob = A.blob + (size_t)b * (size_t)L.stride;
  const int cell0 = b * L.P;                       // L.P <= kThreads: one thread per own cell
  const int n_own = min(L.P, A.n_cells - cell0);
  const int32_t *__restrict__ halo_ids = (const int32_t *)(blob + L.off_halo_ids);

  // ---- everything whose address depends on blockIdx alone is requested at once (one memory latency for all of it):
  // the control block, this patch's flag word in BOTH state buffers (which one is read depends on Control::src) and
  // the flag words of the patch whose tables this block pulls into L2 (below).  The first halo ids of every thread
  // used to be among them: a block that is skipped then waits for a DRAM access it has no use for before it can
  // leave (its blob is in nobody's L2), so they are fetched behind the skip test (profiles/r2aa_contention.md)
  const ulonglong2 *pfa = reinterpret_cast<const ulonglong2 *>(A.pflag_a + (size_t)b * kPflagBytes);
  const ulonglong2 *pfb = reinterpret_cast<const ulonglong2 *>(A.pflag_b + (size_t)b * kPflagBytes);
  StepSlot S0;
  int active, src;
  T dt;
  if (kSelf) { S0 = ctl->slot[A.step_k]; active = 0; src = S0.src; dt = T(0.0); }
  else { active = ctl->active; src = ctl->src; dt = (T)ctl->dt; }
  const ulonglong2 fa0 = pfa[0], fa1 = pfa[1], fb0 = pfb[0], fb1 = pfb[1];
  const int b_pf = b + A.prefetch_dist;            // the block that will run in this block's slot next (about)
  const bool do_pf = A.prefetch_dist > 0 && b_pf < (int)gridDim.x && tid == 0;
  ulonglong2 ga0, ga1, gb0, gb1;
  if (do_pf) {
    const ulonglong2 *qa = reinterpret_cast<const ulonglong2 *>(A.pflag_a + (size_t)b_pf * kPflagBytes);
    const ulonglong2 *qb = reinterpret_cast<const ulonglong2 *>(A.pflag_b + (size_t)b_pf * kPflagBytes);
    ga0 = qa[0]; ga1 = qa[1]; gb0 = qb[0]; gb1 = qb[1];
  }
  const T g = (T)ctl->g, h_dry = (T)ctl->h_dry;
  if constexpr (kSelf) {
    const StepChoice ch = choose_step(S0, ctl->t_end, ctl->cfl, ctl->dt_max);
    active = ch.active; dt = ch.dt;
    if (b == 0) {                // the control duty: next slot, volume bookkeeping (before anything can return)
      const int k1 = (A.step_k + 1) & 3, k2 = (A.step_k + 2) & 3;
      const double vol_out = book_outflow<kThreads>(S0, A.strings, A.n_strings, A.string_M + (size_t)((A.step_k & 1) ^ 1) * A.n_string_edges,
                                                    reinterpret_cast<double *>(smraw + 128));
      if (tid == 0) {
        double vol_in = S0.vol_in;
        if (active)
          for (int s = 0; s < A.n_strings; ++s)
            if (A.strings[s].type == kBcInflowQ) vol_in += ch.dt * hydrograph(A.strings[s].params, A.strings[s].n_params, S0.t);
        StepSlot *N = &ctl->slot[k1];
        N->t = ch.t_new; N->dt_last = active ? ch.dt : S0.dt_last; N->vol_in = vol_in; N->vol_out = vol_out;
        N->steps_left = (active && S0.steps_left > 0) ? S0.steps_left - 1 : S0.steps_left;
        N->steps_done = S0.steps_done + active; N->src = active ? (src ^ 1) : src; N->flags = ch.flags; N->pending = active;
        if (!active) N->rate_bits = S0.rate_bits;       // nothing accumulates into it when the step does no work
        ctl->slot[k2].rate_bits = 0ull;
      }
      __syncthreads();             // the scratch is reused below
    }
  }
  if (!active) return;
  const Rec *__restrict__ in = reinterpret_cast<const Rec *>(src ? A.rec_b : A.rec_a);      // (the args carry untyped record pointers)
  Rec *__restrict__ out = reinterpret_cast<Rec *>(src ? A.rec_a : A.rec_b);
  unsigned char *pf_out_base = src ? A.pflag_a : A.pflag_b;
  const unsigned long long ones = 0x0101010101010101ull;

  // ---- skip test (section 5b): when the own cells of this patch and of every patch that owns one of its halo cells
  // are exactly (0, 0, 0) in the state being read, and no boundary string can feed the patch, every flux of S1 is
  // exactly 0, theta = 1 and S3 returns (+0, 0, 0) for every own cell: write that (unless the target holds it already).
  {
    const ulonglong2 w0 = src ? fb0 : fa0, w1 = src ? fb1 : fa1;
    if (w0.x == ones && w0.y == ones && w1.x == ones && w1.y == ones) {
      // the own flag of the word this patch has in the buffer being written: loaded above with everything else
      const ulonglong2 o1 = src ? fa1 : fb1;
      const unsigned char had = (unsigned char)((o1.y >> (8 * (kPflagOwn - 24))) & 0xffull);
      if (!had) {
        if (tid < n_own) {
          Rec c = in[cell0 + tid];
          c.h = T(0.0); c.qx = T(0.0); c.qy = T(0.0);
          out[cell0 + tid] = c;
          _Pragma("unroll") for (int sp = 0; sp < kMaxSpecies; ++sp) if (sp < n_sp) (src ? A.sc.qa[sp] : A.sc.qb[sp])[cell0 + tid] = 0.0;   // flag: all q_c are 0 too
        }
        __syncthreads();            // every thread has read `had` before the flag changes
        publish_flag<kThreads>(pf_out_base, b, (const int32_t *)(blob + L.off_nbr), (const int32_t *)(blob + L.off_nbr_slot), L.cap_nbr, 1);
      }
      if (tid == 0) atomicAdd(&ctl->patches_skipped, 1ull);
      return;
    }
  }

  const int hid0 = tid < L.cap_halo ? halo_ids[tid] : -1;
  const int hid1 = tid + kThreads < L.cap_halo ? halo_ids[tid + kThreads] : -1;
  const int morph = kMorph ? A.mp.formula : 0;
  const Patch2Smem S = patch2_smem_layout(L, n_sp, morph, kSelf);
  T *sh_qB = (T *)(smraw + S.qB), *sh_fcx = (T *)(smraw + S.fcx), *sh_fcy = (T *)(smraw + S.fcy);
  uint64_t *bar = reinterpret_cast<uint64_t *>(smraw);
  unsigned char *stage = smraw + S.stage;
  Rec *crec = reinterpret_cast<Rec *>(smraw + S.crec);
  T *sh_h = (T *)(smraw + S.h), *sh_u = (T *)(smraw + S.u), *sh_v = (T *)(smraw + S.v), *sh_z = (T *)(smraw + S.z);
  T *sh_th = (T *)(smraw + S.theta), *sh_F1 = (T *)(smraw + S.F1), *sh_F3 = (T *)(smraw + S.F3);
  T *sh_GL = (T *)(smraw + S.GL), *sh_GR = (T *)(smraw + S.GR), *sh_phi = (T *)(smraw + S.phi);
  const int cap_loc = L.cap_loc;

  // ---- the two bulk copies: staged part of the blob, own cell records
  uint32_t *sm_dirty = reinterpret_cast<uint32_t *>(smraw + 16);   // neighbours that read a wet own cell (phase 4)
  uint32_t *sm_marked = reinterpret_cast<uint32_t *>(smraw + 20);  // phase 2 marked a donor cell for phase 3
  if (tid == 0) {
    *sm_dirty = 0u; *sm_marked = 0u;
    mbar_init(bar, 1);
    mbar_expect_tx(bar, (uint32_t)L.stage_bytes + (uint32_t)sizeof(Rec) * (uint32_t)n_own);
    bulk_g2s(stage, blob + L.off_stage, (uint32_t)L.stage_bytes, bar);
    bulk_g2s(crec, in + cell0, (uint32_t)sizeof(Rec) * (uint32_t)n_own, bar);
    // the tables and own records of the patch that will run in this slot next go to L2 now (unless that patch will
    // be skipped): its block then pays L2 latency, not DRAM latency, in the chain flag word -> bulk copy -> phase 1
    if (do_pf) {
      const ulonglong2 v0 = src ? gb0 : ga0, v1 = src ? gb1 : ga1;
      if (!(v0.x == ones && v0.y == ones && v1.x == ones && v1.y == ones)) {
        const int c0n = b_pf * L.P, n_next = min(L.P, A.n_cells - c0n);
        bulk_prefetch_l2(A.blob + (size_t)b_pf * (size_t)L.stride, (uint32_t)(L.off_stage + L.stage_bytes));
        bulk_prefetch_l2(in + c0n, (uint32_t)sizeof(Rec) * (uint32_t)n_next);
      }
    }
  }

  // ---- phase 1a: halo cells (a gather: id -> record), while the bulk copies are in flight; velocities once per cell
  // (R-8: thin films carry no momentum)
  int water = 0;
  for (int j0 = tid; j0 < L.cap_halo; j0 += 2 * kThreads) {
    const int j1 = j0 + kThreads;
    const int id0 = j0 == tid ? hid0 : halo_ids[j0];
    const int id1 = j0 == tid ? hid1 : (j1 < L.cap_halo ? halo_ids[j1] : -1);
    Rec c0, c1;
    if (id0 >= 0) c0 = in[id0];
    if (id1 >= 0) c1 = in[id1];
    if (id0 >= 0) {
      const int l = n_own + j0;
      T u = T(0.0), v = T(0.0);
      if (c0.h > h_dry) { u = c0.qx / c0.h; v = c0.qy / c0.h; }
      sh_h[l] = c0.h; sh_u[l] = u; sh_v[l] = v; sh_z[l] = c0.z;
      if constexpr (kMorph) if (morph == 2) {                // MPM-like law: (g / k^2, cbrt h) as k_cell_update leaves it in Morph::cell
        const T f2 = A.gn2[id0];
        const bool on = c0.h > h_dry && f2 > 0.0;
        sh_fcx[l] = on ? f2 : 0.0; sh_fcy[l] = on ? cbrt_rn(c0.h) : 0.0;
      }
      if (l < L.cap_c1) sh_th[l] = T(1.0);
      water |= (c0.h != T(0.0));
      if constexpr (kScalars)                              // phi = q_c / h where there is water, else 0 (R-19)
        _Pragma("unroll") for (int sp = 0; sp < kMaxSpecies; ++sp) if (sp < n_sp)
          sh_phi[sp * cap_loc + l] = c0.h > 0.0 ? (src ? A.sc.qb[sp] : A.sc.qa[sp])[id0] / c0.h : 0.0;
    }
    if (id1 >= 0) {
      const int l = n_own + j1;
      T u = T(0.0), v = T(0.0);
      if (c1.h > h_dry) { u = c1.qx / c1.h; v = c1.qy / c1.h; }
      sh_h[l] = c1.h; sh_u[l] = u; sh_v[l] = v; sh_z[l] = c1.z;
      if constexpr (kMorph) if (morph == 2) {
        const T f2 = A.gn2[id1];
        const bool on = c1.h > h_dry && f2 > 0.0;
        sh_fcx[l] = on ? f2 : 0.0; sh_fcy[l] = on ? cbrt_rn(c1.h) : 0.0;
      }
      if (l < L.cap_c1) sh_th[l] = T(1.0);
      water |= (c1.h != T(0.0));
      if constexpr (kScalars)
        _Pragma("unroll") for (int sp = 0; sp < kMaxSpecies; ++sp) if (sp < n_sp)
          sh_phi[sp * cap_loc + l] = c1.h > 0.0 ? (src ? A.sc.qb[sp] : A.sc.qa[sp])[id1] / c1.h : 0.0;
    }
  }
  __syncthreads();                 // the mbarrier is initialised for every thread
  mbar_wait(bar, 0);               // both bulk copies have landed

  const BlobHeader H = *reinterpret_cast<const BlobHeader *>(stage + L.s_hdr);
  const int n_c1 = H.n_own + H.n_r1, n_e = H.n_eown + H.n_er1;
  const T *__restrict__ b_halo_area = (const T *)(stage + L.s_halo_area);
  const uint4 *__restrict__ b_pce = (const uint4 *)(stage + L.s_pce);
  const T *__restrict__ b_nx = (const T *)(stage + L.s_nx), *__restrict__ b_ny = (const T *)(stage + L.s_ny);
  const T *__restrict__ b_len = (const T *)(stage + L.s_len);
  const uint32_t *__restrict__ b_lr = (const uint32_t *)(stage + L.s_lr);
  const int32_t *__restrict__ b_aux = (const int32_t *)(stage + L.s_aux);
  const T *__restrict__ b_area = (const T *)(stage + L.s_area);
  const T *__restrict__ b_gn2 = (const T *)(stage + L.s_gn2);

  // ---- phase 1b: own cells, from the records the bulk copy delivered
  T qx_own = T(0.0), qy_own = T(0.0);               // the momenta of this thread's own cell, kept for phase 4
  if (tid < n_own) {
    const Rec c_own = crec[tid];
    qx_own = c_own.qx; qy_own = c_own.qy;
    T u = T(0.0), v = T(0.0);
    if (c_own.h > h_dry) { u = c_own.qx / c_own.h; v = c_own.qy / c_own.h; }
    sh_h[tid] = c_own.h; sh_u[tid] = u; sh_v[tid] = v; sh_z[tid] = c_own.z; sh_th[tid] = T(1.0);
    if constexpr (kMorph) if (morph == 2) {
      const T f2 = b_gn2[tid];
      const bool on = c_own.h > h_dry && f2 > 0.0;
      sh_fcx[tid] = on ? f2 : 0.0; sh_fcy[tid] = on ? cbrt_rn(c_own.h) : 0.0;
    }
    water |= (c_own.h != T(0.0));
    if constexpr (kScalars)
      _Pragma("unroll") for (int sp = 0; sp < kMaxSpecies; ++sp) if (sp < n_sp)
        sh_phi[sp * cap_loc + tid] = c_own.h > 0.0 ? (src ? A.sc.qb[sp] : A.sc.qa[sp])[cell0 + tid] / c_own.h : 0.0;
  }
  // second, exact test on the local cells themselves (the flags above are per whole patch): no water in any
  // local cell and no boundary string -> same result (+0, 0, 0)
  if (!__syncthreads_or(water) && H.n_string_edges == 0) {
    int scalar_mass = 0;
    if (tid < n_own) {
      Rec c; c.h = T(0.0); c.qx = T(0.0); c.qy = T(0.0); c.z = sh_z[tid];
      out[cell0 + tid] = c;
      if constexpr (kScalars) _Pragma("unroll") for (int sp = 0; sp < kMaxSpecies; ++sp) if (sp < n_sp) {          // no flux: scalar mass parked in dry cells stays where it is
        const T q = (src ? A.sc.qb[sp] : A.sc.qa[sp])[cell0 + tid];
        (src ? A.sc.qa[sp] : A.sc.qb[sp])[cell0 + tid] = q;
        scalar_mass |= (q != 0.0);
      }
    }
    scalar_mass = kScalars ? __syncthreads_or(scalar_mass) : 0;
    publish_flag<kThreads>(pf_out_base, b, (const int32_t *)(blob + L.off_nbr), (const int32_t *)(blob + L.off_nbr_slot), L.cap_nbr,
                           scalar_mass ? 0 : 1);
    if (tid == 0) atomicAdd(&ctl->patches_skipped, 1ull);
    return;
  }

  // ---- kSelf: this block owns boundary-string edges -> Q(t^n) and the conveyance sum of every inflow string (R-11),
  // as k_step_control evaluates them: weights from the state being read, fixed-shape pairwise tree in string order
  const BoundaryString *sm_strings = reinterpret_cast<const BoundaryString *>(smraw + S.strs);
  if constexpr (kSelf) if (H.n_string_edges > 0) {
    BoundaryString *st = reinterpret_cast<BoundaryString *>(smraw + S.strs);
    T *v = sh_F1;                               // scratch: the flux arrays (and the own records aliased with them,
                                                     // consumed in phase 1) are not in use before phase 2
    for (int j = tid; j < A.n_strings * (int)(sizeof(BoundaryString) / 8); j += kThreads)
      reinterpret_cast<unsigned long long *>(st)[j] = reinterpret_cast<const unsigned long long *>(A.strings)[j];
    __syncthreads();
    for (int s = 0; s < A.n_strings; ++s) {
      if (st[s].type != kBcInflowQ) continue;
      const int n = st[s].n_edges, first = st[s].first, pow2 = st[s].pow2;
      for (int j = tid; j < pow2; j += kThreads)
        v[j] = j < n ? A.string_lk[first + j] * pow53(in[A.string_cell[first + j]].h) : 0.0;
      const T sum = block_tree_sum(v, pow2);
      if (tid == 0) {
        const T Q = hydrograph(st[s].params, st[s].n_params, S0.t);
        st[s].sumK = sum; st[s].Q = Q;
        // also where k_step_control would leave them (inspection: swe_get_edge_flux re-evaluates this step from them);
        // every block that owns a string edge writes the same two values
        BoundaryString *gs = const_cast<BoundaryString *>(A.strings) + s;
        gs->sumK = sum; gs->Q = Q;
      }
    }
    __syncthreads();
  }

  // ---- phase 2: edge fluxes (two edges per thread and iteration, to interleave their dependent fp64 chains, was
  // measured and is slower: 80 registers with spills, branches keep the streams apart)
  struct EdgeIn { T nx, ny, len, hL, uL, vL, zL, hR, uR, vR, zR; int Lc, Rc; };
  auto load_edge = [&](int e) {
    EdgeIn q;
    const uint32_t lr = b_lr[e];
    q.Lc = (int)(lr & 0xFFFFu); q.Rc = (int)(lr >> 16);
    q.nx = b_nx[e]; q.ny = b_ny[e]; q.len = b_len[e];
    q.hL = sh_h[q.Lc]; q.uL = sh_u[q.Lc]; q.vL = sh_v[q.Lc]; q.zL = sh_z[q.Lc];
    const int Rs = q.Rc != 0xFFFF ? q.Rc : q.Lc;
    q.hR = sh_h[Rs]; q.uR = sh_u[Rs]; q.vR = sh_v[Rs]; q.zR = sh_z[Rs];
    return q;
  };
  auto flux_edge = [&](const EdgeIn &q, int e) {
    Flux o;
    if (q.Rc != 0xFFFF) {
      const T unL = q.uL * q.nx + q.vL * q.ny, utL = q.vL * q.nx - q.uL * q.ny;
      const T unR = q.uR * q.nx + q.vR * q.ny, utR = q.vR * q.nx - q.uR * q.ny;
      o = riemann_nt(g, q.hL, unL, utL, q.zL, q.hR, unR, utR, q.zR);
    } else {
      const BoundaryString *bs = nullptr;
      int code = b_aux[e];
      if (code <= -3) { bs = (kSelf ? sm_strings : A.strings) + A.slot_string[-3 - code]; code = -3; }
      const int gidL = q.Lc < n_own ? cell0 + q.Lc : halo_ids[q.Lc - n_own];
      o = boundary_flux(g, code, bs, reinterpret_cast<const T *>(A.kst), gidL, q.nx, q.ny, q.len, q.hL, q.zL, q.uL, q.vL);
    }
    return o;
  };
  auto store_edge = [&](const EdgeIn &q, int e, const Flux &o) {
    sh_F1[e] = o.F1;
    if (e < H.n_eown) { sh_F3[e] = o.F3; sh_GL[e] = o.GL; sh_GR[e] = o.GR; }
    if constexpr (kMorph) if (e < H.n_eown) {                     // S1m: q_Bij from the state at t^n (Eq. 14-16; R-20)
      const int Rcode = q.Rc != 0xFFFF ? 0 : (b_aux[e] <= -3 ? -3 : b_aux[e]);
      const double2 zero = make_double2(0.0, 0.0);
      const double2 fcL = morph == 2 ? make_double2(sh_fcx[q.Lc], sh_fcy[q.Lc]) : zero;
      const double2 fcR = (morph == 2 && q.Rc != 0xFFFF) ? make_double2(sh_fcx[q.Rc], sh_fcy[q.Rc]) : zero;
      sh_qB[e] = sediment_flux_core(A.mp, g, h_dry, Rcode, q.nx, q.ny, q.hL, q.uL, q.vL, q.zL, fcL, q.hR, q.uR, q.vR, q.zR, fcR);
    }
    // S1c, lazily (R-8b; as in k_edge_flux): theta_i < 1 needs one outgoing edge with dt * o_k > 0.3 h_i |Omega_i|.  Only
    // such donor cells are marked (theta = -1); phase 3 evaluates theta for them and every other cell keeps theta = 1.
    const int d = o.F1 > T(0.0) ? q.Lc : ((o.F1 < T(0.0) && q.Rc != 0xFFFF) ? q.Rc : n_c1);
    if (d < n_c1) {
      const T ad = d < n_own ? b_area[d] : b_halo_area[d - n_own];
      const T hd = d == q.Lc ? q.hL : q.hR;
      if (dt * (q.len * fabs(o.F1)) > T(0.3) * (hd * ad)) { sh_th[d] = -T(1.0); *sm_marked = 1u; }
    }
  };
  for (int e = tid; e < n_e; e += kThreads) {
    const EdgeIn q = load_edge(e);
    const Flux o = flux_edge(q, e);
    store_edge(q, e, o);
  }

  // ---- phase 3 (R-8b): theta_i = min(1, h_i |Omega_i| / (dt * sum of the outgoing l F1)), slots in order -- for the
  // cells marked in phase 2 only; a block that marked none (the rule away from wet/dry fronts) goes on to phase 4
  // without the pass over the cells and its barrier
  __syncthreads();
  const bool any_marked = *sm_marked != 0u;
  if (any_marked) {
  for (int l = tid; l < n_c1; l += kThreads) {
    if (sh_th[l] >= T(0.0)) continue;
    const uint4 pc = b_pce[l];
    const uint32_t w[3] = {pc.x, pc.y, pc.z};
    T o[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      const int e = w[k] & 0x7FFFu;
      const T sM = ((w[k] & 0x8000u) ? T(1.0) : -T(1.0)) * (b_len[e] * sh_F1[e]);
      o[k] = dmax0(sM);
    }
    const T outflow = ((o[0] + o[1]) + o[2]);
    const T avail = sh_h[l] * (l < n_own ? b_area[l] : b_halo_area[l - n_own]);
    T th = T(1.0);
    if (dt * outflow > avail) th = avail / (dt * outflow);
    sh_th[l] = th;
  }
  __syncthreads();
  }

  // ---- phase 4: own cells, one per thread
  T rate = T(0.0);
  int nonzero = 0;
  if (tid < n_own) {
    const int l = tid, i = cell0 + tid;
    const uint4 pc = b_pce[l];
    Rec c_own;
    c_own.h = sh_h[l]; c_own.qx = qx_own; c_own.qy = qy_own; c_own.z = sh_z[l];
    T invA;                                          // 1 / |Omega| as the host forms it for the three-pass step
    if constexpr (sizeof(T) == 8) invA = T(1.0) / b_area[l];
    else invA = reinterpret_cast<const T *>(stage + L.s_inv_area)[l];   // fp64 quotient rounded once (R-21)
    const T f2 = b_gn2[l];
    const uint32_t w[3] = {pc.x, pc.y, pc.z};
    T dH = T(0.0), dX = T(0.0), dY = T(0.0), dB = T(0.0);   // ((d0 + d1) + d2), accumulated in slot order
    T F1k[3], slk[3];                           // kScalars: limited mass flux and sign * length of every slot,
    int up[3];                                       // local id of the upwind cell, or -1 - slot of an inflow-string edge
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      const int e = w[k] & 0x7FFFu;
      const bool isL = (w[k] & 0x8000u) != 0u;
      const uint32_t nb = w[k] >> 16;
      T F1 = sh_F1[e], F3 = sh_F3[e];
      T G = isL ? sh_GL[e] : sh_GR[e];
      // limiter: every component of the edge is scaled by theta of the donor cell (the one F1 leaves)
      if (any_marked) {                             // no donor marked in this block: every theta is 1, x * 1 = x bit for bit
        T th = T(1.0);
        if (F1 > T(0.0)) th = sh_th[isL ? (uint32_t)l : nb];
        else if (F1 < T(0.0) && nb != kPceNoNeighbour) th = sh_th[isL ? nb : (uint32_t)l];
        F1 = th * F1; F3 = th * F3; G = th * G;     // theta = 1: the product is the factor itself, bit for bit
      }
      const T nxk = b_nx[e], nyk = b_ny[e], lenk = b_len[e];
      // s * x with s = +-1 is x or -x exactly: a change of sign instead of a product
      const T dH0 = lenk * F1, dX0 = lenk * (G * nxk - F3 * nyk), dY0 = lenk * (G * nyk + F3 * nxk);
      const T dHk = isL ? dH0 : -dH0, dXk = isL ? dX0 : -dX0, dYk = isL ? dY0 : -dY0;
      if (k == 0) { dH = dHk; dX = dXk; dY = dYk; } else { dH = dH + dHk; dX = dX + dXk; dY = dY + dYk; }
      if constexpr (kMorph) { const T dB0 = lenk * sh_qB[e]; const T dBk = isL ? dB0 : -dB0; dB = k == 0 ? dBk : dB + dBk; }
      if constexpr (kScalars) {
        F1k[k] = F1; slk[k] = lenk;
        const uint32_t Lc = isL ? (uint32_t)l : nb, Rc = isL ? nb : (uint32_t)l;
        up[k] = (int)((F1 >= 0.0 || Rc == kPceNoNeighbour) ? Lc : Rc);   // ghost concentration = the interior cell's
        if (!isL) slk[k] = -lenk;
      }
      if (nb == kPceNoNeighbour) {                  // boundary-string edge: volume bookkeeping of k_step_control
        const int aux = b_aux[e];
        if (aux <= -3) {
          A.string_M[(kSelf ? (size_t)(A.step_k & 1) * A.n_string_edges : (size_t)0) + (-3 - aux)] = lenk * F1;
          if (kScalars && !(F1 >= T(0.0)) && A.strings[A.slot_string[-3 - aux]].type == kBcInflowQ) up[k] = -1 - (-3 - aux);
        }
      }
    }
    const T a = dt * invA;
    T hn = c_own.h - a * dH;
    if (hn < T(0.0)) {                                  // residual negatives (R-8b): clip and count
      atomicAdd(&ctl->vol_clipped, (double)(-hn * b_area[l]));
      hn = T(0.0);
    }
    T qxn = T(0.0), qyn = T(0.0);
    if (hn > h_dry) {
      qxn = c_own.qx - a * dX;
      qyn = c_own.qy - a * dY;
      if (f2 > T(0.0)) {   // R-5/R-6: exact integral of dq/dt = -(g/(k^2 h^(7/3))) |q| q over dt, h frozen at h^{n+1}
        const T D = T(1.0) + ((dt * f2) * sqrt(qxn * qxn + qyn * qyn)) / ((hn * hn) * cbrt_rn(hn));
        qxn = qxn / D;
        qyn = qyn / D;
      }
      // Eq. 21 (R-7) of the new state, for the next dt: max_j lambda_ij / rho_ij
      const T u = qxn / hn, v = qyn / hn;
      const T cel = sqrt(g * hn);
#pragma unroll
      for (int k = 0; k < 3; ++k) {
        const int e = w[k] & 0x7FFFu;
        const T lam = fabs(u * b_nx[e] + v * b_ny[e]) + cel;
        const T val = lam * ((T(0.75) * b_len[e]) * invA);
        if (val > rate) rate = val;
      }
    }
    Rec c = c_own;
    c.h = hn; c.qx = qxn; c.qy = qyn;
    if constexpr (kMorph) c.z = c.z - A.mp.inv1mp * (a * dB);   // Eq. 13, S_b = 0
    out[i] = c;
    nonzero |= (hn != T(0.0)) | (qxn != T(0.0)) | (qyn != T(0.0));
    if constexpr (kScalars) {                                  // Eq. 20, advective part: A_ij = limited F1 x upwind phi (R-19)
      _Pragma("unroll") for (int sp = 0; sp < kMaxSpecies; ++sp) if (sp < n_sp) {
        T dC = 0.0;
#pragma unroll
        for (int k = 0; k < 3; ++k) {
          const T phi = up[k] >= 0 ? sh_phi[sp * cap_loc + up[k]] : A.strings[A.slot_string[-1 - up[k]]].phi_in[sp];
          const T lC = fabs(slk[k]) * (F1k[k] * phi);
          const T Ck = slk[k] < 0.0 ? -lC : lC;
          dC = k == 0 ? Ck : dC + Ck;
        }
        const T qn = (src ? A.sc.qb[sp] : A.sc.qa[sp])[i] - a * dC;
        (src ? A.sc.qa[sp] : A.sc.qb[sp])[i] = qn;
        nonzero |= (qn != 0.0);
      }
    }
  }
  // which neighbour patches read an own cell that is not (0, 0, 0): OR of the masks (fourth word of the slot record)
  {
    const uint32_t mine = (nonzero && tid < n_own) ? reinterpret_cast<const uint32_t *>(b_pce)[4 * tid + 3] : 0u;
    const uint32_t warp_dirty = __reduce_or_sync(0xffffffffu, mine);
    if ((tid & 31) == 0 && warp_dirty) atomicOr(sm_dirty, warp_dirty);
  }
  // block maximum of the rate (non-negative doubles order like their bit patterns): per warp two 32-bit REDUX (high
  // words, then the low words of the lanes that hold the maximal high word) before the barrier that the flag needs
  // anyway, the warps' results by the first warp after it -- no barrier of its own, no shuffle chain at the block's tail
  __shared__ unsigned long long warp_rate[kThreads / 32];
  {
    const unsigned long long rb = (unsigned long long)__double_as_longlong((double)rate);
    const uint32_t hi = (uint32_t)(rb >> 32), mhi = __reduce_max_sync(0xffffffffu, hi);
    const uint32_t mlo = __reduce_max_sync(0xffffffffu, hi == mhi ? (uint32_t)rb : 0u);
    if ((tid & 31) == 0) warp_rate[tid >> 5] = ((unsigned long long)mhi << 32) | mlo;
  }
  nonzero = __syncthreads_or(nonzero);
  publish_flag<kThreads>(pf_out_base, b, (const int32_t *)(stage + L.s_nbr), (const int32_t *)(stage + L.s_nbr_slot), L.cap_nbr,
                         nonzero ? 0 : 1, *sm_dirty);
  if (tid < 32) {
    const unsigned long long rb = tid < kThreads / 32 ? warp_rate[tid] : 0ull;
    const uint32_t hi = (uint32_t)(rb >> 32), mhi = __reduce_max_sync(0xffffffffu, hi);
    const uint32_t mlo = __reduce_max_sync(0xffffffffu, hi == mhi ? (uint32_t)rb : 0u);
    const unsigned long long m = ((unsigned long long)mhi << 32) | mlo;
    if (tid == 0 && m != 0ull) atomicMax(kSelf ? &ctl->slot[(A.step_k + 1) & 3].rate_bits : &ctl->rate_bits, m);
  }
}

// flags after swe_set_state, two launches: (1) own flag of the buffer that holds the newest state from the records
// (the other buffer: unknown = 0); (2) every patch works out its neighbour bytes from its halo cells
template <int kThreads, typename T = double>
__global__ void __launch_bounds__(kThreads)
k_patch2_own_flags(const Control *__restrict__ ctl, const Patch2Args A) {
  const int b = blockIdx.x, cell0 = b * A.L.P, n_own = min(A.L.P, A.n_cells - cell0);
  const CellRecT<T> *__restrict__ rec = reinterpret_cast<const CellRecT<T> *>(ctl->cur ? A.rec_b : A.rec_a);
  int nonzero = 0;
  for (int l = threadIdx.x; l < n_own; l += kThreads) {
    const CellRecT<T> c = rec[cell0 + l];
    nonzero |= !(c.h == T(0.0) && c.qx == T(0.0) && c.qy == T(0.0));
    _Pragma("unroll") for (int sp = 0; sp < kMaxSpecies; ++sp) if (sp < A.sc.n) nonzero |= ((ctl->cur ? A.sc.qb[sp] : A.sc.qa[sp])[cell0 + l] != 0.0);
  }
  nonzero = __syncthreads_or(nonzero);
  if (threadIdx.x == 0) {
    (ctl->cur ? A.pflag_b : A.pflag_a)[(size_t)b * kPflagBytes + kPflagOwn] = nonzero ? 0 : 1;
    (ctl->cur ? A.pflag_a : A.pflag_b)[(size_t)b * kPflagBytes + kPflagOwn] = 0;
  }
}

// one block per patch: neighbour byte j = 1 when every halo cell of this patch that the j-th neighbour owns is
// (0, 0, 0) (and carries no scalar mass) in the newest state; the other buffer: unknown = 0
template <typename T = double>
__global__ void __launch_bounds__(kBlock)
k_patch2_nbr_flags(const Control *__restrict__ ctl, const Patch2Args A, int n_patches) {
  const int p = blockIdx.x;
  if (p >= n_patches) return;
  __shared__ uint32_t s_dirty;
  const unsigned char *blob = A.blob + (size_t)p * (size_t)A.L.stride;
  const BlobHeader H = *reinterpret_cast<const BlobHeader *>(blob);
  const int32_t *nbr = (const int32_t *)(blob + A.L.off_nbr);
  const int32_t *halo_ids = (const int32_t *)(blob + A.L.off_halo_ids);
  const CellRecT<T> *__restrict__ rec = reinterpret_cast<const CellRecT<T> *>(ctl->cur ? A.rec_b : A.rec_a);
  if (threadIdx.x == 0) s_dirty = 0u;
  __syncthreads();
  for (int l = threadIdx.x; l < H.n_r1 + H.n_r2; l += kBlock) {
    const int id = halo_ids[l];
    const CellRecT<T> c = rec[id];
    bool nz = !(c.h == T(0.0) && c.qx == T(0.0) && c.qy == T(0.0));
    _Pragma("unroll") for (int sp = 0; sp < kMaxSpecies; ++sp) if (sp < A.sc.n) nz = nz || ((ctl->cur ? A.sc.qb[sp] : A.sc.qa[sp])[id] != 0.0);
    if (!nz) continue;
    const int owner = id / A.L.P;
    for (int j = 0; j < H.n_nbr && j < kPflagSlots; ++j)
      if (nbr[j] == owner) { atomicOr(&s_dirty, 1u << j); break; }
  }
  __syncthreads();
  unsigned char *cur = (ctl->cur ? A.pflag_b : A.pflag_a), *oth = (ctl->cur ? A.pflag_a : A.pflag_b);
  const int j = threadIdx.x;
  if (j < kPflagSlots) {                          // unused slots never veto
    cur[(size_t)p * kPflagBytes + j] = j < H.n_nbr ? (unsigned char)(((s_dirty >> j) & 1u) ^ 1u) : 1;
    oth[(size_t)p * kPflagBytes + j] = j < H.n_nbr ? 0 : 1;
  }
  if (j == 0) {
    const unsigned char skippable = (H.n_string_edges == 0 && H.n_nbr <= kPflagSlots) ? 1 : 0;
    cur[(size_t)p * kPflagBytes + kPflagSkippable] = skippable;
    oth[(size_t)p * kPflagBytes + kPflagSkippable] = skippable;
  }
}

}  // namespace swe
