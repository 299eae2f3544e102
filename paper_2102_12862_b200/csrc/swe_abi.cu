// C-ABI of include/swe.h: context, workspace carving, upload, CUDA-graph step loop.  Host logic only;
// every step of the numerical path runs in the kernels of swe_kernels.cuh / swe_patch2_kernel.cuh.
//
// Device memory: ONE block, laid out by `Layout` from the sizes a host-only planning pass (`make_plan`) finds --
// the caller's workspace (swe_params.workspace, sized by swe_workspace_bytes, which runs the same planning pass), or,
// when none is lent, one cudaMalloc of that size.  Nothing else is allocated on the device while a context lives.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <limits>
#include <map>
#include <new>
#include <string>
#include <vector>

#include "../../include/swe.h"
#include "mesh_prep.hpp"
#include "patch_blob.hpp"
#include "swe_kernels.cuh"
#include "swe_patch_inst.cuh"
#include "swe_types.h"

using namespace swe;

namespace {

thread_local std::string g_create_error;

constexpr size_t kAlign = 256;
inline size_t align_up(size_t x) { return (x + kAlign - 1) / kAlign * kAlign; }
constexpr int kParamsPool = 16384;        // doubles reserved for the boundary strings' parameter tables (hydrographs)
constexpr size_t kSmemPerSM = 228 * 1024, kSmemPerBlockMax = 227 * 1024, kSmemBlockReserve = 1024;

// What the planning pass finds out about a context: every size that decides the device layout.
struct Sizes {
  int64_t nc = 0, ne = 0;
  int n_species = 0;
  bool morph = false;                     // room for the mobile-bed module (swe_params.morphology)
  bool single = false;                    // swe_params.precision = SWE_PRECISION_SINGLE: 4-byte reals, 16-byte records
  int64_t n_strings = 0, n_string_edges = 0, scratch = 0;
  int64_t n_patches = 0, blob_bytes = 0;  // fused patch step (0: the context has no patch step)
};

// Offsets of the device arrays inside the workspace, in carving order.
struct Layout {
  size_t rec, rec_b, geom, geomR, flux, cell_edge, area, inv_area, gn2, kst, theta, cell_perm, edge_perm, stage, drain_flag;
  size_t ctl, info_part, info_ticket, strings, string_edges, scratch, params, slot_string, string_M, string_lk, string_cell;
  size_t qa[kMaxSpecies], qb[kMaxSpecies], phi_up[kMaxSpecies], scalar_stage;
  size_t blob, pflag;
  size_t qB, mcell;
  size_t total;
  explicit Layout(const Sizes &z) {
    size_t o = 0;
    auto take = [&](size_t bytes) { size_t at = o; o += align_up(std::max<size_t>(bytes, 16)); return at; };
    const size_t nc = (size_t)z.nc, ne = (size_t)z.ne, nse = (size_t)std::max<int64_t>(1, z.n_string_edges);
    const size_t r = z.single ? 4 : 8;      // bytes of a real; records are 4 reals
    rec = take(4 * r * nc);
    rec_b = take(4 * r * nc);                  // second state buffer of the fused patch step
    geom = take(4 * r * ne);
    geomR = z.single ? take(4 * ne) : 0;    // fp32: R of every edge beside the 16-byte geometry record
    flux = take(4 * r * ne);
    cell_edge = take(sizeof(int4) * nc);
    area = take(r * nc); inv_area = take(r * nc); gn2 = take(r * nc); kst = take(r * nc); theta = take(r * nc);
    cell_perm = take(4 * nc); edge_perm = take(4 * ne);
    stage = take(std::max(24 * nc, 16 * ne));           // host <-> device staging of set / get calls
    drain_flag = take(nc + 16);                         // read four bytes at a time
    ctl = take(sizeof(Control));
    info_part = take(sizeof(InfoPartial) * kInfoMaxBlocks);
    info_ticket = take(sizeof(unsigned int));
    strings = take(sizeof(BoundaryString) * (size_t)std::max<int64_t>(1, z.n_strings));
    string_edges = take(4 * nse);
    scratch = take(8 * (size_t)std::max<int64_t>(1, z.scratch));
    params = take(8 * (size_t)kParamsPool);
    slot_string = take(4 * nse);
    string_M = take(2 * 8 * nse);                       // two buffers: the self-controlled patch step alternates
    string_lk = take(8 * nse); string_cell = take(4 * nse);
    for (int sp = 0; sp < kMaxSpecies; ++sp) {
      qa[sp] = qb[sp] = phi_up[sp] = 0;
      if (sp < z.n_species) { qa[sp] = take(8 * nc); qb[sp] = take(8 * nc); phi_up[sp] = take(8 * ne); }
    }
    scalar_stage = z.n_species > 0 ? take(8 * nc) : 0;
    blob = z.n_patches > 0 ? take((size_t)z.blob_bytes) : 0;
    pflag = z.n_patches > 0 ? take(2 * (size_t)kPflagBytes * (size_t)z.n_patches) : 0;
    qB = z.morph ? take(8 * ne) : 0;
    mcell = z.morph ? take(16 * nc) : 0;
    total = o;
  }
};

inline int grid_for(int64_t n) { return (int)((n + kBlock - 1) / kBlock); }

// ---- the fused patch kernel's instantiations: one thread per own cell (P = threads), __launch_bounds__ minimum
// blocks per SM chosen from what the shared memory admits (it only caps the registers)
// (T threads per block >= cells per patch, __launch_bounds__ minimum blocks per SM, getter of the instance for
// [scalars][self-controlled][mobile bed]; the instances live in swe_patch_t*.cu, one translation unit per block size)
struct PatchInst { int T, min_blocks; PatchKernel (*get)(int B, int scalars, int self, int morph); bool f32_only = false; };
const PatchInst kPatchInst[] = {{32, 8, patch_kernel_32}, {64, 8, patch_kernel_64}, {128, 6, patch_kernel_128}, {128, 4, patch_kernel_128},
                                {192, 5, patch_kernel_192}, {192, 4, patch_kernel_192}, {192, 3, patch_kernel_192},
                                {256, 6, patch_kernel_256, true}, {256, 5, patch_kernel_256, true}, {256, 4, patch_kernel_256}, {256, 3, patch_kernel_256},
                                {256, 2, patch_kernel_256}, {384, 2, patch_kernel_384}, {384, 1, patch_kernel_384}, {512, 2, patch_kernel_512}, {512, 1, patch_kernel_512},
                                {1024, 1, patch_kernel_1024}};

inline int patch_threads(int P) {           // the smallest block size of an instance that gives every own cell a thread
  int T = 1 << 30;
  for (const PatchInst &pi : kPatchInst) if (pi.T >= P && pi.T < T) T = pi.T;
  return T;
}

// the instantiation with the most blocks per SM that the shared memory of one block admits (force_blocks > 0: that one)
inline const PatchInst *pick_patch_kernel(int T, size_t smem, int force_blocks, bool single = false) {
  const int fit = (int)(kSmemPerSM / (smem + kSmemBlockReserve));
  const PatchInst *best = nullptr;
  for (const PatchInst &pi : kPatchInst) {
    if (pi.T != T || (pi.f32_only && !single)) continue;
    if (force_blocks > 0) { if (pi.min_blocks == force_blocks) return &pi; continue; }
    if (pi.min_blocks <= std::max(1, fit) && (!best || pi.min_blocks > best->min_blocks)) best = &pi;
  }
  if (!best)
    for (const PatchInst &pi : kPatchInst)
      if (pi.T == T && !(pi.f32_only && !single) && (!best || pi.min_blocks < best->min_blocks)) best = &pi;
  return best;
}

// Everything the host works out before the first CUDA call (shared by swe_workspace_bytes and swe_create)
struct Plan {
  HostMesh hm;
  Sizes z;
  std::vector<BoundaryString> strings;
  std::vector<int32_t> flat;             // string_edges[]: members of all strings, internal edge ids
  std::vector<int32_t> slot_string;      // string id of every position of flat[]
  std::vector<double> string_lk;         // l_e * k_weight(k_st of cell L) of every position of flat[] (R-11)
  std::vector<int32_t> string_cell;      // cell L of every position of flat[]
  std::vector<EdgeGeom> geom;            // internal numbering
  std::vector<int32_t> ce4;
  std::vector<double> area, inv_area, gn2, kst;
  int variant = SWE_VARIANT_THREE_PASS;  // the variant the context starts with
  bool has_patch = false, auto_mode = false;
  PatchBlobs pb;
  size_t patch_smem = 0;
};

}  // namespace

struct swe_ctx {
  int64_t nc = 0, ne = 0;
  swe_params prm{};
  HostMesh hm;
  cudaStream_t stream = nullptr;
  char *ws = nullptr;
  bool own_ws = false;
  // device arrays (inside ws)
  CellRec *rec = nullptr, *rec_b = nullptr; EdgeGeom *geom = nullptr; EdgeFlux *flux = nullptr; int4 *cell_edge = nullptr;
  double *area = nullptr, *inv_area = nullptr, *gn2 = nullptr, *kst = nullptr, *theta = nullptr;
  int *cell_perm = nullptr, *edge_perm = nullptr;
  double *stage = nullptr;
  Control *d_ctl = nullptr;
  Control *h_ctl = nullptr;          // pinned host memory
  BoundaryString *d_strings = nullptr;
  int *d_string_edges = nullptr;
  double *d_scratch = nullptr;
  double *d_params = nullptr;        // pool of kParamsPool doubles; bump-allocated by swe_set_boundary
  int64_t params_used = 0;
  std::vector<BoundaryString> strings;
  std::vector<int64_t> param_off, param_cap;     // per string: its slice of the pool
  // fused patch step (variant SWE_VARIANT_PATCH)
  int variant = 0;
  bool has_patch = false;
  BlobLayout blay{};
  unsigned char *d_blob = nullptr, *d_pflag = nullptr;
  int32_t *d_slot_string = nullptr; double *d_string_M = nullptr;
  double *d_string_lk = nullptr; int32_t *d_string_cell = nullptr;
  bool self_ctl = false;             // fused patch step without k_step_control (every block derives dt itself)
  int64_t step_idx = 0;              // step launches enqueued so far (self_ctl: launch n reads Control::slot[n % 4])
  int64_t n_string_edges = 0;
  int patch_force_blocks = 0;        // SWE_PATCH_MIN_BLOCKS (measurement runs): pin the __launch_bounds__ instance
  int n_patches = 0, patch_threads = 0, patch_prefetch = 0; size_t patch_smem = 0;
  int64_t patch_sum_loc = 0, patch_sum_e = 0; int patch_max_loc = 0, patch_max_e = 0, patch_min_blocks = 0;
  InfoPartial *d_info_part = nullptr; unsigned int *d_info_ticket = nullptr;
  int cell_grid = 148 * 4;           // resident blocks of the persistent k_cell_update
  int edge_grid = 148 * 5;           // resident blocks of the persistent k_edge_flux (set from the occupancy API)
  int base_edge_grid = 0, base_cell_grid = 0, sms = 148;
  Morph mp{};                        // morphodynamics (swe_set_morphology); formula 0 = fixed bed
  bool morph_reserved = false;
  bool single = false;               // single precision: the typed pointers above hold CellRecT<float> etc. (view<T>())
  int32_t *geomR = nullptr;          // fp32: R of every edge
  uint8_t *d_drain_flag = nullptr;   // three-pass step: cells flagged as possible drainers (lazy theta)
  Scalars sc{};                      // passive scalars
  double *d_scalar_stage = nullptr;  // [n_cells] staging of one species for host-pointer set / get
  int64_t alg_bytes_base[2] = {};        // three-pass k_edge_flux / k_cell_update without the mobile bed
  int64_t alg_bytes_v[3][4] = {};        // [variant][kernel]: algorithmic DRAM bytes per launch of the kernels of a step
  int64_t survey_bytes_v[3][4] = {};     // the same on SURVEY.md section 8(d)'s per-cell figures
  bool auto_mode = false;                // AUTO with both variants available: chosen at swe_set_state (wet fraction)
  cudaGraphExec_t graph_exec_v[3] = {nullptr, nullptr, nullptr};   // by variant
  int steps_per_graph = 0;
  int64_t launches = 0;
  double t_host = 0.0;               // t as of the last synchronisation
  std::string err;
};

namespace {

// the precision-dependent device arrays of a context, typed (fp64: the members themselves)
template <typename T> struct View {
  CellRecT<T> *rec, *rec_b; EdgeGeomT<T> *geom; EdgeFluxT<T> *flux; T *area, *inv_area, *gn2, *kst, *theta;
};
template <typename T> View<T> view(const swe_ctx *c) {
  View<T> v;
  v.rec = reinterpret_cast<CellRecT<T> *>(c->rec); v.rec_b = reinterpret_cast<CellRecT<T> *>(c->rec_b);
  v.geom = reinterpret_cast<EdgeGeomT<T> *>(c->geom); v.flux = reinterpret_cast<EdgeFluxT<T> *>(c->flux);
  v.area = reinterpret_cast<T *>(c->area); v.inv_area = reinterpret_cast<T *>(c->inv_area); v.gn2 = reinterpret_cast<T *>(c->gn2);
  v.kst = reinterpret_cast<T *>(c->kst); v.theta = reinterpret_cast<T *>(c->theta);
  return v;
}

#define SWE_CUDA(ctx, call)                                                                       \
  do {                                                                                            \
    cudaError_t e_ = (call);                                                                      \
    if (e_ != cudaSuccess) {                                                                      \
      (ctx)->err = std::string(#call) + ": " + cudaGetErrorString(e_);                            \
      return SWE_ECUDA;                                                                           \
    }                                                                                             \
  } while (0)

// the kernels of one time step, in stream order; ev (nullable) = n_step_kernels + 1 events recorded around them
constexpr int kMaxStepKernels = 4;
const char *const kThreePassNames[4] = {"k_step_control", "k_edge_flux", "k_theta_lazy", "k_cell_update"};
const char *const kPatchNames[2] = {"k_step_control", "k_patch_step"};
const char *const kSelfNames[1] = {"k_patch_step"};

inline bool self_mode(const swe_ctx *c) { return c->variant == SWE_VARIANT_PATCH && c->self_ctl && !c->single && c->mp.formula == 0; }
inline int n_step_kernels(const swe_ctx *c) { return self_mode(c) ? 1 : (c->variant == SWE_VARIANT_PATCH ? 2 : 4); }

Patch2Args patch_args(const swe_ctx *c) {
  Patch2Args a;
  a.blob = c->d_blob; a.L = c->blay;
  a.rec_a = c->rec; a.rec_b = c->rec_b; a.kst = c->kst;
  a.strings = c->d_strings; a.slot_string = c->d_slot_string; a.string_M = c->d_string_M;
  a.pflag_a = c->d_pflag; a.pflag_b = c->d_pflag + (size_t)kPflagBytes * (size_t)c->n_patches;
  a.n_cells = (int32_t)c->nc;
  a.step_k = (int32_t)(c->step_idx & 3); a.n_strings = (int32_t)c->strings.size(); a.n_string_edges = (int32_t)c->n_string_edges;
  a.string_lk = c->d_string_lk; a.string_cell = c->d_string_cell;
  a.prefetch_dist = c->patch_prefetch;
  a.sc = c->sc;
  a.mp = c->mp; a.gn2 = c->gn2;
  return a;
}

// dry flags of the patches from the state as it stands (after swe_set_state / swe_set_scalars / a variant switch)
void launch_patch_flags(swe_ctx *c) {
  const Patch2Args a = patch_args(c);
  if (c->single) {
    k_patch2_own_flags<256, float><<<c->n_patches, 256, 0, c->stream>>>(c->d_ctl, a);
    k_patch2_nbr_flags<float><<<c->n_patches, kBlock, 0, c->stream>>>(c->d_ctl, a, c->n_patches);
  } else {
    k_patch2_own_flags<256><<<c->n_patches, 256, 0, c->stream>>>(c->d_ctl, a);
    k_patch2_nbr_flags<double><<<c->n_patches, kBlock, 0, c->stream>>>(c->d_ctl, a, c->n_patches);
  }
  c->launches += 2;
}

template <typename T>
void launch_control_t(swe_ctx *c, cudaStream_t s, int mode) {
  const View<T> v = view<T>(c);
  k_step_control<T><<<1, kCtlThreads, 0, s>>>(c->d_ctl, c->d_strings, c->d_string_edges, c->d_scratch, v.geom, v.flux,
                                              (const T *)nullptr /* records are limited in place */, v.rec, v.rec_b, v.kst,
                                              c->variant == SWE_VARIANT_PATCH ? c->d_string_M : nullptr, mode);
}
void launch_control(swe_ctx *c, cudaStream_t s, int mode) {
  if (c->single) launch_control_t<float>(c, s, mode); else launch_control_t<double>(c, s, mode);
}

// single precision: the three-pass step in fp32 (16-byte records); no scalars / mobile bed / patch step
void enqueue_three_pass_f32(swe_ctx *c, cudaStream_t s, cudaEvent_t *ev) {
  const View<float> v = view<float>(c);
  k_edge_flux<false, true, false, float><<<std::min(grid_for(c->ne), c->edge_grid), kBlock, 0, s>>>(
      c->d_ctl, v.geom, v.rec, v.kst, c->d_strings, v.flux, (int)c->ne, 0, c->sc, v.area, c->d_drain_flag, Morph{}, c->geomR);
  if (ev) cudaEventRecord(ev[2], s);
  k_theta_lazy<float><<<grid_for((c->nc + 3) / 4), kBlock, 0, s>>>(c->d_ctl, c->cell_edge, v.geom, v.flux, v.rec, v.area, v.theta,
                                                                   c->d_drain_flag, (int)c->nc);
  if (ev) cudaEventRecord(ev[3], s);
  k_cell_update<false, false, float><<<std::min(grid_for(c->nc), c->cell_grid), kBlock, 0, s>>>(
      c->d_ctl, c->cell_edge, v.geom, v.flux, (const float *)nullptr, v.area, v.inv_area, v.gn2, v.rec, (int)c->nc, c->sc);
  if (ev) cudaEventRecord(ev[4], s);
}

// the fused patch kernel of this context: instance by (scalars, self-controlled, mobile bed); the shared memory of a
// block grows with the scalar species and the mobile-bed law
void launch_patch(swe_ctx *c, cudaStream_t s, int self) {
  const int morph = c->mp.formula;
  const size_t smem = (size_t)patch2_smem_layout(c->blay, c->sc.n, morph, self != 0).total;
  // most blocks per SM that fit -- unless the grid cannot fill them: then the instance with the larger register budget
  // (76 instead of 64 registers at 256 threads) is the faster one per block (configs[1]: 10.4 vs 11.8 us per step)
  int force = c->patch_force_blocks;
  if (!force && c->patch_threads == 256 && c->n_patches <= 3 * c->sms) force = 3;
  const PatchInst *pi = pick_patch_kernel(c->patch_threads, smem, force, c->single);
  pi->get(pi->min_blocks, c->sc.n > 0, c->single ? 4 : self, morph != 0)<<<c->n_patches, c->patch_threads, smem, s>>>(c->d_ctl, patch_args(c));
}

// one time step, in stream order.  Self-controlled patch step: the launch number decides the control slot it reads
void enqueue_step(swe_ctx *c, cudaStream_t s, cudaEvent_t *ev = nullptr) {
  if (self_mode(c)) {
    if (ev) cudaEventRecord(ev[0], s);
    launch_patch(c, s, 1);
    if (ev) cudaEventRecord(ev[1], s);
    c->step_idx += 1;
    return;
  }
  c->step_idx += 1;
  if (ev) cudaEventRecord(ev[0], s);
  launch_control(c, s, 0);
  if (ev) cudaEventRecord(ev[1], s);
  if (c->variant == SWE_VARIANT_PATCH) {
    launch_patch(c, s, 0);
    if (ev) cudaEventRecord(ev[2], s);
    return;
  }
  if (c->single) { enqueue_three_pass_f32(c, s, ev); return; }
  const double *no_theta = nullptr;         // the records are limited in place by k_theta_lazy
  if (c->mp.formula && c->sc.n > 0)
    k_edge_flux<true, false, true><<<grid_for(c->ne), kBlock, 0, s>>>(c->d_ctl, c->geom, c->rec, c->kst, c->d_strings, c->flux, (int)c->ne, 0, c->sc,
                                                               c->area, c->d_drain_flag, c->mp);
  else if (c->mp.formula)
    k_edge_flux<false, true, true><<<std::min(grid_for(c->ne), c->edge_grid), kBlock, 0, s>>>(c->d_ctl, c->geom, c->rec, c->kst, c->d_strings, c->flux, (int)c->ne, 0, c->sc,
                                                          c->area, c->d_drain_flag, c->mp);
  else if (c->sc.n > 0)
    k_edge_flux<true, false><<<grid_for(c->ne), kBlock, 0, s>>>(c->d_ctl, c->geom, c->rec, c->kst, c->d_strings, c->flux, (int)c->ne, 0, c->sc,
                                                         c->area, c->d_drain_flag);
  else
    k_edge_flux<false, true><<<std::min(grid_for(c->ne), c->edge_grid), kBlock, 0, s>>>(c->d_ctl, c->geom, c->rec, c->kst, c->d_strings, c->flux, (int)c->ne, 0, c->sc,
                                                          c->area, c->d_drain_flag);
  if (ev) cudaEventRecord(ev[2], s);
  k_theta_lazy<<<grid_for((c->nc + 3) / 4), kBlock, 0, s>>>(c->d_ctl, c->cell_edge, c->geom, c->flux, c->rec, c->area, c->theta,
                                                  c->d_drain_flag, (int)c->nc);
  if (ev) cudaEventRecord(ev[3], s);
  if (c->mp.formula && c->sc.n > 0)
    k_cell_update<true, true><<<std::min(grid_for(c->nc), c->cell_grid), kBlock, 0, s>>>(c->d_ctl, c->cell_edge, c->geom, c->flux, no_theta, c->area,
                                                                 c->inv_area, c->gn2, c->rec, (int)c->nc, c->sc, c->mp);
  else if (c->mp.formula)
    k_cell_update<false, true><<<std::min(grid_for(c->nc), c->cell_grid), kBlock, 0, s>>>(c->d_ctl, c->cell_edge, c->geom, c->flux, no_theta, c->area,
                                                                  c->inv_area, c->gn2, c->rec, (int)c->nc, c->sc, c->mp);
  else if (c->sc.n > 0)
    k_cell_update<true><<<std::min(grid_for(c->nc), c->cell_grid), kBlock, 0, s>>>(c->d_ctl, c->cell_edge, c->geom, c->flux, no_theta, c->area,
                                                           c->inv_area, c->gn2, c->rec, (int)c->nc, c->sc);
  else
    k_cell_update<false><<<std::min(grid_for(c->nc), c->cell_grid), kBlock, 0, s>>>(c->d_ctl, c->cell_edge, c->geom, c->flux, no_theta, c->area,
                                                            c->inv_area, c->gn2, c->rec, (int)c->nc, c->sc);
  if (ev) cudaEventRecord(ev[4], s);
}

int capture_graph(swe_ctx *c) {
  if (c->steps_per_graph <= 0) return SWE_OK;
  cudaStream_t cap;
  SWE_CUDA(c, cudaStreamCreateWithFlags(&cap, cudaStreamNonBlocking));
  SWE_CUDA(c, cudaStreamBeginCapture(cap, cudaStreamCaptureModeThreadLocal));
  const int64_t idx = c->step_idx;     // a graph launch always starts at a launch number that is a multiple of 4
  c->step_idx = 0;
  for (int k = 0; k < c->steps_per_graph; ++k) enqueue_step(c, cap);
  c->step_idx = idx;
  cudaGraph_t g = nullptr;
  SWE_CUDA(c, cudaStreamEndCapture(cap, &g));
  SWE_CUDA(c, cudaGraphInstantiate(&c->graph_exec_v[c->variant], g, 0));
  cudaGraphDestroy(g);
  SWE_CUDA(c, cudaStreamDestroy(cap));
  return SWE_OK;
}

int read_control(swe_ctx *c) {   // device -> pinned host, synchronises the stream
  SWE_CUDA(c, cudaMemcpyAsync(c->h_ctl, c->d_ctl, sizeof(Control), cudaMemcpyDeviceToHost, c->stream));
  SWE_CUDA(c, cudaStreamSynchronize(c->stream));
  c->t_host = c->h_ctl->t;
  return SWE_OK;
}

// start / end of a run of steps (swe_step, swe_profile_step): stop conditions in; bookkeeping of the last step out
void begin_call(swe_ctx *c, long long n_steps, double t_end, double cfl) {
  if (self_mode(c)) k_self_begin<<<1, 1, 0, c->stream>>>(c->d_ctl, n_steps, t_end, cfl, (int)(c->step_idx & 3));
  else k_call_begin<<<1, 1, 0, c->stream>>>(c->d_ctl, n_steps, t_end, cfl);
  c->launches += 1;
}
void end_call(swe_ctx *c, int final) {
  if (self_mode(c))
    k_self_finish<256><<<1, 256, 0, c->stream>>>(c->d_ctl, c->d_strings, (int)c->strings.size(), c->d_string_M, (int)c->n_string_edges,
                                                  (int)(c->step_idx & 3), final);
  else if (final) launch_control(c, c->stream, 1);
  else return;
  c->launches += 1;
}

void release(swe_ctx *c) {
  if (!c) return;
  for (auto &ge : c->graph_exec_v) if (ge) cudaGraphExecDestroy(ge);
  if (c->h_ctl) cudaFreeHost(c->h_ctl);
  if (c->own_ws && c->ws) cudaFree(c->ws);
  delete c;
}

// AUTO: makes `want` the active variant for the state as it is now (no step in flight).  cur = Control::cur as last
// read.  The three-pass step works in place in buffer a; the patch step ping-pongs and needs its dry flags.
int switch_variant(swe_ctx *c, int want, int cur) {
  if (want == c->variant) return SWE_OK;
  const int64_t nc = c->nc;
  if (want == SWE_VARIANT_THREE_PASS && cur == 1) {
    SWE_CUDA(c, cudaMemcpyAsync(c->rec, c->rec_b, (c->single ? sizeof(CellRecT<float>) : sizeof(CellRec)) * nc, cudaMemcpyDeviceToDevice, c->stream));
    for (int sp = 0; sp < c->sc.n; ++sp)
      SWE_CUDA(c, cudaMemcpyAsync(c->sc.qa[sp], c->sc.qb[sp], 8 * nc, cudaMemcpyDeviceToDevice, c->stream));
  }
  c->variant = want;
  k_set_variant<<<1, 1, 0, c->stream>>>(c->d_ctl, want == SWE_VARIANT_PATCH ? 1 : 0, 0);
  c->launches += 1;
  if (want == SWE_VARIANT_PATCH) launch_patch_flags(c);
  if (want == SWE_VARIANT_THREE_PASS && c->mp.formula == 2) {     // the patch step does not keep Morph::cell
    k_sed_cell_init<<<grid_for(nc), kBlock, 0, c->stream>>>(c->d_ctl, c->rec, c->gn2, c->mp.cell, (int)nc);
    c->launches += 1;
  }
  SWE_CUDA(c, cudaGetLastError());
  return SWE_OK;
}

int upload_strings(swe_ctx *c) {
  if (c->strings.empty()) return SWE_OK;
  SWE_CUDA(c, cudaMemcpyAsync(c->d_strings, c->strings.data(), sizeof(BoundaryString) * c->strings.size(),
                              cudaMemcpyHostToDevice, c->stream));
  SWE_CUDA(c, cudaStreamSynchronize(c->stream));
  return SWE_OK;
}

// sum of the member lengths of every string, by the same pairwise tree as the per-step sums
template <typename T>
__global__ void __launch_bounds__(kCtlThreads)
k_string_lengths(BoundaryString *strings, int n_strings, const int *__restrict__ string_edges, double *scratch_,
                 const EdgeGeomT<T> *__restrict__ geom) {
  T *scratch = reinterpret_cast<T *>(scratch_);
  for (int s = 0; s < n_strings; ++s) {
    BoundaryString &bs = strings[s];
    if (bs.n_edges == 0) continue;
    T *v = scratch + bs.scratch;
    for (int j = threadIdx.x; j < bs.pow2; j += blockDim.x) v[j] = j < bs.n_edges ? geom[string_edges[bs.first + j]].len : T(0.0);
    const T sum = block_tree_sum(v, bs.pow2);
    if (threadIdx.x == 0) bs.sumL = (double)sum;
    __syncthreads();
  }
}

// Host part of swe_create: edge tables (given or built), validation + geometry of section 4.1, renumbering.
int host_prepare(const swe_mesh *mesh, int renumber_mode, HostMesh &hm, std::string &err) {
  const int64_t nc = mesh->n_cells, nn = mesh->n_nodes;
  hm.nc = nc; hm.nn = nn;
  if (mesh->edge_cell && mesh->cell_edge) {
    if (mesh->n_edges <= 0 || mesh->n_edges > 3 * nc) { err = "n_edges out of range"; return SWE_EINVAL; }
    hm.ne = mesh->n_edges;
    hm.edge_cell.assign(mesh->edge_cell, mesh->edge_cell + 2 * hm.ne);
    hm.cell_edge.assign(mesh->cell_edge, mesh->cell_edge + 3 * nc);
  } else if (!mesh->edge_cell && !mesh->cell_edge) {
    if (!build_tables(nc, nn, mesh->tri, hm, err)) return SWE_EMESH;
  } else {
    err = "edge_cell and cell_edge must be given together or both be NULL";
    return SWE_EINVAL;
  }
  if (!validate_and_measure(nc, nn, mesh->node_xy, mesh->tri, hm, err)) return SWE_EMESH;
  for (int64_t i = 0; i < nc; ++i) {
    const double k = mesh->kst[i];
    if (!(k > 0.0) || !std::isfinite(mesh->zb[i])) { err = "cell " + std::to_string(i) + ": kst must be > 0 (or +inf), zb finite"; return SWE_EINVAL; }
  }
  if (renumber_mode < 0 || renumber_mode > 2) { err = "unknown renumbering"; return SWE_EINVAL; }
  renumber(renumber_mode, nc, mesh->node_xy, mesh->tri, hm);
  return SWE_OK;
}

int check_args(const swe_mesh *mesh, std::string &err) {
  if (!mesh || !mesh->node_xy || !mesh->tri || !mesh->zb || !mesh->kst) { err = "null argument"; return SWE_EINVAL; }
  if (mesh->n_cells <= 0 || mesh->n_nodes <= 0 || mesh->n_cells > (int64_t)0x7fffffff / 3) { err = "n_cells / n_nodes out of range"; return SWE_EINVAL; }
  return SWE_OK;
}

int check_params(const swe_params &p, std::string &err) {
  if (!(p.g > 0.0) || !(p.h_dry >= 0.0) || !(p.dt_max > 0.0)) { err = "g, h_dry, dt_max out of range"; return SWE_EINVAL; }
  if (p.n_species < 0 || p.n_species > kMaxSpecies) { err = "n_species must be in [0, 5] (P:208)"; return SWE_EINVAL; }
  if (p.variant != SWE_VARIANT_AUTO && p.variant != SWE_VARIANT_THREE_PASS && p.variant != SWE_VARIANT_PATCH) { err = "unknown variant"; return SWE_EINVAL; }
  if (p.precision != SWE_PRECISION_DOUBLE && p.precision != SWE_PRECISION_SINGLE) { err = "unknown precision"; return SWE_EINVAL; }
  if (p.precision == SWE_PRECISION_SINGLE && (p.n_species > 0 || p.morphology)) {
    err = "single precision is built for the hydrodynamic step only (no scalars, no mobile bed)"; return SWE_EINVAL;
  }
  if (p.patch_cells != 0 && (p.patch_cells < 32 || p.patch_cells > 1024)) { err = "patch_cells must be 0 (default) or in [32, 1024]"; return SWE_EINVAL; }
  return SWE_OK;
}

// The planning pass: host preprocessing, boundary strings, internal-numbering tables, patch blobs (emit: with their
// bytes; else capacities only) and from those every size of the device layout.  No CUDA call.
int make_plan(const swe_mesh *mesh, const swe_params &p, bool emit, Plan &pl, std::string &err) {
  int rc = check_args(mesh, err);
  if (rc != SWE_OK) return rc;
  rc = check_params(p, err);
  if (rc != SWE_OK) return rc;
  HostMesh &hm = pl.hm;
  rc = host_prepare(mesh, p.renumber, hm, err);
  if (rc != SWE_OK) return rc;
  const int64_t nc = hm.nc, ne = hm.ne;
  pl.z.nc = nc; pl.z.ne = ne; pl.z.n_species = p.n_species; pl.z.morph = p.morphology != 0;
  pl.z.single = p.precision == SWE_PRECISION_SINGLE;

  // ---- arrays in internal numbering
  pl.geom.resize(ne); pl.ce4.resize((size_t)4 * nc);
  pl.area.resize(nc); pl.inv_area.resize(nc); pl.gn2.resize(nc); pl.kst.resize(nc);
  for (int64_t i = 0; i < nc; ++i) {
    const int32_t o = hm.cell_perm[i];
    for (int k = 0; k < 3; ++k) pl.ce4[4 * i + k] = hm.edge_new[hm.cell_edge[3 * o + k]];
    pl.ce4[4 * i + 3] = 0;
    const double A = hm.area[o], k = mesh->kst[o];
    pl.area[i] = A;
    pl.inv_area[i] = 1.0 / A;
    pl.gn2[i] = std::isfinite(k) ? p.g / (k * k) : 0.0;    // g / k_str^2 (Eq. 2 P:106-111 with Table 1, R-6)
    pl.kst[i] = k;
  }
  for (int64_t e = 0; e < ne; ++e) {
    const int32_t o = hm.edge_perm[e];
    const int32_t L = hm.edge_cell[2 * o], R = hm.edge_cell[2 * o + 1];
    pl.geom[e] = {hm.nx[o], hm.ny[o], hm.len[o], hm.cell_new[L], R >= 0 ? hm.cell_new[R] : R};
  }

  // ---- boundary strings: members in ascending caller edge id ("string order", R-11)
  int max_id = -1;
  for (int64_t e = 0; e < ne; ++e) {
    const int32_t R = hm.edge_cell[2 * e + 1];
    if (R <= -3) max_id = std::max(max_id, -3 - R);
  }
  if (max_id > 65535) { err = "boundary string id too large"; return SWE_EINVAL; }
  pl.strings.assign(max_id + 1, BoundaryString{});
  std::vector<std::vector<int32_t>> members(max_id + 1);
  for (int64_t e = 0; e < ne; ++e) {
    const int32_t R = hm.edge_cell[2 * e + 1];
    if (R <= -3) members[-3 - R].push_back(hm.edge_new[e]);
  }
  size_t scratch = 0;
  for (int s = 0; s <= max_id; ++s) {
    BoundaryString &bs = pl.strings[s];
    bs.n_edges = (int32_t)members[s].size();
    bs.first = (int32_t)pl.flat.size();
    int32_t P2 = 1;
    while (P2 < bs.n_edges) P2 <<= 1;
    bs.pow2 = P2;
    bs.scratch = (int32_t)scratch;
    scratch += P2;
    pl.flat.insert(pl.flat.end(), members[s].begin(), members[s].end());
  }
  pl.slot_string.assign(std::max<size_t>(1, pl.flat.size()), 0);
  for (int s = 0; s <= max_id; ++s)
    for (int32_t j = 0; j < pl.strings[s].n_edges; ++j) pl.slot_string[pl.strings[s].first + j] = s;
  pl.z.n_strings = max_id + 1; pl.z.n_string_edges = (int64_t)pl.flat.size(); pl.z.scratch = (int64_t)scratch;
  pl.string_lk.assign(std::max<size_t>(1, pl.flat.size()), 0.0); pl.string_cell.assign(std::max<size_t>(1, pl.flat.size()), 0);
  for (size_t j = 0; j < pl.flat.size(); ++j) {
    const EdgeGeom &eg = pl.geom[pl.flat[j]];
    const double k = pl.kst[eg.L];
    pl.string_lk[j] = eg.len * (std::isfinite(k) ? k : 1.0);
    pl.string_cell[j] = eg.L;
  }

  // ---- fused patch step: patch blobs, shared-memory size
  pl.variant = p.variant == SWE_VARIANT_THREE_PASS ? SWE_VARIANT_THREE_PASS : SWE_VARIANT_PATCH;
  const int rb = pl.z.single ? 4 : 8;      // bytes of a real in the patch blobs
  if (pl.variant == SWE_VARIANT_PATCH) {
    // default: the largest patch of 240, 232, 224, 208, 192 cells (256 threads each) whose block still fits an SM four
    // times -- 32 warps per SM; the kernel is latency-bound and 4 x 8 warps beat 3 x 8 by 10-13 %, larger patches beat
    // smaller ones by 1-2 % per step of 8 cells (profiles/r2q_patch_size_sweep.md); small meshes get smaller patches, so that
    // the launch-latency-bound step still spreads over the SMs
    std::vector<int32_t> string_pos(ne, -1);
    for (size_t j = 0; j < pl.flat.size(); ++j) string_pos[pl.flat[j]] = (int32_t)j;
    int P = p.patch_cells;
    if (P <= 0 && nc < 148 * 256) P = nc < 148 * 64 ? 32 : (nc < 148 * 128 ? 64 : 128);
    if (P <= 0) {
      const bool self = false;               // (meshes of this size do not run the self-controlled step)
      // (single precision: 34-36 KB per block and 40 registers -- six blocks per SM, patches of up to 256 cells:
      // 95.5 us per step on the river reach against 107.9 at four blocks of 240 cells, profiles/r2u_single_precision.md)
      const int blocks_wanted = pl.z.single ? 6 : 4;
      for (int cand : {256, 248, 240, 232, 224, 208, 192}) {
        if (cand > 240 && !pl.z.single) continue;
        P = cand;
        if (!build_blobs(nc, ne, pl.geom, pl.ce4, pl.area, pl.inv_area, pl.gn2, string_pos, P, false, pl.pb, err, rb)) return SWE_EINVAL;
        const size_t smem = (size_t)patch2_smem_layout(pl.pb.lay, p.n_species, 0, self && nc / P <= 8192).total;
        if (blocks_wanted * (smem + kSmemBlockReserve) <= kSmemPerSM) break;
      }
    }
    if (!build_blobs(nc, ne, pl.geom, pl.ce4, pl.area, pl.inv_area, pl.gn2, string_pos, P, emit, pl.pb, err, rb)) return SWE_EINVAL;
    pl.patch_smem = (size_t)patch2_smem_layout(pl.pb.lay, p.n_species).total;
    // a numbering that is not spatially compact (renumber = NONE on a scattered input order) blows the halos up:
    // more than 2.2 local cells per own cell, or a block that no longer fits an SM twice -> AUTO falls back to the
    // three-pass step (round 1: such patches were 2-3x slower than the three-pass step)
    // (small patches of small meshes have fat halos by geometry: 2.5 local cells per own cell at 32 cells)
    const bool bloated = (double)pl.pb.sum_loc > (P >= 192 ? 2.2 : 4.5) * (double)nc || pl.patch_smem + kSmemBlockReserve > kSmemPerSM / 2;
    if (pl.patch_smem > kSmemPerBlockMax || (p.variant == SWE_VARIANT_AUTO && bloated)) {
      if (p.variant == SWE_VARIANT_AUTO) { pl.variant = SWE_VARIANT_THREE_PASS; pl.pb = PatchBlobs{}; pl.patch_smem = 0; }
      else { err = "patch needs more shared memory than an SM has: lower patch_cells or renumber"; return SWE_EINVAL; }
    }
  }
  pl.has_patch = (pl.variant == SWE_VARIANT_PATCH);
  pl.auto_mode = (p.variant == SWE_VARIANT_AUTO && pl.has_patch);
  if (pl.has_patch) { pl.z.n_patches = pl.pb.n_patches; pl.z.blob_bytes = (int64_t)pl.pb.lay.stride * pl.pb.n_patches; }
  return SWE_OK;
}

int create_impl(const swe_mesh *mesh, const swe_params *params, swe_ctx *c) {
  if (params) c->prm = *params; else swe_params_default(&c->prm);
  const swe_params &p = c->prm;
  c->stream = (cudaStream_t)p.cuda_stream;
  c->steps_per_graph = p.steps_per_graph;

  // ---- host: tables, validation, geometry, numbering, boundary strings, patch blobs, device layout
  Plan pl;
  {
    int rc = make_plan(mesh, p, true, pl, c->err);
    if (rc != SWE_OK) return rc;
  }
  c->hm = std::move(pl.hm);
  const int64_t nc = c->nc = pl.z.nc, ne = c->ne = pl.z.ne;
  const Layout lay(pl.z);

  // ---- workspace: the caller's, or one allocation of the same size
  if (p.workspace) {
    if (p.workspace_bytes < lay.total) { c->err = "workspace too small: need " + std::to_string(lay.total) + " bytes (swe_workspace_bytes)"; return SWE_ENOMEM; }
    if (((uintptr_t)p.workspace) % kAlign != 0) { c->err = "workspace must be 256-byte aligned"; return SWE_EINVAL; }
    c->ws = (char *)p.workspace;
  } else {
    cudaError_t e = cudaMalloc((void **)&c->ws, lay.total);
    if (e == cudaErrorMemoryAllocation) { cudaGetLastError(); c->ws = nullptr; c->err = "out of device memory (" + std::to_string(lay.total) + " bytes)"; return SWE_ENOMEM; }
    SWE_CUDA(c, e);
    c->own_ws = true;
  }
  char *ws = c->ws;
  c->single = pl.z.single;
  if (c->single) c->geomR = (int32_t *)(ws + lay.geomR);
  c->rec = (CellRec *)(ws + lay.rec); c->rec_b = (CellRec *)(ws + lay.rec_b); c->geom = (EdgeGeom *)(ws + lay.geom); c->flux = (EdgeFlux *)(ws + lay.flux);
  c->cell_edge = (int4 *)(ws + lay.cell_edge);
  c->area = (double *)(ws + lay.area); c->inv_area = (double *)(ws + lay.inv_area);
  c->gn2 = (double *)(ws + lay.gn2); c->kst = (double *)(ws + lay.kst); c->theta = (double *)(ws + lay.theta);
  c->cell_perm = (int *)(ws + lay.cell_perm); c->edge_perm = (int *)(ws + lay.edge_perm);
  c->stage = (double *)(ws + lay.stage);
  c->d_drain_flag = (uint8_t *)(ws + lay.drain_flag);
  c->d_ctl = (Control *)(ws + lay.ctl);
  c->d_info_part = (InfoPartial *)(ws + lay.info_part); c->d_info_ticket = (unsigned int *)(ws + lay.info_ticket);
  c->d_strings = (BoundaryString *)(ws + lay.strings); c->d_string_edges = (int *)(ws + lay.string_edges);
  c->d_scratch = (double *)(ws + lay.scratch); c->d_params = (double *)(ws + lay.params);
  c->d_slot_string = (int32_t *)(ws + lay.slot_string); c->d_string_M = (double *)(ws + lay.string_M);
  c->d_string_lk = (double *)(ws + lay.string_lk); c->d_string_cell = (int32_t *)(ws + lay.string_cell);
  c->n_string_edges = (int64_t)std::max<size_t>(1, pl.flat.size());
  c->sc.n = p.n_species;
  for (int sp = 0; sp < c->sc.n; ++sp) {
    c->sc.qa[sp] = (double *)(ws + lay.qa[sp]); c->sc.qb[sp] = (double *)(ws + lay.qb[sp]); c->sc.phi_up[sp] = (double *)(ws + lay.phi_up[sp]);
  }
  if (c->sc.n > 0) c->d_scalar_stage = (double *)(ws + lay.scalar_stage);
  c->morph_reserved = pl.z.morph;
  if (pl.z.morph) { c->mp.qB = (double *)(ws + lay.qB); c->mp.cell = (double2 *)(ws + lay.mcell); }
  SWE_CUDA(c, cudaMallocHost((void **)&c->h_ctl, sizeof(Control)));

  // ---- upload
  {
    auto up = [&](void *dst, const void *src, size_t bytes) { return bytes ? cudaMemcpy(dst, src, bytes, cudaMemcpyHostToDevice) : cudaSuccess; };
    if (!c->single) {
      std::vector<CellRec> rec(nc);
      for (int64_t i = 0; i < nc; ++i) rec[i] = {0.0, 0.0, 0.0, mesh->zb[c->hm.cell_perm[i]]};
      std::vector<double> theta(nc, 1.0);
      SWE_CUDA(c, up(c->rec, rec.data(), sizeof(CellRec) * nc));
      SWE_CUDA(c, up(c->rec_b, rec.data(), sizeof(CellRec) * nc));     // z_B must be valid in both state buffers
      SWE_CUDA(c, up(c->area, pl.area.data(), 8 * nc));
      SWE_CUDA(c, up(c->inv_area, pl.inv_area.data(), 8 * nc));
      SWE_CUDA(c, up(c->gn2, pl.gn2.data(), 8 * nc));
      SWE_CUDA(c, up(c->kst, pl.kst.data(), 8 * nc));
      SWE_CUDA(c, up(c->theta, theta.data(), 8 * nc));
      SWE_CUDA(c, up(c->geom, pl.geom.data(), sizeof(EdgeGeom) * ne));
    } else {
      // single precision (R-21): geometry and constants are the fp64 values rounded ONCE to fp32
      const View<float> v = view<float>(c);
      std::vector<CellRecT<float>> rec(nc);
      std::vector<float> f(nc);
      for (int64_t i = 0; i < nc; ++i) rec[i] = {0.f, 0.f, 0.f, (float)mesh->zb[c->hm.cell_perm[i]]};
      SWE_CUDA(c, up(v.rec, rec.data(), sizeof(CellRecT<float>) * nc));
      SWE_CUDA(c, up(v.rec_b, rec.data(), sizeof(CellRecT<float>) * nc));   // z_B must be valid in both state buffers
      const std::vector<double> *srcs[4] = {&pl.area, &pl.inv_area, &pl.gn2, &pl.kst};
      float *dsts[4] = {v.area, v.inv_area, v.gn2, v.kst};
      for (int a = 0; a < 4; ++a) {
        for (int64_t i = 0; i < nc; ++i) f[i] = (float)(*srcs[a])[i];
        SWE_CUDA(c, up(dsts[a], f.data(), 4 * nc));
      }
      for (int64_t i = 0; i < nc; ++i) f[i] = 1.f;
      SWE_CUDA(c, up(v.theta, f.data(), 4 * nc));
      std::vector<EdgeGeomT<float>> g32(ne);
      std::vector<int32_t> gR(ne);
      for (int64_t e = 0; e < ne; ++e) { g32[e] = {(float)pl.geom[e].nx, (float)pl.geom[e].ny, (float)pl.geom[e].len, pl.geom[e].L}; gR[e] = pl.geom[e].R; }
      SWE_CUDA(c, up(v.geom, g32.data(), sizeof(EdgeGeomT<float>) * ne));
      SWE_CUDA(c, up(c->geomR, gR.data(), 4 * ne));
    }
    SWE_CUDA(c, up(c->cell_edge, pl.ce4.data(), sizeof(int4) * nc));
    SWE_CUDA(c, up(c->cell_perm, c->hm.cell_perm.data(), 4 * nc));
    SWE_CUDA(c, up(c->edge_perm, c->hm.edge_perm.data(), 4 * ne));
    SWE_CUDA(c, cudaMemset(c->flux, 0, (c->single ? sizeof(EdgeFluxT<float>) : sizeof(EdgeFlux)) * ne));
    SWE_CUDA(c, cudaMemset(c->d_drain_flag, 0, (size_t)nc + 16));
    SWE_CUDA(c, cudaMemset(c->d_info_ticket, 0, sizeof(unsigned int)));
    SWE_CUDA(c, up(c->d_string_edges, pl.flat.data(), 4 * pl.flat.size()));
    SWE_CUDA(c, up(c->d_slot_string, pl.slot_string.data(), 4 * pl.slot_string.size()));
    SWE_CUDA(c, cudaMemset(c->d_string_M, 0, 2 * 8 * std::max<size_t>(1, pl.flat.size())));
    SWE_CUDA(c, up(c->d_string_lk, pl.string_lk.data(), 8 * pl.string_lk.size()));
    SWE_CUDA(c, up(c->d_string_cell, pl.string_cell.data(), 4 * pl.string_cell.size()));
    for (int sp = 0; sp < c->sc.n; ++sp) {
      SWE_CUDA(c, cudaMemset(c->sc.qa[sp], 0, 8 * nc));
      SWE_CUDA(c, cudaMemset(c->sc.qb[sp], 0, 8 * nc));
      SWE_CUDA(c, cudaMemset(c->sc.phi_up[sp], 0, 8 * ne));
    }
    if (pl.z.morph) SWE_CUDA(c, cudaMemset(c->mp.qB, 0, 8 * ne));
  }
  c->strings = std::move(pl.strings);
  c->param_off.assign(c->strings.size(), 0); c->param_cap.assign(c->strings.size(), 0);
  if (!c->strings.empty()) {
    SWE_CUDA(c, cudaMemcpy(c->d_strings, c->strings.data(), sizeof(BoundaryString) * c->strings.size(), cudaMemcpyHostToDevice));
    if (c->single) k_string_lengths<float><<<1, kCtlThreads, 0, c->stream>>>(c->d_strings, (int)c->strings.size(), c->d_string_edges, c->d_scratch, view<float>(c).geom);
    else k_string_lengths<double><<<1, kCtlThreads, 0, c->stream>>>(c->d_strings, (int)c->strings.size(), c->d_string_edges, c->d_scratch, c->geom);
    SWE_CUDA(c, cudaGetLastError());
    SWE_CUDA(c, cudaStreamSynchronize(c->stream));
    SWE_CUDA(c, cudaMemcpy(c->strings.data(), c->d_strings, sizeof(BoundaryString) * c->strings.size(), cudaMemcpyDeviceToHost));
  }

  {
    int dev = 0, sms = 148, per_sm = 4;
    SWE_CUDA(c, cudaGetDevice(&dev));
    SWE_CUDA(c, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    SWE_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_edge_flux<false, true>, kBlock, 0));
    c->edge_grid = std::max(1, sms * per_sm);
    if (c->sc.n > 0) SWE_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_cell_update<true>, kBlock, 0));
    else SWE_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_cell_update<false>, kBlock, 0));
    c->cell_grid = std::max(1, sms * per_sm);
    if (c->single) {
      SWE_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_edge_flux<false, true, false, float>, kBlock, 0));
      c->edge_grid = std::max(1, sms * per_sm);
      SWE_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_cell_update<false, false, float>, kBlock, 0));
      c->cell_grid = std::max(1, sms * per_sm);
    }
    c->base_edge_grid = c->edge_grid; c->base_cell_grid = c->cell_grid; c->sms = sms;
  }

  // ---- fused patch step: blobs, flag words, kernel instance
  c->variant = pl.variant;
  c->has_patch = pl.has_patch;
  if (pl.has_patch) {
    const PatchBlobs &pb = pl.pb;
    c->blay = pb.lay;
    c->n_patches = (int)pb.n_patches;
    c->patch_smem = pl.patch_smem;
    c->patch_sum_loc = pb.sum_loc; c->patch_sum_e = pb.sum_e; c->patch_max_loc = pb.max_loc; c->patch_max_e = pb.max_e;
    c->d_blob = (unsigned char *)(ws + lay.blob); c->d_pflag = (unsigned char *)(ws + lay.pflag);
    SWE_CUDA(c, cudaMemcpy(c->d_blob, pb.bytes.data(), pb.bytes.size(), cudaMemcpyHostToDevice));
    SWE_CUDA(c, cudaMemset(c->d_pflag, 0, 2 * (size_t)kPflagBytes * (size_t)c->n_patches));
    if (const char *s = std::getenv("SWE_PATCH_MIN_BLOCKS")) c->patch_force_blocks = std::atoi(s);
    c->patch_threads = patch_threads(pb.lay.P);
    // small meshes whose patches are all resident at once are bound by the latency of one block's chain of phases: one
    // thread per local EDGE instead of one per own cell makes phase 2 (about two edges per cell, each a dependent chain
    // of square roots and a division) a single pass -- configs[0]: 8.7 -> 6.4 us per step (profiles/r2w_small_meshes.md)
    {
      int dev = 0, sms = 148;
      SWE_CUDA(c, cudaGetDevice(&dev));
      SWE_CUDA(c, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
      const int t_edges = pb.lay.cap_e <= 256 ? patch_threads(pb.lay.cap_e) : 0;   // (blocks of up to 256 threads: the instances with >= 4 blocks per SM)
      if (t_edges > c->patch_threads && !c->patch_force_blocks) {
        const size_t smem = (size_t)patch2_smem_layout(pb.lay, c->sc.n, pl.z.morph ? 2 : 0, true).total;
        const PatchInst *pi = pick_patch_kernel(t_edges, smem, 0);
        if (pi && (int64_t)c->n_patches <= (int64_t)sms * pi->min_blocks) c->patch_threads = t_edges;
      }
    }
    c->patch_prefetch = 4 * 148;              // about the blocks resident at a time
    if (const char *s = std::getenv("SWE_PATCH_PREFETCH")) c->patch_prefetch = std::atoi(s);
    // self-controlled steps: at most kCtlPre strings, each string's pairwise tree inside the block's scratch (the
    // flux arrays of the patch, and the 1024 doubles of k_self_finish), graphs a multiple of 4 steps long
    {
      const int64_t cap = std::min<int64_t>(1024, (int64_t)pb.lay.cap_e + 3 * (int64_t)pb.lay.cap_eown);
      // (it saves the control kernel's graph node, 2.3-2.6 us per step: + 20-30 % on meshes up to ~100k cells, nothing
      // measurable from ~2M cells on, where the extra work at the top of 15,000 blocks costs as much: profiles/r2q_patch_size_sweep.md)
      const char *self_env = std::getenv("SWE_PATCH_SELF");           // measurement runs: 0 never, 2 on any mesh size
      const int self_max_patches = (self_env && std::atoi(self_env) == 2) ? (1 << 30) : 8192;
      bool ok = (int)c->strings.size() <= kCtlPre && (c->steps_per_graph % 4) == 0 && c->n_patches <= self_max_patches && c->sc.n == 0 && !c->single;
      for (const BoundaryString &bs : c->strings) ok = ok && bs.pow2 <= cap;
      if (const char *s = std::getenv("SWE_PATCH_SELF")) ok = ok && std::atoi(s) != 0;
      c->self_ctl = ok;
    }
    c->patch_smem = (size_t)patch2_smem_layout(pb.lay, c->sc.n, 0, c->self_ctl).total;
    {
      const PatchInst *pi = pick_patch_kernel(c->patch_threads, c->patch_smem, c->patch_force_blocks, c->single);
      if (!pi) { c->err = "no patch kernel instance for this patch size"; return SWE_EINVAL; }
      c->patch_min_blocks = pi->min_blocks;
    }
    // the attribute belongs to the kernel, not to the context: always raise it to the hardware limit, so that a later
    // context with smaller patches cannot lower it under an earlier context's launches
    {
      const size_t smem_max = (size_t)patch2_smem_layout(pb.lay, c->sc.n, pl.z.morph ? 2 : 0, true).total;
      int dev = 0, optin = 0;
      cudaFuncAttributes fa{};
      SWE_CUDA(c, cudaGetDevice(&dev));
      SWE_CUDA(c, cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
      for (const PatchInst &pi : kPatchInst) {
        if (pi.T != c->patch_threads) continue;
        for (int a = 0; a < 9; ++a) {                  // [scalars][self-controlled][mobile bed], and the single-precision instance
          PatchKernel fn = a < 8 ? pi.get(pi.min_blocks, a & 1, (a >> 1) & 1, (a >> 2) & 1) : pi.get(pi.min_blocks, 0, 4, 0);
          if (!fn) continue;
          SWE_CUDA(c, cudaFuncGetAttributes(&fa, fn));
          const int limit = optin - (int)fa.sharedSizeBytes;
          if ((int)smem_max > limit) { c->err = "patch needs more shared memory than an SM has: lower patch_cells or renumber"; return SWE_EINVAL; }
          SWE_CUDA(c, cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, limit));
        }
      }
    }
    // algorithmic bytes per launch, every datum once (halo re-reads and duplicated edge records NOT counted):
    // state in 32 + state out 32 + slot words 16 + area, g/k^2 16 per cell; 32 bytes of edge data per edge
    int64_t *ab = c->alg_bytes_v[SWE_VARIANT_PATCH];
    ab[0] = 0;
    ab[1] = 96 * nc + 32 * ne + (int64_t)c->sc.n * 16 * nc;         // + q_c in and out per species
    // SURVEY.md section 8(d), one-pass column: 132 B per cell-step (+ 16 per species: q_c in and out)
    c->survey_bytes_v[SWE_VARIANT_PATCH][1] = (132 + 16 * (int64_t)c->sc.n) * nc;
    if (c->single) {   // 16-byte records, 4-byte reals (abs(Omega), 1/abs(Omega), g/k^2; n_x, n_y, l), int32 tables stay
      ab[1] = (16 + 16 + 16 + 12) * nc + (12 + 8) * ne;
      c->survey_bytes_v[SWE_VARIANT_PATCH][1] = (132 - 16) / 2 * nc + 16 * nc;    // reals halve, the slot words stay
    }
  }
  {
    // EdgeGeom read + EdgeFlux written per edge, every CellRec gathered once
    int64_t *ab = c->alg_bytes_v[SWE_VARIANT_THREE_PASS];
    ab[0] = 0;
    ab[1] = 64 * ne + 32 * nc;
    ab[2] = 1 * nc;                                      // k_theta_lazy: one flag byte per cell
    // cell_edge, 1/area, g/k^2, theta read, CellRec read + written per cell; every EdgeGeom and EdgeFlux gathered once
    ab[3] = (16 + 8 + 8 + 64) * nc + 64 * ne;
    ab[1] += (int64_t)c->sc.n * (8 * nc + 8 * ne);       // q_c gathered once, upwind concentration written
    ab[3] += (int64_t)c->sc.n * (16 * nc + 8 * ne);      // q_c read + written, upwind concentration gathered
    if (c->single) {      // 16-byte records, 4-byte reals, R of an edge in its own int32 array
      ab[1] = (16 + 4 + 16) * ne + 16 * nc;
      ab[3] = (16 + 4 + 4 + 32) * nc + 32 * ne;
    }
    c->alg_bytes_base[0] = ab[1]; c->alg_bytes_base[1] = ab[3];
    // SURVEY.md section 8(d), two-kernel column (284 B per cell-step with 1/A read in the edge pass), split as the
    // survey's rows split: edge pass = state 24 + z 8 + 1/A 8 + geometry 36 + edge->cell 12 + flux written 60 = 148;
    // cell pass = state 24 r + 24 w + g/k^2, 1/A 16 + cell->edge 12 + flux read 60 = 136
    int64_t *sb = c->survey_bytes_v[SWE_VARIANT_THREE_PASS];
    sb[1] = 148 * nc; sb[2] = 0; sb[3] = 136 * nc;
    if (c->single) { sb[1] = (148 - 12 - 12) / 2 * nc + 24 * nc; sb[3] = (136 - 12) / 2 * nc + 12 * nc; }   // reals halve, int32 tables stay
  }

  // ---- control block
  Control h{};
  h.g = p.g; h.h_dry = p.h_dry; h.dt_max = p.dt_max;
  h.t_end = std::numeric_limits<double>::infinity(); h.cfl = 0.9;
  h.n_strings = (int32_t)c->strings.size();
  h.ping_pong = (c->variant == SWE_VARIANT_PATCH) ? 1 : 0;
  SWE_CUDA(c, cudaMemcpy(c->d_ctl, &h, sizeof(Control), cudaMemcpyHostToDevice));
  *c->h_ctl = h;
  // AUTO with a compact numbering: both variants stay available (their graphs are captured now) and swe_set_state
  // picks one from the wet fraction of the state -- they compute bit-identical results
  c->auto_mode = pl.auto_mode;
  if (c->auto_mode) {
    c->variant = SWE_VARIANT_THREE_PASS;
    int rc = capture_graph(c);
    c->variant = SWE_VARIANT_PATCH;
    if (rc != SWE_OK) return rc;
  }
  return capture_graph(c);
}

}  // namespace

// =========================================================================================================
// the message swe_last_error(NULL) returns on this thread, for entry points that live in another translation unit
// (swe_static.cu)
namespace swe { void set_thread_error(const char *msg) { g_create_error = msg ? msg : ""; } }

extern "C" {

void swe_params_default(swe_params *p) {
  if (!p) return;
  std::memset(p, 0, sizeof(*p));
  p->g = 9.81;
  p->h_dry = 1e-3;
  p->dt_max = std::numeric_limits<double>::infinity();
  p->renumber = SWE_RENUMBER_MORTON;
  p->state_on_device = 0;
  p->steps_per_graph = 32;
  p->variant = SWE_VARIANT_AUTO;
  p->patch_cells = 0;
  p->n_species = 0;
  p->morphology = 0;
  p->precision = SWE_PRECISION_DOUBLE;
}

size_t swe_workspace_bytes(const swe_mesh *mesh, const swe_params *params) {
  swe_params p;
  if (params) p = *params; else swe_params_default(&p);
  try {
    Plan pl;
    if (make_plan(mesh, p, false, pl, g_create_error) != SWE_OK) return 0;
    return Layout(pl.z).total;
  } catch (const std::bad_alloc &) {
    g_create_error = "out of host memory";
    return 0;
  }
}

int swe_create(const swe_mesh *mesh, const swe_params *params, swe_ctx **out) {
  if (out) *out = nullptr;
  if (!out) { g_create_error = "null argument"; return SWE_EINVAL; }
  swe_ctx *c = new (std::nothrow) swe_ctx;
  if (!c) { g_create_error = "out of host memory"; return SWE_ENOMEM; }
  int rc;
  try {
    rc = create_impl(mesh, params, c);
  } catch (const std::bad_alloc &) {
    c->err = "out of host memory";
    rc = SWE_ENOMEM;
  }
  if (rc != SWE_OK) {
    g_create_error = c->err;
    release(c);
    return rc;
  }
  *out = c;
  return SWE_OK;
}

int swe_set_boundary(swe_ctx *c, int string_id, int type, const double *params, int n_params) {
  if (!c) return SWE_EINVAL;
  if (string_id < 0 || string_id >= (int)c->strings.size() || c->strings[string_id].n_edges == 0) { c->err = "no edge of the mesh belongs to this boundary string"; return SWE_EINVAL; }
  if (n_params < 0 || (n_params > 0 && !params)) { c->err = "bad params"; return SWE_EINVAL; }
  if (type == SWE_BC_INFLOW_Q) {
    if (n_params < 2 || n_params % 2) { c->err = "INFLOW_Q needs a (t, Q) table"; return SWE_EINVAL; }
    for (int k = 0; k < n_params; ++k) if (!std::isfinite(params[k])) { c->err = "hydrograph entries must be finite"; return SWE_EINVAL; }
    for (int k = 2; k < n_params; k += 2) if (!(params[k] > params[k - 2])) { c->err = "hydrograph times must ascend"; return SWE_EINVAL; }
  } else if (type == SWE_BC_OUTFLOW_UNIFORM) {
    if (n_params < 1 || !(params[0] >= 0.0)) { c->err = "OUTFLOW_UNIFORM needs S0 >= 0"; return SWE_EINVAL; }
  } else if (type != SWE_BC_NONE) {
    c->err = "unknown boundary type";
    return SWE_EINVAL;
  }
  // the table goes into the string's slice of the parameter pool (a new slice when it has grown)
  if (n_params > c->param_cap[string_id]) {
    if (c->params_used + n_params > kParamsPool) { c->err = "boundary parameter pool exhausted (16384 doubles per context)"; return SWE_ENOMEM; }
    c->param_off[string_id] = c->params_used; c->param_cap[string_id] = n_params;
    c->params_used += n_params;
  }
  SWE_CUDA(c, cudaStreamSynchronize(c->stream));
  BoundaryString &bs = c->strings[string_id];
  bs.type = type; bs.n_params = n_params; bs.params = nullptr; bs.Q = 0.0; bs.sumK = 0.0;
  bs.S0 = (type == SWE_BC_OUTFLOW_UNIFORM) ? params[0] : 0.0;
  if (n_params > 0) {
    double *dst = c->d_params + c->param_off[string_id];
    SWE_CUDA(c, cudaMemcpy(dst, params, 8 * (size_t)n_params, cudaMemcpyHostToDevice));
    bs.params = dst;
  }
  return upload_strings(c);
}

int swe_set_state(swe_ctx *c, const double *h, const double *hu, const double *hv, double t0) {
  if (!c) return SWE_EINVAL;
  if (!h || !hu || !hv || !std::isfinite(t0)) { c->err = "null state pointer / non-finite t0"; return SWE_EINVAL; }
  const int64_t nc = c->nc;
  const double *dh = h, *dhu = hu, *dhv = hv;
  if (!c->prm.state_on_device) {
    SWE_CUDA(c, cudaMemcpyAsync(c->stage, h, 8 * nc, cudaMemcpyHostToDevice, c->stream));
    SWE_CUDA(c, cudaMemcpyAsync(c->stage + nc, hu, 8 * nc, cudaMemcpyHostToDevice, c->stream));
    SWE_CUDA(c, cudaMemcpyAsync(c->stage + 2 * nc, hv, 8 * nc, cudaMemcpyHostToDevice, c->stream));
    dh = c->stage; dhu = c->stage + nc; dhv = c->stage + 2 * nc;
  }
  if (c->auto_mode) {
    // the fused patch step wins where part of the domain is dry (it skips dry patches), the three-pass step on
    // (almost) all-wet states: count the wet cells of the new state and pick
    k_set_variant<<<1, 1, 0, c->stream>>>(c->d_ctl, 0, 1);
    k_count_wet<<<std::min(grid_for(nc), kInfoMaxBlocks), kBlock, 0, c->stream>>>(c->d_ctl, dh, (int)nc);
    c->launches += 2;
    int rc = read_control(c);
    if (rc != SWE_OK) return rc;
    // with four blocks of the patch kernel per SM it is the faster step at any wet fraction (all-wet 4M: 259.6 vs 266.1 us,
    // 8M: 508 vs 521 us; profiles/r2q_patch_size_sweep.md); with fewer (fat halos, scalar species, large patch_cells) the
    // round-1 crossover holds: three-pass from ~50 % wet cells on (profiles/r1i_auto_threshold.md)
    // (single precision: the three-pass step moves half the bytes and wins on all-wet states, 27.6 vs 23.3 G at 8M cells;
    // the patch step wins while part of the domain is dry, 41.5 vs 29.2 G on the river reach: profiles/r2u_single_precision.md)
    // the crossover: 50 % wet cells in fp64 with fat patches (round 1), 75 % in single precision (71 % wet: 78.8 vs 80.3 us,
    // 85 % wet: 88.0 vs 81.8 us at 2M cells)
    const double wet_limit = c->single ? 0.75 : 0.5;
    const int want = ((c->single || c->patch_min_blocks < 4) && (double)c->h_ctl->n_wet > wet_limit * (double)nc) ? SWE_VARIANT_THREE_PASS : SWE_VARIANT_PATCH;
    if (want != c->variant) {
      if (want == SWE_VARIANT_THREE_PASS && c->h_ctl->cur == 1)      // scalars set earlier live in buffer b: move them
        for (int sp = 0; sp < c->sc.n; ++sp)
          SWE_CUDA(c, cudaMemcpyAsync(c->sc.qa[sp], c->sc.qb[sp], 8 * nc, cudaMemcpyDeviceToDevice, c->stream));
      c->variant = want;
    }
    k_set_variant<<<1, 1, 0, c->stream>>>(c->d_ctl, want == SWE_VARIANT_PATCH ? 1 : 0, 0);
    c->launches += 1;
  }
  if (c->single) { const View<float> v = view<float>(c); k_pack_state<float><<<grid_for(nc), kBlock, 0, c->stream>>>(c->d_ctl, c->cell_perm, dh, dhu, dhv, v.rec, v.rec_b, (int)nc); }
  else k_pack_state<double><<<grid_for(nc), kBlock, 0, c->stream>>>(c->d_ctl, c->cell_perm, dh, dhu, dhv, c->rec, c->rec_b, (int)nc);
  if (c->variant == SWE_VARIANT_PATCH) launch_patch_flags(c);
  if (c->mp.formula == 2 && c->variant == SWE_VARIANT_THREE_PASS) {   // mobile bed, MPM-like law: the per-cell cube roots of the new state
    k_sed_cell_init<<<grid_for(nc), kBlock, 0, c->stream>>>(c->d_ctl, c->rec, c->gn2, c->mp.cell, (int)nc);
    c->launches += 1;
  }
  k_reset<<<1, 1, 0, c->stream>>>(c->d_ctl, t0);
  if (c->single) { const View<float> v = view<float>(c); k_rate<float><<<grid_for(nc), kBlock, 0, c->stream>>>(c->d_ctl, c->cell_edge, v.geom, v.inv_area, v.rec, v.rec_b, (int)nc); }
  else k_rate<double><<<grid_for(nc), kBlock, 0, c->stream>>>(c->d_ctl, c->cell_edge, c->geom, c->inv_area, c->rec, c->rec_b, (int)nc);
  c->launches += 3;
  SWE_CUDA(c, cudaGetLastError());
  c->t_host = t0;
  return SWE_OK;
}

int swe_step(swe_ctx *c, int64_t n_steps, double t_end, double cfl, swe_step_info *info) {
  if (!c) return SWE_EINVAL;
  if (!(cfl > 0.0) || std::isnan(t_end)) { c->err = "cfl must be > 0 and t_end a number"; return SWE_EINVAL; }
  const bool finite_end = std::isfinite(t_end);
  if (n_steps < 0 && !finite_end) { c->err = "either n_steps >= 0 or a finite t_end is needed"; return SWE_EINVAL; }
  begin_call(c, (long long)n_steps, t_end, cfl);
  const int K = c->steps_per_graph;
  int64_t remaining = n_steps < 0 ? std::numeric_limits<int64_t>::max() : n_steps;
  int64_t poll_every = 4;            // graph launches between two reads of t (only when t_end is finite)
  bool done = !(c->t_host < t_end);  // t_end already reached: nothing to do
  while (!done && remaining > 0) {
    int64_t batch_steps = 0;
    if (K > 0 && remaining >= K && self_mode(c) && (c->step_idx & 3) != 0) {
      batch_steps = std::min<int64_t>(remaining, 4 - (c->step_idx & 3));   // plain launches up to a multiple of 4
      for (int64_t j = 0; j < batch_steps; ++j) enqueue_step(c, c->stream);
      SWE_CUDA(c, cudaGetLastError());
    } else if (K > 0 && remaining >= K) {
      int64_t n_graphs = remaining / K;
      if (finite_end) n_graphs = std::min(n_graphs, poll_every);
      for (int64_t j = 0; j < n_graphs; ++j) SWE_CUDA(c, cudaGraphLaunch(c->graph_exec_v[c->variant], c->stream));
      batch_steps = n_graphs * K;
      c->step_idx += batch_steps;
    } else {
      batch_steps = std::min<int64_t>(remaining, 64);   // tail shorter than a graph, or graphs switched off
      for (int64_t j = 0; j < batch_steps; ++j) enqueue_step(c, c->stream);
      SWE_CUDA(c, cudaGetLastError());
    }
    c->launches += batch_steps * n_step_kernels(c);
    remaining -= batch_steps;
    if (finite_end) {                // the only host synchronisation inside the loop: once per batch
      end_call(c, 0);                // (self-controlled steps: snapshot of the newest slot into the fields read here)
      int rc = read_control(c);
      if (rc != SWE_OK) return rc;
      if (!(c->h_ctl->t < t_end) || (c->h_ctl->flags & (SWE_FLAG_DT_UNBOUNDED | SWE_FLAG_STALLED))) done = true;
      poll_every = std::min<int64_t>(poll_every * 2, 64);
    }
  }
  // volume bookkeeping of the last step; then the reductions of swe_step_info
  end_call(c, 1);
  SWE_CUDA(c, cudaGetLastError());
  if (info) {
    if (c->single) { const View<float> v = view<float>(c); k_info<float><<<std::min(grid_for(c->nc), kInfoMaxBlocks), kBlock, 0, c->stream>>>(c->d_ctl, v.rec, v.rec_b, v.area, (int)c->nc, c->d_info_part, c->d_info_ticket); }
    else k_info<double><<<std::min(grid_for(c->nc), kInfoMaxBlocks), kBlock, 0, c->stream>>>(c->d_ctl, c->rec, c->rec_b, c->area, (int)c->nc, c->d_info_part, c->d_info_ticket);
    c->launches += 1;
    int rc = read_control(c);
    if (rc != SWE_OK) return rc;
    const Control &h = *c->h_ctl;
    info->t = h.t; info->dt_last = h.dt_last; info->steps_done = h.steps_done; info->n_wet = h.n_wet;
    info->vol = h.vol; info->vol_clipped = h.vol_clipped; info->vol_in = h.vol_in; info->vol_out = h.vol_out;
    info->flags = h.flags | (h.nonfinite ? SWE_FLAG_NONFINITE : 0);
    if (h.nonfinite) { c->err = "non-finite state value"; return SWE_ENONFINITE; }
    if (c->auto_mode) {   // the wet count is known here: follow a flood that spreads (or recedes), with hysteresis
      const double wet = (double)h.n_wet / (double)c->nc;
      const int want = (c->patch_min_blocks >= 4 && !c->single) ? SWE_VARIANT_PATCH
                                                : (wet > (c->single ? 0.80 : 0.55) ? SWE_VARIANT_THREE_PASS : (wet < (c->single ? 0.70 : 0.45) ? SWE_VARIANT_PATCH : c->variant));
      rc = switch_variant(c, want, h.cur);
      if (rc != SWE_OK) return rc;
    }
  } else if (!finite_end) {
    c->t_host = -std::numeric_limits<double>::infinity();   // unknown until the next read; never blocks stepping
  }
  return SWE_OK;
}

int swe_set_scalars(swe_ctx *c, const double *qc) {
  if (!c) return SWE_EINVAL;
  if (c->sc.n == 0) { c->err = "the context was created with n_species = 0"; return SWE_EINVAL; }
  if (!qc) { c->err = "null scalar pointer"; return SWE_EINVAL; }
  const int64_t nc = c->nc;
  for (int sp = 0; sp < c->sc.n; ++sp) {
    const double *src = qc + (size_t)sp * nc;
    if (!c->prm.state_on_device) {
      SWE_CUDA(c, cudaMemcpyAsync(c->d_scalar_stage, src, 8 * nc, cudaMemcpyHostToDevice, c->stream));
      src = c->d_scalar_stage;
    }
    k_pack_scalar<<<grid_for(nc), kBlock, 0, c->stream>>>(c->d_ctl, c->cell_perm, src, c->sc.qa[sp], c->sc.qb[sp], (int)nc);
    c->launches += 1;
  }
  if (c->variant == SWE_VARIANT_PATCH) launch_patch_flags(c);
  SWE_CUDA(c, cudaGetLastError());
  return SWE_OK;
}

int swe_get_scalars(swe_ctx *c, double *qc) {
  if (!c) return SWE_EINVAL;
  if (c->sc.n == 0) { c->err = "the context was created with n_species = 0"; return SWE_EINVAL; }
  if (!qc) { c->err = "null scalar pointer"; return SWE_EINVAL; }
  const int64_t nc = c->nc;
  for (int sp = 0; sp < c->sc.n; ++sp) {
    double *dst = c->prm.state_on_device ? qc + (size_t)sp * nc : c->d_scalar_stage;
    k_unpack_scalar<<<grid_for(nc), kBlock, 0, c->stream>>>(c->d_ctl, c->cell_perm, c->sc.qa[sp], c->sc.qb[sp], dst, (int)nc);
    c->launches += 1;
    if (!c->prm.state_on_device) {
      SWE_CUDA(c, cudaMemcpyAsync(qc + (size_t)sp * nc, c->d_scalar_stage, 8 * nc, cudaMemcpyDeviceToHost, c->stream));
      SWE_CUDA(c, cudaStreamSynchronize(c->stream));
    }
  }
  SWE_CUDA(c, cudaGetLastError());
  return SWE_OK;
}

// Morphodynamics (include/swe.h): the bed moves from the next step on.  The step becomes the three-pass one with the
// <kMorph> instances of its edge and cell kernels (the fused patch step keeps the bed of its halo cells in tables built
// for a fixed bed); the CUDA graph of the three-pass step is captured again.
int swe_set_morphology(swe_ctx *c, int formula, double alpha, double theta_cr, double s, double d_m, double porosity) {
  if (!c) return SWE_EINVAL;
  if (formula < 0 || formula > 2) { c->err = "formula must be 0 (fixed bed), 1 (Grass-like) or 2 (MPM-like)"; return SWE_EINVAL; }
  if (!(porosity >= 0.0 && porosity < 1.0)) { c->err = "porosity must be in [0, 1)"; return SWE_EINVAL; }
  if (!std::isfinite(alpha) || alpha < 0.0) { c->err = "alpha must be finite and >= 0"; return SWE_EINVAL; }
  if (formula == 2 && !(s > 1.0 && d_m > 0.0 && std::isfinite(s) && std::isfinite(d_m) && std::isfinite(theta_cr))) {
    c->err = "the MPM-like formula needs s > 1, d_m > 0 and a finite theta_cr"; return SWE_EINVAL;
  }
  if (formula && !c->morph_reserved) { c->err = "the context was created without room for the mobile-bed module: set swe_params.morphology = 1"; return SWE_EINVAL; }
  int rc = read_control(c);          // synchronises: no step in flight
  if (rc != SWE_OK) return rc;
  const double g = c->prm.g;
  c->mp.formula = formula; c->mp.alpha = alpha; c->mp.theta_cr = theta_cr;
  c->mp.shields_den = g * ((s - 1.0) * d_m);
  c->mp.Gm = alpha * std::sqrt(((s - 1.0) * g) * (d_m * (d_m * d_m)));
  c->mp.inv1mp = 1.0 / (1.0 - porosity);
  // the fused patch step ping-pongs between two record buffers and leaves the records of skipped (dry) patches alone:
  // both buffers must hold the bed as it is now (afterwards a patch's bed only moves in steps that rewrite its records)
  if (c->has_patch) {
    k_sync_bed<<<grid_for(c->nc), kBlock, 0, c->stream>>>(c->d_ctl, c->rec, c->rec_b, (int)c->nc);
    c->launches += 1;
  }
  if (formula == 2 && c->variant == SWE_VARIANT_THREE_PASS) {   // (g/k^2, cbrt(h)) of the state as it stands; k_cell_update keeps it current
    k_sed_cell_init<<<grid_for(c->nc), kBlock, 0, c->stream>>>(c->d_ctl, c->rec, c->gn2, c->mp.cell, (int)c->nc);
    c->launches += 1;
  }
  SWE_CUDA(c, cudaGetLastError());
  {                                   // algorithmic bytes of the kernels that carry the extra work
    int64_t *ab = c->alg_bytes_v[SWE_VARIANT_THREE_PASS];
    ab[1] = c->alg_bytes_base[0] + (formula ? 8 * c->ne + (formula == 2 ? 16 * c->nc : 0) : 0);
    ab[3] = c->alg_bytes_base[1] + (formula ? 8 * c->ne + (formula == 2 ? 16 * c->nc : 0) : 0);
    if (c->has_patch) c->alg_bytes_v[SWE_VARIANT_PATCH][1] = 96 * c->nc + 32 * c->ne + (int64_t)c->sc.n * 16 * c->nc + (formula == 2 ? 8 * c->nc : 0);
  }
  c->edge_grid = c->base_edge_grid; c->cell_grid = c->base_cell_grid;
  if (formula) {                      // resident grids of the <kMorph> instances
    int per_sm = 3;
    if (c->sc.n > 0) SWE_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_cell_update<true, true>, kBlock, 0));
    else {
      SWE_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_edge_flux<false, true, true>, kBlock, 0));
      c->edge_grid = std::max(1, c->sms * per_sm);
      SWE_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_cell_update<false, true>, kBlock, 0));
    }
    c->cell_grid = std::max(1, c->sms * per_sm);
  }
  // the graphs of both variants launch other kernel instances now: capture them again
  SWE_CUDA(c, cudaStreamSynchronize(c->stream));
  const int keep = c->variant;
  for (int v : {SWE_VARIANT_THREE_PASS, SWE_VARIANT_PATCH}) {
    if (!c->graph_exec_v[v]) continue;
    cudaGraphExecDestroy(c->graph_exec_v[v]);
    c->graph_exec_v[v] = nullptr;
    c->variant = v;
    rc = capture_graph(c);
    if (rc != SWE_OK) { c->variant = keep; return rc; }
  }
  c->variant = keep;
  return SWE_OK;
}

int swe_get_bed(swe_ctx *c, double *zb) {
  if (!c) return SWE_EINVAL;
  if (c->single) { c->err = "swe_get_bed: not built for single precision (the bed is fixed there: it is the caller's zb rounded to fp32)"; return SWE_EINVAL; }
  if (!zb) { c->err = "null bed pointer"; return SWE_EINVAL; }
  const int64_t nc = c->nc;
  double *dst = c->prm.state_on_device ? zb : c->stage;
  k_unpack_bed<<<grid_for(nc), kBlock, 0, c->stream>>>(c->d_ctl, c->cell_perm, c->rec, c->rec_b, dst, (int)nc);
  c->launches += 1;
  SWE_CUDA(c, cudaGetLastError());
  if (!c->prm.state_on_device) {
    SWE_CUDA(c, cudaMemcpyAsync(zb, c->stage, 8 * nc, cudaMemcpyDeviceToHost, c->stream));
    SWE_CUDA(c, cudaStreamSynchronize(c->stream));
  }
  return SWE_OK;
}

int swe_get_sediment_flux(swe_ctx *c, double *qB) {
  if (!c) return SWE_EINVAL;
  if (!qB) { c->err = "null flux pointer"; return SWE_EINVAL; }
  if (!c->morph_reserved) { c->err = "the context has no mobile-bed module (swe_params.morphology)"; return SWE_EINVAL; }
  const int64_t ne = c->ne;
  if (c->variant == SWE_VARIANT_PATCH && c->mp.formula) {
    // the fused step keeps q_Bij in shared memory: re-evaluate the most recent step's with the stand-alone edge kernel,
    // from the state that step read (still intact in the other buffer)
    int rc = read_control(c);
    if (rc != SWE_OK) return rc;
    const CellRec *in = c->h_ctl->src ? c->rec_b : c->rec;
    if (c->mp.formula == 2) k_sed_cell_init<<<grid_for(c->nc), kBlock, 0, c->stream>>>(c->d_ctl, in, c->gn2, c->mp.cell, (int)c->nc);
    k_edge_flux<false, false, true><<<grid_for(ne), kBlock, 0, c->stream>>>(c->d_ctl, c->geom, in, c->kst, c->d_strings, c->flux, (int)ne, 1, Scalars{},
                                                                          c->area, nullptr, c->mp);
    c->launches += 2;
  }
  double *dst = c->prm.state_on_device ? qB : c->stage;       // stage holds 3 n_cells >= n_edges doubles
  k_export_sediment<<<grid_for(ne), kBlock, 0, c->stream>>>(c->edge_perm, c->mp.qB, dst, (int)ne);
  c->launches += 1;
  SWE_CUDA(c, cudaGetLastError());
  if (!c->prm.state_on_device) {
    SWE_CUDA(c, cudaMemcpyAsync(qB, c->stage, 8 * ne, cudaMemcpyDeviceToHost, c->stream));
    SWE_CUDA(c, cudaStreamSynchronize(c->stream));
  }
  return SWE_OK;
}

int swe_set_boundary_scalar(swe_ctx *c, int string_id, const double *phi, int n) {
  if (!c) return SWE_EINVAL;
  if (string_id < 0 || string_id >= (int)c->strings.size() || c->strings[string_id].n_edges == 0) { c->err = "no edge of the mesh belongs to this boundary string"; return SWE_EINVAL; }
  if (n < 0 || n > kMaxSpecies || (n > 0 && !phi)) { c->err = "bad concentration list"; return SWE_EINVAL; }
  SWE_CUDA(c, cudaStreamSynchronize(c->stream));
  for (int sp = 0; sp < kMaxSpecies; ++sp) c->strings[string_id].phi_in[sp] = sp < n ? phi[sp] : 0.0;
  return upload_strings(c);
}

int swe_get_state(swe_ctx *c, double *h, double *hu, double *hv) {
  if (!c) return SWE_EINVAL;
  if (!h || !hu || !hv) { c->err = "null state pointer"; return SWE_EINVAL; }
  const int64_t nc = c->nc;
  if (c->prm.state_on_device) {
    if (c->single) { const View<float> v = view<float>(c); k_unpack_state<float><<<grid_for(nc), kBlock, 0, c->stream>>>(c->d_ctl, c->cell_perm, v.rec, v.rec_b, h, hu, hv, (int)nc); }
    else k_unpack_state<double><<<grid_for(nc), kBlock, 0, c->stream>>>(c->d_ctl, c->cell_perm, c->rec, c->rec_b, h, hu, hv, (int)nc);
    c->launches += 1;
    SWE_CUDA(c, cudaGetLastError());
    return SWE_OK;
  }
  if (c->single) { const View<float> v = view<float>(c); k_unpack_state<float><<<grid_for(nc), kBlock, 0, c->stream>>>(c->d_ctl, c->cell_perm, v.rec, v.rec_b, c->stage, c->stage + nc, c->stage + 2 * nc, (int)nc); }
  else k_unpack_state<double><<<grid_for(nc), kBlock, 0, c->stream>>>(c->d_ctl, c->cell_perm, c->rec, c->rec_b, c->stage, c->stage + nc, c->stage + 2 * nc, (int)nc);
  c->launches += 1;
  SWE_CUDA(c, cudaMemcpyAsync(h, c->stage, 8 * nc, cudaMemcpyDeviceToHost, c->stream));
  SWE_CUDA(c, cudaMemcpyAsync(hu, c->stage + nc, 8 * nc, cudaMemcpyDeviceToHost, c->stream));
  SWE_CUDA(c, cudaMemcpyAsync(hv, c->stage + 2 * nc, 8 * nc, cudaMemcpyDeviceToHost, c->stream));
  SWE_CUDA(c, cudaStreamSynchronize(c->stream));
  return SWE_OK;
}

void swe_destroy(swe_ctx *c) {
  if (!c) return;
  cudaStreamSynchronize(c->stream);
  release(c);
}

const char *swe_last_error(const swe_ctx *c) { return c ? c->err.c_str() : g_create_error.c_str(); }

// ---- inspection ---------------------------------------------------------------------------------------
int swe_get_geometry(swe_ctx *c, double *area, double *nx, double *ny, double *len) {
  if (!c || !area || !nx || !ny || !len) return SWE_EINVAL;
  // read back what the kernels use (device arrays, internal numbering) and undo the renumbering
  SWE_CUDA(c, cudaStreamSynchronize(c->stream));
  if (c->single) {
    std::vector<float> a(c->nc);
    std::vector<EdgeGeomT<float>> g(c->ne);
    SWE_CUDA(c, cudaMemcpy(a.data(), c->area, 4 * c->nc, cudaMemcpyDeviceToHost));
    SWE_CUDA(c, cudaMemcpy(g.data(), c->geom, sizeof(EdgeGeomT<float>) * c->ne, cudaMemcpyDeviceToHost));
    for (int64_t i = 0; i < c->nc; ++i) area[c->hm.cell_perm[i]] = a[i];
    for (int64_t e = 0; e < c->ne; ++e) {
      const int32_t o = c->hm.edge_perm[e];
      nx[o] = g[e].nx; ny[o] = g[e].ny; len[o] = g[e].len;
    }
    return SWE_OK;
  }
  std::vector<double> a(c->nc);
  std::vector<EdgeGeom> g(c->ne);
  SWE_CUDA(c, cudaMemcpy(a.data(), c->area, 8 * c->nc, cudaMemcpyDeviceToHost));
  SWE_CUDA(c, cudaMemcpy(g.data(), c->geom, sizeof(EdgeGeom) * c->ne, cudaMemcpyDeviceToHost));
  for (int64_t i = 0; i < c->nc; ++i) area[c->hm.cell_perm[i]] = a[i];
  for (int64_t e = 0; e < c->ne; ++e) {
    const int32_t o = c->hm.edge_perm[e];
    nx[o] = g[e].nx; ny[o] = g[e].ny; len[o] = g[e].len;
  }
  return SWE_OK;
}

int swe_get_edge_flux(swe_ctx *c, double *F1, double *F3, double *GL, double *GR, double *theta) {
  if (!c || !F1 || !F3 || !GL || !GR) return SWE_EINVAL;
  const int64_t ne = c->ne, nc = c->nc;
  if (c->variant == SWE_VARIANT_PATCH && c->single) {
    c->err = "swe_get_edge_flux: not built for the single-precision patch step (SWE_VARIANT_THREE_PASS exports its fluxes)";
    return SWE_EINVAL;
  }
  if (c->variant == SWE_VARIANT_PATCH) {
    // the fused step keeps edge fluxes in shared memory: re-evaluate S1 and S1c of the most recent step with the
    // stand-alone kernels, from the state that step read (still intact in the other buffer) and its dt
    int rc = read_control(c);
    if (rc != SWE_OK) return rc;
    const CellRec *in = c->h_ctl->src ? c->rec_b : c->rec;
    k_edge_flux<false, false><<<grid_for(ne), kBlock, 0, c->stream>>>(c->d_ctl, c->geom, in, c->kst, c->d_strings, c->flux, (int)ne, 1, Scalars{}, c->area, nullptr);
    k_theta<<<grid_for(nc), kBlock, 0, c->stream>>>(c->d_ctl, c->cell_edge, c->geom, c->flux, in, c->area, c->theta, (int)nc, 1);
    c->launches += 2;
  }
  const double *th_apply = (c->variant == SWE_VARIANT_PATCH) ? c->theta : nullptr;   // three-pass: limited in place
  double *d = c->stage;                                // holds 2 n_edges doubles: export in two halves
  for (int half = 0; half < 2; ++half) {
    double *o1 = half ? nullptr : d, *o2 = half ? nullptr : d + ne, *o3 = half ? d : nullptr, *o4 = half ? d + ne : nullptr;
    if (c->single) { const View<float> v = view<float>(c); k_export_flux<float><<<grid_for(ne), kBlock, 0, c->stream>>>(c->edge_perm, v.geom, v.flux, (const float *)nullptr, o1, o2, o3, o4, (int)ne); }
    else k_export_flux<double><<<grid_for(ne), kBlock, 0, c->stream>>>(c->edge_perm, c->geom, c->flux, th_apply, o1, o2, o3, o4, (int)ne);
    c->launches += 1;
    SWE_CUDA(c, cudaGetLastError());
    SWE_CUDA(c, cudaStreamSynchronize(c->stream));
    SWE_CUDA(c, cudaMemcpy(half ? GL : F1, d, 8 * ne, cudaMemcpyDeviceToHost));
    SWE_CUDA(c, cudaMemcpy(half ? GR : F3, d + ne, 8 * ne, cudaMemcpyDeviceToHost));
  }
  if (theta && c->single) {
    std::vector<float> th(nc);
    SWE_CUDA(c, cudaMemcpy(th.data(), c->theta, 4 * nc, cudaMemcpyDeviceToHost));
    for (int64_t i = 0; i < nc; ++i) theta[c->hm.cell_perm[i]] = th[i];
  } else if (theta) {
    std::vector<double> th(nc);
    SWE_CUDA(c, cudaMemcpy(th.data(), c->theta, 8 * nc, cudaMemcpyDeviceToHost));
    for (int64_t i = 0; i < nc; ++i) theta[c->hm.cell_perm[i]] = th[i];
  }
  return SWE_OK;
}

int swe_peek_dt(swe_ctx *c, double cfl, double t_end, double *dt_out) {
  if (!c || !dt_out || !(cfl > 0.0)) return SWE_EINVAL;
  int rc = read_control(c);
  if (rc != SWE_OK) return rc;
  const Control &h = *c->h_ctl;
  double r;
  std::memcpy(&r, &h.rate_bits, 8);
  double dt = (r > 0.0) ? cfl / r : h.dt_max;
  dt = std::fmin(dt, h.dt_max);
  const double rem = t_end - h.t;
  *dt_out = (dt >= rem) ? rem : dt;
  return SWE_OK;
}

int swe_get_permutation(swe_ctx *c, int32_t *cell_perm, int32_t *edge_perm) {
  if (!c) return SWE_EINVAL;
  if (cell_perm) std::memcpy(cell_perm, c->hm.cell_perm.data(), 4 * c->nc);
  if (edge_perm) std::memcpy(edge_perm, c->hm.edge_perm.data(), 4 * c->ne);
  return SWE_OK;
}

int swe_get_tables(swe_ctx *c, int64_t *n_edges, int32_t *edge_cell, int32_t *cell_edge) {
  if (!c) return SWE_EINVAL;
  if (n_edges) *n_edges = c->ne;
  if (edge_cell) std::memcpy(edge_cell, c->hm.edge_cell.data(), 8 * c->ne);
  if (cell_edge) std::memcpy(cell_edge, c->hm.cell_edge.data(), 12 * c->nc);
  return SWE_OK;
}

int swe_device_cbrt(const double *x, double *y, int64_t n) {
  if (n < 0 || (n > 0 && (!x || !y))) return SWE_EINVAL;
  if (n == 0) return SWE_OK;
  double *d = nullptr;
  if (cudaMalloc((void **)&d, 16 * (size_t)n) != cudaSuccess) return SWE_ECUDA;
  cudaError_t e = cudaMemcpy(d, x, 8 * (size_t)n, cudaMemcpyHostToDevice);
  if (e == cudaSuccess) {
    k_cbrt<<<(unsigned)((n + kBlock - 1) / kBlock), kBlock>>>(d, d + n, (long long)n);
    e = cudaGetLastError();
  }
  if (e == cudaSuccess) e = cudaMemcpy(y, d + n, 8 * (size_t)n, cudaMemcpyDeviceToHost);
  cudaFree(d);
  if (e != cudaSuccess) { g_create_error = std::string("swe_device_cbrt: ") + cudaGetErrorString(e); return SWE_ECUDA; }
  return SWE_OK;
}

int64_t swe_kernel_launches(const swe_ctx *c) { return c ? c->launches : 0; }

int swe_host_preprocess(const swe_mesh *mesh, int renumber_mode, int patch_cells, int64_t *out, int n_out,
                        int32_t *cell_perm, int32_t *edge_perm) {
  if (!mesh || !mesh->node_xy || !mesh->tri || !mesh->zb || !mesh->kst || mesh->n_cells <= 0 || mesh->n_nodes <= 0) {
    g_create_error = "null argument / empty mesh";
    return SWE_EINVAL;
  }
  try {
    HostMesh hm;
    int rc = host_prepare(mesh, renumber_mode, hm, g_create_error);
    if (rc != SWE_OK) return rc;
    int64_t v[10] = {hm.ne, 0, 0, 0, 0, 0, 0, 0, 0, 0};
    if (patch_cells > 0) {
      const int64_t nc = hm.nc, ne = hm.ne;
      std::vector<EdgeGeom> geom(ne); std::vector<int32_t> ce4((size_t)4 * nc); std::vector<double> area(nc), inv_area(nc), gn2(nc, 0.0);
      for (int64_t i = 0; i < nc; ++i) {
        const int32_t o = hm.cell_perm[i];
        for (int k = 0; k < 3; ++k) ce4[4 * i + k] = hm.edge_new[hm.cell_edge[3 * o + k]];
        ce4[4 * i + 3] = 0;
        area[i] = hm.area[o]; inv_area[i] = 1.0 / hm.area[o];
      }
      for (int64_t e = 0; e < ne; ++e) {
        const int32_t o = hm.edge_perm[e];
        const int32_t L = hm.edge_cell[2 * o], R = hm.edge_cell[2 * o + 1];
        geom[e] = {hm.nx[o], hm.ny[o], hm.len[o], hm.cell_new[L], R >= 0 ? hm.cell_new[R] : R};
      }
      std::vector<int32_t> string_pos(ne, -1);
      int32_t n_string = 0;
      for (int64_t e = 0; e < ne; ++e) if (geom[e].R <= -3) string_pos[e] = n_string++;
      PatchBlobs pb;
      if (!build_blobs(nc, ne, geom, ce4, area, inv_area, gn2, string_pos, patch_cells, true, pb, g_create_error)) return SWE_EINVAL;
      // every cell must be an own cell of exactly one patch
      // ... and the emitted blobs must describe what the capacity pass counted: local cells / edges of every header,
      // local indices inside the patch, every slot word pointing at an edge that joins the two cells it names
      int64_t own = 0, covered = 0, hdr_loc = 0, hdr_e = 0;
      std::vector<uint8_t> seen(nc, 0);
      const BlobLayout &BL = pb.lay;
      for (int64_t p = 0; p < pb.n_patches; ++p) {
        const unsigned char *B = pb.bytes.data() + (size_t)BL.stride * (size_t)p;
        const BlobHeader *h = (const BlobHeader *)B;
        own += h->n_own;
        for (int32_t l = 0; l < h->n_own; ++l) { const int64_t cidx = p * patch_cells + l; if (!seen[cidx]) { seen[cidx] = 1; ++covered; } }
        const int32_t n_loc = h->n_own + h->n_r1 + h->n_r2, n_e = h->n_eown + h->n_er1;
        hdr_loc += n_loc; hdr_e += n_e;
        const uint32_t *lr = (const uint32_t *)(B + BL.off_stage + BL.s_lr);
        const uint32_t *pce = (const uint32_t *)(B + BL.off_stage + BL.s_pce);
        for (int32_t j = 0; j < n_e; ++j) {
          const uint32_t Ll = lr[j] & 0xFFFFu, Rl = lr[j] >> 16;
          if ((int32_t)Ll >= n_loc || (Rl != 0xFFFFu && (int32_t)Rl >= n_loc)) { g_create_error = "patch blob: local cell index out of range"; return SWE_EINVAL; }
        }
        for (int32_t l = 0; l < h->n_own + h->n_r1; ++l)
          for (int k = 0; k < 3; ++k) {
            const uint32_t wd = pce[4 * l + k], e = wd & 0x7FFFu, nb = wd >> 16;
            const bool isL = (wd & 0x8000u) != 0u;
            if ((int32_t)e >= n_e) { g_create_error = "patch blob: slot word names an edge outside the patch"; return SWE_EINVAL; }
            const uint32_t Ll = lr[e] & 0xFFFFu, Rl = lr[e] >> 16;
            if ((isL ? Ll : Rl) != (uint32_t)l || (isL ? Rl : Ll) != nb) { g_create_error = "patch blob: slot word and edge record disagree"; return SWE_EINVAL; }
          }
      }
      // the reader masks (fourth word of an own cell's slot record: bit j = the j-th neighbour patch reads the cell; the exact
      // skip flags rest on them): every halo entry of every patch has its bit in the owner's mask, and there are no others
      int64_t halo_entries = 0, mask_bits = 0;
      for (int64_t p = 0; p < pb.n_patches; ++p) {
        const unsigned char *B = pb.bytes.data() + (size_t)BL.stride * (size_t)p;
        const BlobHeader *h = (const BlobHeader *)B;
        const int32_t *halo = (const int32_t *)(B + BL.off_halo_ids);
        for (int32_t j = 0; j < h->n_r1 + h->n_r2; ++j) {
          const int64_t cidx = halo[j], o = cidx / patch_cells;
          const unsigned char *Bo = pb.bytes.data() + (size_t)BL.stride * (size_t)o;
          const BlobHeader *ho = (const BlobHeader *)Bo;
          const int32_t *nbr_o = (const int32_t *)(Bo + BL.off_nbr);
          int32_t slot = -1;
          for (int32_t k = 0; k < ho->n_nbr; ++k) if (nbr_o[k] == (int32_t)p) { slot = k; break; }
          if (slot < 0) { g_create_error = "patch blob: a patch reads a cell of a patch that does not list it as a neighbour"; return SWE_EINVAL; }
          if (slot >= 32) continue;
          ++halo_entries;
          const uint32_t *pce_o = (const uint32_t *)(Bo + BL.off_stage + BL.s_pce);
          if (!((pce_o[4 * (cidx - o * patch_cells) + 3] >> slot) & 1u)) { g_create_error = "patch blob: reader mask misses a neighbour that reads the cell"; return SWE_EINVAL; }
        }
        const uint32_t *pce = (const uint32_t *)(B + BL.off_stage + BL.s_pce);
        for (int32_t l = 0; l < h->n_own; ++l) mask_bits += __builtin_popcount(pce[4 * l + 3]);
      }
      if (mask_bits != halo_entries) { g_create_error = "patch blob: reader masks name neighbours that do not read the cell"; return SWE_EINVAL; }
      if (hdr_loc != pb.sum_loc || hdr_e != pb.sum_e) { g_create_error = "patch blob: headers disagree with the capacity pass"; return SWE_EINVAL; }
      v[1] = pb.n_patches; v[2] = pb.sum_loc; v[3] = pb.sum_e; v[4] = pb.max_loc; v[5] = pb.max_e;
      v[6] = (int64_t)patch2_smem_layout(pb.lay, 0).total;
      v[7] = own; v[8] = covered; v[9] = pb.sum_nbr;
    }
    for (int k = 0; k < n_out && k < 10; ++k) out[k] = v[k];
    if (cell_perm) std::memcpy(cell_perm, hm.cell_perm.data(), 4 * hm.nc);
    if (edge_perm) std::memcpy(edge_perm, hm.edge_perm.data(), 4 * hm.ne);
  } catch (const std::bad_alloc &) {
    g_create_error = "out of host memory";
    return SWE_ENOMEM;
  }
  return SWE_OK;
}

int swe_step_kernel_count(const swe_ctx *c) { return c ? n_step_kernels(c) : 0; }

const char *swe_step_kernel_name(const swe_ctx *c, int k) {
  if (!c || k < 0 || k >= n_step_kernels(c)) return nullptr;
  return self_mode(c) ? kSelfNames[k] : (c->variant == SWE_VARIANT_PATCH ? kPatchNames[k] : kThreePassNames[k]);
}

int64_t swe_algorithmic_bytes(const swe_ctx *c, int k) { return (c && k >= 0 && k < n_step_kernels(c)) ? c->alg_bytes_v[c->variant][self_mode(c) ? k + 1 : k] : 0; }

int64_t swe_survey_bytes(const swe_ctx *c, int k) { return (c && k >= 0 && k < n_step_kernels(c)) ? c->survey_bytes_v[c->variant][self_mode(c) ? k + 1 : k] : 0; }

int swe_get_patch_stats(swe_ctx *c, int64_t *out, int n_out) {
  if (!c || !out || n_out < 1) return SWE_EINVAL;
  int rc = read_control(c);
  if (rc != SWE_OK) return rc;
  const int64_t v[12] = {c->variant, c->n_patches, c->blay.P, (int64_t)c->patch_smem, c->patch_sum_loc, c->patch_sum_e,
                         c->patch_max_loc, c->patch_max_e, (int64_t)c->h_ctl->patches_skipped, c->patch_min_blocks,
                         c->blay.stride, c->blay.stage_bytes};
  for (int k = 0; k < n_out && k < 12; ++k) out[k] = v[k];
  return SWE_OK;
}

int swe_profile_step(swe_ctx *c, int64_t n_steps, double cfl, double *ms, int n_ms) {
  if (!c) return SWE_EINVAL;
  if (n_steps < 1 || !(cfl > 0.0) || !ms || n_ms < 1) { c->err = "swe_profile_step: bad argument"; return SWE_EINVAL; }
  constexpr int kBatch = 32;                       // steps between two synchronisations
  constexpr int kEv = kMaxStepKernels + 1;
  const int nk = n_step_kernels(c);
  std::vector<cudaEvent_t> ev((size_t)kBatch * kEv, nullptr);
  for (auto &e : ev) SWE_CUDA(c, cudaEventCreate(&e));
  double sum[kMaxStepKernels] = {0.0};
  begin_call(c, (long long)n_steps, std::numeric_limits<double>::infinity(), cfl);
  cudaError_t rc = cudaSuccess;
  for (int64_t done = 0; done < n_steps && rc == cudaSuccess; done += kBatch) {
    const int nb = (int)std::min<int64_t>(kBatch, n_steps - done);
    for (int j = 0; j < nb; ++j) enqueue_step(c, c->stream, ev.data() + (size_t)j * kEv);
    c->launches += (int64_t)nb * nk;
    rc = cudaStreamSynchronize(c->stream);
    for (int j = 0; j < nb && rc == cudaSuccess; ++j)
      for (int k = 0; k < nk && rc == cudaSuccess; ++k) {
        float t = 0.f;
        rc = cudaEventElapsedTime(&t, ev[(size_t)j * kEv + k], ev[(size_t)j * kEv + k + 1]);
        sum[k] += t;
      }
  }
  for (auto &e : ev) cudaEventDestroy(e);
  SWE_CUDA(c, rc);
  end_call(c, 1);
  SWE_CUDA(c, cudaGetLastError());
  for (int k = 0; k < n_ms; ++k) ms[k] = k < nk ? sum[k] / (double)n_steps : 0.0;
  c->t_host = -std::numeric_limits<double>::infinity();
  return SWE_OK;
}

}  // extern "C"
