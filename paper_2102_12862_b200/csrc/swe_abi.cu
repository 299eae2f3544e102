// C-ABI of include/swe.h: context, workspace carving, upload, CUDA-graph step loop.  Host logic only;
// every step of the numerical path runs in the kernels of swe_kernels.cuh.
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
#include "patch_prep.hpp"
#include "swe_kernels.cuh"
#include "swe_patch_kernel.cuh"
#include "swe_types.h"

using namespace swe;

namespace {

thread_local std::string g_create_error;

constexpr size_t kAlign = 256;
inline size_t align_up(size_t x) { return (x + kAlign - 1) / kAlign * kAlign; }

// Sizes of the O(N) device arrays carved out of the workspace, in carving order.
struct Layout {
  size_t rec, rec_b, geom, flux, cell_edge, area, inv_area, gn2, kst, theta, cell_perm, edge_perm, stage, total;
  Layout(int64_t nc, int64_t ne) {
    size_t o = 0;
    auto take = [&](size_t bytes) { size_t at = o; o += align_up(bytes); return at; };
    rec = take(sizeof(CellRec) * nc);
    rec_b = take(sizeof(CellRec) * nc);     // second state buffer of the fused patch step
    geom = take(sizeof(EdgeGeom) * ne);
    flux = take(sizeof(EdgeFlux) * ne);
    cell_edge = take(sizeof(int4) * nc);
    area = take(8 * nc); inv_area = take(8 * nc); gn2 = take(8 * nc); kst = take(8 * nc); theta = take(8 * nc);
    cell_perm = take(4 * nc); edge_perm = take(4 * ne);
    stage = take(24 * nc);
    total = o;
  }
};

inline int grid_for(int64_t n) { return (int)((n + kBlock - 1) / kBlock); }

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
  // small device allocations owned by the library
  Control *d_ctl = nullptr;
  Control *h_ctl = nullptr;          // pinned
  BoundaryString *d_strings = nullptr;
  int *d_string_edges = nullptr;
  double *d_scratch = nullptr;
  std::vector<BoundaryString> strings;
  std::vector<double *> d_params;
  // fused patch step (variant SWE_VARIANT_PATCH): tables built by patch_prep.hpp, allocated by the library
  int variant = 0;
  PatchTables pt;                    // host copy (headers kept for statistics; the big vectors are released)
  PatchHeader *d_hdr = nullptr; int32_t *d_halo_ids = nullptr; double *d_halo_area = nullptr;
  PatchEdge *d_pedge = nullptr; uint4 *d_pce = nullptr; int32_t *d_slot_string = nullptr; double *d_string_M = nullptr;
  InfoPartial *d_info_part = nullptr; unsigned int *d_info_ticket = nullptr;
  int cell_grid = 148 * 4;           // resident blocks of the persistent k_cell_update
  int edge_grid = 148 * 5;           // resident blocks of the persistent k_edge_flux (set from the occupancy API)
  int base_edge_grid = 0, base_cell_grid = 0, sms = 148;
  Morph mp{};                        // morphodynamics (swe_set_morphology); formula 0 = fixed bed
  uint8_t *d_drain_flag = nullptr;   // three-pass step: cells flagged as possible drainers (lazy theta)
  Scalars sc{};                      // passive scalars: device arrays owned by the library (cudaMalloc)
  double *d_scalar_stage = nullptr;  // [n_cells] staging of one species for host-pointer set / get
  int32_t *d_patch_nbr = nullptr; uint8_t *d_dry = nullptr;   // d_dry: [2][n_patches]
  int n_patches = 0; size_t patch_smem = 0;
  void (*patch_kernel)(Control *, PatchArgs) = nullptr;
  int64_t alg_bytes_base[2] = {};        // three-pass k_edge_flux / k_cell_update without the mobile bed
  int64_t alg_bytes_v[3][4] = {};        // [variant][kernel]: algorithmic DRAM bytes per launch of the kernels of a step
  bool auto_mode = false;                // AUTO with both variants available: chosen at swe_set_state (wet fraction)
  cudaGraph_t graph = nullptr;
  cudaGraphExec_t graph_exec_v[3] = {nullptr, nullptr, nullptr};   // by variant
  int steps_per_graph = 0;
  int64_t launches = 0;
  double t_host = 0.0;               // t as of the last synchronisation
  std::string err;
};

namespace {

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
// (two edges per thread, i.e. two gather chains in flight, needs 80 registers: measured slower)
constexpr int kPatchThreads = 256;
const char *const kThreePassNames[4] = {"k_step_control", "k_edge_flux", "k_theta_lazy", "k_cell_update"};
const char *const kPatchNames[2] = {"k_step_control", "k_patch_step"};

inline int n_step_kernels(const swe_ctx *c) { return c->variant == SWE_VARIANT_PATCH ? 2 : 4; }

PatchArgs patch_args(const swe_ctx *c) {
  PatchArgs a;
  a.hdr = c->d_hdr; a.halo_ids = c->d_halo_ids; a.halo_area = c->d_halo_area; a.pedge = c->d_pedge; a.pce = c->d_pce;
  a.rec_a = c->rec; a.rec_b = c->rec_b; a.area = c->area; a.inv_area = c->inv_area; a.gn2 = c->gn2; a.kst = c->kst;
  a.strings = c->d_strings; a.slot_string = c->d_slot_string; a.string_M = c->d_string_M;
  a.patch_nbr = c->d_patch_nbr; a.dry_a = c->d_dry; a.dry_b = c->d_dry + c->n_patches;
  a.sc = c->sc;
  a.max_loc = c->pt.max_loc; a.max_c1 = c->pt.max_c1; a.max_e = c->pt.max_e; a.max_eown = c->pt.max_eown;
  return a;
}

void launch_control(swe_ctx *c, cudaStream_t s, int mode) {
  k_step_control<<<1, kCtlThreads, 0, s>>>(c->d_ctl, c->d_strings, c->d_string_edges, c->d_scratch, c->geom, c->flux,
                                           nullptr /* records are limited in place */, c->rec, c->rec_b, c->kst,
                                           c->variant == SWE_VARIANT_PATCH ? c->d_string_M : nullptr, mode);
}

void enqueue_step(swe_ctx *c, cudaStream_t s, cudaEvent_t *ev = nullptr) {
  if (ev) cudaEventRecord(ev[0], s);
  launch_control(c, s, 0);
  if (ev) cudaEventRecord(ev[1], s);
  if (c->variant == SWE_VARIANT_PATCH) {
    c->patch_kernel<<<c->n_patches, kPatchThreads, c->patch_smem, s>>>(c->d_ctl, patch_args(c));
    if (ev) cudaEventRecord(ev[2], s);
    return;
  }
  if (c->mp.formula)
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
  if (c->mp.formula)
    k_cell_update<false, true><<<std::min(grid_for(c->nc), c->cell_grid), kBlock, 0, s>>>(c->d_ctl, c->cell_edge, c->geom, c->flux, nullptr, c->area,
                                                                  c->inv_area, c->gn2, c->rec, (int)c->nc, c->sc, c->mp);
  else if (c->sc.n > 0)
    k_cell_update<true><<<std::min(grid_for(c->nc), c->cell_grid), kBlock, 0, s>>>(c->d_ctl, c->cell_edge, c->geom, c->flux, nullptr, c->area,
                                                           c->inv_area, c->gn2, c->rec, (int)c->nc, c->sc);
  else
    k_cell_update<false><<<std::min(grid_for(c->nc), c->cell_grid), kBlock, 0, s>>>(c->d_ctl, c->cell_edge, c->geom, c->flux, nullptr, c->area,
                                                            c->inv_area, c->gn2, c->rec, (int)c->nc, c->sc);
  if (ev) cudaEventRecord(ev[4], s);
}

int capture_graph(swe_ctx *c) {
  if (c->steps_per_graph <= 0) return SWE_OK;
  cudaStream_t cap;
  SWE_CUDA(c, cudaStreamCreateWithFlags(&cap, cudaStreamNonBlocking));
  SWE_CUDA(c, cudaStreamBeginCapture(cap, cudaStreamCaptureModeThreadLocal));
  for (int k = 0; k < c->steps_per_graph; ++k) enqueue_step(c, cap);
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

void release(swe_ctx *c) {
  if (!c) return;
  for (auto &ge : c->graph_exec_v) if (ge) cudaGraphExecDestroy(ge);
  if (c->graph) cudaGraphDestroy(c->graph);
  for (double *p : c->d_params) if (p) cudaFree(p);
  if (c->d_ctl) cudaFree(c->d_ctl);
  if (c->h_ctl) cudaFreeHost(c->h_ctl);
  if (c->d_strings) cudaFree(c->d_strings);
  if (c->d_string_edges) cudaFree(c->d_string_edges);
  if (c->d_scratch) cudaFree(c->d_scratch);
  if (c->d_hdr) cudaFree(c->d_hdr);
  if (c->d_halo_ids) cudaFree(c->d_halo_ids);
  if (c->d_halo_area) cudaFree(c->d_halo_area);
  if (c->d_pedge) cudaFree(c->d_pedge);
  if (c->d_pce) cudaFree(c->d_pce);
  if (c->d_slot_string) cudaFree(c->d_slot_string);
  if (c->d_string_M) cudaFree(c->d_string_M);
  if (c->d_info_part) cudaFree(c->d_info_part);
  if (c->d_info_ticket) cudaFree(c->d_info_ticket);
  for (int sp = 0; sp < kMaxSpecies; ++sp) {
    if (c->sc.qa[sp]) cudaFree(c->sc.qa[sp]);
    if (c->sc.qb[sp]) cudaFree(c->sc.qb[sp]);
    if (c->sc.phi_up[sp]) cudaFree(c->sc.phi_up[sp]);
  }
  if (c->d_scalar_stage) cudaFree(c->d_scalar_stage);
  if (c->d_drain_flag) cudaFree(c->d_drain_flag);
  if (c->mp.qB) cudaFree(c->mp.qB);
  if (c->mp.cell) cudaFree(c->mp.cell);
  if (c->d_patch_nbr) cudaFree(c->d_patch_nbr);
  if (c->d_dry) cudaFree(c->d_dry);
  if (c->own_ws && c->ws) cudaFree(c->ws);
  delete c;
}

// AUTO: makes `want` the active variant for the state as it is now (no step in flight).  cur = Control::cur as last
// read.  The three-pass step works in place in buffer a; the patch step ping-pongs and needs its dry flags.
int switch_variant(swe_ctx *c, int want, int cur) {
  if (want == c->variant) return SWE_OK;
  const int64_t nc = c->nc;
  if (want == SWE_VARIANT_THREE_PASS && cur == 1) {
    SWE_CUDA(c, cudaMemcpyAsync(c->rec, c->rec_b, sizeof(CellRec) * nc, cudaMemcpyDeviceToDevice, c->stream));
    for (int sp = 0; sp < c->sc.n; ++sp)
      SWE_CUDA(c, cudaMemcpyAsync(c->sc.qa[sp], c->sc.qb[sp], 8 * nc, cudaMemcpyDeviceToDevice, c->stream));
  }
  c->variant = want;
  k_set_variant<<<1, 1, 0, c->stream>>>(c->d_ctl, want == SWE_VARIANT_PATCH ? 1 : 0, 0);
  c->launches += 1;
  if (want == SWE_VARIANT_PATCH) {
    k_patch_flags<kPatchThreads><<<c->n_patches, kPatchThreads, 0, c->stream>>>(c->d_ctl, c->d_hdr, c->rec, c->rec_b, c->d_dry,
                                                                             c->d_dry + c->n_patches, c->sc);
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
__global__ void __launch_bounds__(kCtlThreads)
k_string_lengths(BoundaryString *strings, int n_strings, const int *__restrict__ string_edges, double *scratch,
                 const EdgeGeom *__restrict__ geom) {
  for (int s = 0; s < n_strings; ++s) {
    BoundaryString &bs = strings[s];
    if (bs.n_edges == 0) continue;
    double *v = scratch + bs.scratch;
    for (int j = threadIdx.x; j < bs.pow2; j += blockDim.x) v[j] = j < bs.n_edges ? geom[string_edges[bs.first + j]].len : 0.0;
    const double sum = block_tree_sum(v, bs.pow2);
    if (threadIdx.x == 0) bs.sumL = sum;
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

// internal-numbering edge geometry and slot table, as uploaded by swe_create
void internal_tables(const HostMesh &hm, std::vector<EdgeGeom> &geom, std::vector<int32_t> &ce4, std::vector<double> &area) {
  const int64_t nc = hm.nc, ne = hm.ne;
  geom.resize(ne); ce4.resize((size_t)4 * nc); area.resize(nc);
  for (int64_t i = 0; i < nc; ++i) {
    const int32_t o = hm.cell_perm[i];
    for (int k = 0; k < 3; ++k) ce4[4 * i + k] = hm.edge_new[hm.cell_edge[3 * o + k]];
    ce4[4 * i + 3] = 0;
    area[i] = hm.area[o];
  }
  for (int64_t e = 0; e < ne; ++e) {
    const int32_t o = hm.edge_perm[e];
    const int32_t L = hm.edge_cell[2 * o], R = hm.edge_cell[2 * o + 1];
    geom[e] = {hm.nx[o], hm.ny[o], hm.len[o], hm.cell_new[L], R >= 0 ? hm.cell_new[R] : R};
  }
}

int create_impl(const swe_mesh *mesh, const swe_params *params, swe_ctx *c) {
  const int64_t nc = mesh->n_cells;
  c->nc = nc;
  if (params) c->prm = *params; else swe_params_default(&c->prm);
  const swe_params &p = c->prm;
  if (!(p.g > 0.0) || !(p.h_dry >= 0.0) || !(p.dt_max > 0.0)) { c->err = "g, h_dry, dt_max out of range"; return SWE_EINVAL; }
  c->stream = (cudaStream_t)p.cuda_stream;
  c->steps_per_graph = p.steps_per_graph;

  // ---- tables, validation, geometry, numbering (host)
  HostMesh &hm = c->hm;
  {
    int rc = host_prepare(mesh, p.renumber, hm, c->err);
    if (rc != SWE_OK) return rc;
  }
  const int64_t ne = c->ne = hm.ne;

  // ---- workspace
  const Layout lay(nc, ne);
  if (p.workspace) {
    if (p.workspace_bytes < lay.total) { c->err = "workspace too small: need " + std::to_string(lay.total) + " bytes"; return SWE_ENOMEM; }
    if (((uintptr_t)p.workspace) % kAlign != 0) { c->err = "workspace must be 256-byte aligned"; return SWE_EINVAL; }
    c->ws = (char *)p.workspace;
  } else {
    SWE_CUDA(c, cudaMalloc((void **)&c->ws, lay.total));
    c->own_ws = true;
  }
  c->rec = (CellRec *)(c->ws + lay.rec); c->rec_b = (CellRec *)(c->ws + lay.rec_b); c->geom = (EdgeGeom *)(c->ws + lay.geom); c->flux = (EdgeFlux *)(c->ws + lay.flux);
  c->cell_edge = (int4 *)(c->ws + lay.cell_edge);
  c->area = (double *)(c->ws + lay.area); c->inv_area = (double *)(c->ws + lay.inv_area);
  c->gn2 = (double *)(c->ws + lay.gn2); c->kst = (double *)(c->ws + lay.kst); c->theta = (double *)(c->ws + lay.theta);
  c->cell_perm = (int *)(c->ws + lay.cell_perm); c->edge_perm = (int *)(c->ws + lay.edge_perm);
  c->stage = (double *)(c->ws + lay.stage);

  // ---- arrays in internal numbering
  std::vector<int4> ce(nc);
  std::vector<double> area(nc);
  std::vector<EdgeGeom> geom(ne);
  {
    std::vector<CellRec> rec(nc);
    std::vector<double> inv_area(nc), gn2(nc), kst(nc), theta(nc, 1.0);
    for (int64_t i = 0; i < nc; ++i) {
      const int32_t o = hm.cell_perm[i];
      rec[i] = {0.0, 0.0, 0.0, mesh->zb[o]};
      ce[i] = make_int4(hm.edge_new[hm.cell_edge[3 * o]], hm.edge_new[hm.cell_edge[3 * o + 1]],
                        hm.edge_new[hm.cell_edge[3 * o + 2]], 0);
      const double A = hm.area[o], k = mesh->kst[o];
      area[i] = A;
      inv_area[i] = 1.0 / A;
      gn2[i] = std::isfinite(k) ? p.g / (k * k) : 0.0;    // g / k_str^2 (Eq. 2 P:106-111 with Table 1, R-6)
      kst[i] = k;
    }
    for (int64_t e = 0; e < ne; ++e) {
      const int32_t o = hm.edge_perm[e];
      const int32_t L = hm.edge_cell[2 * o], R = hm.edge_cell[2 * o + 1];
      geom[e] = {hm.nx[o], hm.ny[o], hm.len[o], hm.cell_new[L], R >= 0 ? hm.cell_new[R] : R};
    }
    auto up = [&](void *dst, const void *src, size_t bytes) { return cudaMemcpy(dst, src, bytes, cudaMemcpyHostToDevice); };
    SWE_CUDA(c, up(c->rec, rec.data(), sizeof(CellRec) * nc));
    SWE_CUDA(c, up(c->rec_b, rec.data(), sizeof(CellRec) * nc));     // z_B must be valid in both state buffers
    SWE_CUDA(c, up(c->cell_edge, ce.data(), sizeof(int4) * nc));
    SWE_CUDA(c, up(c->area, area.data(), 8 * nc));
    SWE_CUDA(c, up(c->inv_area, inv_area.data(), 8 * nc));
    SWE_CUDA(c, up(c->gn2, gn2.data(), 8 * nc));
    SWE_CUDA(c, up(c->kst, kst.data(), 8 * nc));
    SWE_CUDA(c, up(c->theta, theta.data(), 8 * nc));
    SWE_CUDA(c, up(c->geom, geom.data(), sizeof(EdgeGeom) * ne));
    SWE_CUDA(c, up(c->cell_perm, hm.cell_perm.data(), 4 * nc));
    SWE_CUDA(c, up(c->edge_perm, hm.edge_perm.data(), 4 * ne));
    SWE_CUDA(c, cudaMemset(c->flux, 0, sizeof(EdgeFlux) * ne));
  }

  // ---- boundary strings: members in ascending caller edge id ("string order", R-11)
  int max_id = -1;
  for (int64_t e = 0; e < ne; ++e) {
    const int32_t R = hm.edge_cell[2 * e + 1];
    if (R <= -3) max_id = std::max(max_id, -3 - R);
  }
  if (max_id > 65535) { c->err = "boundary string id too large"; return SWE_EINVAL; }
  c->strings.assign(max_id + 1, BoundaryString{});
  c->d_params.assign(max_id + 1, nullptr);
  std::vector<std::vector<int32_t>> members(max_id + 1);
  for (int64_t e = 0; e < ne; ++e) {
    const int32_t R = hm.edge_cell[2 * e + 1];
    if (R <= -3) members[-3 - R].push_back(hm.edge_new[e]);
  }
  std::vector<int32_t> flat;
  size_t scratch = 0;
  for (int s = 0; s <= max_id; ++s) {
    BoundaryString &bs = c->strings[s];
    bs.n_edges = (int32_t)members[s].size();
    bs.first = (int32_t)flat.size();
    int32_t P = 1;
    while (P < bs.n_edges) P <<= 1;
    bs.pow2 = P;
    bs.scratch = (int32_t)scratch;
    scratch += P;
    flat.insert(flat.end(), members[s].begin(), members[s].end());
  }
  SWE_CUDA(c, cudaMalloc((void **)&c->d_ctl, sizeof(Control)));
  SWE_CUDA(c, cudaMalloc((void **)&c->d_info_part, sizeof(InfoPartial) * kInfoMaxBlocks));
  SWE_CUDA(c, cudaMalloc((void **)&c->d_info_ticket, sizeof(unsigned int)));
  SWE_CUDA(c, cudaMemset(c->d_info_ticket, 0, sizeof(unsigned int)));
  SWE_CUDA(c, cudaMallocHost((void **)&c->h_ctl, sizeof(Control)));
  SWE_CUDA(c, cudaMalloc((void **)&c->d_strings, sizeof(BoundaryString) * std::max<size_t>(1, c->strings.size())));
  SWE_CUDA(c, cudaMalloc((void **)&c->d_string_edges, 4 * std::max<size_t>(1, flat.size())));
  SWE_CUDA(c, cudaMalloc((void **)&c->d_scratch, 8 * std::max<size_t>(1, scratch)));
  if (!flat.empty()) SWE_CUDA(c, cudaMemcpy(c->d_string_edges, flat.data(), 4 * flat.size(), cudaMemcpyHostToDevice));
  if (!c->strings.empty()) {
    SWE_CUDA(c, cudaMemcpy(c->d_strings, c->strings.data(), sizeof(BoundaryString) * c->strings.size(), cudaMemcpyHostToDevice));
    k_string_lengths<<<1, kCtlThreads, 0, c->stream>>>(c->d_strings, (int)c->strings.size(), c->d_string_edges, c->d_scratch, c->geom);
    SWE_CUDA(c, cudaGetLastError());
    SWE_CUDA(c, cudaStreamSynchronize(c->stream));
    SWE_CUDA(c, cudaMemcpy(c->strings.data(), c->d_strings, sizeof(BoundaryString) * c->strings.size(), cudaMemcpyDeviceToHost));
  }

  SWE_CUDA(c, cudaMalloc((void **)&c->d_drain_flag, (size_t)nc + 16));           // read four bytes at a time
  SWE_CUDA(c, cudaMemset(c->d_drain_flag, 0, (size_t)nc + 16));
  {
    int dev = 0, sms = 148, per_sm = 4;
    SWE_CUDA(c, cudaGetDevice(&dev));
    SWE_CUDA(c, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    SWE_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_edge_flux<false, true>, kBlock, 0));
    c->edge_grid = std::max(1, sms * per_sm);
    if (c->sc.n > 0) SWE_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_cell_update<true>, kBlock, 0));
    else SWE_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_cell_update<false>, kBlock, 0));
    c->cell_grid = std::max(1, sms * per_sm);
    c->base_edge_grid = c->edge_grid; c->base_cell_grid = c->cell_grid; c->sms = sms;
  }
  // ---- passive scalars (R-19): state per species (both buffers), per-edge upwind concentrations of the three-pass step
  if (p.n_species < 0 || p.n_species > kMaxSpecies) { c->err = "n_species must be in [0, 5] (P:208)"; return SWE_EINVAL; }
  c->sc.n = p.n_species;
  for (int sp = 0; sp < c->sc.n; ++sp) {
    SWE_CUDA(c, cudaMalloc((void **)&c->sc.qa[sp], 8 * nc));
    SWE_CUDA(c, cudaMalloc((void **)&c->sc.qb[sp], 8 * nc));
    SWE_CUDA(c, cudaMalloc((void **)&c->sc.phi_up[sp], 8 * ne));
    SWE_CUDA(c, cudaMemset(c->sc.qa[sp], 0, 8 * nc));
    SWE_CUDA(c, cudaMemset(c->sc.qb[sp], 0, 8 * nc));
    SWE_CUDA(c, cudaMemset(c->sc.phi_up[sp], 0, 8 * ne));
  }
  if (c->sc.n > 0) SWE_CUDA(c, cudaMalloc((void **)&c->d_scalar_stage, 8 * nc));

  // ---- fused patch step: patch tables (host build, upload), shared-memory size
  c->variant = (p.variant == SWE_VARIANT_THREE_PASS) ? SWE_VARIANT_THREE_PASS : SWE_VARIANT_PATCH;
  if (p.variant != SWE_VARIANT_AUTO && p.variant != SWE_VARIANT_THREE_PASS && p.variant != SWE_VARIANT_PATCH) {
    c->err = "unknown variant"; return SWE_EINVAL;
  }
  if (c->variant == SWE_VARIANT_PATCH) {
    // default: 384 cells (3 blocks/SM: fastest in the round-1 sweep); small meshes get smaller patches, so that the
    // launch-latency-bound step still spreads over ~256 blocks (4k cells: 9.3 us/step at 64 cells vs 14.5 at 384)
    int pc = p.patch_cells > 0 ? p.patch_cells : 384;
    if (p.patch_cells <= 0 && nc < 256 * 384) pc = std::max<int>(64, (int)((nc / 256 + 31) / 32 * 32));
    if (pc < 32 || pc > 8192) { c->err = "patch_cells must be in [32, 8192]"; return SWE_EINVAL; }
    std::vector<int32_t> string_pos(ne, -1);
    for (size_t j = 0; j < flat.size(); ++j) string_pos[flat[j]] = (int32_t)j;
    std::vector<int32_t> ce4((size_t)4 * nc);
    for (int64_t i = 0; i < nc; ++i) { ce4[4 * i] = ce[i].x; ce4[4 * i + 1] = ce[i].y; ce4[4 * i + 2] = ce[i].z; ce4[4 * i + 3] = 0; }
    PatchTables &pt = c->pt;
    if (!build_patches(nc, ne, geom, ce4, area, string_pos, pc, pt, c->err)) return SWE_EINVAL;
    c->n_patches = (int)pt.hdr.size();
    c->patch_smem = sizeof(double) * (size_t)patch_smem_layout(pt.max_loc, pt.max_c1, pt.max_e, pt.max_eown, c->sc.n).total;
    // 3 blocks per SM need <= 75 KB each; a numbering that is not spatially compact (renumber = NONE on a
    // scattered input order) blows the halos up: AUTO then falls back to the three-pass step
    // (with scalar species the block is fatter anyway: 2 blocks per SM, <= 113 KB, still beat the three-pass step)
    const size_t auto_limit = (c->sc.n > 0 ? 113 : 75) * 1024;
    if (c->patch_smem > 227 * 1024 || (p.variant == SWE_VARIANT_AUTO && c->patch_smem > auto_limit)) {
      if (p.variant == SWE_VARIANT_AUTO) { c->variant = SWE_VARIANT_THREE_PASS; c->pt = PatchTables{}; c->n_patches = 0; c->patch_smem = 0; }
      else { c->err = "patch needs more shared memory than an SM has: lower patch_cells or renumber"; return SWE_EINVAL; }
    }
  }
  if (c->variant == SWE_VARIANT_PATCH) {
    PatchTables &pt = c->pt;
    std::vector<int32_t> slot_string(std::max<size_t>(1, flat.size()), 0);
    for (int s = 0; s <= max_id; ++s)
      for (int32_t j = 0; j < c->strings[s].n_edges; ++j) slot_string[c->strings[s].first + j] = s;
    // default patch size on a compact numbering: shared-memory arrays with compile-time capacities; anything else
    // (other patch sizes, fatter halos) runs the same kernel with run-time capacities
    constexpr int kCapLoc = 640, kCapC1 = 544, kCapE = 864, kCapEown = 704;
    if (c->sc.n > 0) {               // scalar module: run-time capacities (the concentrations enlarge the block)
      c->patch_kernel = c->patch_smem <= 75 * 1024 ? k_patch_step<kPatchThreads, 3, 0, 0, 0, 0, true>
                                                   : k_patch_step<kPatchThreads, 2, 0, 0, 0, 0, true>;
    } else if (pt.max_loc <= kCapLoc && pt.max_c1 <= kCapC1 && pt.max_e <= kCapE && pt.max_eown <= kCapEown) {
      c->patch_kernel = k_patch_step<kPatchThreads, 3, kCapLoc, kCapC1, kCapE, kCapEown>;
      c->patch_smem = sizeof(double) * (size_t)patch_smem_layout(kCapLoc, kCapC1, kCapE, kCapEown).total;
    } else {
      // 3 blocks/SM while the patch fits 75 KB (the round-1 sweep: 2 blocks are slower, 4 need 64 registers and spill)
      c->patch_kernel = c->patch_smem <= 75 * 1024 ? k_patch_step<kPatchThreads, 3, 0, 0, 0, 0> : k_patch_step<kPatchThreads, 2, 0, 0, 0, 0>;
    }
    // the attribute belongs to the kernel, not to the context: always raise it to the hardware limit, so that a later
    // context with smaller patches cannot lower it under an earlier context's launches
    {
      int dev = 0, optin = 0;
      cudaFuncAttributes fa{};
      SWE_CUDA(c, cudaGetDevice(&dev));
      SWE_CUDA(c, cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
      SWE_CUDA(c, cudaFuncGetAttributes(&fa, c->patch_kernel));
      const int limit = optin - (int)fa.sharedSizeBytes;
      if ((int)c->patch_smem > limit) { c->err = "patch needs more shared memory than an SM has: lower patch_cells or renumber"; return SWE_EINVAL; }
      SWE_CUDA(c, cudaFuncSetAttribute(c->patch_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, limit));
    }
    auto dup = [&](void **dst, const void *src, size_t bytes) {
      cudaError_t e = cudaMalloc(dst, std::max<size_t>(bytes, 16));
      if (e == cudaSuccess && bytes) e = cudaMemcpy(*dst, src, bytes, cudaMemcpyHostToDevice);
      return e;
    };
    SWE_CUDA(c, dup((void **)&c->d_hdr, pt.hdr.data(), sizeof(PatchHeader) * pt.hdr.size()));
    SWE_CUDA(c, dup((void **)&c->d_halo_ids, pt.halo_ids.data(), 4 * pt.halo_ids.size()));
    SWE_CUDA(c, dup((void **)&c->d_halo_area, pt.halo_area.data(), 8 * pt.halo_area.size()));
    SWE_CUDA(c, dup((void **)&c->d_pedge, pt.pedge.data(), sizeof(PatchEdge) * pt.pedge.size()));
    SWE_CUDA(c, dup((void **)&c->d_pce, pt.pce.data(), 4 * pt.pce.size()));
    SWE_CUDA(c, dup((void **)&c->d_slot_string, slot_string.data(), 4 * slot_string.size()));
    SWE_CUDA(c, dup((void **)&c->d_patch_nbr, pt.patch_nbr.data(), 4 * pt.patch_nbr.size()));
    SWE_CUDA(c, cudaMalloc((void **)&c->d_dry, 2 * (size_t)c->n_patches));
    SWE_CUDA(c, cudaMemset(c->d_dry, 0, 2 * (size_t)c->n_patches));
    SWE_CUDA(c, cudaMalloc((void **)&c->d_string_M, 8 * std::max<size_t>(1, flat.size())));
    SWE_CUDA(c, cudaMemset(c->d_string_M, 0, 8 * std::max<size_t>(1, flat.size())));
    // algorithmic bytes per launch, every datum once (halo re-reads and duplicated edge records NOT counted):
    // state in 32 + state out 32 + pce 16 + area, 1/area, g/k^2 24 per cell; one 32-byte edge record per edge
    int64_t *ab = c->alg_bytes_v[SWE_VARIANT_PATCH];
    ab[0] = 0;
    ab[1] = 104 * nc + 32 * ne + (int64_t)c->sc.n * 16 * nc;        // + q_c in and out per species
    pt.halo_ids = {}; pt.halo_area = {}; pt.pedge = {}; pt.pce = {}; pt.patch_nbr = {};   // host copies no longer needed
  }
  {
    // EdgeGeom read + EdgeFlux written per edge, every CellRec gathered once
    int64_t *ab = c->alg_bytes_v[SWE_VARIANT_THREE_PASS];
    ab[0] = 0;
    ab[1] = 64 * ne + 32 * nc;
    // cell_edge, CellRec, area read + theta written per cell; every EdgeGeom and EdgeFlux gathered once
    ab[2] = 1 * nc;                                      // k_theta_lazy: one flag byte per cell
    // cell_edge, 1/area, g/k^2, theta read, CellRec read + written per cell; every EdgeGeom and EdgeFlux gathered once
    ab[3] = (16 + 8 + 8 + 64) * nc + 64 * ne;
    ab[1] += (int64_t)c->sc.n * (8 * nc + 8 * ne);       // q_c gathered once, upwind concentration written
    ab[3] += (int64_t)c->sc.n * (16 * nc + 8 * ne);      // q_c read + written, upwind concentration gathered
    c->alg_bytes_base[0] = ab[1]; c->alg_bytes_base[1] = ab[3];
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
  c->auto_mode = (p.variant == SWE_VARIANT_AUTO && c->variant == SWE_VARIANT_PATCH);
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
}

size_t swe_workspace_bytes(int64_t n_cells, int64_t n_edges) {
  if (n_cells < 0) return 0;
  if (n_edges <= 0) n_edges = 3 * n_cells;
  return Layout(n_cells, n_edges).total;
}

int swe_create(const swe_mesh *mesh, const swe_params *params, swe_ctx **out) {
  if (out) *out = nullptr;
  if (!mesh || !out || !mesh->node_xy || !mesh->tri || !mesh->zb || !mesh->kst) { g_create_error = "null argument"; return SWE_EINVAL; }
  if (mesh->n_cells <= 0 || mesh->n_nodes <= 0 || mesh->n_cells > (int64_t)0x7fffffff / 3) { g_create_error = "n_cells / n_nodes out of range"; return SWE_EINVAL; }
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
    for (int k = 2; k < n_params; k += 2) if (!(params[k] > params[k - 2])) { c->err = "hydrograph times must ascend"; return SWE_EINVAL; }
  } else if (type == SWE_BC_OUTFLOW_UNIFORM) {
    if (n_params < 1 || !(params[0] >= 0.0)) { c->err = "OUTFLOW_UNIFORM needs S0 >= 0"; return SWE_EINVAL; }
  } else if (type != SWE_BC_NONE) {
    c->err = "unknown boundary type";
    return SWE_EINVAL;
  }
  SWE_CUDA(c, cudaStreamSynchronize(c->stream));
  BoundaryString &bs = c->strings[string_id];
  if (c->d_params[string_id]) { cudaFree(c->d_params[string_id]); c->d_params[string_id] = nullptr; }
  bs.type = type; bs.n_params = n_params; bs.params = nullptr; bs.Q = 0.0; bs.sumK = 0.0;
  bs.S0 = (type == SWE_BC_OUTFLOW_UNIFORM) ? params[0] : 0.0;
  if (n_params > 0) {
    SWE_CUDA(c, cudaMalloc((void **)&c->d_params[string_id], 8 * (size_t)n_params));
    SWE_CUDA(c, cudaMemcpy(c->d_params[string_id], params, 8 * (size_t)n_params, cudaMemcpyHostToDevice));
    bs.params = c->d_params[string_id];
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
    // measured crossover on the river reach filled to different stages: ~52 % wet cells (profiles/r1i_auto_threshold.md)
    const int want = (double)c->h_ctl->n_wet > 0.5 * (double)nc ? SWE_VARIANT_THREE_PASS : SWE_VARIANT_PATCH;
    if (want != c->variant) {
      if (want == SWE_VARIANT_THREE_PASS && c->h_ctl->cur == 1)      // scalars set earlier live in buffer b: move them
        for (int sp = 0; sp < c->sc.n; ++sp)
          SWE_CUDA(c, cudaMemcpyAsync(c->sc.qa[sp], c->sc.qb[sp], 8 * nc, cudaMemcpyDeviceToDevice, c->stream));
      c->variant = want;
    }
    k_set_variant<<<1, 1, 0, c->stream>>>(c->d_ctl, want == SWE_VARIANT_PATCH ? 1 : 0, 0);
    c->launches += 1;
  }
  k_pack_state<<<grid_for(nc), kBlock, 0, c->stream>>>(c->d_ctl, c->cell_perm, dh, dhu, dhv, c->rec, c->rec_b, (int)nc);
  if (c->variant == SWE_VARIANT_PATCH) {
    k_patch_flags<kPatchThreads><<<c->n_patches, kPatchThreads, 0, c->stream>>>(c->d_ctl, c->d_hdr, c->rec, c->rec_b, c->d_dry,
                                                                             c->d_dry + c->n_patches, c->sc);
    c->launches += 1;
  }
  if (c->mp.formula == 2) {           // mobile bed, MPM-like law: the per-cell cube roots of the new state
    k_sed_cell_init<<<grid_for(nc), kBlock, 0, c->stream>>>(c->d_ctl, c->rec, c->gn2, c->mp.cell, (int)nc);
    c->launches += 1;
  }
  k_reset<<<1, 1, 0, c->stream>>>(c->d_ctl, t0);
  k_rate<<<grid_for(nc), kBlock, 0, c->stream>>>(c->d_ctl, c->cell_edge, c->geom, c->inv_area, c->rec, c->rec_b, (int)nc);
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
  k_call_begin<<<1, 1, 0, c->stream>>>(c->d_ctl, (long long)n_steps, t_end, cfl);
  c->launches += 1;
  const int K = c->steps_per_graph;
  int64_t remaining = n_steps < 0 ? std::numeric_limits<int64_t>::max() : n_steps;
  int64_t poll_every = 4;            // graph launches between two reads of t (only when t_end is finite)
  bool done = !(c->t_host < t_end);  // t_end already reached: nothing to do
  while (!done && remaining > 0) {
    int64_t batch_steps = 0;
    if (K > 0 && remaining >= K) {
      int64_t n_graphs = remaining / K;
      if (finite_end) n_graphs = std::min(n_graphs, poll_every);
      for (int64_t j = 0; j < n_graphs; ++j) SWE_CUDA(c, cudaGraphLaunch(c->graph_exec_v[c->variant], c->stream));
      batch_steps = n_graphs * K;
    } else {
      batch_steps = std::min<int64_t>(remaining, 64);   // tail shorter than a graph, or graphs switched off
      for (int64_t j = 0; j < batch_steps; ++j) enqueue_step(c, c->stream);
      SWE_CUDA(c, cudaGetLastError());
    }
    c->launches += batch_steps * n_step_kernels(c);
    remaining -= batch_steps;
    if (finite_end) {                // the only host synchronisation inside the loop: once per batch
      int rc = read_control(c);
      if (rc != SWE_OK) return rc;
      if (!(c->h_ctl->t < t_end) || (c->h_ctl->flags & SWE_FLAG_DT_UNBOUNDED)) done = true;
      poll_every = std::min<int64_t>(poll_every * 2, 64);
    }
  }
  // volume bookkeeping of the last step; then the reductions of swe_step_info
  launch_control(c, c->stream, 1);
  c->launches += 1;
  SWE_CUDA(c, cudaGetLastError());
  if (info) {
    k_info<<<std::min(grid_for(c->nc), kInfoMaxBlocks), kBlock, 0, c->stream>>>(c->d_ctl, c->rec, c->rec_b, c->area, (int)c->nc,
                                                                               c->d_info_part, c->d_info_ticket);
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
      const int want = wet > 0.55 ? SWE_VARIANT_THREE_PASS : (wet < 0.45 ? SWE_VARIANT_PATCH : c->variant);
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
  if (c->variant == SWE_VARIANT_PATCH) {
    k_patch_flags<kPatchThreads><<<c->n_patches, kPatchThreads, 0, c->stream>>>(c->d_ctl, c->d_hdr, c->rec, c->rec_b, c->d_dry,
                                                                             c->d_dry + c->n_patches, c->sc);
    c->launches += 1;
  }
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
  if (formula && c->sc.n > 0) { c->err = "passive scalars and a mobile bed in one context are not built"; return SWE_EINVAL; }
  if (formula && !c->auto_mode && c->variant == SWE_VARIANT_PATCH) {
    c->err = "the fused patch step has no mobile bed: create the context with SWE_VARIANT_AUTO or SWE_VARIANT_THREE_PASS";
    return SWE_EINVAL;
  }
  int rc = read_control(c);          // synchronises: no step in flight
  if (rc != SWE_OK) return rc;
  if (formula) {
    if (c->variant == SWE_VARIANT_PATCH) {
      rc = switch_variant(c, SWE_VARIANT_THREE_PASS, c->h_ctl->cur);
      if (rc != SWE_OK) return rc;
    }
    c->auto_mode = false;            // stays three-pass from here on
    if (!c->mp.qB) {
      SWE_CUDA(c, cudaMalloc((void **)&c->mp.qB, 8 * (size_t)c->ne));
      SWE_CUDA(c, cudaMemsetAsync(c->mp.qB, 0, 8 * (size_t)c->ne, c->stream));
    }
  }
  const double g = c->prm.g;
  c->mp.formula = formula; c->mp.alpha = alpha; c->mp.theta_cr = theta_cr;
  c->mp.shields_den = g * ((s - 1.0) * d_m);
  c->mp.Gm = alpha * std::sqrt(((s - 1.0) * g) * (d_m * (d_m * d_m)));
  c->mp.inv1mp = 1.0 / (1.0 - porosity);
  if (formula == 2) {                 // (g/k^2, cbrt(h)) of the state as it stands; k_cell_update keeps it current
    if (!c->mp.cell) SWE_CUDA(c, cudaMalloc((void **)&c->mp.cell, 16 * (size_t)c->nc));
    k_sed_cell_init<<<grid_for(c->nc), kBlock, 0, c->stream>>>(c->d_ctl, c->rec, c->gn2, c->mp.cell, (int)c->nc);
    c->launches += 1;
    SWE_CUDA(c, cudaGetLastError());
  }
  {                                   // algorithmic bytes of the two kernels that carry the extra work
    int64_t *ab = c->alg_bytes_v[SWE_VARIANT_THREE_PASS];
    ab[1] = c->alg_bytes_base[0] + (formula ? 8 * c->ne + (formula == 2 ? 16 * c->nc : 0) : 0);
    ab[3] = c->alg_bytes_base[1] + (formula ? 8 * c->ne + (formula == 2 ? 16 * c->nc : 0) : 0);
  }
  c->edge_grid = c->base_edge_grid; c->cell_grid = c->base_cell_grid;
  if (formula) {                      // resident grids of the <kMorph> instances
    int per_sm = 3;
    SWE_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_edge_flux<false, true, true>, kBlock, 0));
    c->edge_grid = std::max(1, c->sms * per_sm);
    SWE_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_cell_update<false, true>, kBlock, 0));
    c->cell_grid = std::max(1, c->sms * per_sm);
  }
  if (c->graph_exec_v[SWE_VARIANT_THREE_PASS]) {
    SWE_CUDA(c, cudaStreamSynchronize(c->stream));
    cudaGraphExecDestroy(c->graph_exec_v[SWE_VARIANT_THREE_PASS]);
    c->graph_exec_v[SWE_VARIANT_THREE_PASS] = nullptr;
  }
  if (c->variant == SWE_VARIANT_THREE_PASS) return capture_graph(c);
  const int keep = c->variant;        // fixed bed again on a context that steps with the patch kernel
  c->variant = SWE_VARIANT_THREE_PASS;
  rc = capture_graph(c);
  c->variant = keep;
  return rc;
}

int swe_get_bed(swe_ctx *c, double *zb) {
  if (!c) return SWE_EINVAL;
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
  if (!c->mp.qB) { c->err = "morphodynamics was never switched on"; return SWE_EINVAL; }
  const int64_t ne = c->ne;
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
    k_unpack_state<<<grid_for(nc), kBlock, 0, c->stream>>>(c->d_ctl, c->cell_perm, c->rec, c->rec_b, h, hu, hv, (int)nc);
    c->launches += 1;
    SWE_CUDA(c, cudaGetLastError());
    return SWE_OK;
  }
  k_unpack_state<<<grid_for(nc), kBlock, 0, c->stream>>>(c->d_ctl, c->cell_perm, c->rec, c->rec_b, c->stage, c->stage + nc,
                                                         c->stage + 2 * nc, (int)nc);
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
  std::vector<double> a(c->nc);
  std::vector<EdgeGeom> g(c->ne);
  SWE_CUDA(c, cudaStreamSynchronize(c->stream));
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
  double *d = nullptr;
  SWE_CUDA(c, cudaMalloc((void **)&d, 8 * 4 * ne));
  const double *th_apply = (c->variant == SWE_VARIANT_PATCH) ? c->theta : nullptr;   // three-pass: limited in place
  k_export_flux<<<grid_for(ne), kBlock, 0, c->stream>>>(c->edge_perm, c->geom, c->flux, th_apply, d, d + ne, d + 2 * ne,
                                                        d + 3 * ne, (int)ne);
  c->launches += 1;
  cudaError_t e1 = cudaStreamSynchronize(c->stream);
  if (e1 == cudaSuccess) e1 = cudaMemcpy(F1, d, 8 * ne, cudaMemcpyDeviceToHost);
  if (e1 == cudaSuccess) e1 = cudaMemcpy(F3, d + ne, 8 * ne, cudaMemcpyDeviceToHost);
  if (e1 == cudaSuccess) e1 = cudaMemcpy(GL, d + 2 * ne, 8 * ne, cudaMemcpyDeviceToHost);
  if (e1 == cudaSuccess) e1 = cudaMemcpy(GR, d + 3 * ne, 8 * ne, cudaMemcpyDeviceToHost);
  cudaFree(d);
  SWE_CUDA(c, e1);
  if (theta) {
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
      std::vector<EdgeGeom> geom; std::vector<int32_t> ce4; std::vector<double> area;
      internal_tables(hm, geom, ce4, area);
      std::vector<int32_t> string_pos(hm.ne, -1);
      int32_t n_string = 0;
      for (int64_t e = 0; e < hm.ne; ++e) if (geom[e].R <= -3) string_pos[e] = n_string++;
      PatchTables pt;
      if (!build_patches(hm.nc, hm.ne, geom, ce4, area, string_pos, patch_cells, pt, g_create_error)) return SWE_EINVAL;
      int64_t own = 0, covered = 0;
      std::vector<uint8_t> seen(hm.nc, 0);
      for (const PatchHeader &h : pt.hdr) {
        own += h.n_own;
        for (int32_t l = 0; l < h.n_own; ++l) if (!seen[h.cell0 + l]) { seen[h.cell0 + l] = 1; ++covered; }
      }
      v[1] = (int64_t)pt.hdr.size(); v[2] = pt.sum_loc; v[3] = pt.sum_e; v[4] = pt.max_loc; v[5] = pt.max_e;
      v[6] = (int64_t)sizeof(double) * patch_smem_layout(pt.max_loc, pt.max_c1, pt.max_e, pt.max_eown).total;
      v[7] = own; v[8] = covered; v[9] = (int64_t)pt.patch_nbr.size();
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
  return c->variant == SWE_VARIANT_PATCH ? kPatchNames[k] : kThreePassNames[k];
}

int64_t swe_algorithmic_bytes(const swe_ctx *c, int k) { return (c && k >= 0 && k < n_step_kernels(c)) ? c->alg_bytes_v[c->variant][k] : 0; }

int swe_get_patch_stats(swe_ctx *c, int64_t *out, int n_out) {
  if (!c || !out || n_out < 1) return SWE_EINVAL;
  int rc = read_control(c);
  if (rc != SWE_OK) return rc;
  const int64_t v[9] = {c->variant, c->n_patches, c->pt.patch_cells, (int64_t)c->patch_smem, c->pt.sum_loc, c->pt.sum_e,
                        c->pt.max_loc, c->pt.max_e, (int64_t)c->h_ctl->patches_skipped};
  for (int k = 0; k < n_out && k < 9; ++k) out[k] = v[k];
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
  k_call_begin<<<1, 1, 0, c->stream>>>(c->d_ctl, (long long)n_steps, std::numeric_limits<double>::infinity(), cfl);
  c->launches += 1;
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
  launch_control(c, c->stream, 1);
  c->launches += 1;
  SWE_CUDA(c, cudaGetLastError());
  for (int k = 0; k < n_ms; ++k) ms[k] = k < nk ? sum[k] / (double)n_steps : 0.0;
  c->t_host = -std::numeric_limits<double>::infinity();
  return SWE_OK;
}

}  // extern "C"
