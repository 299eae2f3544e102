/* include/swe.h -- C-ABI of the B200-native shallow-water hot path (libswe_b200.so).
 *
 * One thing is exported: the explicit finite-volume time step of the 2-D depth-averaged
 * shallow-water equations on an unstructured triangular mesh, as BASEMENT v3 (arxiv 2102.12862)
 * states it.  "P:n" below is line n of the paper text; "R-k" are the readings of points
 * the paper leaves open, listed in DESIGN.md section 2.
 *
 *   per time step n (state U^n = (h, q_x, q_y) per cell, fp64):
 *     S0  dt = min(CFL / max_i max_j(lambda_ij / rho_ij), t_end - t, dt_max)         Eq. 21
 *     S1  per edge: hydrostatic ("modified-state") face depths + HLLC flux
 *     S1c per cell: draining-time factor theta_i; edge flux x theta of its donor     R-8b
 *     S2  per cell: sum_j l_ij F_ij in slot order                                    Eq. 12
 *     S3  explicit Euler update + split Strickler friction                           Eq. 12; Eq. 2 P:106-111;
 *                                                                                    Table 1
 *     S4  t += dt
 *
 * Every step of the path runs in CUDA kernels compiled for sm_100a; there is no CPU fallback.  All
 * functions return SWE_OK (0) or a negative error code; nothing throws or exits across this boundary.
 * One context must be used by one host thread at a time.
 */
#ifndef SWE_B200_H
#define SWE_B200_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct swe_ctx swe_ctx; /* opaque; created by swe_create, freed by swe_destroy */

enum {
  SWE_OK = 0,
  SWE_EINVAL = -1,     /* null / out-of-range argument                                             */
  SWE_EMESH = -2,      /* non-CCW or zero-area cell, non-conforming mesh, inconsistent tables       */
  SWE_ENOMEM = -3,     /* host or device allocation failed, or the lent workspace is too small      */
  SWE_ECUDA = -4,      /* a CUDA call failed (no device, launch error, ...); see swe_last_error     */
  SWE_ENONFINITE = -5  /* swe_step found a non-finite state value at the end of the call            */
};

/* Boundary codes in edge_cell[e][1] (P:332 wall is the default of every external edge) */
enum { SWE_EDGE_WALL = -1, SWE_EDGE_TRANSMISSIVE = -2 /* , -3 - s = member of boundary string s */ };
/* Boundary-string types for swe_set_boundary (types named at P:342; formulas are readings R-11, R-12) */
enum { SWE_BC_NONE = 0 /* string behaves as wall */, SWE_BC_INFLOW_Q = 1, SWE_BC_OUTFLOW_UNIFORM = 2 };
/* Cell / edge renumbering applied inside the library (invisible at this boundary) */
enum { SWE_RENUMBER_NONE = 0, SWE_RENUMBER_MORTON = 1, SWE_RENUMBER_RCM = 2 /* reverse Cuthill-McKee */ };
/* Step variant: both compute bit-identical states.  AUTO keeps both ready: the fused patch step
 * whenever four of its blocks fit an SM (the faster variant at every wet fraction then); with
 * larger patches it chooses at every swe_set_state from the wet fraction of the new state (patch step below 50 % wet
 * cells, three-pass step above); on a numbering that is not spatially compact it is the three-pass step. */
enum { SWE_VARIANT_AUTO = 0, SWE_VARIANT_THREE_PASS = 1 /* edge flux -> theta -> CSR gather + update */,
       SWE_VARIANT_PATCH = 2 /* one fused kernel per step over shared-memory mesh patches */ };
/* Arithmetic ("single or double"; R-21).  SINGLE: state, geometry and every flux / update operation in
 * fp32 (16-byte records); time, dt = CFL / rate, the hydrograph lookup and the volume bookkeeping stay fp64; built for the
 * hydrodynamic step only (SWE_EINVAL with scalars or mobile bed), in both step variants; AUTO: fused patch step below
 * 75 % wet cells, three-pass step above (it moves half the bytes in fp32 and wins on all-wet states).  swe_get_edge_flux
 * is not built for the single-precision patch step.  The arrays at this boundary stay fp64 in both cases (rounded once
 * on the way in, exact on the way out). */
enum { SWE_PRECISION_DOUBLE = 0, SWE_PRECISION_SINGLE = 1 };
/* swe_step_info.flags */
enum { SWE_FLAG_NONFINITE = 1, SWE_FLAG_DT_UNBOUNDED = 2 /* whole domain dry and dt_max = +inf */,
       SWE_FLAG_STALLED = 4 /* Eq. 21 gave dt <= 0 or t + dt == t (a rate of +inf from a non-finite state, or dt below
                               ulp(t)): swe_step stops stepping and returns, with this flag in info */ };

/* The mesh (section 4.1, Fig. 2): conforming triangulation, cell i with neighbours j = 1..3
 * across edges Gamma_ij.  All pointers are HOST pointers; everything is copied during swe_create and
 * the caller may free the arrays as soon as it returns. */
typedef struct {
  int64_t n_nodes, n_cells, n_edges;
  const double *node_xy;    /* [n_nodes][2]  metres                                                  */
  const int32_t *tri;       /* [n_cells][3]  counter-clockwise node ids                              */
  const int32_t *edge_cell; /* [n_edges][2]  [0] = L >= 0; [1] = R >= 0, or a boundary code < 0.
                               The stored unit normal of an edge points from L to R.  May be NULL
                               together with cell_edge: both tables are then built by the library,
                               every boundary edge a wall, and n_edges is ignored.                   */
  const int32_t *cell_edge; /* [n_cells][3]  slot k = edge between tri[k] and tri[(k+1)%3]           */
  const double *zb;         /* [n_cells]     cell-mean bed elevation z_B (R-13)                      */
  const double *kst;        /* [n_cells]     Strickler k_str (Table 1); +inf = frictionless   */
} swe_mesh;

typedef struct {
  double g;             /* gravity; default 9.81                                                     */
  double h_dry;         /* wet/dry threshold (R-8): cells with h <= h_dry carry no momentum; 1e-3    */
  double dt_max;        /* upper bound of dt, used when the whole domain is dry; default +inf        */
  int renumber;         /* SWE_RENUMBER_*; default MORTON                                            */
  int state_on_device;  /* 0: swe_set_state/swe_get_state take HOST pointers (default);
                           1: they take DEVICE pointers (e.g. torch tensors), read/written on stream  */
  int steps_per_graph;  /* time steps captured per CUDA graph launch; default 32; 0 = no graph       */
  int variant;          /* SWE_VARIANT_*; default AUTO                                               */
  int patch_cells;      /* cells per patch of the fused step, 32..1024 (at least one thread per own cell);
                           0 = default (the largest of 240..192 that runs four blocks per SM; less
                           on meshes that would not fill the SMs)                                    */
  int n_species;        /* passive scalar species advected with the flow (0..5); default 0    */
  int morphology;       /* 1: reserve room for the mobile-bed module (swe_set_morphology); default 0 */
  int precision;        /* SWE_PRECISION_*; default DOUBLE                                           */
  void *cuda_stream;    /* cudaStream_t all work is enqueued on; NULL = the legacy default stream    */
  void *workspace;      /* DEVICE memory lent by the caller for the context's lifetime (e.g. a torch
                           uint8 tensor), 256-byte aligned: EVERY device array of the context is carved
                           from it (state, tables, patch blobs, scalars, mobile bed, control block).
                           NULL: the library makes one cudaMalloc of the same size instead.          */
  size_t workspace_bytes; /* size of workspace; must be >= swe_workspace_bytes(mesh, params)         */
} swe_params;

typedef struct {
  double t, dt_last;           /* simulation time; dt of the most recent step                        */
  int64_t steps_done, n_wet;   /* steps since swe_set_state; cells with h > h_dry                    */
  double vol;                  /* sum_i h_i |Omega_i|                                                 */
  double vol_clipped;          /* volume created by clipping residual negative depths (R-8b)         */
  double vol_in, vol_out;      /* volume through INFLOW_Q / OUTFLOW_UNIFORM strings since set_state  */
  int flags;                   /* SWE_FLAG_*                                                          */
} swe_step_info;

/* Fills *p with the defaults named above. */
void swe_params_default(swe_params *p);

/* Device bytes a context for this mesh and these parameters needs (params == NULL: defaults; workspace / stream
 * fields are ignored).  Runs the host part of swe_create (validation, renumbering, patch tables) to size every
 * array, with no CUDA call; returns 0 when swe_create would reject the arguments (swe_last_error(NULL)). */
size_t swe_workspace_bytes(const swe_mesh *mesh, const swe_params *params);

/* Validates the mesh (CCW, positive area, both tables consistent and conforming), computes the geometry
 * of section 4.1 (areas, edge lengths, unit normals L->R), renumbers cells and edges (Morton order of the
 * centroids; slot order and L/R orientation are kept, R-15), uploads everything and captures the step graph.
 * params == NULL: defaults.  On failure *out is NULL and swe_last_error(NULL) describes the reason. */
int swe_create(const swe_mesh *mesh, const swe_params *params, swe_ctx **out);

/* Sets type and parameters of boundary string s (the edges whose code is -3 - s).
 *   SWE_BC_INFLOW_Q (R-11):        params = hydrograph table (t_0, Q_0, t_1, Q_1, ...), n_params even, t ascending;
 *                                  Q(t) piecewise linear, clamped at both ends; Q in m^3/s over the whole string.
 *   SWE_BC_OUTFLOW_UNIFORM (R-12): params = (S_0), the bed slope of the normal-depth condition.
 * The parameters are copied. */
int swe_set_boundary(swe_ctx *ctx, int string_id, int type, const double *params, int n_params);

/* Sets the state (h, hu, hv) [n_cells] in the CALLER's cell numbering and the time t0; resets steps_done and
 * the volume counters.  Host or device pointers according to swe_params.state_on_device. */
int swe_set_state(swe_ctx *ctx, const double *h, const double *hu, const double *hv, double t0);

/* Advances until n_steps steps are done (n_steps < 0: no limit) or t reaches t_end (+inf: no limit),
 * whichever comes first; the last step is shortened to land on t_end exactly.  cfl in (0, 1] (default
 * 0.9 in the paper).  With the literal rho_ij of Eq. 21 the first-order scheme is linearly stable only up to
 * cfl ~ 0.75 on regular right-triangle meshes (bounded transverse noise above that: DESIGN.md R-7,
 * tests/test_oracle_analytic.py::test_config1_noise_at_cfl_09_and_07); irregular Delaunay meshes run clean at 0.9.  All steps run on the device without host synchronisation per step; the call synchronises
 * the stream once per chunk of steps when t_end is finite, and once at the end if info != NULL.
 * info may be NULL.  Returns SWE_ENONFINITE if info was requested and the state holds NaN/inf. */
int swe_step(swe_ctx *ctx, int64_t n_steps, double t_end, double cfl, swe_step_info *info);

/* Passive scalars (section 3.3, Eq. 8, advective part; update Eq. 20 P:298-304 with A_ij = limited mass flux
 * x concentration on the upwind side of the contact wave; R-19).  qc = [n_species][n_cells] specific masses
 * q_c = h * phi_c in the CALLER's cell numbering (host or device pointers as for swe_set_state).  They are advanced by
 * every step of swe_step; swe_set_state does not touch them (new contexts hold q_c = 0). */
int swe_set_scalars(swe_ctx *ctx, const double *qc);
int swe_get_scalars(swe_ctx *ctx, double *qc);
/* concentrations phi[0..n) of the water entering through SWE_BC_INFLOW_Q string string_id (default 0) */
int swe_set_boundary_scalar(swe_ctx *ctx, int string_id, const double *phi, int n);

/* Morphodynamics (section 3.2, Eq. 3; section 4.3, Eq. 13-16; Table 2; R-20).
 * From the next step on the bed elevation of every cell moves, with the hydrodynamic time step ("synchronous-decoupled",
 * P:256), by Eq. 13 with S_b = 0 and the HLL-type sediment flux of Eq. 14-16 evaluated from the state at t^n:
 *   formula 0  fixed bed (switches the module off again)
 *   formula 1  Grass-like   |q_B| = alpha |u|^3                              (m = 3, u_cr = 0)
 *   formula 2  MPM-like     |q_B| = alpha (theta - theta_cr)^1.5 sqrt((s-1) g d_m^3), theta = |u|^2 / (k_st^2 h^(1/3) (s-1) d_m)
 * theta_cr, s, d_m are read by formula 2 only; porosity p in [0, 1).  No transport through walls or where a side of an
 * interface is dry (h <= h_dry); through every open boundary the interior cell's own flux passes (equilibrium).
 * Both step variants carry the module (three-pass: the edge kernel also writes q_Bij, 8 B per edge, the cell kernel gathers it
 * and writes z_B with the record it writes anyway; fused patch step: q_Bij of the patch's own edges in shared memory), with
 * or without scalar species, bit-identical to each other; AUTO keeps choosing between them.  The context must have been
 * created with swe_params.morphology = 1 (room for q_Bij and the per-cell record of the MPM-like law), else SWE_EINVAL; not
 * built for single precision.  The bed persists across swe_set_state (there is no call that resets it; create a new
 * context for the initial bed).  Synchronises the stream and captures the CUDA graphs of the step again (once per call). */
int swe_set_morphology(swe_ctx *ctx, int formula, double alpha, double theta_cr, double s, double d_m, double porosity);
/* bed elevation z_B [n_cells] in the caller's cell numbering (host or device pointer as for swe_get_state) */
int swe_get_bed(swe_ctx *ctx, double *zb);
/* inspection: q_Bij [n_edges] of the most recent step, caller edge numbering, positive from L to R */
int swe_get_sediment_flux(swe_ctx *ctx, double *qB);

/* Reads the state in the caller's cell numbering (host or device pointers as for swe_set_state). */
int swe_get_state(swe_ctx *ctx, double *h, double *hu, double *hv);

void swe_destroy(swe_ctx *ctx);

/* Message of the most recent error of ctx, or of the most recent failed swe_create if ctx == NULL.
 * The pointer stays valid until the next failing call on the same context / thread. */
const char *swe_last_error(const swe_ctx *ctx);

/* ---- inspection entry points (used by the parity tests; HOST pointers, caller numbering, they synchronise) */
/* area [n_cells]; nx, ny, len [n_edges]: geometry of section 4.1 as the kernels use it */
int swe_get_geometry(swe_ctx *ctx, double *area, double *nx, double *ny, double *len);
/* per-edge results of the most recent step, after the limiter: F1 (mass), F3 (tangential momentum),
 * GL, GR (normal momentum minus each side's hydrostatic pressure) [n_edges]; theta [n_cells] (may be NULL) */
int swe_get_edge_flux(swe_ctx *ctx, double *F1, double *F3, double *GL, double *GR, double *theta);
/* dt that S0 would choose now for (cfl, t_end), without advancing */
int swe_peek_dt(swe_ctx *ctx, double cfl, double t_end, double *dt);
/* internal numbering: cell_perm[new] = caller cell id [n_cells]; edge_perm[new] = caller edge id [n_edges] */
int swe_get_permutation(swe_ctx *ctx, int32_t *cell_perm, int32_t *edge_perm);
/* edge tables as used (identical to the caller's when those were given): for meshes passed without tables */
int swe_get_tables(swe_ctx *ctx, int64_t *n_edges, int32_t *edge_cell, int32_t *cell_edge);
/* y[i] = cube root of x[i] rounded to nearest, evaluated on the device by the function the kernels use (R-14);
 * x, y: HOST pointers [n]; uses the current device and the legacy default stream; needs no context */
int swe_device_cbrt(const double *x, double *y, int64_t n);
/* The HOST part of swe_create alone (no CUDA call, works without a GPU): validation, edge tables, geometry,
 * renumbering and -- when patch_cells > 0 -- the patch tables of the fused step.  out[0..9] = edges, patches, sum of
 * local cells, sum of local edges, largest local cell count, largest local edge count, shared memory per block
 * [bytes], sum of own cells, distinct own cells, entries of the patch-neighbour lists.  cell_perm / edge_perm (may be
 * NULL): internal -> caller numbering.  Returns the same error codes as swe_create (swe_last_error(NULL)). */
int swe_host_preprocess(const swe_mesh *mesh, int renumber, int patch_cells, int64_t *out, int n_out,
                        int32_t *cell_perm, int32_t *edge_perm);
/* number of kernel launches enqueued by this context since swe_create (graph nodes count individually) */
int64_t swe_kernel_launches(const swe_ctx *ctx);
/* Measurement (bench.py roofline): advances n_steps >= 1 time steps with plain launches, every kernel of the step
 * bracketed by CUDA events on the context's stream; ms[k] = mean device time of kernel k per step, in
 * milliseconds, for k < min(n_ms, swe_step_kernel_count()).  Results are those of swe_step(n_steps, +inf, cfl).
 * It synchronises. */
int swe_profile_step(swe_ctx *ctx, int64_t n_steps, double cfl, double *ms, int n_ms);
/* kernels per time step of this context's variant, and the name of kernel k of the step (NULL if out of range) */
int swe_step_kernel_count(const swe_ctx *ctx);
const char *swe_step_kernel_name(const swe_ctx *ctx, int k);
/* algorithmic DRAM bytes per launch of kernel k of the step: every datum the kernel needs counted once at the size
 * of the record that carries it; re-reads of halo cells / duplicated records are NOT counted */
int64_t swe_algorithmic_bytes(const swe_ctx *ctx, int k);
/* the same on the per-cell figures of SURVEY.md section 8(d) ("Algorithmic bytes per cell-step"): 132 B x n_cells for
 * the one-pass fused step; 284 B x n_cells for the edge-flux -> gather design, split 148 (edge pass) + 136 (cell pass);
 * + 16 B per cell and scalar species.  bench.py reports the roofline fraction on both counts. */
int64_t swe_survey_bytes(const swe_ctx *ctx, int k);
/* out[0..11] = variant, patches, cells per patch, dynamic shared memory per block [bytes], sum over patches of local
 * cells, sum over patches of local edges, largest local cell count, largest local edge count, the number of
 * patch-steps since swe_create in which a block found its whole patch dry and skipped the flux work, the
 * __launch_bounds__ minimum blocks per SM of the kernel instance, bytes per patch blob, bytes of a blob that are
 * staged into shared memory.  It synchronises. */
int swe_get_patch_stats(swe_ctx *ctx, int64_t *out, int n_out);

/* ---- an entry point that allocates nothing -----------------------------------------------------------------
 * The reductions of swe_step_info (vol = sum_i h_i |Omega_i|, the quantity whose conservation P:591 promises; n_wet =
 * cells with h > h_dry, R-8; non-finite check) of a state given as plain arrays, for callers that cannot call
 * cudaMalloc: code under CUDA graph capture, tight serving loops, harnesses that forbid it.  It needs no context and no
 * workspace: the per-block partial results and the ticket that swe_step keeps in the context's workspace live in a
 * file-scope __device__ array of 98,560 bytes, which every GPU that loads the library holds until the process exits.
 * It calls no cudaMalloc / cudaFree / allocating routine, does not synchronise, and enqueues one 4-byte memset and one
 * kernel on `cuda_stream` (NULL = the legacy default stream) of the CURRENT device.
 *   h, hu, hv, area : DEVICE pointers, [n_cells] doubles each, read only; any cell numbering (the same in all four)
 *   n_cells         : 1 .. SWE_SUMMARY_STATIC_MAX_CELLS; beyond that SWE_EINVAL (the array holds one partial per 4096
 *                     cells) and swe_last_error(NULL) names the limit -- use swe_step's info for larger meshes
 *   out             : DEVICE pointer to one swe_state_summary, written by the kernel (valid once the stream has
 *                     reached that point); owned by the caller
 * vol is summed in a fixed order (independent of scheduling): the same inputs give the same bits; it differs from
 * swe_step_info.vol, which sums in the library's internal numbering, by rounding only (<= 1e-12 relative).
 * ALL calls share the one array per GPU: calls that overlap on the GPU (two streams, two host threads) race on it and
 * give wrong sums -- the caller serialises them.  The first call on a device resolves the array's device address
 * (cudaGetSymbolAddress); make that first call outside graph capture. */
#define SWE_SUMMARY_STATIC_MAX_CELLS 16777216 /* 2^24 */
typedef struct {
  double vol;        /* sum_i h_i |Omega_i|                */
  int64_t n_wet;     /* cells with h > h_dry                */
  int32_t nonfinite; /* 1 if any h, hu or hv is inf or NaN  */
  int32_t pad_;
} swe_state_summary;
int swe_state_summary_static(const double *h, const double *hu, const double *hv, const double *area, int64_t n_cells,
                             double h_dry, void *cuda_stream, swe_state_summary *out);

#ifdef __cplusplus
}
#endif
#endif
