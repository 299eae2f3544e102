/* oracle/swe_ref.h -- TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * Plain single-threaded fp64 C++ oracle of the explicit finite-volume shallow-water step of
 * BASEMENT v3 (arxiv 2102.12862), written from the paper and SURVEY.md section 8(c) only.
 * It shares no code, header, table or helper with the CUDA path under paper_2102_12862_b200/.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * load this library.
 *
 * What is computed, per time step n (PAPER.md line / equation in brackets):
 *   S0  dt  = min(CFL / max_i max_j (lambda_ij / rho_ij), t_end - t, dt_max)      [Eq. 21, PAPER.md:306-312]
 *   S1  per edge: hydrostatic "modified-state" reconstruction [PAPER.md:254, ref 69]
 *       + HLLC flux (HLL mass/normal momentum + upwinded tangential momentum)     [PAPER.md:252, ref 18 ch.10]
 *   S2  per cell: sum over j=1..3 of l_ij F_ij                                    [Eq. 12, PAPER.md:244-250]
 *   S3  explicit Euler update of (h, q_x, q_y) + split friction source            [Eq. 12; Eq. 2, Table 1
 *       Strickler row PAPER.md:106-123; splitting PAPER.md:254]
 *   S4  t += dt
 * Readings of every point the paper leaves open are listed in DESIGN.md (R-1 ... R-18).
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): hand-computed fluxes, literal Eq. 10/11 H-form
 * identity, geometry closed forms, Ritter and Stoker dam breaks, lake at rest, mass conservation,
 * uniform-flow normal depth, permutation invariance, restart, T6 rest level 0.364 m.
 * Morphodynamics (tests/test_oracle_morph.py): Table 2 by hand, psi of Eq. 16 by finite differences, Vieta's relations
 * of Eq. 16, HLL special cases of Eq. 14-15, Eq. 13 re-assembled with numpy, porosity factor, sediment volume in a closed
 * box, flat bed under a uniform stream, bed-hump celerity under the Grass-like law.
 * Draining-time limiter with moving water: tests/golden/limiter_moving_water.txt (hand-computed: F1, F3, GL, GR all scaled).
 * Builds of this one source (oracle/build.py): fp64 single-threaded (the default; every parity test), single precision
 * (-DSWE_REF_REAL=float; R-21; pinned by tests/test_oracle_f32.py: golden values to fp32 round-off, mass, lake
 * at rest, dam-break errors against the fp64 build), and an OpenMP build of the fp64 source for bench.py's optional
 * cpu_baseline omp line (bit-identical results; no test depends on it).
 * "parity unpinned" items: none of the functions; but the *choice* of readings R-2 (HLLC form) and
 * R-11 (inflow distribution) cannot be pinned against BASEMENT itself (closed source).
 */
#ifndef SWE_REF_H
#define SWE_REF_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct swe_ref_ctx swe_ref_ctx;

typedef struct {
  int64_t n_nodes, n_cells, n_edges;
  const double *node_xy;      /* [n_nodes][2] */
  const int32_t *tri;         /* [n_cells][3] CCW */
  const int32_t *edge_cell;   /* [n_edges][2] L, R (R<0: -1 wall, -2 transmissive, -3-s string s) */
  const int32_t *cell_edge;   /* [n_cells][3] slot k = edge (tri[k], tri[(k+1)%3]) */
  const double *zb;           /* [n_cells] */
  const double *kst;          /* [n_cells] Strickler k, +inf = frictionless */
} swe_ref_mesh;

typedef struct { double g, h_dry, dt_max; } swe_ref_params;

typedef struct {
  double t, dt_last;
  int64_t steps_done, n_wet;
  double vol, vol_clipped, vol_in, vol_out;
  int flags;
} swe_ref_info;

enum { SWE_REF_BC_INFLOW_Q = 1, SWE_REF_BC_OUTFLOW_UNIFORM = 2 };

int swe_ref_create(const swe_ref_mesh *m, const swe_ref_params *p, swe_ref_ctx **out);
int swe_ref_set_boundary(swe_ref_ctx *c, int string_id, int type, const double *params, int n_params);
int swe_ref_set_state(swe_ref_ctx *c, const double *h, const double *hu, const double *hv, double t0);
/* Passive scalars (Eq. 8, advective part only; update Eq. 20 PAPER.md:298-304 with A_ij = F1 * phi of
 * the upwind side; R-19).  qc = [n_species][n_cells] specific masses q_c = h * phi_c, n_species <= 5. */
int swe_ref_set_scalars(swe_ref_ctx *c, int n_species, const double *qc);
int swe_ref_get_scalars(swe_ref_ctx *c, double *qc);
/* concentrations phi[0..n) carried by the water that enters through INFLOW_Q string string_id (default 0) */
int swe_ref_set_boundary_scalar(swe_ref_ctx *c, int string_id, const double *phi, int n);
/* Morphodynamics (Eq. 3; Eq. 13-16; Table 2; R-20):
 * formula 0 = fixed bed, 1 = Grass-like alpha |u|^3, 2 = MPM-like alpha (theta - theta_cr)^1.5 sqrt((s-1) g d_m^3).
 * From the next step on the bed z_B of every cell moves by Eq. 13 with the HLL-type sediment flux of Eq. 14-16. */
int swe_ref_set_morphology(swe_ref_ctx *c, int formula, double alpha, double theta_cr, double sdens, double dm,
                           double porosity);
int swe_ref_get_bed(swe_ref_ctx *c, double *zb);
int swe_ref_get_sediment_flux(swe_ref_ctx *c, double *qB);   /* q_Bij [n_edges] of the most recent step */
/* inspection: one cell seen from one interface (Table 2 + Eq. 16), and Eq. 14-15 for one interface */
void swe_ref_sediment_state(int formula, double alpha, double theta_cr, double sdens, double dm, double g,
                            double h, double u, double v, double gn2, double nx, double ny,
                            double *qBn, double *psi, double *lam1, double *lam2);
double swe_ref_sediment_flux(double qBi, double l1i, double l2i, double zi, double qBj, double l1j, double l2j, double zj);
int swe_ref_step(swe_ref_ctx *c, int64_t n_steps, double t_end, double cfl, swe_ref_info *info);
int swe_ref_get_state(swe_ref_ctx *c, double *h, double *hu, double *hv);
void swe_ref_destroy(swe_ref_ctx *c);
const char *swe_ref_last_error(const swe_ref_ctx *c);

/* --- inspection entry points used by the pins (not part of the 5-call boundary) --------------- */
/* One interior-edge evaluation of S1: in = effective depths/velocities/bed of both sides and the
 * unit normal (L -> R); out = F1 (mass), F3 (tangential momentum), GL, GR (normal momentum minus
 * each side's hydrostatic pressure). */
void swe_ref_edge_flux(double g, double heL, double uL, double vL, double zL,
                       double heR, double uR, double vR, double zR, double nx, double ny,
                       double *F1, double *F3, double *GL, double *GR);
/* wall flux evaluated through the interior solver with a mirror ghost state (pin for the closed form) */
void swe_ref_wall_flux_via_ghost(double g, double he, double un, double ut, double *F1, double *F3, double *G);
/* geometry of the context: area [n_cells]; nx, ny, len [n_edges] (normal from L to R) */
int swe_ref_get_geometry(swe_ref_ctx *c, double *area, double *nx, double *ny, double *len);
/* per-edge outputs of the most recent step: F1, F3, GL, GR [n_edges] each */
int swe_ref_get_edge_flux(swe_ref_ctx *c, double *F1, double *F3, double *GL, double *GR);
/* cube root rounded to nearest (R-14): the only non-IEEE-basic operation of the scheme */
double swe_ref_cbrt(double x);
/* dt that S0 would choose now for (cfl, t_end) without advancing */
double swe_ref_peek_dt(swe_ref_ctx *c, double cfl, double t_end);

#ifdef __cplusplus
}
#endif
#endif
