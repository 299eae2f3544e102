// oracle/swe_ref.cpp -- TEST INFRASTRUCTURE, NOT PRODUCT. See oracle/swe_ref.h for scope, citations and pins.
//
// Plain, single-threaded, fp64. Compile with -O2 -ffp-contract=off (no FMA contraction) so that the
// parenthesisation written here IS the arithmetic (R-14). No blocking, no fusion, no
// reordering beyond what SURVEY.md 8(c) S0-S4 states; loops run over edges and cells in index order.
#include "swe_ref.h"

#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <limits>
#include <map>
#include <string>
#include <vector>

// Optional OpenMP build (oracle/build.py build_omp(): -fopenmp -DSWE_REF_OMP), the analogue of the paper's `omp`
// backend (Table 3) for bench.py's cpu_baseline_omp line ONLY: the loops below are race-free as written
// (per-edge outputs in the edge loops, per-cell outputs in the cell loops, gather in slot order), so the same source
// runs them in parallel with identical results.  The default build, which every test uses, is single-threaded.
#if defined(SWE_REF_OMP)
#define SWE_REF_PARALLEL_FOR _Pragma("omp parallel for schedule(static)")
#define SWE_REF_PARALLEL_MAX(r) _Pragma("omp parallel for schedule(static) reduction(max : r)")
#define SWE_REF_ATOMIC _Pragma("omp atomic")
#else
#define SWE_REF_PARALLEL_FOR
#define SWE_REF_PARALLEL_MAX(r)
#define SWE_REF_ATOMIC
#endif

// Precision switch ("single or double"): the SAME source builds the fp64
// oracle (default) and, with -DSWE_REF_REAL=float (oracle/build.py build_f32()), the single-precision oracle.  `real`
// is the type of the state, the geometry and every flux / update operation; RL(x) is the literal x in that type.  What
// stays fp64 in both builds: time and the time step (t, dt = cfl / rate, t_end), the hydrograph lookup, the volume
// bookkeeping, and the mesh geometry as computed from the node coordinates (rounded once to `real` when stored).
// The cube root of a `real` is the correctly rounded fp64 cube root rounded to `real` (R-14, R-21).
#ifndef SWE_REF_REAL
#define SWE_REF_REAL double
#endif
typedef SWE_REF_REAL real;
#define RL(x) (static_cast<real>(x))

namespace {

struct BString {
  int type = 0;
  std::vector<double> params;
  std::vector<int32_t> edges;  // members in ascending (caller) edge id = "string order"
  std::vector<double> phi_in;  // scalar concentrations carried by an INFLOW_Q string, one per species (default 0)
  // values fixed at t^n by eval_strings():
  real Q = 0, sumK = 0, sumL = 0;
};

thread_local std::string g_create_error;

}  // namespace

struct swe_ref_ctx {
  int64_t nc = 0, ne = 0;
  real g = RL(9.81), h_dry = RL(1e-3);
  double dt_max = std::numeric_limits<double>::infinity();
  std::vector<real> area, invA, gn2, zb, kst;
  std::vector<int32_t> eL, eR, ce;      // ce[3*i+k]
  std::vector<real> nx, ny, len;        // per edge, normal from L to R  [PAPER.md:228]
  std::vector<real> h, qx, qy;
  std::vector<real> F1, F3, GL, GR;     // per edge, most recent step (after the limiter)
  std::vector<real> theta;              // per cell, most recent step
  // passive scalars (section 3.3, Eq. 8 advective part; Eq. 20 with A_ij only): specific mass q_c = h phi_c
  int n_species = 0;
  std::vector<std::vector<real>> qc;    // [species][cell]
  std::vector<std::vector<real>> Ac;    // [species][edge] advective scalar flux of the most recent step
  // morphodynamics (section 3.2 Eq. 3, section 4.3 Eq. 13-16; R-20): 0 = fixed bed
  int morph_formula = 0;
  double morph_alpha = 0.0, morph_theta_cr = 0.047, morph_s = 2.65, morph_dm = 1e-3, morph_p = 0.4;
  std::vector<real> qB;                 // per edge: normal sediment flux q_Bij of the most recent step
  std::map<int, BString> strings;
  double t = 0.0, dt_last = 0.0, vol_clipped = 0.0, vol_in = 0.0, vol_out = 0.0;
  int64_t steps_done = 0;
  int flags = 0;
  std::string err;
};

// ------------------------------------------------------------------------------------------------
// S1, interior edge. PAPER.md:252 (HLLC, "Chapter 10 of [18]"), PAPER.md:254 (modified-state bed
// slope of ref [69]); arithmetic exactly as SURVEY.md 8(c) S1 / DESIGN.md R-1, R-2, R-3.
// ------------------------------------------------------------------------------------------------
static void riemann_nt(real g, real heL, real unL, real utL, real zL,
                       real heR, real unR, real utR, real zR,
                       real *F1o, real *F3o, real *GLo, real *GRo) {
  const real dz = zR - zL;
  const real hsL = std::fmax(RL(0.0), heL - std::fmax(RL(0.0), dz));    // face depths over z* = max(zL, zR)
  const real hsR = std::fmax(RL(0.0), heR - std::fmax(RL(0.0), -dz));
  if (hsL == RL(0.0) && hsR == RL(0.0)) {
    *F1o = RL(0.0); *F3o = RL(0.0); *GLo = RL(0.0); *GRo = RL(0.0);
    return;
  }
  const real cL = std::sqrt(g * hsL), cR = std::sqrt(g * hsR);
  real SL, SR;
  if (hsL > RL(0.0) && hsR > RL(0.0)) {                  // two-rarefaction estimates
    const real us = RL(0.5) * (unL + unR) + (cL - cR);
    const real cs = RL(0.5) * (cL + cR) + RL(0.25) * (unL - unR);
    SL = std::fmin(unL - cL, us - cs);
    SR = std::fmax(unR + cR, us + cs);
  } else if (hsR == RL(0.0)) {                       // dry bed on the right
    SL = unL - cL;
    SR = unL + RL(2.0) * cL;
  } else {                                       // dry bed on the left
    SL = unR - RL(2.0) * cR;
    SR = unR + cR;
  }
  const real qsL = hsL * unL, qsR = hsR * unR;
  const real pL = (RL(0.5) * g) * (hsL * hsL), pR = (RL(0.5) * g) * (hsR * hsR);
  const real FL1 = qsL, FL2 = qsL * unL + pL;
  const real FR1 = qsR, FR2 = qsR * unR + pR;
  real F1, F2;
  if (SL >= RL(0.0)) {
    F1 = FL1; F2 = FL2;
  } else if (SR <= RL(0.0)) {
    F1 = FR1; F2 = FR2;
  } else {                                       // HLL written as F_L + increment
    const real inv = RL(1.0) / (SR - SL);
    F1 = FL1 + (SL * (SR * (hsR - hsL) - (FR1 - FL1))) * inv;
    F2 = FL2 + (SL * (SR * (qsR - qsL) - (FR2 - FL2))) * inv;
  }
  const real F3 = F1 * (F1 >= RL(0.0) ? utL : utR);  // contact wave: upwind tangential velocity
  *F1o = F1;
  *F3o = F3;
  *GLo = F2 - pL;                                  // per-side hydrostatic (bed-slope) correction
  *GRo = F2 - pR;
}

// one interior edge from the cell states: rotation into the (normal, tangential) frame of the edge, then riemann_nt
static void edge_flux(real g, real heL, real uL, real vL, real zL, real heR, real uR, real vR, real zR, real nx, real ny,
                      real *F1o, real *F3o, real *GLo, real *GRo) {
  const real unL = uL * nx + vL * ny, utL = vL * nx - uL * ny;
  const real unR = uR * nx + vR * ny, utR = vR * nx - uR * ny;
  riemann_nt(g, heL, unL, utL, zL, heR, unR, utR, zR, F1o, F3o, GLo, GRo);
}

extern "C" void swe_ref_edge_flux(double g, double heL, double uL, double vL, double zL,
                                  double heR, double uR, double vR, double zR, double nx, double ny,
                                  double *F1o, double *F3o, double *GLo, double *GRo) {
  real F1, F3, GL, GR;
  edge_flux(RL(g), RL(heL), RL(uL), RL(vL), RL(zL), RL(heR), RL(uR), RL(vR), RL(zR), RL(nx), RL(ny), &F1, &F3, &GL, &GR);
  *F1o = F1; *F3o = F3; *GLo = GL; *GRo = GR;
}

// wall evaluated through the solver with a mirror ghost (u_n -> -u_n): used only by the pin that
// checks the closed form in boundary_flux() against it.
extern "C" void swe_ref_wall_flux_via_ghost(double g, double he, double un, double ut,
                                            double *F1o, double *F3o, double *Go) {
  real F1, F3, G, GR;
  riemann_nt(RL(g), RL(he), RL(un), RL(ut), RL(0.0), RL(he), -RL(un), RL(ut), RL(0.0), &F1, &F3, &G, &GR);
  *F1o = F1; *F3o = F3; *Go = G;
}

// ------------------------------------------------------------------------------------------------
// Cube root, CORRECTLY ROUNDED (round to nearest) -- DESIGN.md R-14.  The friction term needs
// h^(7/3) (Eq. 2 with the Strickler row of Table 1) and the conveyance weights
// h^(5/3); a library cbrt is only good to 1 ulp and differs between libraries, which a 100-step
// run amplifies.  "The nearest double to the real cube root" is a definition, not an algorithm,
// so both sides can meet it independently.  Here it is found the slow, checkable way:
//   x = M * 2^E (M a 53-bit integer).  Pick s in {107,108,109} with (E - s) divisible by 3 and let
//   X = M * 2^s, an integer in [2^159, 2^162).  T = floor(X^(1/3)) is a 54-bit integer in
//   [2^53, 2^54): one bit more than a double holds.  T is found from a library estimate and then
//   corrected with exact 192-bit integer cubes until T^3 <= X < (T+1)^3.  X^(1/3) is never a
//   half-way point (an odd T has an odd cube, X is even), so rounding T's last bit is exact:
//   mantissa K = (T + 1) >> 1, result K * 2^((E - s)/3 + 1).
// ------------------------------------------------------------------------------------------------
struct U192 { uint64_t w[3]; };   // little-endian limbs

static U192 cube_u64(uint64_t t) {   // t < 2^55: t^3 < 2^165
  typedef unsigned __int128 u128;
  const u128 sq = (u128)t * t;                         // < 2^110
  const uint64_t sq_lo = (uint64_t)sq, sq_hi = (uint64_t)(sq >> 64);
  const u128 a = (u128)sq_lo * t;                      // contributes at limb 0
  const u128 b = (u128)sq_hi * t;                      // contributes at limb 1
  U192 r;
  r.w[0] = (uint64_t)a;
  const u128 mid = (a >> 64) + (u128)(uint64_t)b;
  r.w[1] = (uint64_t)mid;
  r.w[2] = (uint64_t)(b >> 64) + (uint64_t)(mid >> 64);
  return r;
}

static bool less_equal(const U192 &a, const U192 &b) {  // a <= b
  for (int k = 2; k >= 0; --k) {
    if (a.w[k] < b.w[k]) return true;
    if (a.w[k] > b.w[k]) return false;
  }
  return true;
}

extern "C" double swe_ref_cbrt(double x) {
  if (x == 0.0 || !std::isfinite(x)) return x;
  if (x < 0.0) return -swe_ref_cbrt(-x);
  int ex;
  const double fr = std::frexp(x, &ex);                  // x = fr * 2^ex, fr in [0.5, 1); exact, also for subnormals
  const uint64_t M = (uint64_t)std::ldexp(fr, 53);       // 53-bit integer, x = M * 2^E
  const int E = ex - 53;
  int s = 107;
  while (((E - s) % 3) != 0) ++s;                        // s in {107, 108, 109}
  const int q = (E - s) / 3;                             // x^(1/3) = X^(1/3) * 2^q
  U192 X;                                                // X = M << s
  X.w[0] = 0;
  X.w[1] = M << (s - 64);
  X.w[2] = M >> (128 - s);
  // estimate of T from the library cube root of X / 2^159 in [1, 8)
  uint64_t T = (uint64_t)std::ldexp(std::cbrt(std::ldexp((double)M, s - 159)), 53);
  while (!less_equal(cube_u64(T), X)) --T;               // now T^3 <= X
  while (less_equal(cube_u64(T + 1), X)) ++T;            // now X < (T+1)^3
  const uint64_t K = (T + 1) >> 1;                       // round to 53 bits; never a tie
  return std::ldexp((double)K, q + 1);
}

namespace {

// fixed-shape pairwise tree in string order (R-11): pad to a power of two with zeros,
// then add neighbours at stride 1, 2, 4, ...
real tree_sum(std::vector<real> v) {
  if (v.empty()) return RL(0.0);
  size_t P = 1;
  while (P < v.size()) P <<= 1;
  v.resize(P, RL(0.0));
  for (size_t s = 1; s < P; s <<= 1)
    for (size_t i = 0; i + s < P; i += 2 * s) v[i] = v[i] + v[i + s];
  return v[0];
}

inline real cbrt_real(real x) { return RL(swe_ref_cbrt((double)x)); }   // fp64: swe_ref_cbrt itself

inline real pow53(real he) {           // he^(5/3)
  const real c3 = cbrt_real(he);
  return (he * c3) * c3;
}

inline real kweight(real k) { return std::isfinite(k) ? k : RL(1.0); }

double hydrograph(const std::vector<double> &p, double t) {  // piecewise linear, clamped
  const size_t m = p.size() / 2;
  if (m == 0) return 0.0;
  if (t <= p[0]) return p[1];
  if (t >= p[2 * (m - 1)]) return p[2 * (m - 1) + 1];
  size_t k = 0;
  while (!(p[2 * k] <= t && t < p[2 * (k + 1)])) ++k;
  const double tk = p[2 * k], Qk = p[2 * k + 1], tk1 = p[2 * k + 2], Qk1 = p[2 * k + 3];
  return Qk + (Qk1 - Qk) * ((t - tk) / (tk1 - tk));
}

// R-8: a cell with h <= h_dry (a thin film) keeps its water and still takes part in the hydrostatic
// reconstruction with its depth, but carries no momentum: its velocity is 0 and it is left out of Eq. 21.
inline bool is_wet(const swe_ref_ctx *c, int64_t i) { return c->h[i] > c->h_dry; }

// S0 -- Eq. 21: rho_ij = 2 * dist(centroid, edge j) = 4|Omega_i| / (3 l_ij)
real max_rate(const swe_ref_ctx *c) {
  real r = RL(0.0);
  SWE_REF_PARALLEL_MAX(r)
  for (int64_t i = 0; i < c->nc; ++i) {
    if (!(c->h[i] > c->h_dry)) continue;
    const real u = c->qx[i] / c->h[i], v = c->qy[i] / c->h[i];
    const real cel = std::sqrt(c->g * c->h[i]);
    for (int k = 0; k < 3; ++k) {
      const int32_t e = c->ce[3 * i + k];
      const real lam = std::fabs(u * c->nx[e] + v * c->ny[e]) + cel;
      const real val = lam * ((RL(0.75) * c->len[e]) * c->invA[i]);
      if (val > r) r = val;
    }
  }
  return r;
}

struct DtChoice { double dt, t_new; bool unbounded; };

DtChoice choose_dt(const swe_ref_ctx *c, double cfl, double t_end) {
  const double r = (double)max_rate(c);
  double dt = (r > 0.0) ? cfl / r : c->dt_max;
  dt = std::fmin(dt, c->dt_max);
  const double rem = t_end - c->t;
  DtChoice o;
  if (dt >= rem) { o.dt = rem; o.t_new = t_end; }
  else           { o.dt = dt;  o.t_new = c->t + dt; }
  o.unbounded = !std::isfinite(o.dt);
  return o;
}

// boundary strings at t^n (R-11, R-12; types named at PAPER.md:342)
void eval_strings(swe_ref_ctx *c) {
  for (auto &kv : c->strings) {
    BString &s = kv.second;
    s.Q = s.sumK = s.sumL = RL(0.0);
    std::vector<real> a, b;
    if (s.type == SWE_REF_BC_INFLOW_Q) {
      s.Q = RL(hydrograph(s.params, c->t));
      for (int32_t e : s.edges) {
        const int64_t L = c->eL[e];
        a.push_back((c->len[e] * kweight(c->kst[L])) * pow53(c->h[L]));
        b.push_back(c->len[e]);
      }
      s.sumK = tree_sum(a);
      s.sumL = tree_sum(b);
    }
  }
}

void boundary_flux(swe_ref_ctx *c, int64_t e) {
  const int64_t L = c->eL[e];
  const int code = c->eR[e];
  const real nx = c->nx[e], ny = c->ny[e];
  const real he = c->h[L];
  real u = RL(0.0), v = RL(0.0);
  if (is_wet(c, L)) { u = c->qx[L] / c->h[L]; v = c->qy[L] / c->h[L]; }
  real F1 = RL(0.0), F3 = RL(0.0), GL = RL(0.0), GR = RL(0.0);
  const BString *s = nullptr;
  if (code <= -3) {
    auto it = c->strings.find(-3 - code);
    if (it != c->strings.end() && it->second.type != 0) s = &it->second;
  }
  if (code == -2) {
    // transmissive: ghost = copy of the interior state (R-10)
    edge_flux(c->g, he, u, v, c->zb[L], he, u, v, c->zb[L], nx, ny, &F1, &F3, &GL, &GR);
  } else if (s && s->type == SWE_REF_BC_INFLOW_Q) {
    real qe;
    if (s->sumK > RL(0.0)) {
      const real Ke = (c->len[e] * kweight(c->kst[L])) * pow53(he);
      qe = ((s->Q * Ke) / s->sumK) / c->len[e];
    } else {
      qe = s->Q / s->sumL;
    }
    F1 = -qe;
    GL = (he > RL(0.0)) ? (qe * qe) / he : RL(0.0);
    F3 = RL(0.0);
  } else if (s && s->type == SWE_REF_BC_OUTFLOW_UNIFORM) {
    if (he > RL(0.0)) {
      const real sqrtS0 = std::sqrt(s->params.empty() ? RL(0.0) : RL(s->params[0]));
      const real qn = (kweight(c->kst[L]) * pow53(he)) * sqrtS0;
      const real ut = v * nx - u * ny;
      F1 = qn;
      GL = (qn * qn) / he;
      F3 = qn * ut;
    }
  } else {
    // wall (default): reflective; closed form of the mirror-ghost Riemann problem (R-9):
    // F1 = 0, F3 = 0, G = h u_n (u_n + S), S = max(c - u_n, c + u_n/2)
    if (he > RL(0.0)) {
      const real un = u * nx + v * ny;
      const real cel = std::sqrt(c->g * he);
      const real S = std::fmax(cel - un, cel + RL(0.5) * un);
      GL = (he * un) * (un + S);
    }
  }
  c->F1[e] = F1; c->F3[e] = F3; c->GL[e] = GL; c->GR[e] = RL(0.0);
  (void)GR;
}

}  // namespace

// ---- section 3.2.1 Table 2 + Eq. 16, R-20 ------------------------
// One cell seen from one interface with unit normal (nx, ny): normal sediment flux q_B.n, the derivative
// psi = d(q_B,n)/d(q_n) (q_n = h u_n; h and the tangential velocity held fixed) and the two speeds of Eq. 16.
//   formula 1, Grass-like:  |q_B| = alpha |u|^3 (m = 3, u_cr = 0), along u
//   formula 2, MPM-like:    |q_B| = alpha (theta - theta_cr)^1.5 sqrt((s-1) g d_m^3) for theta > theta_cr, along u, with the
//                           Shields parameter theta = tau_B / (rho g (s-1) d_m) and the Strickler bed shear stress of
//                           Table 1, tau_B / rho = g |u|^2 / (k_st^2 h^(1/3))   (gn2 = g / k_st^2)
extern "C" void swe_ref_sediment_state(int formula, double alpha, double theta_cr, double sdens, double dm, double g,
                                       double h, double u, double v, double gn2, double nx, double ny,
                                       double *qBn, double *psi, double *lam1, double *lam2) {
  const double un = u * nx + v * ny, ut = v * nx - u * ny;
  const double sp2 = u * u + v * v;
  double q = 0.0, ps = 0.0;
  if (formula == 1) {
    q = alpha * (sp2 * un);
    ps = (alpha * (sp2 + 2.0 * (un * un))) / h;
  } else if (formula == 2) {
    const double th = (gn2 * sp2) / (swe_ref_cbrt(h) * (g * ((sdens - 1.0) * dm)));
    const double x = th - theta_cr;
    if (x > 0.0 && sp2 > 0.0) {
      const double Gm = alpha * std::sqrt(((sdens - 1.0) * g) * (dm * (dm * dm)));
      const double rx = std::sqrt(x), spd = std::sqrt(sp2);
      q = (Gm * (x * rx)) * (un / spd);
      ps = (Gm * (((3.0 * rx) * th) * (un * un) + (x * rx) * (ut * ut))) / ((sp2 * spd) * h);
    }
  }
  const double cel = std::sqrt(g * h);
  const double a = un - cel;
  const double disc = std::sqrt(a * a + 4.0 * (ps * (cel * cel)));
  *qBn = q; *psi = ps; *lam1 = 0.5 * (a - disc); *lam2 = 0.5 * (a + disc);
}

// Eq. 14-15: HLL-type sediment flux through the interface between cell i (left) and cell j (right)
extern "C" double swe_ref_sediment_flux(double qBi, double l1i, double l2i, double zi,
                                        double qBj, double l1j, double l2j, double zj) {
  const double sm = std::fmin(l1i, l1j), sp = std::fmax(l2i, l2j);
  if (!(sp - sm > 0.0)) return 0.0;
  return ((sp * qBi - sm * qBj) + (sp * sm) * (zj - zi)) / (sp - sm);
}

namespace {

// S1m: q_Bij of every edge from the state at t^n (synchronous-decoupled).  R-20: no transport where a
// cell is dry (h <= h_dry), so an interface with a dry side carries none; walls carry none; through every open
// boundary the interior cell's own flux leaves or enters (equilibrium boundary: q_Bij = q_Bi . n).
void sediment_fluxes(swe_ref_ctx *c) {
  SWE_REF_PARALLEL_FOR
  for (int64_t e = 0; e < c->ne; ++e) {
    const int64_t L = c->eL[e], R = c->eR[e];
    c->qB[e] = RL(0.0);
    if (!is_wet(c, L) || R == -1) continue;
    double qi, psi, l1i, l2i;
    swe_ref_sediment_state(c->morph_formula, c->morph_alpha, c->morph_theta_cr, c->morph_s, c->morph_dm, c->g, c->h[L],
                           c->qx[L] / c->h[L], c->qy[L] / c->h[L], c->gn2[L], c->nx[e], c->ny[e], &qi, &psi, &l1i, &l2i);
    if (R < 0) { c->qB[e] = RL(qi); continue; }
    if (!is_wet(c, R)) continue;
    double qj, l1j, l2j;
    swe_ref_sediment_state(c->morph_formula, c->morph_alpha, c->morph_theta_cr, c->morph_s, c->morph_dm, c->g, c->h[R],
                           c->qx[R] / c->h[R], c->qy[R] / c->h[R], c->gn2[R], c->nx[e], c->ny[e], &qj, &psi, &l1j, &l2j);
    c->qB[e] = RL(swe_ref_sediment_flux(qi, l1i, l2i, c->zb[L], qj, l1j, l2j, c->zb[R]));
  }
}

void one_step(swe_ref_ctx *c, const double dt_, const double t_new) {
  const real g = c->g;
  const real dt = RL(dt_);          // the step in the precision of the state (fp64: dt_ itself)
  eval_strings(c);
  // ---- S1 / S1b
  SWE_REF_PARALLEL_FOR
  for (int64_t e = 0; e < c->ne; ++e) {
    const int64_t L = c->eL[e], R = c->eR[e];
    if (R < 0) { boundary_flux(c, e); continue; }
    const real heL = c->h[L], heR = c->h[R];
    real uL = 0, vL = 0, uR = 0, vR = 0;
    if (is_wet(c, L)) { uL = c->qx[L] / c->h[L]; vL = c->qy[L] / c->h[L]; }
    if (is_wet(c, R)) { uR = c->qx[R] / c->h[R]; vR = c->qy[R] / c->h[R]; }
    edge_flux(g, heL, uL, vL, c->zb[L], heR, uR, vR, c->zb[R], c->nx[e], c->ny[e],
              &c->F1[e], &c->F3[e], &c->GL[e], &c->GR[e]);
  }
  if (c->morph_formula) sediment_fluxes(c);
  // ---- S1c draining-time limiter (R-8b): a cell may not lose more water than it holds.
  //      theta_i = min(1, h_i |Omega_i| / (dt * sum of its outgoing l F1)); every flux component of
  //      an edge is scaled by theta of the edge's donor cell (the cell the mass flux leaves).
  SWE_REF_PARALLEL_FOR
  for (int64_t i = 0; i < c->nc; ++i) {
    real o[3];
    for (int k = 0; k < 3; ++k) {
      const int32_t e = c->ce[3 * i + k];
      const real sM = (c->eL[e] == i ? RL(1.0) : -RL(1.0)) * (c->len[e] * c->F1[e]);
      o[k] = std::fmax(RL(0.0), sM);
    }
    const real out = ((o[0] + o[1]) + o[2]);
    const real avail = c->h[i] * c->area[i];
    c->theta[i] = (dt * out > avail) ? avail / (dt * out) : RL(1.0);
  }
  SWE_REF_PARALLEL_FOR
  for (int64_t e = 0; e < c->ne; ++e) {
    const int64_t L = c->eL[e], R = c->eR[e];
    real th = RL(1.0);
    if (c->F1[e] > RL(0.0)) th = c->theta[L];
    else if (c->F1[e] < RL(0.0) && R >= 0) th = c->theta[R];
    if (th < RL(1.0)) { c->F1[e] = th * c->F1[e]; c->F3[e] = th * c->F3[e]; c->GL[e] = th * c->GL[e]; c->GR[e] = th * c->GR[e]; }
  }
  // ---- scalar advection, PAPER.md:204-208 (Eq. 8), PAPER.md:298-304 (Eq. 20, advective part A_ij): "the HLLC solver
  //      ... provides the advective component of the scalar fluxes" = the mass flux times the concentration on the
  //      upwind side of the contact wave, sign(S*) = sign(F1) (R-19, same upwinding as F3 in R-2).
  //      phi_i = q_c,i / h_i where h_i > 0, else 0; F1 is the limited mass flux, so a cell never loses more scalar
  //      mass than it holds.  Ghost concentrations: transmissive, wall, outflow = phi of the interior cell; an
  //      INFLOW_Q string carries the concentrations set with swe_ref_set_boundary_scalar.
  for (int sp = 0; sp < c->n_species; ++sp) {
    const std::vector<real> &q = c->qc[sp];
    for (int64_t e = 0; e < c->ne; ++e) {
      const int64_t L = c->eL[e], R = c->eR[e];
      const real phiL = c->h[L] > RL(0.0) ? q[L] / c->h[L] : RL(0.0);
      real phiR = phiL;
      if (R >= 0) phiR = c->h[R] > RL(0.0) ? q[R] / c->h[R] : RL(0.0);
      else if (R <= -3) {
        auto it = c->strings.find(-3 - (int)R);
        if (it != c->strings.end() && it->second.type == SWE_REF_BC_INFLOW_Q)
          phiR = sp < (int)it->second.phi_in.size() ? RL(it->second.phi_in[sp]) : RL(0.0);
      }
      c->Ac[sp][e] = c->F1[e] * (c->F1[e] >= RL(0.0) ? phiL : phiR);
    }
  }
  // ---- S2 + S3 (in place: the fluxes of step n are already stored per edge)
  SWE_REF_PARALLEL_FOR
  for (int64_t i = 0; i < c->nc; ++i) {
    real M[3], X[3], Y[3], s[3];
    for (int k = 0; k < 3; ++k) {
      const int32_t e = c->ce[3 * i + k];
      const bool isL = (c->eL[e] == i);
      const real G = isL ? c->GL[e] : c->GR[e];
      const real l = c->len[e], nx = c->nx[e], ny = c->ny[e];
      s[k] = isL ? RL(1.0) : -RL(1.0);
      M[k] = l * c->F1[e];
      X[k] = l * (G * nx - c->F3[e] * ny);
      Y[k] = l * (G * ny + c->F3[e] * nx);
    }
    const real dH = ((s[0] * M[0] + s[1] * M[1]) + s[2] * M[2]);
    const real dX = ((s[0] * X[0] + s[1] * X[1]) + s[2] * X[2]);
    const real dY = ((s[0] * Y[0] + s[1] * Y[1]) + s[2] * Y[2]);
    const real a = dt * c->invA[i];
    real hn = c->h[i] - a * dH;
    if (hn < RL(0.0)) {
      SWE_REF_ATOMIC
      c->vol_clipped += (double)(-hn * c->area[i]);
      hn = RL(0.0);
    }
    real qxn = RL(0.0), qyn = RL(0.0);
    if (hn > c->h_dry) {
      qxn = c->qx[i] - a * dX;
      qyn = c->qy[i] - a * dY;
      if (c->gn2[i] > RL(0.0)) {   // split friction, exact integral of dq/dt = -gamma |q| q (R-5, R-6)
        const real D = RL(1.0) + ((dt * c->gn2[i]) * std::sqrt(qxn * qxn + qyn * qyn)) / ((hn * hn) * cbrt_real(hn));
        qxn = qxn / D;
        qyn = qyn / D;
      }
    }
    c->h[i] = hn; c->qx[i] = qxn; c->qy[i] = qyn;
    for (int sp = 0; sp < c->n_species; ++sp) {     // Eq. 20, advective part: same gather, same slot order
      real C[3];
      for (int k = 0; k < 3; ++k) { const int32_t e = c->ce[3 * i + k]; C[k] = c->len[e] * c->Ac[sp][e]; }
      const real dC = ((s[0] * C[0] + s[1] * C[1]) + s[2] * C[2]);
      c->qc[sp][i] = c->qc[sp][i] - a * dC;
    }
  }
  // ---- Eq. 13, S_b = 0: z_B <- z_B - 1/(1-p) * dt/|Omega| * sum_j l_ij q_Bij, slots in order
  if (c->morph_formula) {
    const real inv1mp = RL(1.0 / (1.0 - c->morph_p));
    SWE_REF_PARALLEL_FOR
    for (int64_t i = 0; i < c->nc; ++i) {
      real B[3], s[3];
      for (int k = 0; k < 3; ++k) {
        const int32_t e = c->ce[3 * i + k];
        s[k] = (c->eL[e] == i) ? RL(1.0) : -RL(1.0);
        B[k] = c->len[e] * c->qB[e];
      }
      const real dB = ((s[0] * B[0] + s[1] * B[1]) + s[2] * B[2]);
      c->zb[i] = c->zb[i] - inv1mp * ((dt * c->invA[i]) * dB);
    }
  }
  for (auto &kv : c->strings) {      // bookkeeping from the (limited) fluxes actually applied
    BString &s = kv.second;
    if (s.type == SWE_REF_BC_INFLOW_Q) c->vol_in += dt_ * (double)s.Q;
    if (s.type == SWE_REF_BC_OUTFLOW_UNIFORM) {
      std::vector<real> a;
      for (int32_t e : s.edges) a.push_back(c->len[e] * c->F1[e]);
      c->vol_out += dt_ * (double)tree_sum(a);
    }
  }
  // ---- S4
  c->t = t_new;
  c->dt_last = dt_;
  c->steps_done += 1;
}

void fill_info(swe_ref_ctx *c, swe_ref_info *info) {
  if (!info) return;
  double vol = 0.0;
  int64_t nwet = 0;
  bool bad = false;
  for (int64_t i = 0; i < c->nc; ++i) {
    vol += (double)c->h[i] * (double)c->area[i];
    if (c->h[i] > c->h_dry) ++nwet;
    if (!std::isfinite(c->h[i]) || !std::isfinite(c->qx[i]) || !std::isfinite(c->qy[i])) bad = true;
  }
  if (bad) c->flags |= 1;
  info->t = c->t; info->dt_last = c->dt_last; info->steps_done = c->steps_done; info->n_wet = nwet;
  info->vol = vol; info->vol_clipped = c->vol_clipped; info->vol_in = c->vol_in; info->vol_out = c->vol_out;
  info->flags = c->flags;
}

}  // namespace

extern "C" int swe_ref_create(const swe_ref_mesh *m, const swe_ref_params *p, swe_ref_ctx **out) {
  if (!m || !out || !m->node_xy || !m->tri || !m->edge_cell || !m->cell_edge || !m->zb || !m->kst) {
    g_create_error = "null argument";
    return -1;
  }
  swe_ref_ctx *c = new swe_ref_ctx;
  c->nc = m->n_cells; c->ne = m->n_edges;
  const double g64 = p ? p->g : 9.81;
  if (p) { c->g = RL(p->g); c->h_dry = RL(p->h_dry); c->dt_max = p->dt_max; }
  const int64_t nc = c->nc, ne = c->ne;
  c->area.resize(nc); c->invA.resize(nc); c->gn2.resize(nc);
  c->zb.resize(nc); c->kst.resize(nc);
  for (int64_t i = 0; i < nc; ++i) { c->zb[i] = RL(m->zb[i]); c->kst[i] = RL(m->kst[i]); }
  c->ce.assign(m->cell_edge, m->cell_edge + 3 * nc);
  c->eL.resize(ne); c->eR.resize(ne); c->nx.resize(ne); c->ny.resize(ne); c->len.resize(ne);
  c->h.assign(nc, RL(0.0)); c->qx.assign(nc, RL(0.0)); c->qy.assign(nc, RL(0.0));
  c->theta.assign(nc, RL(1.0));
  c->F1.assign(ne, RL(0.0)); c->F3.assign(ne, RL(0.0)); c->GL.assign(ne, RL(0.0)); c->GR.assign(ne, RL(0.0));
  for (int64_t e = 0; e < ne; ++e) { c->eL[e] = m->edge_cell[2 * e]; c->eR[e] = m->edge_cell[2 * e + 1]; }
  // geometry, PAPER.md:226-228 (section 4.1, Fig. 2)
  for (int64_t i = 0; i < nc; ++i) {
    const int32_t *t = m->tri + 3 * i;
    const double x0 = m->node_xy[2 * t[0]], y0 = m->node_xy[2 * t[0] + 1];
    const double x1 = m->node_xy[2 * t[1]], y1 = m->node_xy[2 * t[1] + 1];
    const double x2 = m->node_xy[2 * t[2]], y2 = m->node_xy[2 * t[2] + 1];
    const double A = 0.5 * ((x1 - x0) * (y2 - y0) - (x2 - x0) * (y1 - y0));
    if (!(A > 0.0)) { g_create_error = "cell " + std::to_string(i) + " is not counter-clockwise / has no area"; delete c; return -2; }
    c->area[i] = RL(A);                  // geometry and constants: computed in fp64, rounded once to `real`
    c->invA[i] = RL(1.0 / A);
    const double k = m->kst[i];
    c->gn2[i] = std::isfinite(k) ? RL(g64 / (k * k)) : RL(0.0);
    for (int s = 0; s < 3; ++s) {
      const int32_t e = c->ce[3 * i + s];
      if (e < 0 || e >= ne) { g_create_error = "cell_edge out of range"; delete c; return -2; }
      if (c->eL[e] == i) {               // the edge's stored normal and length come from its L cell's slot
        const int32_t a = t[s], b = t[(s + 1) % 3];
        const double dx = m->node_xy[2 * b] - m->node_xy[2 * a], dy = m->node_xy[2 * b + 1] - m->node_xy[2 * a + 1];
        const double l = std::sqrt(dx * dx + dy * dy);
        c->len[e] = RL(l); c->nx[e] = RL(dy / l); c->ny[e] = RL(-dx / l);
      } else if (c->eR[e] != i) {
        g_create_error = "edge_cell / cell_edge tables are inconsistent at cell " + std::to_string(i);
        delete c; return -2;
      }
    }
  }
  for (int64_t e = 0; e < ne; ++e)
    if (c->eR[e] <= -3) c->strings[-3 - c->eR[e]].edges.push_back((int32_t)e);
  *out = c;
  return 0;
}

extern "C" int swe_ref_set_boundary(swe_ref_ctx *c, int string_id, int type, const double *params, int n_params) {
  if (!c || string_id < 0) return -1;
  BString &s = c->strings[string_id];
  s.type = type;
  s.params.assign(params, params + n_params);
  return 0;
}

extern "C" int swe_ref_set_state(swe_ref_ctx *c, const double *h, const double *hu, const double *hv, double t0) {
  if (!c || !h || !hu || !hv) return -1;
  for (int64_t i = 0; i < c->nc; ++i) { c->h[i] = RL(h[i]); c->qx[i] = RL(hu[i]); c->qy[i] = RL(hv[i]); }
  c->t = t0; c->dt_last = 0.0; c->steps_done = 0; c->vol_clipped = c->vol_in = c->vol_out = 0.0; c->flags = 0;
  return 0;
}

extern "C" int swe_ref_set_scalars(swe_ref_ctx *c, int n_species, const double *qc) {
  if (!c || n_species < 0 || n_species > 5 || (n_species > 0 && !qc)) return -1;   // "up to a maximum of 5"
  c->n_species = n_species;
  c->qc.assign(n_species, std::vector<real>(c->nc, RL(0.0)));
  c->Ac.assign(n_species, std::vector<real>(c->ne, RL(0.0)));
  for (int sp = 0; sp < n_species; ++sp)
    for (int64_t i = 0; i < c->nc; ++i) c->qc[sp][i] = RL(qc[(size_t)sp * c->nc + i]);
  return 0;
}

extern "C" int swe_ref_get_scalars(swe_ref_ctx *c, double *qc) {
  if (!c || !qc) return -1;
  for (int sp = 0; sp < c->n_species; ++sp)
    for (int64_t i = 0; i < c->nc; ++i) qc[(size_t)sp * c->nc + i] = c->qc[sp][i];
  return 0;
}

extern "C" int swe_ref_set_boundary_scalar(swe_ref_ctx *c, int string_id, const double *phi, int n) {
  if (!c || string_id < 0 || n < 0 || (n > 0 && !phi)) return -1;
  c->strings[string_id].phi_in.assign(phi, phi + n);
  return 0;
}

extern "C" int swe_ref_set_morphology(swe_ref_ctx *c, int formula, double alpha, double theta_cr, double sdens,
                                      double dm, double porosity) {
  if (formula < 0 || formula > 2) { c->err = "formula must be 0 (fixed bed), 1 (Grass-like) or 2 (MPM-like)"; return 1; }
  if (!(porosity >= 0.0 && porosity < 1.0)) { c->err = "porosity must be in [0, 1)"; return 1; }
  if (formula == 2 && !(sdens > 1.0 && dm > 0.0)) { c->err = "MPM-like formula needs s > 1 and d_m > 0"; return 1; }
  c->morph_formula = formula; c->morph_alpha = alpha; c->morph_theta_cr = theta_cr; c->morph_s = sdens; c->morph_dm = dm;
  c->morph_p = porosity;
  c->qB.assign(c->ne, RL(0.0));
  return 0;
}

extern "C" int swe_ref_get_bed(swe_ref_ctx *c, double *zb) {
  for (int64_t i = 0; i < c->nc; ++i) zb[i] = c->zb[i];
  return 0;
}

extern "C" int swe_ref_get_sediment_flux(swe_ref_ctx *c, double *qB) {
  if (c->qB.empty()) { c->err = "morphodynamics is off"; return 1; }
  for (int64_t e = 0; e < c->ne; ++e) qB[e] = c->qB[e];
  return 0;
}

extern "C" int swe_ref_step(swe_ref_ctx *c, int64_t n_steps, double t_end, double cfl, swe_ref_info *info) {
  if (!c || !(cfl > 0.0)) return -1;
  int64_t done = 0;
  while ((n_steps < 0 || done < n_steps) && c->t < t_end) {
    const DtChoice d = choose_dt(c, cfl, t_end);
    if (d.unbounded) { c->flags |= 2; break; }
    one_step(c, d.dt, d.t_new);
    ++done;
  }
  fill_info(c, info);
  return 0;
}

extern "C" int swe_ref_get_state(swe_ref_ctx *c, double *h, double *hu, double *hv) {
  if (!c) return -1;
  for (int64_t i = 0; i < c->nc; ++i) { h[i] = c->h[i]; hu[i] = c->qx[i]; hv[i] = c->qy[i]; }
  return 0;
}

extern "C" void swe_ref_destroy(swe_ref_ctx *c) { delete c; }

extern "C" const char *swe_ref_last_error(const swe_ref_ctx *c) { return c ? c->err.c_str() : g_create_error.c_str(); }

extern "C" int swe_ref_get_geometry(swe_ref_ctx *c, double *area, double *nx, double *ny, double *len) {
  if (!c) return -1;
  for (int64_t i = 0; i < c->nc; ++i) area[i] = c->area[i];
  for (int64_t e = 0; e < c->ne; ++e) { nx[e] = c->nx[e]; ny[e] = c->ny[e]; len[e] = c->len[e]; }
  return 0;
}

extern "C" int swe_ref_get_edge_flux(swe_ref_ctx *c, double *F1, double *F3, double *GL, double *GR) {
  if (!c) return -1;
  for (int64_t e = 0; e < c->ne; ++e) { F1[e] = c->F1[e]; F3[e] = c->F3[e]; GL[e] = c->GL[e]; GR[e] = c->GR[e]; }
  return 0;
}

extern "C" double swe_ref_peek_dt(swe_ref_ctx *c, double cfl, double t_end) { return choose_dt(c, cfl, t_end).dt; }
