// CUDA kernels (sm_100a) of the explicit finite-volume shallow-water step.  fp64 throughout; compiled with
// -fmad=false so that the parenthesisation written here IS the arithmetic (R-14).
//
//   k_step_control  S0/S4: dt from the max rate of U^n, t += dt, boundary-string values at t^n, volume bookkeeping
//   k_edge_flux     S1/S1b: hydrostatic reconstruction + HLLC per edge; boundary edges
//   k_theta         S1c: draining-time factor per cell
//   k_cell_update   S2+S3 (+S0 of the next step): gather in slot order, Euler update, friction, wet/dry,
//                   local wave speed -> warp-shuffle + block max -> one atomicMax per block
//
// "P:n" = PAPER.md line n; R-k = DESIGN.md section 2.
#pragma once
#include <cuda_runtime.h>

#include "swe_cbrt.cuh"
#include "swe_types.h"

namespace swe {

constexpr int kBlock = 256;           // threads per block of the mesh kernels
constexpr int kCtlThreads = 1024;     // the single block of k_step_control
constexpr int kTreeCap = 4096;        // boundary-string members whose pairwise tree fits the block's shared memory

// boundary codes / string types (values of include/swe.h, restated so that device code needs no host header)
constexpr int kEdgeTransmissive = -2;
constexpr int kBcInflowQ = 1, kBcOutflowUniform = 2;
constexpr int kFlagUnbounded = 2, kFlagStalled = 4;

// ---------------------------------------------------------------------------------------------------------
// S1, one edge in the (normal, tangential) frame.  P:252 HLLC ("Chapter 10 of [18]"): HLL for mass and normal
// momentum with two-rarefaction wave speeds and dry-bed limits (R-2, R-3), contact wave = upwinded tangential
// momentum; P:254 bed slope by the modified-state approach of ref [69] (R-1): face bed z* = max(zL, zR), face
// depths hs_K = max(0, h_K + z_K - z*), per-side pressure correction G_K = F2 - 1/2 g hs_K^2.
// ---------------------------------------------------------------------------------------------------------
// min / max of finite doubles as one compare + select (fmin / fmax also order NaNs and signed zeros, which costs
// several more instructions; here a zero of either sign leads to the same branch and the same values)
template <typename T> __device__ __forceinline__ T dmax0(T x) { return x > T(0.0) ? x : T(0.0); }
// fp64: the compiler turns the line above into its fmax sequence (DSETP.MAX + NaN quieting, ~7 instructions); a test of
// the sign bit gives the same value for every x that is not a NaN (-0 and negatives -> +0) in 3
template <> __device__ __forceinline__ double dmax0<double>(double x) { return __double2hiint(x) < 0 ? 0.0 : x; }
template <typename T> __device__ __forceinline__ T dmin2(T a, T b) { return a < b ? a : b; }
template <typename T> __device__ __forceinline__ T dmax2(T a, T b) { return a > b ? a : b; }

template <typename T>
__device__ __forceinline__ EdgeFluxT<T> riemann_nt(T g, T hL, T unL, T utL, T zL,
                                               T hR, T unR, T utR, T zR) {
  EdgeFluxT<T> o;
  const T dz = zR - zL;
  const T hsL = dmax0(hL - dmax0(dz));
  const T hsR = dmax0(hR - dmax0(-dz));
  if (hsL == T(0.0) && hsR == T(0.0)) {
    o.F1 = T(0.0); o.F3 = T(0.0); o.GL = T(0.0); o.GR = T(0.0);
    return o;
  }
  const T cL = sqrt(g * hsL), cR = sqrt(g * hsR);
  T SL, SR;
  if (hsL > T(0.0) && hsR > T(0.0)) {
    const T us = T(0.5) * (unL + unR) + (cL - cR);
    const T cs = T(0.5) * (cL + cR) + T(0.25) * (unL - unR);
    SL = dmin2(unL - cL, us - cs);
    SR = dmax2(unR + cR, us + cs);
  } else if (hsR == T(0.0)) {
    SL = unL - cL;
    SR = unL + T(2.0) * cL;
  } else {
    SL = unR - T(2.0) * cR;
    SR = unR + cR;
  }
  const T qsL = hsL * unL, qsR = hsR * unR;
  const T pL = (T(0.5) * g) * (hsL * hsL), pR = (T(0.5) * g) * (hsR * hsR);
  const T FL2 = qsL * unL + pL, FR2 = qsR * unR + pR;
  T F1, F2;
  if (SL >= T(0.0)) {
    F1 = qsL; F2 = FL2;
  } else if (SR <= T(0.0)) {
    F1 = qsR; F2 = FR2;
  } else {
    const T inv = T(1.0) / (SR - SL);
    F1 = qsL + (SL * (SR * (hsR - hsL) - (qsR - qsL))) * inv;
    F2 = FL2 + (SL * (SR * (qsR - qsL) - (FR2 - FL2))) * inv;
  }
  o.F1 = F1;
  o.F3 = F1 * (F1 >= T(0.0) ? utL : utR);
  o.GL = F2 - pL;
  o.GR = F2 - pR;
  return o;
}

template <typename T>
__device__ __forceinline__ T pow53(T h) {  // h^(5/3), Strickler conveyance (Table 1)
  const T c3 = cbrt_rn(h);
  return (h * c3) * c3;
}

template <typename T> __device__ __forceinline__ T k_weight(T k) { return isfinite(k) ? k : T(1.0); }

// S1b, boundary edge (only the L side exists).  P:332 wall; P:342 zero-gradient, inflow hydrograph, uniform outflow.
// code: -1 wall, -2 transmissive; s: the boundary string the edge belongs to (nullptr if none); kL = k_str of cell L
// is read only for string edges.
template <typename T>
__device__ __forceinline__ EdgeFluxT<T> boundary_flux(T g, int code, const BoundaryString *__restrict__ s,
                                                  const T *__restrict__ kst, int L, T nx, T ny,
                                                  T len, T he, T z, T u, T v) {
  EdgeFluxT<T> o;
  o.F1 = T(0.0); o.F3 = T(0.0); o.GL = T(0.0); o.GR = T(0.0);
  const int type = s ? s->type : 0;
  if (code == kEdgeTransmissive) {            // R-10: ghost = copy of the interior state
    const T un = u * nx + v * ny, ut = v * nx - u * ny;
    o = riemann_nt(g, he, un, ut, z, he, un, ut, z);
    o.GR = T(0.0);
  } else if (type == kBcInflowQ) {            // R-11: Q(t) distributed by conveyance l k h^(5/3)
    T qe;
    if ((T)s->sumK > T(0.0)) {
      const T Ke = (len * k_weight(kst[L])) * pow53(he);
      qe = (((T)s->Q * Ke) / (T)s->sumK) / len;
    } else {
      qe = (T)s->Q / (T)s->sumL;
    }
    o.F1 = -qe;
    o.GL = (he > T(0.0)) ? (qe * qe) / he : T(0.0);
  } else if (type == kBcOutflowUniform) {     // R-12: normal depth, q_n = k h^(5/3) sqrt(S0)
    if (he > T(0.0)) {
      const T qn = (k_weight(kst[L]) * pow53(he)) * sqrt((T)s->S0);
      const T ut = v * nx - u * ny;
      o.F1 = qn;
      o.GL = (qn * qn) / he;
      o.F3 = qn * ut;
    }
  } else {                                    // R-9: reflective wall, closed form of the mirror-ghost problem
    if (he > T(0.0)) {
      const T un = u * nx + v * ny;
      const T cel = sqrt(g * he);
      const T S = dmax2(cel - un, cel + T(0.5) * un);
      o.GL = (he * un) * (un + S);
    }
  }
  return o;
}

// ---------------------------------------------------------------------------------------------------------
// S1: one thread per edge.  Reads one EdgeGeom record (coalesced 256-bit), gathers the two CellRec records
// (one sector each), writes one EdgeFlux record (coalesced 256-bit).
// ---------------------------------------------------------------------------------------------------------
// R of an edge: inside the fp64 geometry record; a separate array beside the 16-byte fp32 record
__device__ __forceinline__ int edge_R(const EdgeGeomT<double> &eg, const int32_t *, int) { return eg.R; }
__device__ __forceinline__ int edge_R(const EdgeGeomT<float> &, const int32_t *__restrict__ geomR, int e) { return geomR[e]; }

template <bool kScalars, typename T>
__device__ __forceinline__ void
edge_process(const Control *__restrict__ ctl, T g, T h_dry, int e, const EdgeGeomT<T> &eg, const int egR, const CellRecT<T> &a,
             const CellRecT<T> &b, const CellRecT<T> *__restrict__ rec, const T *__restrict__ kst,
             const BoundaryString *__restrict__ strings, EdgeFluxT<T> *__restrict__ flux, const Scalars &sc,
             const T *__restrict__ area, uint8_t *__restrict__ drain_flag, T (&vel)[4]) {
  T uL = T(0.0), vL = T(0.0);
  if (a.h > h_dry) { uL = a.qx / a.h; vL = a.qy / a.h; }   // R-8: thin films carry no momentum
  vel[0] = uL; vel[1] = vL; vel[2] = T(0.0); vel[3] = T(0.0);    // handed to the sediment flux of the <kMorph> instance
  EdgeFluxT<T> o;
  if (egR >= 0) {
    T uR = T(0.0), vR = T(0.0);
    if (b.h > h_dry) { uR = b.qx / b.h; vR = b.qy / b.h; }
    vel[2] = uR; vel[3] = vR;
    const T unL = uL * eg.nx + vL * eg.ny, utL = vL * eg.nx - uL * eg.ny;
    const T unR = uR * eg.nx + vR * eg.ny, utR = vR * eg.nx - uR * eg.ny;
    o = riemann_nt(g, a.h, unL, utL, a.z, b.h, unR, utR, b.z);
  } else {
    const BoundaryString *bs = (egR <= -3 && (-3 - egR) < ctl->n_strings) ? strings + (-3 - egR) : nullptr;
    o = boundary_flux(g, egR, bs, kst, eg.L, eg.nx, eg.ny, eg.len, a.h, a.z, uL, vL);
  }
  flux[e] = o;
  // S1c, lazily (R-8b): theta_i < 1 needs dt * (o_0 + o_1 + o_2) > h_i |Omega_i|, hence at least one outgoing edge with
  // dt * o_k > 0.3 h_i |Omega_i| (0.3 * 3 * (1 + rounding) < 1).  Only such donor cells are flagged; k_theta_lazy evaluates
  // theta exactly for them and every other cell keeps theta = 1 without being visited.
  if (drain_flag) {
    const int d = o.F1 > T(0.0) ? eg.L : ((o.F1 < T(0.0) && egR >= 0) ? egR : -1);
    if (d >= 0) {
      const T hd = (d == eg.L) ? a.h : b.h;
      if ((T)ctl->dt * (eg.len * fabs(o.F1)) > T(0.3) * (hd * area[d])) drain_flag[d] = 1;
    }
  }
  // passive scalars (Eq. 8 / Eq. 20 advective part, R-19): concentration on the upwind side of the contact wave
  if (kScalars)
  _Pragma("unroll") for (int sp = 0; sp < kMaxSpecies; ++sp) if (sp < sc.n) {
    const T phiL = a.h > T(0.0) ? sc.qa[sp][eg.L] / a.h : T(0.0);
    T phiR = phiL;
    if (egR >= 0) {
      phiR = b.h > T(0.0) ? sc.qa[sp][egR] / b.h : T(0.0);
    } else if (egR <= -3 && (-3 - egR) < ctl->n_strings && strings[-3 - egR].type == kBcInflowQ) {
      phiR = strings[-3 - egR].phi_in[sp];
    }
    sc.phi_up[sp][e] = o.F1 >= T(0.0) ? phiL : phiR;
  }
}

// ---------------------------------------------------------------------------------------------------------
// Morphodynamics, S1m (section 4.3; R-20): Table 2's transport law and the two speeds of Eq. 16 for one
// cell seen from one interface, then Eq. 14-15.
// ---------------------------------------------------------------------------------------------------------
struct SedState { double q, l1, l2; };

__device__ __forceinline__ SedState sed_state(const Morph &mp, double g, double h, double u, double v, double2 fc,
                                              double nx, double ny) {
  const double un = u * nx + v * ny, ut = v * nx - u * ny;
  const double sp2 = u * u + v * v;
  double q = 0.0, ps = 0.0;
  if (mp.formula == 1) {                       // Grass-like, m = 3, u_cr = 0 (Table 2)
    q = mp.alpha * (sp2 * un);
    ps = (mp.alpha * (sp2 + 2.0 * (un * un))) / h;
  } else {                                     // MPM-like, m = 1.5 (Table 2); Shields parameter from Table 1's
    // Strickler shear stress; fc = (g / k_st^2, cbrt_rn(h)) from Morph::cell; no friction law: theta = 0 / (..) = 0
    const double th = fc.x > 0.0 ? (fc.x * sp2) / (fc.y * mp.shields_den) : 0.0;
    const double x = th - mp.theta_cr;
    if (x > 0.0 && sp2 > 0.0) {
      const double rx = sqrt(x), spd = sqrt(sp2);
      q = (mp.Gm * (x * rx)) * (un / spd);
      ps = (mp.Gm * (((3.0 * rx) * th) * (un * un) + (x * rx) * (ut * ut))) / ((sp2 * spd) * h);
    }
  }
  const double cel = sqrt(g * h);
  const double a = un - cel;                   // Eq. 16 as printed: (u_n - c) in both roots
  const double disc = sqrt(a * a + 4.0 * (ps * (cel * cel)));
  SedState o;
  o.q = q; o.l1 = 0.5 * (a - disc); o.l2 = 0.5 * (a + disc);
  return o;
}

// q_Bij of edge e from the two cell records of t^n: nothing where a side is dry or at a wall; through open boundaries
// the interior cell's own flux (equilibrium boundary)
// vel = (u, v) of L and R as edge_process formed them (q / h where h > h_dry): the same quotients the oracle forms
// (R: >= 0 interior edge, < 0 boundary code; fcL / fcR: (g / k_st^2, cbrt(h)) of the two cells, MPM-like law only)
__device__ __forceinline__ double sediment_flux_core(const Morph &mp, double g, double h_dry, int R, double nx, double ny,
                                                     double hL, double uL, double vL, double zL, double2 fcL,
                                                     double hR, double uR, double vR, double zR, double2 fcR) {
  if (!(hL > h_dry) || R == -1) return 0.0;
  const SedState si = sed_state(mp, g, hL, uL, vL, fcL, nx, ny);
  if (R < 0) return si.q;
  if (!(hR > h_dry)) return 0.0;
  const SedState sj = sed_state(mp, g, hR, uR, vR, fcR, nx, ny);
  const double sm = dmin2(si.l1, sj.l1), sp = dmax2(si.l2, sj.l2);        // Eq. 15
  if (!(sp - sm > 0.0)) return 0.0;
  return ((sp * si.q - sm * sj.q) + (sp * sm) * (zR - zL)) / (sp - sm);    // Eq. 14
}

__device__ __forceinline__ double sediment_edge(const Morph &mp, double g, double h_dry, const EdgeGeom &eg,
                                                const CellRec &a, const CellRec &b, const double (&vel)[4]) {
  const double2 zero = make_double2(0.0, 0.0);
  const double2 fcL = (mp.formula == 2 && a.h > h_dry && eg.R != -1) ? mp.cell[eg.L] : zero;
  const double2 fcR = (mp.formula == 2 && a.h > h_dry && eg.R >= 0 && b.h > h_dry) ? mp.cell[eg.R] : zero;
  return sediment_flux_core(mp, g, h_dry, eg.R, eg.nx, eg.ny, a.h, vel[0], vel[1], a.z, fcL, b.h, vel[2], vel[3], b.z, fcR);
}

// kPersistent = false: one edge per thread.  kPersistent = true: a grid of resident blocks strides over the edges and
// the (streamed) geometry record of a thread's next edge is loaded while the current edge is worked on, so that the
// geom -> cell record gather chain of an edge pays one memory latency instead of two (profiles/r1f: the kernel's
// stalls are exactly these two loads).
template <bool kScalars, bool kPersistent, bool kMorph = false, typename T = double>
__global__ void __launch_bounds__(kBlock, kMorph ? 3 : 0)
k_edge_flux(const Control *__restrict__ ctl, const EdgeGeomT<T> *__restrict__ geom, const CellRecT<T> *__restrict__ rec,
            const T *__restrict__ kst, const BoundaryString *__restrict__ strings,
            EdgeFluxT<T> *__restrict__ flux, int n_edges, int force, const Scalars sc,
            const T *__restrict__ area, uint8_t *__restrict__ drain_flag, const Morph mp = Morph{},
            const int32_t *__restrict__ geomR = nullptr) {
  if (!ctl->active && !force) return;
  const T g = (T)ctl->g, h_dry = (T)ctl->h_dry;
  int e = blockIdx.x * kBlock + threadIdx.x;
  if (e >= n_edges) return;
  if (!kPersistent) {
    const EdgeGeomT<T> eg = geom[e];
    const int R = edge_R(eg, geomR, e);
    const CellRecT<T> a = rec[eg.L];
    CellRecT<T> b = a;
    if (R >= 0) b = rec[R];
    T vel[4];
    edge_process<kScalars>(ctl, g, h_dry, e, eg, R, a, b, rec, kst, strings, flux, sc, area, drain_flag, vel);
    if constexpr (kMorph) mp.qB[e] = sediment_edge(mp, g, h_dry, eg, a, b, vel);
    return;
  }
  const int stride = gridDim.x * kBlock;
  EdgeGeomT<T> eg_next = geom[e];
  int R_next = edge_R(eg_next, geomR, e);
  for (; e < n_edges; e += stride) {
    const EdgeGeomT<T> eg = eg_next;
    const int R = R_next;
    const CellRecT<T> a = rec[eg.L];
    CellRecT<T> b = a;
    if (R >= 0) b = rec[R];
    if (e + stride < n_edges) { eg_next = geom[e + stride]; R_next = edge_R(eg_next, geomR, e + stride); }
    T vel[4];
    edge_process<kScalars>(ctl, g, h_dry, e, eg, R, a, b, rec, kst, strings, flux, sc, area, drain_flag, vel);
    if constexpr (kMorph) mp.qB[e] = sediment_edge(mp, g, h_dry, eg, a, b, vel);
  }
}

// ---------------------------------------------------------------------------------------------------------
// S1c (R-8b): theta_i = min(1, h_i |Omega_i| / (dt * sum of the outgoing l F1 of cell i)), slots in order.
// ---------------------------------------------------------------------------------------------------------
static __global__ void __launch_bounds__(kBlock)
k_theta(const Control *__restrict__ ctl, const int4 *__restrict__ cell_edge, const EdgeGeom *__restrict__ geom,
        const EdgeFlux *__restrict__ flux, const CellRec *__restrict__ rec, const double *__restrict__ area,
        double *__restrict__ theta, int n_cells, int force) {
  if (!ctl->active && !force) return;
  const int i = blockIdx.x * kBlock + threadIdx.x;
  if (i >= n_cells) return;
  const double dt = ctl->dt;
  const int4 ce = cell_edge[i];
  const int es[3] = {ce.x, ce.y, ce.z};
  double o[3];
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    const EdgeGeom eg = geom[es[k]];
    const double F1 = flux[es[k]].F1;
    const double sM = (eg.L == i ? 1.0 : -1.0) * (eg.len * F1);
    o[k] = dmax0(sM);
  }
  const double out = ((o[0] + o[1]) + o[2]);
  const double avail = rec[i].h * area[i];
  theta[i] = (dt * out > avail) ? avail / (dt * out) : 1.0;
}

// S1c for the flagged cells only (see k_edge_flux): theta_i exactly as in k_theta; when theta_i < 1 the cell scales the
// records of its own outgoing edges in place -- every edge has exactly one donor, so no two cells touch one record,
// and a neighbour that reads the same record for its own theta sees it as an inflow (o_k = 0) before and after.
// flag bits: 1 = flagged by k_edge_flux in this step, 2 = theta[i] holds a value < 1 from an earlier step.
template <typename T = double>
__global__ void __launch_bounds__(kBlock)
k_theta_lazy(const Control *__restrict__ ctl, const int4 *__restrict__ cell_edge, const EdgeGeomT<T> *__restrict__ geom,
             EdgeFluxT<T> *__restrict__ flux, const CellRecT<T> *__restrict__ rec, const T *__restrict__ area,
             T *__restrict__ theta, uint8_t *__restrict__ drain_flag, int n_cells) {
  if (!ctl->active) return;
  // four flag bytes per thread: almost every word is 0 and the thread leaves after one 4-byte load
  const int i4 = (blockIdx.x * kBlock + threadIdx.x) * 4;
  if (i4 >= n_cells) return;
  const uint32_t f4 = *reinterpret_cast<const uint32_t *>(drain_flag + i4);     // the array is padded to 4 bytes
  if (f4 == 0u) return;
  for (int j = 0; j < 4; ++j) {
  const int i = i4 + j;
  const uint8_t fl = (uint8_t)(f4 >> (8 * j));
  if (fl == 0 || i >= n_cells) continue;
  T th = T(1.0);
  if (fl & 1) {
    const T dt = (T)ctl->dt;
    const int4 ce = cell_edge[i];
    const int es[3] = {ce.x, ce.y, ce.z};
    T o[3];
    bool isL[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      const EdgeGeomT<T> eg = geom[es[k]];
      isL[k] = (eg.L == i);
      const T sM = (isL[k] ? T(1.0) : -T(1.0)) * (eg.len * flux[es[k]].F1);
      o[k] = dmax0(sM);
    }
    const T out = ((o[0] + o[1]) + o[2]);
    const T avail = rec[i].h * area[i];
    if (dt * out > avail) th = avail / (dt * out);
    if (th < T(1.0)) {
#pragma unroll
      for (int k = 0; k < 3; ++k)
        if (o[k] > T(0.0)) {
          EdgeFluxT<T> f = flux[es[k]];
          f.F1 = th * f.F1; f.F3 = th * f.F3; f.GL = th * f.GL; f.GR = th * f.GR;
          flux[es[k]] = f;
        }
    }
  }
  theta[i] = th;
  drain_flag[i] = th < T(1.0) ? 2 : 0;
  }
}

// block-wide max of non-negative doubles -> one atomicMax on the bit pattern (order-preserving for x >= 0)
template <int kThreads = kBlock>
__device__ __forceinline__ void block_max_to_global(double r, unsigned long long *dst) {
  __shared__ double warp_max[kThreads / 32];
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) {
    const double other = __shfl_xor_sync(0xffffffffu, r, off);
    r = (other > r) ? other : r;
  }
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  if (lane == 0) warp_max[wid] = r;
  __syncthreads();
  if (wid == 0) {
    r = (lane < kThreads / 32) ? warp_max[lane] : 0.0;
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {          // all 32 lanes: the warp count need not be a power of two
      const double other = __shfl_xor_sync(0xffffffffu, r, off);
      r = (other > r) ? other : r;
    }
    if (lane == 0 && r > 0.0) atomicMax(dst, (unsigned long long)__double_as_longlong(r));
  }
}

// Eq. 21 (R-7) for one cell: max_j lambda_ij / rho_ij with rho_ij = 4|Omega_i| / (3 l_ij)
template <typename T>
__device__ __forceinline__ T cell_rate(T g, T h, T qx, T qy, T invA,
                                            const T nx[3], const T ny[3], const T len[3]) {
  const T u = qx / h, v = qy / h;
  const T cel = sqrt(g * h);
  T r = T(0.0);
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    const T lam = fabs(u * nx[k] + v * ny[k]) + cel;
    const T val = lam * ((T(0.75) * len[k]) * invA);
    if (val > r) r = val;
  }
  return r;
}

// ---------------------------------------------------------------------------------------------------------
// S2 + S3, and S0 of the NEXT step fused in: one thread per cell.
// ---------------------------------------------------------------------------------------------------------
template <bool kScalars, bool kMorph = false, typename T = double>
__global__ void __launch_bounds__(kBlock, (kScalars || kMorph) ? 3 : 4)      // 4 blocks/SM = 64 registers: measured faster than 3
k_cell_update(Control *__restrict__ ctl, const int4 *__restrict__ cell_edge, const EdgeGeomT<T> *__restrict__ geom,
              const EdgeFluxT<T> *__restrict__ flux, const T *__restrict__ theta,
              const T *__restrict__ area, const T *__restrict__ inv_area,
              const T *__restrict__ gn2, CellRecT<T> *__restrict__ rec, int n_cells, const Scalars sc,
              const Morph mp = Morph{}) {
  if (!ctl->active) return;
  // a grid of resident blocks strides over the cells; the (streamed) slot record of a thread's next cell is loaded
  // while the current cell is worked on: its cell_edge -> (geometry, flux) gather chain pays one latency, not two
  T rate = T(0.0);
  const int stride = gridDim.x * kBlock;
  int i = blockIdx.x * kBlock + threadIdx.x;
  int4 ce_next = make_int4(0, 0, 0, 0);
  if (i < n_cells) ce_next = cell_edge[i];
  const T dt = (T)ctl->dt, g = (T)ctl->g, h_dry = (T)ctl->h_dry;
  for (; i < n_cells; i += stride) {
    const int4 ce = ce_next;
    if (i + stride < n_cells) ce_next = cell_edge[i + stride];
    const int es[3] = {ce.x, ce.y, ce.z};
    T nx[3], ny[3], len[3];
    T dHk[3], dXk[3], dYk[3], sgn[3], F1lim[3], dBk[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      const EdgeGeomT<T> eg = geom[es[k]];
      EdgeFluxT<T> f = flux[es[k]];
      const bool isL = (eg.L == i);
      // limiter: every component of the edge is scaled by theta of the donor cell (the one F1 leaves)
      T G = isL ? f.GL : f.GR;
      if constexpr (sizeof(T) == 8) if (theta) {     // eager variant (fp64 inspection only); nullptr: k_theta_lazy has limited the records
        T th = T(1.0);
        if (f.F1 > T(0.0)) th = theta[eg.L];
        else if (f.F1 < T(0.0) && eg.R >= 0) th = theta[eg.R];
        if (th < T(1.0)) { f.F1 = th * f.F1; f.F3 = th * f.F3; G = th * G; }
      }
      const T s = isL ? T(1.0) : -T(1.0);
      nx[k] = eg.nx; ny[k] = eg.ny; len[k] = eg.len;
      if (kScalars) { sgn[k] = s; F1lim[k] = f.F1; }
      if constexpr (kMorph) dBk[k] = s * (eg.len * mp.qB[es[k]]);
      dHk[k] = s * (eg.len * f.F1);
      dXk[k] = s * (eg.len * (G * eg.nx - f.F3 * eg.ny));
      dYk[k] = s * (eg.len * (G * eg.ny + f.F3 * eg.nx));
    }
    const T dH = ((dHk[0] + dHk[1]) + dHk[2]);
    const T dX = ((dXk[0] + dXk[1]) + dXk[2]);
    const T dY = ((dYk[0] + dYk[1]) + dYk[2]);
    CellRecT<T> c = rec[i];
    const T invA = inv_area[i];
    const T a = dt * invA;
    T hn = c.h - a * dH;
    if (hn < T(0.0)) {                                  // residual negatives (R-8b): clip and count
      atomicAdd(&ctl->vol_clipped, (double)(-hn * area[i]));
      hn = T(0.0);
    }
    T qxn = T(0.0), qyn = T(0.0);
    double2 fc = make_double2(T(0.0), T(0.0));             // <kMorph>, MPM-like law: (g/k^2, cbrt(h^{n+1})) for the next step's edges
    if (hn > h_dry) {
      qxn = c.qx - a * dX;
      qyn = c.qy - a * dY;
      const T f2 = gn2[i];
      if (f2 > T(0.0)) {   // R-5/R-6: exact integral of dq/dt = -(g/(k^2 h^(7/3))) |q| q over dt, h frozen at h^{n+1}
        const T cb = cbrt_rn(hn);
        const T D = T(1.0) + ((dt * f2) * sqrt(qxn * qxn + qyn * qyn)) / ((hn * hn) * cb);
        qxn = qxn / D;
        qyn = qyn / D;
        fc = make_double2(f2, cb);
      }
      const T r = cell_rate(g, hn, qxn, qyn, invA, nx, ny, len);
      if (r > rate) rate = r;
    }
    c.h = hn; c.qx = qxn; c.qy = qyn;
    if constexpr (kMorph) {                          // Eq. 13, S_b = 0: the bed rides in the same record
      c.z = c.z - mp.inv1mp * (a * ((dBk[0] + dBk[1]) + dBk[2]));
      if (mp.formula == 2) mp.cell[i] = fc;
    }
    rec[i] = c;
    if (kScalars)                                    // Eq. 20, advective part: same gather, same slot order (R-19)
    _Pragma("unroll") for (int sp = 0; sp < kMaxSpecies; ++sp) if (sp < sc.n) {
      T Ck[3];
#pragma unroll
      for (int k = 0; k < 3; ++k) Ck[k] = sgn[k] * (len[k] * (F1lim[k] * sc.phi_up[sp][es[k]]));
      const T dC = ((Ck[0] + Ck[1]) + Ck[2]);
      sc.qa[sp][i] = sc.qa[sp][i] - a * dC;
    }
  }
  block_max_to_global((double)rate, &ctl->rate_bits);
}

// Eq. 21 on the current state (after swe_set_state): same arithmetic as the fused part of k_cell_update
template <typename T = double>
__global__ void __launch_bounds__(kBlock)
k_rate(Control *__restrict__ ctl, const int4 *__restrict__ cell_edge, const EdgeGeomT<T> *__restrict__ geom,
       const T *__restrict__ inv_area, const CellRecT<T> *rec_a, const CellRecT<T> *rec_b, int n_cells) {
  const CellRecT<T> *__restrict__ rec = ctl->cur ? rec_b : rec_a;
  const int i = blockIdx.x * kBlock + threadIdx.x;
  T rate = T(0.0);
  if (i < n_cells) {
    const CellRecT<T> c = rec[i];
    if (c.h > (T)ctl->h_dry) {
      const int4 ce = cell_edge[i];
      const int es[3] = {ce.x, ce.y, ce.z};
      T nx[3], ny[3], len[3];
#pragma unroll
      for (int k = 0; k < 3; ++k) {
        const EdgeGeomT<T> eg = geom[es[k]];
        nx[k] = eg.nx; ny[k] = eg.ny; len[k] = eg.len;
      }
      rate = cell_rate((T)ctl->g, c.h, c.qx, c.qy, inv_area[i], nx, ny, len);
    }
  }
  block_max_to_global((double)rate, &ctl->rate_bits);
}

// ---------------------------------------------------------------------------------------------------------
// Step control: one block.  Fixed-shape pairwise tree in string order (R-11): pad to a power of two with zeros,
// add neighbours at stride 1, 2, 4, ... -- the same pairs whatever the thread count, hence bit-reproducible.
// ---------------------------------------------------------------------------------------------------------
template <typename T>
__device__ __forceinline__ T block_tree_sum(T *v, int pow2) {
  for (int s = 1; s < pow2; s <<= 1) {
    __syncthreads();
    for (int j = threadIdx.x; 2 * s * j + s < pow2; j += blockDim.x) v[2 * s * j] = v[2 * s * j] + v[2 * s * j + s];
  }
  __syncthreads();
  const T sum = v[0];
  __syncthreads();                    // v may be refilled by the caller right away
  return sum;
}

__device__ __forceinline__ double hydrograph(const double *p, int n_params, double t) {  // piecewise linear, clamped
  const int m = n_params / 2;
  if (m == 0) return 0.0;
  if (t <= p[0]) return p[1];
  if (t >= p[2 * (m - 1)]) return p[2 * (m - 1) + 1];
  int k = 0;
  while (k < m - 2 && !(p[2 * k] <= t && t < p[2 * (k + 1)])) ++k;   // bounded: entries are finite and ascending (swe_set_boundary)
  const double tk = p[2 * k], Qk = p[2 * k + 1], tk1 = p[2 * k + 2], Qk1 = p[2 * k + 3];
  return Qk + (Qk1 - Qk) * ((t - tk) / (tk1 - tk));
}

// mode 0: start of a step.  mode 1: end of an swe_step call (bookkeeping of the last step only; zeroes the
// accumulators of k_info).
constexpr int kCtlPre = 4;            // boundary strings whose members k_step_control gathers up front (one per thread)

template <typename T = double>
__global__ void __launch_bounds__(kCtlThreads, 1)
k_step_control(Control *ctl, BoundaryString *strings, const int *__restrict__ string_edges, double *scratch_,
               const EdgeGeomT<T> *__restrict__ geom, const EdgeFluxT<T> *__restrict__ flux,
               const T *__restrict__ theta, const CellRecT<T> *rec_a, const CellRecT<T> *rec_b,
               const T *__restrict__ kst, const double *__restrict__ string_M, int mode) {
  // T: the precision of the state; the string sums run in T (fixed-shape trees, R-11), time / dt / volumes in fp64
  T *scratch = reinterpret_cast<T *>(scratch_);
  // the pairwise trees run in shared memory when the string fits (same pairs, same order as in global scratch)
  __shared__ T s_tree[kTreeCap];
  __shared__ double s_Q[kCtlPre];
  __shared__ int s_active;
  __shared__ double s_t_old;
  // This block sits on the critical path between two steps, and what it does is a chain of dependent global loads
  // (control word -> string descriptor -> member list -> geometry -> cell record).  Everything that depends only on
  // what is in memory when the kernel starts is therefore loaded NOW, by all threads at once: the control fields
  // (thread 0), every string member's term of both sums (thread j: member j of each string; the conveyance weights
  // use the state the step will read, buffer `cur` before the flip), the hydrographs (one thread per string).
  const int ns = ctl->n_strings, pending = ctl->pending, cur = ctl->cur;
  const double dt_prev = ctl->dt_last, t_now = ctl->t;
  double c_tend = 0.0, c_cfl = 0.0, c_dtmax = 0.0;
  long long c_left = 0, c_done = 0;
  int c_flags = 0, c_pp = 0;
  unsigned long long c_rate = 0ull;
  if (threadIdx.x == 0) {
    c_tend = ctl->t_end; c_cfl = ctl->cfl; c_dtmax = ctl->dt_max; c_left = ctl->steps_left; c_done = ctl->steps_done;
    c_flags = ctl->flags; c_pp = ctl->ping_pong; c_rate = ctl->rate_bits;
  }
  const CellRecT<T> *__restrict__ rec = cur ? rec_b : rec_a;
  auto term_out = [&](const BoundaryString &bs, int j) -> T {   // l * (limited F1) of member j (bookkeeping)
    if (string_M) return (T)string_M[bs.first + j];         // fused patch step: written by the owning patch
    const int e = string_edges[bs.first + j];
    const EdgeGeomT<T> eg = geom[e];
    T F1 = flux[e].F1;
    if (theta && F1 > T(0.0)) {                              // nullptr: the records are limited already (k_theta_lazy)
      const T th = theta[eg.L];
      if (th < T(1.0)) F1 = th * F1;
    }
    return eg.len * F1;
  };
  auto term_in = [&](const BoundaryString &bs, int j) -> T {    // conveyance weight of member j (R-11)
    const int e = string_edges[bs.first + j];
    const EdgeGeomT<T> eg = geom[e];
    return (eg.len * k_weight(kst[eg.L])) * pow53(rec[eg.L].h);
  };
  bool fast = ns <= kCtlPre;                             // block-uniform: every thread reads the same descriptors
  T pre[kCtlPre];
#pragma unroll
  for (int s = 0; s < kCtlPre; ++s) {
    pre[s] = T(0.0);
    if (s < ns) {
      const BoundaryString &bs = strings[s];
      if (bs.pow2 > (int)blockDim.x) fast = false;
      else if ((int)threadIdx.x < bs.n_edges) {
        if (bs.type == kBcOutflowUniform) { if (pending) pre[s] = term_out(bs, threadIdx.x); }
        else if (bs.type == kBcInflowQ && mode == 0) pre[s] = term_in(bs, threadIdx.x);
      }
      if (bs.type == kBcInflowQ && mode == 0 && threadIdx.x == blockDim.x - 1 - s)
        s_Q[s] = (double)(T)hydrograph(bs.params, bs.n_params, t_now);   // Q(t^n) in the precision of the state
    }
  }
  if (fast) {
    // every string's pairwise tree at once, out of registers: xor-free shuffle tree inside each warp (lane 0 ends up
    // with v[i] + v[i+1], then + (v[i+2] + v[i+3]), ...: the same pairs in the same order as block_tree_sum; the
    // padding zeros beyond pow2 add nothing), the warp sums to shared memory, warp s finishes string s.
    __shared__ T s_part[kCtlPre][32];
    __shared__ T s_sum[kCtlPre];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int s = 0; s < kCtlPre; ++s) {
      T x = pre[s];
#pragma unroll
      for (int off = 1; off < 32; off <<= 1) x = x + __shfl_down_sync(0xffffffffu, x, off);
      if (lane == 0) s_part[s][wid] = x;
    }
    __syncthreads();
    if (wid < kCtlPre) {
      T x = (lane < (int)(blockDim.x >> 5)) ? s_part[wid][lane] : T(0.0);
#pragma unroll
      for (int off = 1; off < 32; off <<= 1) x = x + __shfl_down_sync(0xffffffffu, x, off);
      if (lane == 0) s_sum[wid] = x;
    }
    __syncthreads();
    if (threadIdx.x != 0) return;
    if (pending)
      for (int s = 0; s < ns; ++s) {
        if (strings[s].type == kBcInflowQ) ctl->vol_in += dt_prev * strings[s].Q;
        else if (strings[s].type == kBcOutflowUniform) ctl->vol_out += dt_prev * (double)s_sum[s & (kCtlPre - 1)];
      }
    if (mode == 1) { ctl->pending = 0; ctl->vol = 0.0; ctl->n_wet = 0; ctl->nonfinite = 0; return; }
    int active = 0, new_pending = 0;
    const double t = t_now, t_end = c_tend;
    if (c_left != 0 && t < t_end && !(c_flags & (kFlagUnbounded | kFlagStalled))) {
      const double r = __longlong_as_double((long long)c_rate);
      double dt = (r > 0.0) ? c_cfl / r : c_dtmax;
      dt = fmin(dt, c_dtmax);
      const double rem = t_end - t;
      double t_new;
      if (dt >= rem) { dt = rem; t_new = t_end; } else { t_new = t + dt; }
      if (!isfinite(dt)) {
        ctl->flags = c_flags | kFlagUnbounded;
      } else if (!(dt > 0.0) || !(t_new > t)) {   // the clock cannot advance (a rate of +inf, or dt below ulp(t)):
        ctl->flags = c_flags | kFlagStalled;      // stop instead of stepping in place for ever
      } else {
        active = 1;
        ctl->dt = dt; ctl->dt_last = dt; ctl->t = t_new;
        ctl->rate_bits = 0ull;
        ctl->src = cur;                      // the step reads the newest state ...
        ctl->cur = cur ^ c_pp;               // ... and, when it ping-pongs, writes the other buffer
        ctl->steps_done = c_done + 1;
        if (c_left > 0) ctl->steps_left = c_left - 1;
        new_pending = 1;
      }
    }
    ctl->pending = new_pending;
    ctl->active = active;
    if (active)                              // boundary strings at t^n (R-11): Q(t^n) and the conveyance sum
      for (int s = 0; s < ns; ++s)
        if (strings[s].type == kBcInflowQ) { strings[s].sumK = (double)s_sum[s & (kCtlPre - 1)]; strings[s].Q = s_Q[s & (kCtlPre - 1)]; }
    return;
  }
  // ---- general path (more than kCtlPre strings, or a string with more members than the block has threads)
  // ---- volume bookkeeping of the previous step, from the (limited) fluxes actually applied
  if (pending) {
    for (int s = 0; s < ns; ++s) {
      BoundaryString &bs = strings[s];
      if (bs.type == kBcInflowQ) {
        if (threadIdx.x == 0) ctl->vol_in += dt_prev * bs.Q;
      } else if (bs.type == kBcOutflowUniform) {
        T *v = bs.pow2 <= kTreeCap ? s_tree : scratch + bs.scratch;
        for (int j = threadIdx.x; j < bs.pow2; j += blockDim.x) {
          T a = T(0.0);
          if (j < bs.n_edges) a = term_out(bs, j);
          v[j] = a;
        }
        const T sum = block_tree_sum(v, bs.pow2);
        if (threadIdx.x == 0) ctl->vol_out += dt_prev * (double)sum;
      }
    }
  }
  __syncthreads();
  if (mode == 1) {
    if (threadIdx.x == 0) { ctl->pending = 0; ctl->vol = 0.0; ctl->n_wet = 0; ctl->nonfinite = 0; }
    return;
  }
  // ---- S0: dt from the rate of U^n; S4: t += dt (t_end is hit exactly)
  if (threadIdx.x == 0) {
    int active = 0, new_pending = 0;
    const double t = t_now, t_end = c_tend;
    if (c_left != 0 && t < t_end && !(c_flags & (kFlagUnbounded | kFlagStalled))) {
      const double r = __longlong_as_double((long long)c_rate);
      double dt = (r > 0.0) ? c_cfl / r : c_dtmax;
      dt = fmin(dt, c_dtmax);
      const double rem = t_end - t;
      double t_new;
      if (dt >= rem) { dt = rem; t_new = t_end; } else { t_new = t + dt; }
      if (!isfinite(dt)) {
        ctl->flags = c_flags | kFlagUnbounded;
      } else if (!(dt > 0.0) || !(t_new > t)) {   // the clock cannot advance (a rate of +inf, or dt below ulp(t)):
        ctl->flags = c_flags | kFlagStalled;      // stop instead of stepping in place for ever
      } else {
        active = 1;
        ctl->dt = dt; ctl->dt_last = dt; ctl->t = t_new;
        ctl->rate_bits = 0ull;
        ctl->src = cur;                      // the step reads the newest state ...
        ctl->cur = cur ^ c_pp;               // ... and, when it ping-pongs, writes the other buffer
        ctl->steps_done = c_done + 1;
        if (c_left > 0) ctl->steps_left = c_left - 1;
        new_pending = 1;
      }
    }
    ctl->pending = new_pending;
    ctl->active = active;
    s_active = active;
    s_t_old = t;
  }
  __syncthreads();
  if (!s_active) return;
  // ---- boundary strings at t^n (R-11): Q(t^n) and the conveyance sum over the string
  for (int s = 0; s < ns; ++s) {
    BoundaryString &bs = strings[s];
    if (bs.type != kBcInflowQ) continue;
    T *v = bs.pow2 <= kTreeCap ? s_tree : scratch + bs.scratch;
    for (int j = threadIdx.x; j < bs.pow2; j += blockDim.x) {
      T a = T(0.0);
      if (j < bs.n_edges) a = term_in(bs, j);
      v[j] = a;
    }
    const T sum = block_tree_sum(v, bs.pow2);
    if (threadIdx.x == 0) {
      bs.sumK = (double)sum;
      bs.Q = (double)(T)hydrograph(bs.params, bs.n_params, s_t_old);
    }
  }
}

// AUTO variant choice at swe_set_state: number of cells with h > h_dry in the caller's array
static __global__ void __launch_bounds__(kBlock)
k_count_wet(Control *__restrict__ ctl, const double *__restrict__ h, int n_cells) {
  long long wet = 0;
  const double h_dry = ctl->h_dry;
  for (int i = blockIdx.x * kBlock + threadIdx.x; i < n_cells; i += gridDim.x * kBlock) wet += (h[i] > h_dry);
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) wet += __shfl_xor_sync(0xffffffffu, wet, off);
  if ((threadIdx.x & 31) == 0 && wet) atomicAdd((unsigned long long *)&ctl->n_wet, (unsigned long long)wet);
}

// switches the step variant (both compute bit-identical states): the three-pass step works in place in buffer a
static __global__ void k_set_variant(Control *ctl, int ping_pong, int zero_wet) {
  if (zero_wet) { ctl->n_wet = 0; return; }
  ctl->ping_pong = ping_pong;
  if (!ping_pong) { ctl->cur = 0; ctl->src = 0; }
}

// start of an swe_step call: the stop conditions of this call
static __global__ void k_call_begin(Control *ctl, long long n_steps, double t_end, double cfl) {
  ctl->steps_left = n_steps;
  ctl->t_end = t_end;
  ctl->cfl = cfl;
  ctl->flags &= ~(kFlagUnbounded | kFlagStalled);
}

static __global__ void k_reset(Control *ctl, double t0) {
  ctl->t = t0; ctl->dt = 0.0; ctl->dt_last = 0.0;
  ctl->vol_in = 0.0; ctl->vol_out = 0.0; ctl->vol_clipped = 0.0;
  ctl->rate_bits = 0ull; ctl->steps_left = 0; ctl->steps_done = 0;
  ctl->active = 0; ctl->pending = 0; ctl->flags = 0;
  ctl->src = ctl->cur;
}

// swe_step_info reductions: volume, wet count, non-finite check.  Deterministic (the same sum order every call):
// fixed cell -> thread assignment, xor-shuffle tree per warp, warps in order per block, one partial per block, and the
// block that finishes last adds the partials in block order.
constexpr int kInfoMaxBlocks = 148 * 8;
struct InfoPartial { double vol; long long wet; int bad; int pad_; };

template <typename T = double>
__global__ void __launch_bounds__(kBlock)
k_info(Control *__restrict__ ctl, const CellRecT<T> *rec_a, const CellRecT<T> *rec_b, const T *__restrict__ area,
       int n_cells, InfoPartial *__restrict__ part, unsigned int *__restrict__ ticket) {
  const CellRecT<T> *__restrict__ rec = ctl->cur ? rec_b : rec_a;
  double vol = 0.0;
  long long wet = 0;
  int bad = 0;
  const double h_dry = ctl->h_dry;
  for (int i = blockIdx.x * kBlock + threadIdx.x; i < n_cells; i += gridDim.x * kBlock) {
    const CellRecT<T> c = rec[i];
    vol += (double)c.h * (double)area[i];
    wet += (c.h > (T)h_dry);
    bad |= !(isfinite(c.h) && isfinite(c.qx) && isfinite(c.qy));
  }
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) {
    vol += __shfl_xor_sync(0xffffffffu, vol, off);
    wet += __shfl_xor_sync(0xffffffffu, wet, off);
    bad |= __shfl_xor_sync(0xffffffffu, bad, off);
  }
  __shared__ double s_vol[kBlock / 32];
  __shared__ long long s_wet[kBlock / 32];
  __shared__ int s_bad[kBlock / 32];
  __shared__ bool s_last;
  if ((threadIdx.x & 31) == 0) { s_vol[threadIdx.x >> 5] = vol; s_wet[threadIdx.x >> 5] = wet; s_bad[threadIdx.x >> 5] = bad; }
  __syncthreads();
  if (threadIdx.x == 0) {
    InfoPartial p; p.vol = 0.0; p.wet = 0; p.bad = 0; p.pad_ = 0;
    for (int k = 0; k < kBlock / 32; ++k) { p.vol += s_vol[k]; p.wet += s_wet[k]; p.bad |= s_bad[k]; }
    part[blockIdx.x] = p;
    __threadfence();
    s_last = (atomicAdd(ticket, 1u) == gridDim.x - 1);
  }
  __syncthreads();
  if (!s_last) return;
  __threadfence();
  if (threadIdx.x == 0) {
    double v = 0.0; long long w = 0; int b = 0;
    for (unsigned k = 0; k < gridDim.x; ++k) { const InfoPartial p = part[k]; v += p.vol; w += p.wet; b |= p.bad; }
    ctl->vol = v; ctl->n_wet = w; ctl->nonfinite = b;
    *ticket = 0u;
  }
}

// caller numbering <-> internal numbering (cell_perm[new] = caller id)
template <typename T = double>
__global__ void __launch_bounds__(kBlock)
k_pack_state(const Control *__restrict__ ctl, const int *__restrict__ cell_perm, const double *__restrict__ h,
             const double *__restrict__ hu, const double *__restrict__ hv, CellRecT<T> *rec_a, CellRecT<T> *rec_b, int n_cells) {
  CellRecT<T> *__restrict__ rec = ctl->cur ? rec_b : rec_a;
  const int i = blockIdx.x * kBlock + threadIdx.x;
  if (i >= n_cells) return;
  const int o = cell_perm[i];
  CellRecT<T> c = rec[i];
  c.h = (T)h[o]; c.qx = (T)hu[o]; c.qy = (T)hv[o];      // the caller's arrays are fp64; rounded once when T = float
  rec[i] = c;
}

template <typename T = double>
__global__ void __launch_bounds__(kBlock)
k_unpack_state(const Control *__restrict__ ctl, const int *__restrict__ cell_perm, const CellRecT<T> *rec_a,
               const CellRecT<T> *rec_b, double *__restrict__ h, double *__restrict__ hu, double *__restrict__ hv,
               int n_cells) {
  const CellRecT<T> *__restrict__ rec = ctl->cur ? rec_b : rec_a;
  const int i = blockIdx.x * kBlock + threadIdx.x;
  if (i >= n_cells) return;
  const int o = cell_perm[i];
  const CellRecT<T> c = rec[i];
  h[o] = c.h; hu[o] = c.qx; hv[o] = c.qy;
}

// Morph::cell of the state as it stands (after swe_set_morphology / swe_set_state): what k_cell_update leaves behind
static __global__ void __launch_bounds__(kBlock)
k_sed_cell_init(const Control *__restrict__ ctl, const CellRec *__restrict__ rec, const double *__restrict__ gn2,
                double2 *__restrict__ cell, int n_cells) {
  const int i = blockIdx.x * kBlock + threadIdx.x;
  if (i >= n_cells) return;
  const double h = rec[i].h, f2 = gn2[i];
  cell[i] = (h > ctl->h_dry && f2 > 0.0) ? make_double2(f2, cbrt_rn(h)) : make_double2(0.0, 0.0);
}

// both record buffers of the fused patch step hold the bed of the newest state (swe_set_morphology)
static __global__ void __launch_bounds__(kBlock)
k_sync_bed(const Control *__restrict__ ctl, CellRec *rec_a, CellRec *rec_b, int n_cells) {
  const int i = blockIdx.x * kBlock + threadIdx.x;
  if (i >= n_cells) return;
  if (ctl->cur) rec_a[i].z = rec_b[i].z; else rec_b[i].z = rec_a[i].z;
}

// bed elevation z_B (swe_get_bed), newest state buffer, caller numbering
static __global__ void __launch_bounds__(kBlock)
k_unpack_bed(const Control *__restrict__ ctl, const int *__restrict__ cell_perm, const CellRec *rec_a,
             const CellRec *rec_b, double *__restrict__ zb, int n_cells) {
  const CellRec *__restrict__ rec = ctl->cur ? rec_b : rec_a;
  const int i = blockIdx.x * kBlock + threadIdx.x;
  if (i < n_cells) zb[cell_perm[i]] = rec[i].z;
}

// q_Bij of the most recent step in caller edge numbering (swe_get_sediment_flux); the sign follows the caller's L -> R
static __global__ void __launch_bounds__(kBlock)
k_export_sediment(const int *__restrict__ edge_perm, const double *__restrict__ qB, double *__restrict__ out, int n_edges) {
  const int e = blockIdx.x * kBlock + threadIdx.x;
  if (e < n_edges) out[edge_perm[e]] = qB[e];
}

// one scalar species, caller numbering <-> internal numbering, newest state buffer
static __global__ void __launch_bounds__(kBlock)
k_pack_scalar(const Control *__restrict__ ctl, const int *__restrict__ cell_perm, const double *__restrict__ src,
              double *qa, double *qb, int n_cells) {
  const int i = blockIdx.x * kBlock + threadIdx.x;
  if (i < n_cells) (ctl->cur ? qb : qa)[i] = src[cell_perm[i]];
}

static __global__ void __launch_bounds__(kBlock)
k_unpack_scalar(const Control *__restrict__ ctl, const int *__restrict__ cell_perm, const double *qa, const double *qb,
                double *__restrict__ dst, int n_cells) {
  const int i = blockIdx.x * kBlock + threadIdx.x;
  if (i < n_cells) dst[cell_perm[i]] = (ctl->cur ? qb : qa)[i];
}

// inspection (swe_device_cbrt): the cube root of R-14 as the kernels evaluate it
static __global__ void __launch_bounds__(kBlock)
k_cbrt(const double *__restrict__ x, double *__restrict__ y, long long n) {
  const long long i = (long long)blockIdx.x * kBlock + threadIdx.x;
  if (i < n) y[i] = cbrt_rn(x[i]);
}

// inspection (swe_get_edge_flux): per-edge records after the limiter, in caller edge numbering
template <typename T = double>
__global__ void __launch_bounds__(kBlock)
k_export_flux(const int *__restrict__ edge_perm, const EdgeGeomT<T> *__restrict__ geom, const EdgeFluxT<T> *__restrict__ flux,
              const T *__restrict__ theta, double *__restrict__ F1, double *__restrict__ F3,
              double *__restrict__ GL, double *__restrict__ GR, int n_edges) {
  const int e = blockIdx.x * kBlock + threadIdx.x;
  if (e >= n_edges) return;
  const EdgeGeomT<T> eg = geom[e];
  EdgeFluxT<T> f = flux[e];
  if constexpr (sizeof(T) == 8) if (theta) {                                       // nullptr: the records are limited already (k_theta_lazy)
    double th = 1.0;
    if (f.F1 > 0.0) th = theta[eg.L];
    else if (f.F1 < 0.0 && eg.R >= 0) th = theta[eg.R];
    if (th < 1.0) { f.F1 = th * f.F1; f.F3 = th * f.F3; f.GL = th * f.GL; f.GR = th * f.GR; }
  }
  const int o = edge_perm[e];
  if (F1) { F1[o] = f.F1; F3[o] = f.F3; }             // the caller exports in two halves (staging holds 2 n_edges doubles)
  if (GL) { GL[o] = f.GL; GR[o] = f.GR; }
}

}  // namespace swe
