// Fused patch step (sm_100a): one thread block advances one patch of consecutive (Morton-ordered) cells by a whole
// time step -- S1 edge fluxes, S1c limiter, S2 gather, S3 update + friction, and Eq. 21 of the new state for the
// next dt -- out of shared memory.  Edge fluxes never go to DRAM; the state ping-pongs between two buffers because
// neighbouring patches read the old state of this patch's cells.  Arithmetic and parenthesisation are those of the
// three-pass kernels in swe_kernels.cuh (R-14), so both variants give bit-identical states.
//
// Phases (separated by __syncthreads):
//   1  states of the local cells (own, ring 1, ring 2) -> shared memory as (h, u, v, z)
//   2  every local edge: hydrostatic reconstruction + HLLC, boundary edges
//   3  theta of own and ring-1 cells (R-8b)
//   4  own cells: limited fluxes in slot order (Eq. 12), update, friction (Eq. 2), Eq. 21 rate
#pragma once
#include "swe_kernels.cuh"

namespace swe {

struct PatchSmem {          // offsets (in doubles) into the dynamic shared memory; the same for every block
  int h, u, v, z, theta, area, F1, len, F3, GL, GR, nx, ny, phi, total;
};

__host__ __device__ inline PatchSmem patch_smem_layout(int max_loc, int max_c1, int max_e, int max_eown,
                                                       int n_species = 0) {
  PatchSmem s;
  int o = 0;
  s.h = o; o += max_loc; s.u = o; o += max_loc; s.v = o; o += max_loc; s.z = o; o += max_loc;
  s.theta = o; o += max_c1;
  s.area = o; o += max_c1;                      // |Omega| of own and ring-1 cells (limiter)
  s.F1 = o; o += max_e; s.len = o; o += max_e;
  s.F3 = o; o += max_eown; s.GL = o; o += max_eown; s.GR = o; o += max_eown;
  s.nx = o; o += max_eown; s.ny = o; o += max_eown;
  s.phi = o; o += n_species * max_loc;          // concentrations of the local cells, species-major
  s.total = o;
  return s;
}

struct PatchArgs {
  const PatchHeader *hdr;
  const int32_t *halo_ids;
  const double *halo_area;
  const PatchEdge *pedge;
  const uint4 *pce;
  CellRec *rec_a, *rec_b;
  const double *area, *inv_area, *gn2, *kst;
  const BoundaryString *strings;
  const int32_t *slot_string;     // string id of every position of string_edges[]
  double *string_M;               // l * (limited F1) of every boundary-string edge, by position in string_edges[]
  const int32_t *patch_nbr;       // PatchHeader::nbr_off / n_nbr
  uint8_t *dry_a, *dry_b;         // per state buffer and patch: 1 = every own cell of the patch is exactly (0, 0, 0)
  int max_loc, max_c1, max_e, max_eown;
  Scalars sc;                     // passive scalars (kScalars instantiation only)
};

// Loads are software-pipelined: the record an iteration needs is loaded one iteration (or one phase) ahead, so that
// the global-memory latency overlaps the arithmetic of the current item instead of stalling its first use.
// kCap* != 0: the shared-memory arrays have these compile-time capacities (every offset becomes an immediate of the
// LDS / STS instructions); kCap* == 0: capacities come from PatchArgs at run time (any patch size).
// kScalars: the passive-scalar module (R-19) is on: concentrations of the local cells in shared memory, one more
// gather per species in phase 4 (always with run-time capacities).
template <int kThreads, int kMinBlocks, int kCapLoc, int kCapC1, int kCapE, int kCapEown, bool kScalars = false>
__global__ void __launch_bounds__(kThreads, kMinBlocks)
k_patch_step(Control *__restrict__ ctl, const PatchArgs A) {
  if (!ctl->active) return;
  extern __shared__ double sm[];
  const int n_sp = kScalars ? A.sc.n : 0;
  const int cap_loc = kCapLoc ? kCapLoc : A.max_loc;
  const PatchSmem S = kCapLoc ? patch_smem_layout(kCapLoc, kCapC1, kCapE, kCapEown)
                              : patch_smem_layout(A.max_loc, A.max_c1, A.max_e, A.max_eown, n_sp);
  double *sh_phi = sm + S.phi;
  double *sh_h = sm + S.h, *sh_u = sm + S.u, *sh_v = sm + S.v, *sh_z = sm + S.z, *sh_th = sm + S.theta;
  double *sh_F1 = sm + S.F1, *sh_len = sm + S.len, *sh_F3 = sm + S.F3, *sh_GL = sm + S.GL, *sh_GR = sm + S.GR;
  double *sh_nx = sm + S.nx, *sh_ny = sm + S.ny, *sh_area = sm + S.area;

  const PatchHeader H = A.hdr[blockIdx.x];
  const int src = ctl->src;
  const CellRec *__restrict__ in = src ? A.rec_b : A.rec_a;
  CellRec *__restrict__ out = src ? A.rec_a : A.rec_b;
  const double dt = ctl->dt, g = ctl->g, h_dry = ctl->h_dry;
  const int tid = threadIdx.x;
  const int n_loc = H.n_own + H.n_r1 + H.n_r2, n_c1 = H.n_own + H.n_r1, n_e = H.n_eown + H.n_er1;
  const PatchEdge *__restrict__ pedge = A.pedge + H.edge_off;
  const uint4 *__restrict__ pce = A.pce + H.pce_off;
  const int32_t *__restrict__ halo_ids = A.halo_ids + H.halo_off - H.n_own;     // indexed by local cell id >= n_own
  const double *__restrict__ halo_area = A.halo_area + H.halo_off - H.n_own;

  // ---- dry patch: when the own cells of this patch and of every patch that owns one of its halo cells are exactly
  // (0, 0, 0) in the state being read, and no boundary string can feed the patch, every flux of S1 is exactly 0,
  // theta = 1 and S3 returns (+0, 0, 0) for every own cell: write that (unless the target buffer holds it already).
  const uint8_t *__restrict__ dry_in = src ? A.dry_b : A.dry_a;
  uint8_t *__restrict__ dry_out = src ? A.dry_a : A.dry_b;
  {
    int wet = 1;
    if (H.n_string_edges == 0 && H.n_nbr < kThreads) {
      wet = 0;
      if (tid <= H.n_nbr) wet = !dry_in[tid == 0 ? (int)blockIdx.x : A.patch_nbr[H.nbr_off + tid - 1]];
    }
    if (!__syncthreads_or(wet)) {
      if (!dry_out[blockIdx.x]) {
        for (int l = tid; l < H.n_own; l += kThreads) {
          CellRec c = in[H.cell0 + l];
          c.h = 0.0; c.qx = 0.0; c.qy = 0.0;
          out[H.cell0 + l] = c;
          _Pragma("unroll") for (int sp = 0; sp < kMaxSpecies; ++sp) if (sp < n_sp) (src ? A.sc.qa[sp] : A.sc.qb[sp])[H.cell0 + l] = 0.0;   // flag: all q_c are 0 too
        }
        __syncthreads();
        if (tid == 0) dry_out[blockIdx.x] = 1;
      }
      if (tid == 0) atomicAdd(&ctl->patches_skipped, 1ull);
      return;
    }
  }

  // ---- the patch's streamed tables are contiguous: pull them into L2 now (no registers held), so that the loads of
  // phases 2-4 pay L2 latency instead of DRAM latency
  {
    auto prefetch_range = [&](const void *base, int bytes) {
      const char *p = (const char *)base;
      for (int off = tid * 128; off < bytes; off += kThreads * 128) asm volatile("prefetch.global.L2 [%0];" ::"l"(p + off));
    };
    prefetch_range(pedge, n_e * (int)sizeof(PatchEdge));
    prefetch_range(pce, n_c1 * (int)sizeof(uint4));
    prefetch_range(A.area + H.cell0, H.n_own * 8);
    prefetch_range(A.inv_area + H.cell0, H.n_own * 8);
    prefetch_range(A.gn2 + H.cell0, H.n_own * 8);
    prefetch_range(halo_area + H.n_own, H.n_r1 * 8);
  }

  // ---- phase 1: local cell states; velocities once per cell (R-8: thin films carry no momentum).  Three records per
  // thread are in flight at a time (the halo part is a dependent id -> record gather).
  PatchEdge pe_next;
  if (tid < n_e) pe_next = pedge[tid];                 // first record of phase 2, in flight during phase 1
  {
    int water = 0;
    int l;
    for (int base = tid; base < n_loc; base += 3 * kThreads) {
      int gid[3];
      CellRec c[3];
#pragma unroll
      for (int j = 0; j < 3; ++j) {
        l = base + j * kThreads;
        gid[j] = l < H.n_own ? H.cell0 + l : (l < n_loc ? halo_ids[l] : -1);
      }
#pragma unroll
      for (int j = 0; j < 3; ++j)
        if (gid[j] >= 0) c[j] = in[gid[j]];
#pragma unroll
      for (int j = 0; j < 3; ++j) {
        l = base + j * kThreads;
        if (gid[j] >= 0) {
          double u = 0.0, v = 0.0;
          if (c[j].h > h_dry) { u = c[j].qx / c[j].h; v = c[j].qy / c[j].h; }
          sh_h[l] = c[j].h; sh_u[l] = u; sh_v[l] = v; sh_z[l] = c[j].z;
          if (l < n_c1) { sh_th[l] = 1.0; sh_area[l] = l < H.n_own ? A.area[gid[j]] : halo_area[l]; }
          water |= (c[j].h != 0.0);
          if (kScalars)                              // phi = q_c / h where there is water, else 0 (R-19)
            _Pragma("unroll") for (int sp = 0; sp < kMaxSpecies; ++sp) if (sp < n_sp)
              sh_phi[sp * cap_loc + l] = c[j].h > 0.0 ? (src ? A.sc.qb[sp] : A.sc.qa[sp])[gid[j]] / c[j].h : 0.0;
        }
      }
    }
    // second, exact test on the local cells themselves (the flags above are per whole patch): no water in any
    // local cell and no boundary string -> same result (+0, 0, 0)
    if (!__syncthreads_or(water) && H.n_string_edges == 0) {
      int scalar_mass = 0;
      for (l = tid; l < H.n_own; l += kThreads) {
        CellRec c; c.h = 0.0; c.qx = 0.0; c.qy = 0.0; c.z = sh_z[l];
        out[H.cell0 + l] = c;
        _Pragma("unroll") for (int sp = 0; sp < kMaxSpecies; ++sp) if (sp < n_sp) {          // no flux: scalar mass parked in dry cells stays where it is
          const double q = (src ? A.sc.qb[sp] : A.sc.qa[sp])[H.cell0 + l];
          (src ? A.sc.qa[sp] : A.sc.qb[sp])[H.cell0 + l] = q;
          scalar_mass |= (q != 0.0);
        }
      }
      scalar_mass = kScalars ? __syncthreads_or(scalar_mass) : 0;
      if (tid == 0) { dry_out[blockIdx.x] = scalar_mass ? 0 : 1; atomicAdd(&ctl->patches_skipped, 1ull); }
      return;
    }
  }
  uint4 pc_next = make_uint4(0u, 0u, 0u, 0u);          // slot record of this thread's first own cell (phase 4)
  if (tid < H.n_own) pc_next = pce[tid];

  // ---- phase 2: edge fluxes
  for (int e = tid; e < n_e; e += kThreads) {
    const PatchEdge pe = pe_next;
    if (e + kThreads < n_e) pe_next = pedge[e + kThreads];
    const int L = pe.L;
    const double hL = sh_h[L], uL = sh_u[L], vL = sh_v[L], zL = sh_z[L];
    EdgeFlux o;
    if (pe.R != 0xFFFF) {
      const int R = pe.R;
      const double hR = sh_h[R], uR = sh_u[R], vR = sh_v[R], zR = sh_z[R];
      const double unL = uL * pe.nx + vL * pe.ny, utL = vL * pe.nx - uL * pe.ny;
      const double unR = uR * pe.nx + vR * pe.ny, utR = vR * pe.nx - uR * pe.ny;
      o = riemann_nt(g, hL, unL, utL, zL, hR, unR, utR, zR);
    } else {
      const BoundaryString *bs = nullptr;
      int code = pe.aux;
      if (code <= -3) { bs = A.strings + A.slot_string[-3 - code]; code = -3; }
      const int gidL = L < H.n_own ? H.cell0 + L : halo_ids[L];
      o = boundary_flux(g, code, bs, A.kst, gidL, pe.nx, pe.ny, pe.len, hL, zL, uL, vL);
    }
    sh_F1[e] = o.F1; sh_len[e] = pe.len;
    if (e < H.n_eown) { sh_F3[e] = o.F3; sh_GL[e] = o.GL; sh_GR[e] = o.GR; sh_nx[e] = pe.nx; sh_ny[e] = pe.ny; }
    // S1c, lazily (R-8b; as in k_edge_flux): theta_i < 1 needs one outgoing edge with dt * o_k > 0.3 h_i |Omega_i|.  Only
    // such donor cells are marked (theta = -1); phase 3 evaluates theta for them and every other cell keeps theta = 1.
    const int d = o.F1 > 0.0 ? L : ((o.F1 < 0.0 && pe.R != 0xFFFF) ? (int)pe.R : n_c1);
    if (d < n_c1 && dt * (pe.len * fabs(o.F1)) > 0.3 * (sh_h[d] * sh_area[d])) sh_th[d] = -1.0;
  }
  // first own cell of this thread in phase 4: its record and constants, in flight during phase 3
  const uint4 pc4_first = pc_next;
  CellRec c4_next;
  double invA_next = 0.0, gn2_next = 0.0;
  if (tid < H.n_own) { c4_next = in[H.cell0 + tid]; invA_next = A.inv_area[H.cell0 + tid]; gn2_next = A.gn2[H.cell0 + tid]; }
  __syncthreads();

  // ---- phase 3 (R-8b): theta_i = min(1, h_i |Omega_i| / (dt * sum of the outgoing l F1)), slots in order -- for the
  // cells marked in phase 2 only
  for (int l = tid; l < n_c1; l += kThreads) {
    if (sh_th[l] >= 0.0) continue;
    const uint4 pc = pce[l];
    const uint32_t w[3] = {pc.x, pc.y, pc.z};
    double o[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      const int e = w[k] & 0x7FFFu;
      const double sM = ((w[k] & 0x8000u) ? 1.0 : -1.0) * (sh_len[e] * sh_F1[e]);
      o[k] = dmax0(sM);
    }
    const double outflow = ((o[0] + o[1]) + o[2]);
    const double avail = sh_h[l] * sh_area[l];
    double th = 1.0;
    if (dt * outflow > avail) th = avail / (dt * outflow);
    sh_th[l] = th;
  }
  __syncthreads();

  // ---- phase 4: own cells
  double rate = 0.0;
  int nonzero = 0;
  uint4 pc4 = pc4_first;
  for (int l = tid; l < H.n_own; l += kThreads) {
    const int i = H.cell0 + l;
    const uint4 pc = pc4;
    CellRec c = c4_next;
    const double invA = invA_next, f2 = gn2_next;
    const int ln = l + kThreads;
    if (ln < H.n_own) { pc4 = pce[ln]; c4_next = in[i + kThreads]; invA_next = A.inv_area[i + kThreads]; gn2_next = A.gn2[i + kThreads]; }
    const uint32_t w[3] = {pc.x, pc.y, pc.z};
    double dH = 0.0, dX = 0.0, dY = 0.0;             // ((d0 + d1) + d2), accumulated in slot order
    double F1k[3], slk[3];                           // kScalars: limited mass flux and sign * length of every slot,
    int up[3];                                       // local id of the upwind cell, or -1 - slot of an inflow-string edge
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      const int e = w[k] & 0x7FFFu;
      const bool isL = (w[k] & 0x8000u) != 0u;
      const uint32_t nb = w[k] >> 16;
      double F1 = sh_F1[e], F3 = sh_F3[e];
      double G = isL ? sh_GL[e] : sh_GR[e];
      // limiter: every component of the edge is scaled by theta of the donor cell (the one F1 leaves)
      double th = 1.0;
      if (F1 > 0.0) th = sh_th[isL ? (uint32_t)l : nb];
      else if (F1 < 0.0 && nb != kPceNoNeighbour) th = sh_th[isL ? nb : (uint32_t)l];
      if (th < 1.0) { F1 = th * F1; F3 = th * F3; G = th * G; }
      const double s = isL ? 1.0 : -1.0;
      const double nxk = sh_nx[e], nyk = sh_ny[e], lenk = sh_len[e];
      const double dHk = s * (lenk * F1);
      const double dXk = s * (lenk * (G * nxk - F3 * nyk));
      const double dYk = s * (lenk * (G * nyk + F3 * nxk));
      if (k == 0) { dH = dHk; dX = dXk; dY = dYk; } else { dH = dH + dHk; dX = dX + dXk; dY = dY + dYk; }
      if (kScalars) {
        F1k[k] = F1; slk[k] = lenk;
        const uint32_t Lc = isL ? (uint32_t)l : nb, Rc = isL ? nb : (uint32_t)l;
        up[k] = (int)((F1 >= 0.0 || Rc == kPceNoNeighbour) ? Lc : Rc);   // ghost concentration = the interior cell's
        if (!isL) slk[k] = -lenk;
      }
      if (nb == kPceNoNeighbour) {                  // boundary-string edge: volume bookkeeping of k_step_control
        const int aux = pedge[e].aux;
        if (aux <= -3) {
          A.string_M[-3 - aux] = lenk * F1;
          if (kScalars && !(F1 >= 0.0) && A.strings[A.slot_string[-3 - aux]].type == kBcInflowQ) up[k] = -1 - (-3 - aux);
        }
      }
    }
    const double a = dt * invA;
    double hn = c.h - a * dH;
    if (hn < 0.0) {                                  // residual negatives (R-8b): clip and count
      atomicAdd(&ctl->vol_clipped, -hn * A.area[i]);
      hn = 0.0;
    }
    double qxn = 0.0, qyn = 0.0;
    if (hn > h_dry) {
      qxn = c.qx - a * dX;
      qyn = c.qy - a * dY;
      if (f2 > 0.0) {   // R-5/R-6: exact integral of dq/dt = -(g/(k^2 h^(7/3))) |q| q over dt, h frozen at h^{n+1}
        const double D = 1.0 + ((dt * f2) * sqrt(qxn * qxn + qyn * qyn)) / ((hn * hn) * cbrt_rn(hn));
        qxn = qxn / D;
        qyn = qyn / D;
      }
      // Eq. 21 (R-7) of the new state, for the next dt: max_j lambda_ij / rho_ij
      const double u = qxn / hn, v = qyn / hn;
      const double cel = sqrt(g * hn);
#pragma unroll
      for (int k = 0; k < 3; ++k) {
        const int e = w[k] & 0x7FFFu;
        const double lam = fabs(u * sh_nx[e] + v * sh_ny[e]) + cel;
        const double val = lam * ((0.75 * sh_len[e]) * invA);
        if (val > rate) rate = val;
      }
    }
    c.h = hn; c.qx = qxn; c.qy = qyn;
    out[i] = c;
    nonzero |= (hn != 0.0) | (qxn != 0.0) | (qyn != 0.0);
    if (kScalars) {                                  // Eq. 20, advective part: A_ij = limited F1 x upwind phi (R-19)
      _Pragma("unroll") for (int sp = 0; sp < kMaxSpecies; ++sp) if (sp < n_sp) {
        double dC = 0.0;
#pragma unroll
        for (int k = 0; k < 3; ++k) {
          const double phi = up[k] >= 0 ? sh_phi[sp * cap_loc + up[k]] : A.strings[A.slot_string[-1 - up[k]]].phi_in[sp];
          const double lC = fabs(slk[k]) * (F1k[k] * phi);
          const double Ck = slk[k] < 0.0 ? -lC : lC;
          dC = k == 0 ? Ck : dC + Ck;
        }
        const double qn = (src ? A.sc.qb[sp] : A.sc.qa[sp])[i] - a * dC;
        (src ? A.sc.qa[sp] : A.sc.qb[sp])[i] = qn;
        nonzero |= (qn != 0.0);
      }
    }
  }
  nonzero = __syncthreads_or(nonzero);
  if (tid == 0) dry_out[blockIdx.x] = nonzero ? 0 : 1;
  block_max_to_global<kThreads>(rate, &ctl->rate_bits);
}

// dry flags of the state buffer that holds the newest state (after swe_set_state); the other buffer's are cleared
template <int kThreads>
__global__ void __launch_bounds__(kThreads)
k_patch_flags(const Control *__restrict__ ctl, const PatchHeader *__restrict__ hdr, const CellRec *rec_a,
              const CellRec *rec_b, uint8_t *dry_a, uint8_t *dry_b, const Scalars sc) {
  const PatchHeader H = hdr[blockIdx.x];
  const CellRec *__restrict__ rec = ctl->cur ? rec_b : rec_a;
  int nonzero = 0;
  for (int l = threadIdx.x; l < H.n_own; l += kThreads) {
    const CellRec c = rec[H.cell0 + l];
    nonzero |= !(c.h == 0.0 && c.qx == 0.0 && c.qy == 0.0);
    _Pragma("unroll") for (int sp = 0; sp < kMaxSpecies; ++sp) if (sp < sc.n) nonzero |= ((ctl->cur ? sc.qb[sp] : sc.qa[sp])[H.cell0 + l] != 0.0);
  }
  nonzero = __syncthreads_or(nonzero);
  if (threadIdx.x == 0) {
    (ctl->cur ? dry_b : dry_a)[blockIdx.x] = nonzero ? 0 : 1;
    (ctl->cur ? dry_a : dry_b)[blockIdx.x] = 0;
  }
}

}  // namespace swe
