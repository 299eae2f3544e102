"""Pins for the oracle's edge flux (S1): hand values, textbook properties, and the literal H-form of
the paper's Eq. 10/11/12.  CPU only."""
import os
from decimal import Decimal as D, getcontext

import numpy as np
import pytest

from workloads import configs as C

G = 9.81
HERE = os.path.dirname(os.path.abspath(__file__))


def load_golden():
    out = {}
    with open(os.path.join(HERE, "golden", "hand_fluxes.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            case, q, v = line.split()
            out[(case, q)] = float(v)
    return out


def close_digits(a, b, digits=12):
    return abs(a - b) <= 10.0 ** (-digits) * max(1.0, abs(b)) * 5


# ---------------------------------------------------------------- independent textbook HLL (Decimal)
def hll_textbook_decimal(hL, unL, hR, unR, SL, SR, g):
    """(SR*FL - SL*FR + SL*SR*(UR-UL))/(SR-SL), Toro ch. 10 eq. of the HLL flux, in 50-digit decimals."""
    getcontext().prec = 50
    hL, unL, hR, unR, SL, SR, g = map(lambda x: D(repr(float(x))), (hL, unL, hR, unR, SL, SR, g))
    FL = (hL * unL, hL * unL * unL + g * hL * hL / 2)
    FR = (hR * unR, hR * unR * unR + g * hR * hR / 2)
    UL = (hL, hL * unL)
    UR = (hR, hR * unR)
    return tuple(float((SR * FL[k] - SL * FR[k] + SL * SR * (UR[k] - UL[k])) / (SR - SL)) for k in range(2))


def test_hand_values_interior(ref):
    gold = load_golden()
    # edge n = (1,0); L: h=2, u=(1,0.5), z=0; R: h=1, u=0, z=0.5
    F1, F3, GL, GR = ref.edge_flux(G, 2.0, 1.0, 0.5, 0.0, 1.0, 0.0, 0.0, 0.5, 1.0, 0.0)
    assert close_digits(F1, gold[("interior", "F1")])
    assert close_digits(F3, gold[("interior", "F3")])
    assert close_digits(GL, gold[("interior", "GL")])
    assert close_digits(GR, gold[("interior", "GR")])
    # re-derive by the textbook form: face depths over z* = max(zL, zR) = 0.5 -> 1.5 and 1.0
    hsL, hsR = 1.5, 1.0
    cL, cR = np.sqrt(G * hsL), np.sqrt(G * hsR)
    us = 0.5 * (1.0 + 0.0) + cL - cR
    cs = 0.5 * (cL + cR) + 0.25 * (1.0 - 0.0)
    SL, SR = min(1.0 - cL, us - cs), max(0.0 + cR, us + cs)
    assert close_digits(SL, gold[("interior", "SL")]) and close_digits(SR, gold[("interior", "SR")])
    F1t, F2t = hll_textbook_decimal(hsL, 1.0, hsR, 0.0, SL, SR, G)
    assert close_digits(F2t, gold[("interior", "F2")])
    assert abs(F1 - F1t) < 1e-14 * abs(F1t)
    assert abs(GL - (F2t - 0.5 * G * hsL ** 2)) < 1e-13
    assert abs(GR - (F2t - 0.5 * G * hsR ** 2)) < 1e-13
    assert abs(F3 - F1t * 0.5) < 1e-14          # F1 > 0: upwind tangential velocity is the left one (0.5)


def test_hand_values_rest_dry_blocked_wall(ref):
    gold = load_golden()
    # rest state over a step, n = (0.6, 0.8): both face depths 1.5 -> every output bit-zero
    out = ref.edge_flux(G, 2.0, 0.0, 0.0, 0.0, 1.5, 0.0, 0.0, 0.5, 0.6, 0.8)
    assert out == (0.0, 0.0, 0.0, 0.0)
    # dry right: SL = -c, SR = 2c, F1 = 2/3 c h, GL = F2 - p = -g h^2 / 6
    F1, F3, GL, GR = ref.edge_flux(G, 1.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 1.0, 0.0)
    assert close_digits(F1, gold[("dryright", "F1")]) and close_digits(GL, gold[("dryright", "GL")])
    assert abs(F1 - 2.0 / 3.0 * np.sqrt(G)) < 1e-14 and abs(GL + G / 6.0) < 1e-14 and F3 == 0.0
    # wet cell below a dry neighbour whose bed is above its surface: blocked, contributes nothing
    assert ref.edge_flux(G, 1.0, 0.3, -0.2, 0.0, 0.0, 0.0, 0.0, 1.5, 0.8, -0.6) == (0.0, 0.0, 0.0, 0.0)
    # wall: mirror ghost through the solver vs closed form h un (un + S), S = max(c - un, c + un/2)
    he, un = 1.5, 0.7
    F1w, F3w, Gw = ref.wall_flux_via_ghost(G, he, un, 0.3)
    c = np.sqrt(G * he)
    closed = he * un * (un + max(c - un, c + 0.5 * un))
    assert close_digits(closed, gold[("wall", "G")])
    assert abs(F1w) < 1e-15 and abs(F3w) < 1e-15 and abs(Gw - closed) < 1e-13


def test_wall_boundary_edge_uses_closed_form(ref):
    """A 2-cell mesh with walls all round: the stored boundary-edge record must be (0, 0, closed form)."""
    w = C.tiny_mesh("two-cells")
    w.h[:] = 1.5
    w.hu[:] = 1.5 * 0.7
    w.hv[:] = 1.5 * -0.2
    s = ref.RefSolver(w)
    s.step(n_steps=1, cfl=1e-9)      # tiny dt: state essentially unchanged, fluxes are those of U^0
    F1, F3, GL, GR = s.edge_fluxes()
    area, nx, ny, ln = s.geometry()
    c = np.sqrt(G * 1.5)
    for e in np.nonzero(w.edge_cell[:, 1] < 0)[0]:
        un = 0.7 * nx[e] - 0.2 * ny[e]
        assert F1[e] == 0.0 and F3[e] == 0.0
        assert abs(GL[e] - 1.5 * un * (un + max(c - un, c + 0.5 * un))) < 1e-13


@pytest.mark.parametrize("seed", range(5))
def test_consistency_and_symmetries(ref, seed):
    rng = np.random.default_rng(100 + seed)
    for _ in range(200):
        h, u, v, z = rng.uniform(0.05, 3), rng.uniform(-3, 3), rng.uniform(-3, 3), rng.uniform(-1, 1)
        th = rng.uniform(0, 2 * np.pi)
        nx, ny = np.cos(th), np.sin(th)
        # consistency: F(U,U) is the physical flux (Toro ch. 10: any approximate Riemann flux)
        F1, F3, GL, GR = ref.edge_flux(G, h, u, v, z, h, u, v, z, nx, ny)
        un, ut = u * nx + v * ny, v * nx - u * ny
        assert abs(F1 - h * un) < 1e-13 * (1 + abs(h * un))
        assert abs(GL - h * un * un) < 1e-12 * (1 + h * un * un) and abs(GL - GR) < 1e-12
        assert abs(F3 - h * un * ut) < 1e-12 * (1 + abs(h * un * ut))
        # mirror: swapping the two cells and reversing the normal gives the same physical exchange
        h2, u2, v2, z2 = rng.uniform(0.0, 3), rng.uniform(-3, 3), rng.uniform(-3, 3), rng.uniform(-1, 1)
        if h2 < 0.05:
            h2, u2, v2 = 0.0, 0.0, 0.0
        a = ref.edge_flux(G, h, u, v, z, h2, u2, v2, z2, nx, ny)
        b = ref.edge_flux(G, h2, u2, v2, z2, h, u, v, z, -nx, -ny)
        assert abs(a[0] + b[0]) < 1e-12 * (1 + abs(a[0]))          # mass flux reverses
        # F3 multiplies ut, and ut = v nx - u ny changes sign with n, while F1 changes sign too:
        assert abs(a[1] - b[1]) < 1e-12 * (1 + abs(a[1]))
        assert abs(a[2] - b[3]) < 1e-12 * (1 + abs(a[2]))          # GL <-> GR
        assert abs(a[3] - b[2]) < 1e-12 * (1 + abs(a[3]))
        # rotation invariance: rotate velocities and normal by the same angle
        ph = rng.uniform(0, 2 * np.pi)
        cph, sph = np.cos(ph), np.sin(ph)
        rot = lambda x, y: (cph * x - sph * y, sph * x + cph * y)
        c_ = ref.edge_flux(G, h, *rot(u, v), z, h2, *rot(u2, v2), z2, *rot(nx, ny))
        for k in range(4):
            assert abs(a[k] - c_[k]) < 1e-11 * (1 + abs(a[k]))


# ---------------------------------------------------------------- literal H-form, Eq. 10 / 11 / 12
def hll_standard(UL, UR, FL, FR, SL, SR):
    if SL >= 0:
        return FL
    if SR <= 0:
        return FR
    return (SR * FL - SL * FR + SL * SR * (UR - UL)) / (SR - SL)


def h_form_increment(g, cell, nbrs, normals, lens, area):
    """-(1/|Omega|) sum_j l_ij F_ij + S_bed for cell i in the paper's variables U = (H, qx, qy), with the
    flux of Eq. 10 (q_n^2/h + g H^2/2 - g H z_B) and the source of Eq. 11 (-g H grad z_B, Green-Gauss with
    the face bed z* = max(z_i, z_j)), evaluated on the modified face states eta* = h* + z*.  Written
    independently of the oracle: standard-form HLL on (eta, q_n), numpy floats.  Valid where the face
    bed is not above either water surface (the blocked case is a separate hand value)."""
    hi, ui, vi, zi = cell
    Hi = hi + zi
    dU = np.zeros(3)
    src = np.zeros(2)
    for (hj, uj, vj, zj), (nx, ny), l in zip(nbrs, normals, lens):
        zs = max(zi, zj)
        assert zs <= Hi + 1e-15 and zs <= hj + zj + 1e-15
        hsi, hsj = max(0.0, hi + zi - zs), max(0.0, hj + zj - zs)
        src += -g * Hi * zs * np.array([nx, ny]) * l          # Eq. 11, S_bed = -g H grad z_B
        uni, uti = ui * nx + vi * ny, vi * nx - ui * ny
        unj, utj = uj * nx + vj * ny, vj * nx - uj * ny
        ci, cj = np.sqrt(g * hsi), np.sqrt(g * hsj)
        if hsi > 0 and hsj > 0:
            us, cs = 0.5 * (uni + unj) + ci - cj, 0.5 * (ci + cj) + 0.25 * (uni - unj)
            SL, SR = min(uni - ci, us - cs), max(unj + cj, us + cs)
        elif hsj == 0:
            SL, SR = uni - ci, uni + 2 * ci
        else:
            SL, SR = unj - 2 * cj, unj + cj
        eta_i, eta_j = hsi + zs, hsj + zs
        # Eq. 10 normal flux on the face states: (q_n, q_n^2/h + g eta^2/2 - g eta z*)
        FLv = np.array([hsi * uni, hsi * uni * uni + 0.5 * g * eta_i ** 2 - g * eta_i * zs])
        FRv = np.array([hsj * unj, hsj * unj * unj + 0.5 * g * eta_j ** 2 - g * eta_j * zs])
        F = hll_standard(np.array([eta_i, hsi * uni]), np.array([eta_j, hsj * unj]), FLv, FRv, SL, SR)
        Ft = F[0] * (uti if F[0] >= 0 else utj)
        dU[0] += l * F[0]
        dU[1] += l * (F[1] * nx - Ft * ny)
        dU[2] += l * (F[1] * ny + Ft * nx)
    inc = -dU / area
    inc[1:] += src / area
    return inc


@pytest.mark.parametrize("seed", range(4))
def test_h_form_identity(ref, seed):
    """SURVEY O-2 / DESIGN R-1: the h-form hydrostatic reconstruction used by the oracle gives the same
    cell increment as the paper's H-form (Eq. 10, 11, 12) on the modified states -- in every case where
    the neighbour's bed does not rise above cell i's surface (z* <= H_i; the fully-blocked case is the
    separate 'blocked' hand value)."""
    rng = np.random.default_rng(7000 + seed)
    for _ in range(60):
        # a random triangle (cell 0) with one neighbour triangle on each edge
        p = rng.uniform(-1, 1, (3, 2)) + np.array([[0, 0], [3, 0], [1.5, 3]])
        ctr = p.mean(0)
        outer = []
        for k in range(3):
            a, b = p[k], p[(k + 1) % 3]
            mid = 0.5 * (a + b)
            outer.append(mid + (mid - ctr) * rng.uniform(0.6, 1.4))
        node_xy = np.vstack([p, np.array(outer)])
        tri = np.array([[0, 1, 2], [1, 0, 3], [2, 1, 4], [0, 2, 5]], dtype=np.int32)
        from workloads import mesh as M
        tri = M.orient_ccw(node_xy, tri).astype(np.int32)
        ec, ce = M.build_edge_tables(tri, 6)
        zb = rng.uniform(-0.1, 0.1, 4)
        h = rng.uniform(0.25, 2.0, 4)
        if rng.uniform() < 0.4:
            j = rng.integers(1, 4)
            h[j] = 0.0                                   # a dry neighbour...
            zb[j] = zb[0] + h[0] * rng.uniform(0.1, 0.9)  # ...whose bed lies between cell 0's bed and surface
        u = rng.uniform(-2, 2, 4)
        v = rng.uniform(-2, 2, 4)
        u[h == 0] = 0
        v[h == 0] = 0
        w4 = C.Workload("stencil", node_xy, tri, ec, ce, zb, np.full(4, np.inf), h, h * u, h * v)
        s = ref.RefSolver(w4)
        dt = 1e-4
        area, nx, ny, ln = s.geometry()
        h0 = h.copy()
        info = s.step(n_steps=1, t_end=dt, cfl=1e9)      # dt forced to t_end
        assert abs(info["dt_last"] - dt) < 1e-18
        h1, hu1, hv1 = s.get_state()
        inc_oracle = np.array([h1[0] - h0[0], hu1[0] - h0[0] * u[0], hv1[0] - h0[0] * v[0]]) / dt
        # literal H-form for cell 0
        nbrs, normals, lens = [], [], []
        for k in range(3):
            e = ce[0, k]
            Lc, Rc = ec[e]
            other = Rc if Lc == 0 else Lc
            sgn = 1.0 if Lc == 0 else -1.0
            nbrs.append((h[other], u[other], v[other], zb[other]))
            normals.append((sgn * nx[e], sgn * ny[e]))
            lens.append(ln[e])
        inc_H = h_form_increment(G, (h[0], u[0], v[0], zb[0]), nbrs, normals, lens, area[0])
        scale = G * 4.0 * np.sum(lens) / area[0]
        assert np.all(np.abs(inc_oracle - inc_H) < 1e-9 * scale), (inc_oracle, inc_H)
