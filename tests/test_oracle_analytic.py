"""System-level pins of the oracle: analytic dam breaks (Ritter, Stoker), the two-rarefaction problem of
the paper's T5, lake at rest, mass conservation, steady uniform flow, permutation
invariance and the printed rest depth of T6.  CPU only."""
import os

import numpy as np
import pytest
from scipy.optimize import brentq

from workloads import configs as C
from workloads import mesh as M

G = 9.81
HERE = os.path.dirname(os.path.abspath(__file__))


def golden(name):
    out = {}
    with open(os.path.join(HERE, "golden", name)) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            k, v = line.split()[:2]
            out[k] = float(v)
    return out


# ------------------------------------------------------------------------------------------ Ritter
def ritter(x, t, h0=1.0, x0=50.0):
    c0 = np.sqrt(G * h0)
    xi = (x - x0) / t
    h = np.where(xi < -c0, h0, np.where(xi > 2 * c0, 0.0, (2 * c0 - xi) ** 2 / (9 * G)))
    u = np.where((xi > -c0) & (xi < 2 * c0), 2.0 / 3.0 * (c0 + xi), 0.0)
    return h, u


def test_ritter_constants_golden():
    g = golden("analytic_dam_break.txt")
    c0 = np.sqrt(G)
    assert abs(c0 - g["ritter_c0"]) < 5e-9
    assert abs(50 - 4 * c0 - g["ritter_tail_x"]) < 5e-5 and abs(50 + 8 * c0 - g["ritter_front_x"]) < 5e-5
    assert abs(8.0 / 27.0 * c0 - g["ritter_q_dam"]) < 5e-7


@pytest.mark.slow
def test_ritter_convergence(ref):
    """SURVEY O-4 / BASELINE configs[0]: L1(h), L1(hu) fall under refinement with observed order in
    [0.5, 1.1]; volume conserved; nothing clipped beyond round-off; CFL 0.9."""
    errs_h, errs_q, dxs = [], [], []
    for refine in (0.25, 0.5, 1.0, 2.0):
        w = C.config1(refine=refine)
        s = ref.RefSolver(w)
        area = s.geometry()[0]
        v0 = (w.h * area).sum()
        info = s.step(t_end=4.0, cfl=0.9)
        assert info["t"] == 4.0 and info["flags"] == 0
        h, hu, hv = s.get_state()
        x = M.centroids(w.node_xy, w.tri)[:, 0]
        he, ue = ritter(x, 4.0)
        errs_h.append(float((np.abs(h - he) * area).sum() / area.sum()))
        errs_q.append(float((np.abs(hu - he * ue) * area).sum() / area.sum()))
        dxs.append(100.0 / w.meta["nx"])
        assert abs(info["vol"] - v0) < 1e-13 * v0 * 10
        assert info["vol_clipped"] < 1e-12 * v0
        if refine == 1.0:
            # bulk of the wave: where the exact depth is 0.05 m the computed depth is within 2 cells' reach
            i_lvl = np.argmin(np.abs(he - 0.05))
            x_num = x[(h > 0.05)].max()
            assert abs(x_num - x[i_lvl]) < 2.5
            # dam section: h = 4/9, q = 8/27 c0 h0 (constant in time)
            m = np.abs(x - 50.0) < 0.15
            assert abs(h[m].mean() - 4.0 / 9.0) < 0.02 and abs(hu[m].mean() - 8.0 / 27.0 * np.sqrt(G)) < 0.02
    assert all(b < a for a, b in zip(errs_h, errs_h[1:])), errs_h
    assert all(b < a for a, b in zip(errs_q, errs_q[1:])), errs_q
    order_h = np.polyfit(np.log(dxs), np.log(errs_h), 1)[0]
    order_q = np.polyfit(np.log(dxs), np.log(errs_q), 1)[0]
    assert 0.5 <= order_h <= 1.1 and 0.5 <= order_q <= 1.1, (order_h, order_q)


# ------------------------------------------------------------------------------------------ Stoker
def stoker(hL, hR):
    cL = np.sqrt(G * hL)
    f = lambda hm: 2 * (cL - np.sqrt(G * hm)) - (hm - hR) * np.sqrt(G * (hm + hR) / (2 * hm * hR))
    hm = brentq(f, hR * (1 + 1e-12), hL)
    um = 2 * (cL - np.sqrt(G * hm))
    S = hm * um / (hm - hR)
    return hm, um, S


def test_stoker_constants_golden():
    g = golden("analytic_dam_break.txt")
    for tag, hL, hR in (("a", 1.0, 0.1), ("b", 10.0, 1.0), ("c", 1.0, 0.5)):
        hm, um, S = stoker(hL, hR)
        assert abs(hm - g[f"stoker_{tag}_hm"]) < 5e-8 * hL
        assert abs(um - g[f"stoker_{tag}_um"]) < 5e-8 * 10
        assert abs(S - g[f"stoker_{tag}_S"]) < 5e-8 * 10


@pytest.mark.parametrize("hR", [0.1, 0.5])
def test_stoker_plateau_and_shock(ref, hR):
    """SURVEY O-5: plateau (h_m, u_m) within 1 %, shock within 2 cells of S t on the 500x4 mesh, CFL 0.9."""
    hm, um, S = stoker(1.0, hR)
    w = C.dam_break_channel(h_right=hR)
    s = ref.RefSolver(w)
    info = s.step(t_end=4.0, cfl=0.9)
    h, hu, hv = s.get_state()
    x = M.centroids(w.node_xy, w.tri)[:, 0]
    # plateau between the fan head (x0 + (um - cm) t) and the shock (x0 + S t)
    cm = np.sqrt(G * hm)
    lo, hi = 50 + (um - cm) * 4 + 2.0, 50 + S * 4 - 2.0
    m = (x > lo) & (x < hi)
    assert abs(h[m].mean() - hm) < 0.01 * hm
    assert abs((hu[m] / h[m]).mean() - um) < 0.01 * um
    # shock position: where h crosses the mean of plateau and downstream depth
    lvl = 0.5 * (hm + hR)
    x_shock = x[h > lvl].max()
    assert abs(x_shock - (50 + S * 4)) < 2 * 0.2 + 0.2
    assert info["vol_clipped"] == 0.0


def test_two_rarefactions_t5(ref):
    """Hydrodynamic half of T5 (Eq. 22): h = 1, q = -/+ 3, transparent ends, CFL 0.95,
    t = 2.5 s.  Exact (Toro ch. 10): middle state u* = 0, c* = c0 - 1.5, h* = c*^2/g = 0.2715 m."""
    w = C.dam_break_channel(nx=681, ny=1, lx=100.0, ly=0.1, h_left=1.0, h_right=1.0, q_left=-3.0, q_right=3.0,
                            transmissive_ends=True, t_end=2.5, cfl=0.95)
    assert w.n_cells == 1362                       # the paper's cell count
    s = ref.RefSolver(w)
    info = s.step(t_end=2.5, cfl=0.95)
    h, hu, hv = s.get_state()
    x = M.centroids(w.node_xy, w.tri)[:, 0]
    c0 = np.sqrt(G)
    cstar = c0 - 1.5
    hstar = cstar ** 2 / G
    assert abs(hstar - 0.2715) < 1e-4
    m = np.abs(x - 50.0) < 0.6 * cstar * 2.5          # inside the middle state (tails at +-c* t)
    assert abs(h[m].mean() - hstar) < 0.03 * hstar + 0.01
    # exact fan: left rarefaction between x0 + (-3 - c0) t and x0 - c* t :  u - 2c = -3 - 2 c0 ... check L1
    xi = (x - 50.0) / 2.5
    he = np.where(np.abs(xi) < cstar, hstar,
                  np.where(np.abs(xi) < 3 + c0, ((np.abs(xi) - 3 + 2 * c0) / 3.0) ** 2 / G, 1.0))
    assert np.abs(h - he).mean() < 0.01
    assert info["vol_clipped"] == 0.0


# ------------------------------------------------------------------------------------------ invariants
@pytest.mark.slow
def test_lake_at_rest_config2(ref):
    """SURVEY O-6 / BASELINE configs[1]: 1000 steps, |u|,|v| <= 1e-12, volume drift <= 1e-13, mask unchanged."""
    w = C.config2()
    assert 75000 < w.n_cells <= 80000 and np.any(w.h == 0.0)
    s = ref.RefSolver(w)
    area = s.geometry()[0]
    v0 = (w.h * area).sum()
    wet0 = w.h > w.h_dry
    umax = 0.0
    for _ in range(4):
        info = s.step(n_steps=250)
        h, hu, hv = s.get_state()
        wet = h > w.h_dry
        assert np.array_equal(wet, wet0)
        umax = max(umax, np.abs(hu[wet] / h[wet]).max(), np.abs(hv[wet] / h[wet]).max())
    assert info["steps_done"] == 1000
    assert umax <= 1e-12, umax
    assert abs(info["vol"] - v0) <= 1e-13 * v0
    assert np.abs(h - w.h).max() <= 1e-13 * 2.0
    assert info["vol_clipped"] == 0.0


def test_mass_closed_box_with_friction(ref):
    """SURVEY O-7: closed channel, several wall reflections, k = 30: volume conserved to round-off."""
    w = C.dam_break_channel(nx=125, ny=1, h_right=0.0, kst=30.0)
    s = ref.RefSolver(w)
    area = s.geometry()[0]
    v0 = (w.h * area).sum()
    info = s.step(t_end=60.0, cfl=0.9)
    assert info["t"] == 60.0
    assert abs(info["vol"] - v0) <= 1e-13 * v0 * 20
    assert info["vol_clipped"] <= 1e-13 * v0
    h, hu, hv = s.get_state()
    assert h.min() >= 0.0 and np.isfinite(hu).all()


@pytest.mark.parametrize("case", ["config3", "config4-strings"])
def test_permutation_invariance(ref, case):
    """SURVEY O-9 / R-15: renumbering cells and edges (slot order, L/R and the order of boundary-string members
    kept) leaves the result bit-identical."""
    w = C.config3(target_cells=3000, lx=110.0) if case == "config3" else C.by_id(4, 0.002)
    wp, cp = w.permuted(seed=3)
    a, b = ref.RefSolver(w), ref.RefSolver(wp)
    ia, ib = a.step(n_steps=40), b.step(n_steps=40)
    assert ia["t"] == ib["t"] and ia["dt_last"] == ib["dt_last"]
    for x, y in zip(a.get_state(), b.get_state()):
        assert np.array_equal(x[cp], y)


@pytest.mark.slow
def test_uniform_flow_normal_depth(ref):
    """SURVEY O-8: sloped prismatic channel, INFLOW_Q + OUTFLOW_UNIFORM: steady depth = (q/(k sqrt(S0)))^(3/5)
    (Strickler/Manning uniform flow; Eq. 2 + Table 1), and the volume balance closes."""
    w = C.uniform_flow_channel()
    hn = (w.meta["q"] / (w.meta["kst"] * np.sqrt(w.meta["slope"]))) ** 0.6
    assert abs(hn - 1.5644) < 1e-4
    w.h[:] = hn * 0.9                      # start off the steady state; the transient leaves a slowly
    s = ref.RefSolver(w)                    # damped long wave, so the pin uses the median over the reach
    area = s.geometry()[0]
    v0 = (w.h * area).sum()
    # CFL 0.7: on this regular right-triangle mesh the first-order scheme with Eq. 21's rho = 4A/(3l) is
    # linearly stable only up to CFL ~ 0.75 (R-7 note); the pin is about friction + boundaries.
    info = s.step(t_end=3000.0, cfl=0.7)
    h, hu, hv = s.get_state()
    x = M.centroids(w.node_xy, w.tri)[:, 0]
    mid = (x > 250.0) & (x < 750.0)
    assert abs(np.median(h[mid]) - hn) < 0.005 * hn
    assert np.abs(h[mid] - hn).max() < 0.05 * hn
    assert abs(np.median(hu[mid]) - w.meta["q"]) < 0.01 * w.meta["q"]
    bal = info["vol"] - v0 - info["vol_in"] + info["vol_out"] - info["vol_clipped"]
    assert abs(bal) < 1e-9 * v0
    # the outlet holds normal depth too (R-12)
    out = x > 990.0
    assert np.abs(h[out] - hn).max() < 0.05 * hn
    # started exactly at normal depth, the state stays there (steady solution of scheme + both boundaries)
    w.h[:] = hn
    s = ref.RefSolver(w)
    s.step(t_end=500.0, cfl=0.7)
    h = s.get_state()[0]
    assert np.abs(h - hn).max() < 0.01 * hn


def test_t6_rest_level(ref):
    """PAPER.md:591 prints the rest depth h = 0.364 m for T6.  With Eq. 24's 'h' read as surface elevation
    over the bed of Eq. 23 (DESIGN R-18), the closed-domain volume fixes the rest level by volume balance;
    the oracle's volume (sum h |Omega|) is the one used."""
    w = C.t6_cones(spacing=0.25)
    s = ref.RefSolver(w)
    info = s.step(n_steps=0)
    vol = info["vol"]
    assert abs(vol - 619.35) < 0.01 * 619.35
    # rest level L solves integral max(0, L - eta) dA = vol over the same discrete bed
    area = s.geometry()[0]
    f = lambda L: (np.maximum(0.0, L - w.zb) * area).sum() - vol
    L = brentq(f, 0.1, 1.0)
    assert abs(L - 0.364) < 1.5e-3


def test_config1_noise_at_cfl_09_and_07(ref):
    """DESIGN R-7 / R-8b in numbers: on the structured split-quad mesh of B:configs[0] the literal Eq. 21 time step at the
    paper's default CFL 0.9 leaves transverse noise in the 1-D dam break (the thin fast precursor film ahead of the front;
    the scheme is linearly stable only up to CFL ~0.75 on regular right triangles), bounded but visible: transverse
    momentum up to ~9 % of the longitudinal one and 0.05 m of depth spread across the 8 triangles of a column, against
    0.9 % at CFL 0.7.  The pin keeps both numbers from growing unnoticed."""
    w = C.config1()
    x = M.centroids(w.node_xy, w.tri)[:, 0]
    cols = np.floor(x / 0.2).astype(int)
    out = {}
    for cfl in (0.9, 0.7):
        s = ref.RefSolver(w)
        info = s.step(t_end=4.0, cfl=cfl)
        h, hu, hv = s.get_state()
        spread = np.array([np.ptp(h[cols == c]) for c in range(500)])
        out[cfl] = (np.abs(hv).max() / np.abs(hu).max(), spread.max(), info["vol_clipped"])
        assert np.all(np.isfinite(h)) and info["vol_clipped"] < 1e-15
    assert out[0.9][0] < 0.15 and out[0.9][1] < 0.06
    assert out[0.7][0] < 0.02 and out[0.7][1] < 0.03
    assert out[0.7][0] < 0.25 * out[0.9][0]
