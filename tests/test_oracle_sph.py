"""Pins for the oracle's neighbour sets, kernel, density/h iteration, forces, timestep and leapfrog -- CPU only.

Nothing here re-types the oracle's formulas to compare them with themselves: the checks are brute force written
independently in NumPy, closed forms, invariants (conservation identities, Galilean invariance, unique root of
the h equation), the lattice constants of tests/golden/lattice_constants.txt and the exact Riemann solution.
"""
import math
import os

import numpy as np
import pytest

import oracle as O
from paper_2503_09713_b200 import workloads as W

GOLD = os.path.join(os.path.dirname(__file__), "golden")


# ---------------------------------------------------------------- neighbour sets (O5)

def _numpy_sets(pos, h, L, periodic, chi):
    d = pos[:, :, None] - pos[:, None, :]
    for c in range(3):
        if periodic[c]:
            d[c] = np.where(d[c] > 0.5 * L[c], d[c] - L[c], np.where(d[c] < -0.5 * L[c], d[c] + L[c], d[c]))
    d2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2]
    rc = 2.0 * chi * np.maximum(h[:, None], h[None, :])
    return d2 < rc * rc


@pytest.mark.parametrize("periodic", [True, False])
def test_neighbours_brute_vs_numpy(periodic):
    w = W.random_cloud(700, seed=11, periodic=periodic)
    box = O.make_box(w.box_lo, w.box_hi, w.periodic)
    offs, idx = O.neighbours(w.pos, w.h0, box, 1.1, "brute")
    adj = _numpy_sets(w.pos, w.h0, (1.0, 1.0, 1.0), w.periodic, 1.1)
    assert offs[-1] == adj.sum()
    for a in range(w.n):
        assert np.array_equal(idx[offs[a]:offs[a + 1]], np.nonzero(adj[a])[0])
    assert np.array_equal(adj, adj.T)  # symmetric criterion
    assert np.all(np.diag(adj))  # self included


@pytest.mark.parametrize("make", [lambda: W.config(0), lambda: W.random_cloud(4096, seed=2),
                                  lambda: W.random_cloud(3000, seed=4, periodic=False),
                                  lambda: W.sod(16, 12)])
def test_neighbours_grid_equals_brute(make):
    w = make()
    box = O.make_box(w.box_lo, w.box_hi, w.periodic)
    ob, ib = O.neighbours(w.pos, w.h0, box, 1.1, "brute")
    og, ig = O.neighbours(w.pos, w.h0, box, 1.1, "grid")
    assert np.array_equal(ob, og) and np.array_equal(ib, ig)


def test_neighbour_counts_lattice_and_continuum():
    """PAPER.md:101 (~60 neighbours for M4, h_fact = 1.2); exact lattice counts from the golden file."""
    gold = dict(l.split()[:2] for l in open(os.path.join(GOLD, "lattice_constants.txt")) if not l.startswith("#"))
    w = W.cube(10, jitter=0.0, vel_amp=0.0)
    box = O.make_box(w.box_lo, w.box_hi, w.periodic)
    for chi, key in ((1.0, "neighbours_chi_1.0"), (1.1, "neighbours_chi_1.1")):
        offs, _ = O.neighbours(w.pos, w.h0, box, chi, "brute")
        assert np.all(np.diff(offs) == int(gold[key]))
    w = W.cube(16, jitter=0.3, vel_amp=0.0, seed=5)
    offs, _ = O.neighbours(w.pos, w.h0, box, 1.1, "grid")
    assert abs(np.diff(offs).mean() - 4.0 / 3.0 * math.pi * (2 * 1.2 * 1.1) ** 3) < 1.0


def test_group_criterion_is_conservative():
    """E8 hierarchy: if any particle of a tree node interacts with a, then
    r_a lies in the node box extended by R_kern * chi * max(hmax_node, h_a) (non-periodic case)."""
    w = W.random_cloud(400, seed=8, periodic=False)
    box = O.make_box(w.box_lo, w.box_hi, w.periodic)
    skey, perm = O.sort_keys(O.morton_keys(w.pos, box))
    ps, hs = w.pos[:, perm], w.h0[perm]
    t = O.tree(skey)
    box6, hmax = O.aabb(t, ps, hs)
    adj = _numpy_sets(ps, hs, (1, 1, 1), (0, 0, 0), 1.1)
    for i in range(w.n - 1):
        inter = adj[:, t["rlo"][i]:t["rhi"][i] + 1].any(axis=1)
        ext = 2.0 * 1.1 * np.maximum(hmax[i], hs)
        inside = np.all((ps >= box6[i, :3, None] - ext) & (ps <= box6[i, 3:, None] + ext), axis=0)
        assert np.all(inside[inter])


# ---------------------------------------------------------------- kernel (O6)

@pytest.mark.parametrize("kernel,radius,f0,cnorm", [(0, 2.0, 1.0, 1.0 / math.pi), (1, 2.5, 14.375, 1.0 / (20.0 * math.pi)),
                                                     (2, 3.0, 66.0, 1.0 / (120.0 * math.pi)),
                                                     (3, 2.0, 1.0, 21.0 / (16.0 * math.pi)), (4, 2.0, 1.0, 495.0 / (256.0 * math.pi)),
                                                     (5, 2.0, 1.0, 1365.0 / (512.0 * math.pi))],
                         ids=["M4", "M5", "M6", "WendlandC2", "WendlandC4", "WendlandC6"])
def test_kernel_closed_forms(kernel, radius, f0, cnorm):
    """B-spline kernels M4, M5, M6 and Wendland functions C2, C4, C6: unit volume integral (pins the 3-D normalisations 1/pi, 1/(20 pi),
    1/(120 pi)), closed-form central values (1, 115/8, 66), compact support, continuity of f and f' at the knots,
    F and dW/dh against finite differences of W."""
    L = O.lib()
    O.set_kernel(kernel)
    try:
        r = np.linspace(0.0, radius, 300001)
        f = np.array([L.orc_f(q) for q in r])
        assert abs(np.trapezoid(4.0 * math.pi * r * r * f * cnorm, r) - 1.0) < 1e-9           # int W dV with h = 1
        assert L.orc_W(0.0, 0.7) == pytest.approx(f0 * cnorm / 0.7 ** 3, rel=1e-15)
        for q in np.arange(radius, 0.0, -1.0):
            assert L.orc_f(q - 1e-12) == pytest.approx(L.orc_f(q + 1e-12), abs=1e-9)
            assert L.orc_df(q - 1e-12) == pytest.approx(L.orc_df(q + 1e-12), abs=1e-9)
        assert L.orc_f(radius + 0.5) == 0.0 and L.orc_df(radius + 0.5) == 0.0 and L.orc_f(radius - 1e-3) > 0.0
        for rr, h in ((0.3, 0.5), (0.7, 0.5), (0.2, 1.3)):
            eps = 1e-6
            assert L.orc_F(rr, h) == pytest.approx((L.orc_W(rr + eps, h) - L.orc_W(rr - eps, h)) / (2 * eps), rel=1e-7)
            assert L.orc_dWdh(rr, h) == pytest.approx((L.orc_W(rr, h + eps) - L.orc_W(rr, h - eps)) / (2 * eps), rel=1e-7)
        assert all(L.orc_df(q) < 0 for q in (0.25, 0.75, 1.5, radius - 0.2)) and L.orc_df(0.0) == 0.0
    finally:
        O.set_kernel(0)


def test_m6_lattice_and_conservation():
    """M6 with h_fact = 1.0 (the paper's physics-test setting: ~113 neighbours): uniform density on a
    lattice, h from the unique-root bisection, momentum and energy identities."""
    w = W.cube(10, jitter=0.03, vel_amp=0.05, seed=4)
    w.hfact, w.kernel = 1.0, 2
    w.h0 = np.full(w.n, 1.0 / 10)
    box, p = O.workload_box_params(w)
    ev = O.evaluate(w.pos, w.vel, w.mass, w.u, w.h0, box, p, "brute")
    assert 105 < ev["n_neigh"] / w.n < 160 and abs(ev["rho"].mean() - 1.0) < 2e-3
    hb = O.h_bisect(w.pos, w.mass, box, p.hfact, 0.5 * ev["h"], 2.0 * ev["h"], kernel=2)
    assert np.max(np.abs(hb / ev["h"] - 1)) < 1e-6
    ma = (w.mass * ev["acc"]).sum(axis=1)
    assert np.all(np.abs(ma) < 1e-13 * np.abs(w.mass * ev["acc"]).sum(axis=1).max())
    de = (w.mass * ((w.vel * ev["acc"]).sum(axis=0) + ev["dudt"])).sum()
    assert abs(de) < 1e-12 * (w.mass * np.abs(ev["dudt"])).sum()
    O.set_kernel(0)


# ---------------------------------------------------------------- density / h (O7)

def test_lattice_constants():
    gold = {l.split()[0]: l.split()[1:] for l in open(os.path.join(GOLD, "lattice_constants.txt"))
            if not l.startswith("#")}
    for n_side in (10, 12):
        w = W.cube(n_side, jitter=0.0, vel_amp=0.0)
        box, p = O.workload_box_params(w)
        ev = O.evaluate(w.pos, w.vel, w.mass, w.u, w.h0, box, p, "grid")
        rho0 = 1.0
        assert np.ptp(ev["rho"]) < 1e-13 and np.ptp(ev["h"]) < 1e-14
        assert abs(ev["rho"][0] / rho0 - 1 - float(gold["rho_over_rho0_minus_1"][0])) < float(gold["rho_over_rho0_minus_1"][2])
        assert abs(ev["h"][0] * n_side - float(gold["h_over_spacing"][0])) < float(gold["h_over_spacing"][2])
        assert abs(ev["omega"][0] - float(gold["omega"][0])) < float(gold["omega"][2])
        assert ev["restarts"] == 0
        assert np.abs(ev["acc"]).max() < 1e-12 * ev["rho"][0] * (2.0 / 3.0) * n_side  # symmetric cancellation


@pytest.mark.parametrize("make", [lambda: W.cube(8, jitter=0.2, vel_amp=0.0, seed=9),
                                  lambda: W.random_cloud(500, seed=6)])
def test_h_is_the_unique_root_bisection(make):
    """Reading A5b: h_a is the unique root of g_a(h) = sum_b m_b C f(r/h) - m_a hfact^3."""
    w = make()
    box, p = O.workload_box_params(w)
    ev = O.evaluate(w.pos, w.vel, w.mass, w.u, w.h0, box, p, "grid")
    hb = O.h_bisect(w.pos, w.mass, box, w.hfact, 0.2 * ev["h"], 5.0 * ev["h"])
    # Newton stops at |dh|/h <= 1e-6 and converges quadratically: the result is far inside 1e-10
    assert np.max(np.abs(ev["h"] / hb - 1.0)) < 1e-10
    assert np.all(ev["h"] > 0)
    # rho is F1 evaluated at h
    assert np.allclose(ev["rho"], w.mass * (w.hfact / ev["h"]) ** 3, rtol=1e-15)


def test_newton_literal_vs_exact_derivative():
    """Reading A5: Alg. 7 line 9 as printed (3 rho_sum / h) and the exact derivative share the fixed point."""
    w = W.cube(10, jitter=0.1, vel_amp=0.0, seed=2)
    box, p = O.workload_box_params(w)
    box, pl = O.workload_box_params(w, newton_literal=1)
    a = O.evaluate(w.pos, w.vel, w.mass, w.u, w.h0, box, p, "grid")
    b = O.evaluate(w.pos, w.vel, w.mass, w.u, w.h0, box, pl, "grid")
    assert np.max(np.abs(a["h"] / b["h"] - 1)) < 1e-10


def test_chi_restart_and_clamp():
    """h may grow by at most chi per pass; a too-small guess triggers restarts and still converges
    to the same root; h stays positive."""
    w = W.cube(8, jitter=0.1, vel_amp=0.0, seed=4)
    box, p = O.workload_box_params(w)
    good = O.evaluate(w.pos, w.vel, w.mass, w.u, w.h0, box, p, "grid")
    small = O.evaluate(w.pos, w.vel, w.mass, w.u, 0.7 * w.h0, box, p, "grid")
    assert good["restarts"] == 0 and small["restarts"] >= 3
    assert np.max(np.abs(small["h"] / good["h"] - 1)) < 1e-10
    offs, idx = O.neighbours(w.pos, 0.7 * w.h0, box, 1.1, "grid")
    one = O.density(w.pos, w.mass, 0.7 * w.h0, offs, idx, box, p)
    assert one["n_exceeded"] > 0
    assert np.all(one["h"] <= 0.7 * w.h0 * 1.1 * (1 + 1e-15))
    assert np.all(one["h"][one["exceeded"] == 1] == (0.7 * w.h0 * 1.1)[one["exceeded"] == 1])


# ---------------------------------------------------------------- forces / dt (O8, O9)

def _random_state(n_side=9, seed=7):
    w = W.cube(n_side, jitter=0.15, vel_amp=0.0, seed=seed)
    idx = np.arange(w.n, dtype=np.uint64)
    w.vel = np.stack([0.6 * (W.splitmix_u01(seed + 10, idx, k) - 0.5) for k in range(3)])
    w.u = 0.5 + W.splitmix_u01(seed + 11, idx, 0)
    return w


def test_momentum_and_energy_identities():
    """momentum to machine precision; sum m (v.a + du/dt) = 0 fixes the sign garble G1 and G2."""
    w = _random_state()
    box, p = O.workload_box_params(w)
    ev = O.evaluate(w.pos, w.vel, w.mass, w.u, w.h0, box, p, "grid")
    acc, du = ev["acc"], ev["dudt"]
    amax = np.abs(acc).max()
    assert np.all(np.abs((w.mass * acc).sum(axis=1)) < 1e-14 * amax)
    de = (w.mass * ((w.vel * acc).sum(axis=0) + du)).sum()
    assert abs(de) < 1e-13 * (w.mass * np.abs(du)).sum()
    # flipping the sign of a (the equation as extracted, without the minus) breaks the identity at O(1)
    de_wrong = (w.mass * (-(w.vel * acc).sum(axis=0) + du)).sum()
    assert abs(de_wrong) > 0.1 * (w.mass * np.abs(du)).sum()


def test_galilean_invariance():
    """a and du/dt depend on velocity differences only."""
    w = _random_state(seed=3)
    box, p = O.workload_box_params(w)
    a = O.evaluate(w.pos, w.vel, w.mass, w.u, w.h0, box, p, "grid")
    b = O.evaluate(w.pos, w.vel + np.array([[3.0], [-2.0], [1.0]]), w.mass, w.u, w.h0, box, p, "grid")
    assert np.max(np.abs(a["acc"] - b["acc"])) < 1e-12 * np.abs(a["acc"]).max()
    assert np.max(np.abs(a["dudt"] - b["dudt"])) < 1e-12 * np.abs(a["dudt"]).max()
    assert a["dt"] == pytest.approx(b["dt"], rel=1e-12)


def test_pressure_pushes_outwards_and_conduction_cools():
    w = W.cube(10, jitter=0.0, vel_amp=0.0)
    c = w.pos - 0.5
    r = np.sqrt((c * c).sum(axis=0))
    w.u = 1.0 + 4.0 * np.exp(-(r / 0.15) ** 2)
    box, p = O.workload_box_params(w)
    ev = O.evaluate(w.pos, w.vel, w.mass, w.u, w.h0, box, p, "grid")
    shell = (r > 0.1) & (r < 0.25)
    assert np.all((ev["acc"] * c).sum(axis=0)[shell] > 0)          # high -> low pressure
    box, p0 = O.workload_box_params(w, beta_u=0.0)
    ev0 = O.evaluate(w.pos, w.vel, w.mass, w.u, w.h0, box, p0, "grid")
    assert np.all(ev0["dudt"] == 0.0)                              # v = 0: only conduction changes u
    hot = r < 0.08
    assert np.all(ev["dudt"][hot] < 0)                             # u_a > u_b => Lambda_cond cools a


def test_viscosity_only_for_approaching_pairs():
    """Eq. 5: q = 0 when v_ab.r_ab >= 0; compression heats, and AV is dissipative."""
    w = W.cube(8, jitter=0.0, vel_amp=0.0)
    box, p = O.workload_box_params(w, beta_u=0.0)
    wexp = np.array(w.vel)
    wexp[0] = 0.3 * np.sin(2 * math.pi * w.pos[0])
    ev_av = O.evaluate(w.pos, wexp, w.mass, w.u, w.h0, box, p, "grid")
    box, pn = O.workload_box_params(w, beta_u=0.0, alpha_av=0.0, beta_av=0.0)
    ev_no = O.evaluate(w.pos, wexp, w.mass, w.u, w.h0, box, pn, "grid")
    comp = np.abs(w.pos[0] - 0.5) < 0.1      # dv/dx < 0: converging
    expa = (w.pos[0] < 0.1) | (w.pos[0] > 0.9)  # diverging
    assert np.all(ev_av["dudt"][comp] > ev_no["dudt"][comp])
    assert np.allclose(ev_av["dudt"][expa], ev_no["dudt"][expa], rtol=1e-12, atol=1e-15)


def test_cfl_timestep_definition():
    """G8 on a static uniform lattice: a = 0, so dt = C_cour h / c_s."""
    w = W.cube(10, jitter=0.0, vel_amp=0.0)
    box, p = O.workload_box_params(w)
    ev = O.evaluate(w.pos, w.vel, w.mass, w.u, w.h0, box, p, "grid")
    cs = math.sqrt(w.gamma * (w.gamma - 1.0) * 1.0)
    assert ev["dt"] == pytest.approx(0.3 * ev["h"][0] / cs, rel=1e-10)


def test_point_mass_and_isothermal_eos():
    """BASELINE config 3 switches: a_ext = -GM d/(d^2+eps^2)^(3/2); du/dt = 0; P = cs(R)^2 rho."""
    w = W.disc(3000, seed=1)
    box, p = O.workload_box_params(w)
    box, p_nogm = O.workload_box_params(w)
    p_nogm.GM = 0.0
    a = O.evaluate(w.pos, w.vel, w.mass, w.u, w.h0, box, p, "grid")
    b = O.evaluate(w.pos, w.vel, w.mass, w.u, w.h0, box, p_nogm, "grid")
    d2 = (w.pos ** 2).sum(axis=0) + 0.01
    assert np.allclose(a["acc"] - b["acc"], -w.pos / d2 ** 1.5, rtol=1e-9, atol=1e-12)
    assert np.all(a["dudt"] == 0.0)
    assert a["restarts"] >= 1 and np.all(a["h"] > 0)


# ---------------------------------------------------------------- leapfrog (O10)

def _energy(s):
    return float((s.m * (0.5 * (s.vel ** 2).sum(axis=0) + s.u)).sum())


def test_energy_and_momentum_over_10_steps():
    """PAPER.md:208 (energy drift <= 1e-6 relative in the paper's M6 tests; momentum to machine precision).
    With M4, constant alpha and the default CFL the drift observed here over 10 steps is ~5e-6 (DESIGN.md
    "Readings"); the pin is the bound 1e-5, the dt^2 convergence of the drift on a smooth problem, and exact
    momentum conservation."""
    drift = {}
    for f, n in ((1.0, 10), (0.5, 20), (0.25, 40)):
        w = W.cube(10, jitter=0.0, vel_amp=0.05, seed=1)
        s = O.State(w, "grid")
        e0, p0 = _energy(s), (s.m * s.vel).sum(axis=1)
        dt = f * s.dt
        for _ in range(n):
            s.step(dt)
        drift[f] = abs(_energy(s) / e0 - 1)
        assert np.all(np.abs((s.m * s.vel).sum(axis=1) - p0) < 1e-15)
        assert np.all((s.pos >= 0) & (s.pos < 1))
    assert drift[1.0] < 1e-5
    assert drift[0.5] < drift[1.0] / 3 and drift[0.25] < drift[0.5] / 3
    w = W.cube(10, jitter=0.05, vel_amp=0.0, seed=1)          # C0-like noisy lattice, CFL dt
    s = O.State(w, "grid")
    e0 = _energy(s)
    for _ in range(10):
        s.step()
    assert abs(_energy(s) / e0 - 1) < 1e-5


def test_leapfrog_time_reversible():
    """KDK (G1-G5) with fixed dt is time-reversible when a depends on positions only: isothermal EOS
    (P = cs0^2 rho, du/dt = 0), no viscosity. (With the adiabatic EOS a depends on u, whose predictor uses the
    first-order v*, and exact reversibility is not expected.)"""
    w = W.cube(8, jitter=0.05, vel_amp=0.0, seed=3)
    w.vel[0] = 1e-2 * np.sin(2 * math.pi * w.pos[0])
    w.eos_isothermal = (1.0, 1.0, 0.0)
    s = O.State(w, "grid", alpha_av=0.0, beta_av=0.0, beta_u=0.0)
    pos0, vel0 = s.pos.copy(), s.vel.copy()
    dt = 0.5 * s.dt
    for _ in range(5):
        s.step(dt)
    assert np.max(np.abs(s.pos - pos0)) > 1e-5
    s.vel *= -1.0
    for _ in range(5):
        s.step(dt)
    assert np.max(np.abs(s.pos - pos0)) < 1e-12
    assert np.max(np.abs(-s.vel - vel0)) < 1e-10


# ---------------------------------------------------------------- Sod tube vs exact Riemann solution

def _riemann_exact(xi, gamma=1.4, left=(1.0, 0.0, 1.0), right=(0.125, 0.0, 0.1)):
    """Exact solution of the Riemann problem (two-rarefaction/shock pressure function, Newton on p*), sampled
    at xi = x/t. Textbook algorithm (e.g. Toro, ch. 4), restated here independently of the oracle."""
    rl, ul, pl = left
    rr, ur, pr = right
    g = gamma
    cl, cr = math.sqrt(g * pl / rl), math.sqrt(g * pr / rr)

    def fk(p, rk, pk, ck):
        if p > pk:
            A, B = 2.0 / ((g + 1) * rk), (g - 1) / (g + 1) * pk
            return (p - pk) * math.sqrt(A / (p + B)), math.sqrt(A / (p + B)) * (1 - 0.5 * (p - pk) / (B + p))
        return 2 * ck / (g - 1) * ((p / pk) ** ((g - 1) / (2 * g)) - 1), 1.0 / (rk * ck) * (p / pk) ** (-(g + 1) / (2 * g))

    p = 0.5 * (pl + pr)
    for _ in range(100):
        fl, dl = fk(p, rl, pl, cl)
        fr, dr = fk(p, rr, pr, cr)
        pn = max(1e-12, p - (fl + fr + ur - ul) / (dl + dr))
        if abs(pn - p) < 1e-14 * p:
            p = pn
            break
        p = pn
    us = 0.5 * (ul + ur) + 0.5 * (fk(p, rr, pr, cr)[0] - fk(p, rl, pl, cl)[0])
    rho = np.empty_like(xi)
    vel = np.empty_like(xi)
    prs = np.empty_like(xi)
    rls = rl * (p / pl) ** (1 / g)            # left rarefaction (p < pl for Sod)
    cls = cl * (p / pl) ** ((g - 1) / (2 * g))
    rrs = rr * ((p / pr + (g - 1) / (g + 1)) / ((g - 1) / (g + 1) * p / pr + 1))   # right shock
    S = ur + cr * math.sqrt((g + 1) / (2 * g) * p / pr + (g - 1) / (2 * g))
    for i, s in enumerate(xi):
        if s < ul - cl:
            rho[i], vel[i], prs[i] = rl, ul, pl
        elif s < us - cls:
            c = 2 / (g + 1) * (cl + (g - 1) / 2 * (ul - s))
            rho[i], vel[i], prs[i] = rl * (c / cl) ** (2 / (g - 1)), 2 / (g + 1) * (cl + (g - 1) / 2 * ul + s), pl * (c / cl) ** (2 * g / (g - 1))
        elif s < us:
            rho[i], vel[i], prs[i] = rls, us, p
        elif s < S:
            rho[i], vel[i], prs[i] = rrs, us, p
        else:
            rho[i], vel[i], prs[i] = rr, ur, pr
    return rho, vel, prs


@pytest.mark.slow
def test_sod_tube_against_exact_riemann():
    """PAPER.md:229 (Sod tube). The paper's L2 ~1e-3/1e-4 is for M6 + alpha switch + HCP at t/D ~ 100 spacings;
    an oracle-sized run (64x12x12 + 32x6x6, t = 0.1, i.e. t/D = 13 left spacings) leaves the star region between
    contact and shock under-resolved (about 3 h wide), so the pins are the quantities that do not depend on
    resolving it: the momentum budget (P_L - P_R) t per unit area (exact for a conservative scheme: fixes the
    sign and normalisation of Eq. 3), the rarefaction head/upper fan (EOS, sound speed), the undisturbed states,
    the shock position, and loose L1 norms against the exact solution."""
    w = W.sod(64, 12)
    s = O.State(w, "grid")
    t_end = 0.1
    while s.t < t_end - 1e-12:
        s.step(min(s.dt, t_end - s.t))
    x, xi = s.pos[0], s.pos[0] / s.t
    sel = np.abs(x) < 0.25                       # the discontinuity at x = 0 (the seam at +-1/2 mirrors it)
    area = (w.box_hi[1] - w.box_lo[1]) ** 2
    mom = (s.m * s.vel[0])[sel].sum() / area
    assert mom == pytest.approx((1.0 - 0.1) * s.t, rel=0.03)
    assert abs((s.m * s.vel[0]).sum()) < 1e-15   # the mirrored problem at the seam cancels it exactly
    rho_e, v_e, p_e = _riemann_exact(xi[sel])
    P = (w.gamma - 1) * s.rho * s.u
    fan = (xi[sel] > -1.05) & (xi[sel] < -0.8)
    assert np.max(np.abs(s.vel[0][sel][fan] - v_e[fan])) < 0.03
    assert np.max(np.abs(s.rho[sel][fan] - rho_e[fan])) < 0.03
    quiet = sel & ((xi < -1.45) | (xi > 2.3))
    assert np.abs(s.vel[0][quiet]).max() < 0.01
    assert np.all(s.vel[0][sel & (xi > -1.0) & (xi < 1.5)] > 0.05)       # gas flows from high to low pressure
    right = sel & (xi > 1.0)
    shock = xi[right][np.argmin(np.abs(s.rho[right] - 0.19))]            # exact: 1.7522
    assert 1.5 < shock < 2.0
    l1 = lambda a, b: np.mean(np.abs(a - b))
    assert l1(s.rho[sel], rho_e) < 0.04 and l1(s.vel[0][sel], v_e) < 0.06 and l1(P[sel], p_e) < 0.04
    assert np.abs(s.vel[1:]).max() < 0.01


def test_corrector_recycle_pins():
    """Leapfrog corrector check / re-cycle (G6-G7, reading A15) and CFL multiplier (G9-G10).
    Pins that do not restate the code: (i) with the check switched off, or a threshold nothing can reach, the step
    is bit-identical to the plain G1-G5 step; (ii) re-cycling is the fixed-point iteration of the implicit corrector
    v = v* + dt/2 (a(v) - a^n): the change between k and k+1 forced re-cycles shrinks geometrically; (iii) the
    multiplier halves after a step that re-cycled and relaxes as (1 + s m)/(1 + s) otherwise."""
    import oracle as O
    from paper_2503_09713_b200 import workloads as W
    w = W.sedov(12, cfl=0.3)

    def run(steps, **kw):
        s = O.State(w, "grid", **kw)
        out = []
        for _ in range(steps):
            s.step()
            out.append((s.recycles, s.cfl_mult))
        return s, out

    plain, _ = run(2)
    off, rec = run(2, eps_v=1e30)
    assert np.array_equal(plain.vel, off.vel) and np.array_equal(plain.u, off.u) and np.array_equal(plain.pos, off.pos)
    assert [r for r, _ in rec] == [0, 0] and rec[-1][1] == 1.0
    # (ii) force exactly k re-cycles in the first step
    vk = []
    for k in range(5):
        s, rec = run(1, eps_v=1e-300, max_recycle=k)
        assert rec[0][0] == k
        vk.append(s.vel.copy())
    d = [np.abs(vk[k + 1] - vk[k]).max() for k in range(4)]
    assert d[0] > 0 and all(d[k + 1] < 0.5 * d[k] for k in range(3))
    # (iii) multiplier
    s, rec = run(6, eps_v=1e-2, lambda_stiff=2.0)
    m = 1.0
    for r, mult in rec:
        m = 0.5 * m if r > 0 else (1.0 + 2.0 * m) / 3.0
        assert mult == pytest.approx(m, rel=1e-15)
    assert any(r > 0 for r, _ in rec) and any(r == 0 for r, _ in rec)


@pytest.mark.parametrize("kernel", [3, 4, 5], ids=["WendlandC2", "WendlandC4", "WendlandC6"])
def test_wendland_factored_derivative_lattice_and_conservation(kernel):
    """Wendland C2/C4/C6: f' in its factored closed form (-5 q t^3, -(7/3) q t^5 (2 + 5q),
    -(11/4) q t^7 (2 + 7q + 8q^2), t = 1 - q/2: f' <= 0 everywhere, zero at q = 0 and q = 2), near-uniform density on a
    jittered lattice, h from the unique-root bisection, momentum and energy identities."""
    L = O.lib()
    O.set_kernel(kernel)
    try:
        for q in np.linspace(0.0, 2.0, 41):
            t = 1.0 - 0.5 * q
            ref = {3: -5.0 * q * t ** 3, 4: -(7.0 / 3.0) * q * t ** 5 * (2.0 + 5.0 * q),
                   5: -2.75 * q * t ** 7 * (2.0 + 7.0 * q + 8.0 * q * q)}[kernel]
            assert L.orc_df(float(q)) == pytest.approx(ref, rel=1e-12, abs=1e-15)
        w = W.cube(10, jitter=0.03, vel_amp=0.05, seed=4)
        w.kernel = kernel
        box, p = O.workload_box_params(w)
        ev = O.evaluate(w.pos, w.vel, w.mass, w.u, w.h0, box, p, "brute")
        # the self term over-estimates rho at ~58 neighbours, more for the more peaked functions (C2 < C4 < C6)
        assert 0.0 < ev["rho"].mean() - 1.0 < (0.02, 0.03, 0.05)[kernel - 3] and ev["omega"].min() > 0.5
        hb = O.h_bisect(w.pos, w.mass, box, p.hfact, 0.5 * ev["h"], 2.0 * ev["h"], kernel=kernel)
        assert np.max(np.abs(hb / ev["h"] - 1)) < 1e-6
        ma = (w.mass * ev["acc"]).sum(axis=1)
        assert np.all(np.abs(ma) < 1e-13 * np.abs(w.mass * ev["acc"]).sum(axis=1).max())
        de = (w.mass * ((w.vel * ev["acc"]).sum(axis=0) + ev["dudt"])).sum()
        assert abs(de) < 1e-12 * (w.mass * np.abs(ev["dudt"])).sum()
    finally:
        O.set_kernel(0)
