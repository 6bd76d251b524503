"""Pins for the oracle's shock switch (G11-G13; reading A18 for alpha_loc and tau) -- CPU only.

What PAPER.md fixes is pinned against it: the implicit update G13 in closed form (decay on a quiescent lattice, instant
rise, limits dt -> 0 and dt -> infinity), the runscript constants and the recovery of the constant-
alpha scheme. What the reading adds (the gradient estimates behind alpha_loc) is pinned against analytic velocity fields,
and the whole against the Sod tube: alpha reaches alpha_max at the shock and stays small away from it.
"""
import math

import numpy as np
import pytest

import oracle as O
from paper_2503_09713_b200 import workloads as W


def _state(w, **kw):
    box, p = O.workload_box_params(w, av_switch=1, **kw)
    ev = O.evaluate(w.pos, w.vel, w.mass, w.u, w.h0, box, p, "grid")
    offs, idx = O.neighbours(w.pos, ev["h"], box, 1.0, "grid")     # any superset of the kernel support will do
    return box, p, ev, offs, idx


def test_constant_alpha_is_recovered():
    """alpha_a = alpha for every particle gives the constant-alpha forces of reading A10 bit for bit."""
    w = W.cube(9, jitter=0.15, vel_amp=0.0, seed=7)
    w.vel = np.stack([0.6 * (W.splitmix_u01(17, np.arange(w.n, dtype=np.uint64), k) - 0.5) for k in range(3)])
    box, p, ev, offs, idx = _state(w)
    a0 = O.forces(w.pos, w.vel, w.mass, ev["h"], ev["rho"], ev["omega"], w.u, offs, idx, box, p)
    a1 = O.forces(w.pos, w.vel, w.mass, ev["h"], ev["rho"], ev["omega"], w.u, offs, idx, box, p, alpha=np.full(w.n, 1.0))
    assert np.array_equal(a0[0], a1[0]) and np.array_equal(a0[1], a1[1]) and a0[2] == a1[2]
    a2 = O.forces(w.pos, w.vel, w.mass, ev["h"], ev["rho"], ev["omega"], w.u, offs, idx, box, p, alpha=np.zeros(w.n))
    box, p0 = O.workload_box_params(w, alpha_av=0.0)
    a3 = O.forces(w.pos, w.vel, w.mass, ev["h"], ev["rho"], ev["omega"], w.u, offs, idx, box, p0)
    assert np.array_equal(a2[0], a3[0]) and np.array_equal(a2[1], a3[1])


def test_g13_closed_form_on_a_quiescent_lattice():
    """v = 0, a = 0: alpha_loc = alpha_min = 0 and G13 reads alpha^{n+1} = alpha^n / (1 + dt/tau), tau = h / (sigma c_s),
    sigma_decay = 0.1: monotone decay, alpha_k = alpha_0 (1 + dt/tau)^-k; dt = 0 leaves alpha alone and
    dt -> infinity gives alpha_loc; alpha never drops below alpha_loc (the max of G13)."""
    w = W.cube(8, jitter=0.0, vel_amp=0.0)
    box, p, ev, offs, idx = _state(w)
    assert (p.alpha_min, p.alpha_max, p.sigma_decay) == (0.0, 1.0, 0.1)
    cs = math.sqrt(w.gamma * (w.gamma - 1.0) * 1.0)
    zero = np.zeros((3, w.n))
    alpha = np.full(w.n, 0.7)
    dt = 0.05
    x = dt * 0.1 * cs / ev["h"][0]
    for k in range(1, 6):
        out = O.alpha_update(w.pos, zero, zero, w.mass, ev["h"], ev["rho"], ev["omega"], w.u, offs, idx, box, p, dt, alpha)
        assert np.all(out["alpha_loc"] == 0.0) and np.all(np.abs(out["divv"]) < 1e-12)
        assert np.allclose(out["alpha"], 0.7 / (1.0 + x) ** k, rtol=1e-13)
        assert np.all(out["alpha"] < alpha)
        alpha = out["alpha"]
    same = O.alpha_update(w.pos, zero, zero, w.mass, ev["h"], ev["rho"], ev["omega"], w.u, offs, idx, box, p, 0.0, alpha)
    assert np.array_equal(same["alpha"], alpha)
    far = O.alpha_update(w.pos, zero, zero, w.mass, ev["h"], ev["rho"], ev["omega"], w.u, offs, idx, box, p, 1e12, alpha)
    assert np.all(far["alpha"] < 1e-9)
    box, pm = O.workload_box_params(w, av_switch=1, alpha_min=0.2)
    low = O.alpha_update(w.pos, zero, zero, w.mass, ev["h"], ev["rho"], ev["omega"], w.u, offs, idx, box, pm, 1e12, alpha)
    assert np.allclose(low["alpha"], 0.2, rtol=1e-9)          # decays to alpha_loc = alpha_min, not below


def test_gradient_estimates_and_instant_rise():
    """v_x = A sin(2 pi x) on a periodic lattice, a^n = 0: div v = 2 pi A cos(2 pi x), curl v = 0, d(div v)/dt =
    -(d_x v_x)^2, so alpha_loc = min(10 h^2 (2 pi A cos)^2 / c_s^2, alpha_max) to the accuracy of the SPH derivative
    estimate ((k h)^2 ~ 5 % on 24 sites); alpha below alpha_loc jumps to it at once (G13's max), whatever dt."""
    n = 24
    w = W.cube(n, jitter=0.0, vel_amp=0.0)
    A = 0.8
    w.vel[0] = A * np.sin(2 * math.pi * w.pos[0])
    box, p, ev, offs, idx = _state(w)
    zero = np.zeros((3, w.n))
    out = O.alpha_update(w.pos, w.vel, zero, w.mass, ev["h"], ev["rho"], ev["omega"], w.u, offs, idx, box, p, 0.01, np.zeros(w.n))
    div_exact = 2 * math.pi * A * np.cos(2 * math.pi * w.pos[0])
    assert np.max(np.abs(out["divv"] - div_exact)) < 0.08 * 2 * math.pi * A
    assert np.max(out["curlv"]) < 1e-10 * 2 * math.pi * A
    cs2 = w.gamma * (w.gamma - 1.0)
    aloc_exact = np.minimum(10.0 * ev["h"] ** 2 * div_exact ** 2 / cs2, 1.0)
    assert np.max(np.abs(out["alpha_loc"] - aloc_exact)) < 0.15 * aloc_exact.max()
    assert np.array_equal(out["alpha"], out["alpha_loc"]) and out["alpha"].max() > 0.3
    # expanding and compressing regions alike: A depends on (d_x v_x)^2 only when a^n = 0
    hi = O.alpha_update(w.pos, w.vel, zero, w.mass, ev["h"], ev["rho"], ev["omega"], w.u, offs, idx, box, p, 0.01, np.ones(w.n))
    assert np.all(hi["alpha"] >= hi["alpha_loc"]) and np.all(hi["alpha"] <= 1.0)


def test_limiter_suppresses_the_switch_in_shear():
    """v = (-k x + S y, 0, 0) in the interior of an open lattice: div v = -k, |curl v| = S, d(div v)/dt = -k^2 (a = 0), so
    alpha_loc = 10 h^2 xi k^2 / c_s^2 with xi = k^2 / (k^2 + S^2): strong shear switches the viscosity off."""
    n = 14
    w = W.cube(n, jitter=0.0, vel_amp=0.0)
    w.periodic = (0, 0, 0)
    k = 1.5
    res = {}
    for S in (0.0, 6.0):
        w.vel = np.zeros((3, w.n))
        w.vel[0] = -k * (w.pos[0] - 0.5) + S * (w.pos[1] - 0.5)
        box, p, ev, offs, idx = _state(w)
        out = O.alpha_update(w.pos, w.vel, np.zeros((3, w.n)), w.mass, ev["h"], ev["rho"], ev["omega"], w.u, offs, idx, box, p,
                             0.0, np.zeros(w.n))
        inner = np.all(np.abs(w.pos - 0.5) < 0.2, axis=0)
        assert np.max(np.abs(out["divv"][inner] + k)) < 0.02 * k
        assert np.max(np.abs(out["curlv"][inner] - S)) < 0.02 * max(S, k)
        cs2 = w.gamma * (w.gamma - 1.0)
        expect = 10.0 * ev["h"][inner] ** 2 * (k * k / (k * k + S * S)) * k * k / cs2
        assert np.allclose(out["alpha_loc"][inner], expect, rtol=0.06)
        res[S] = out["alpha_loc"][inner].mean()
    assert res[6.0] < 0.08 * res[0.0]


@pytest.mark.slow
def test_sod_alpha_peaks_at_the_shock():
    """Sod tube with the switch on (alpha_min = 0, alpha_max = 1, sigma_decay = 0.1): alpha rises to
    alpha_max in the shock, stays small in the undisturbed gas, and the solution keeps the momentum budget of the exact
    Riemann problem."""
    w = W.sod(64, 12)
    w.av_switch = 1
    s = O.State(w, "grid")
    assert s.alpha is not None
    t_end = 0.1
    while s.t < t_end - 1e-12:
        s.step(min(s.dt, t_end - s.t))
    x, xi = s.pos[0], s.pos[0] / s.t
    sel = np.abs(x) < 0.25
    shock = sel & (xi > 1.45) & (xi < 2.0)                       # exact shock speed 1.7522
    quiet = sel & ((xi < -1.6) | (xi > 2.6))
    assert s.alpha[shock].max() > 0.8
    assert s.alpha[quiet].max() < 0.05
    assert np.all((s.alpha >= 0.0) & (s.alpha <= 1.0))
    area = (w.box_hi[1] - w.box_lo[1]) ** 2
    assert (s.m * s.vel[0])[sel].sum() / area == pytest.approx((1.0 - 0.1) * s.t, rel=0.03)
