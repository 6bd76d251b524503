"""Pins for orc_forces on hand-worked two-particle cases (tests/golden/pair_forces.txt) -- CPU only.

The conservation identities of tests/test_oracle_sph.py hold for any magnitude of the artificial viscosity (Eq. 5-6)
and of the conductivity (Eq. 8-9), and its CFL test never has the force term or the pair maximum of v_sig^dt as the
minimum. The golden file derives, on paper, from Eq. 3-6, 8-10 and G8, the
accelerations, du/dt split into pressure, viscous and conductive parts, and dt for five pairs; a factor 1 instead of
1/2 in Eq. 5 or Eq. 8, beta applied to c_s, rho_a + rho_b for the mean density, F_ab(h_a) and F_ab(h_b) swapped, or a
Courant-only timestep each fail here.
"""
import math
import os

import numpy as np
import pytest

import oracle as O

GOLD = os.path.join(os.path.dirname(__file__), "golden", "pair_forces.txt")


def _gold():
    out = {}
    for line in open(GOLD):
        if line.startswith("#") or not line.strip():
            continue
        case, name, unit, val = line.split()
        out[(case, name)] = float(val) / (4.0 * math.pi) if unit == "x4pi" else float(val)
    return out


# the inputs of each case as stated in the golden file's comments: (h0, h1, r, m0, m1, v0x)
CASES = {"A": (1.0, 1.0, 1.0, 2.0, 3.0, 1.0), "B": (1.0, 1.0, 1.0, 2.0, 3.0, -1.0), "C": (1.0, 1.0, 1.0, 20.0, 30.0, 0.0),
         "D": (1.0, 2.0, 1.0, 2.0, 3.0, 1.0), "E": (1.0, 1.0, 2.1, 2.0, 3.0, 1.0)}


def _run(case, **kw):
    h0, h1, r, m0, m1, v0x = CASES[case]
    pos = np.array([[0.0, r], [0.0, 0.0], [0.0, 0.0]])
    vel = np.array([[v0x, 0.0], [0.0, 0.0], [0.0, 0.0]])
    box = O.make_box((-10.0,) * 3, (10.0,) * 3, (0, 0, 0))
    p = O.make_params(gamma=2.0, **kw)
    offs = np.array([0, 2, 4], dtype=np.uint64)
    idx = np.array([0, 1, 0, 1], dtype=np.uint32)          # both lists: self and the partner
    return O.forces(pos, vel, np.array([m0, m1]), np.array([h0, h1]), np.array([1.0, 3.0]), np.array([1.0, 0.5]),
                    np.array([8.0, 2.0]), offs, idx, box, p)


@pytest.mark.parametrize("case", sorted(CASES))
def test_pair_forces_against_hand_derivation(case):
    g = _gold()
    acc, du, dt = _run(case)                                              # everything on
    acc_nl, du_nl, _ = _run(case, beta_u=0.0)                            # no conductivity
    acc_p, du_p, _ = _run(case, beta_u=0.0, alpha_av=0.0, beta_av=0.0)   # pressure only
    tol = 1e-14 * 840.0 / (4.0 * math.pi)
    for a in (0, 1):
        assert acc[0, a] == pytest.approx(g[(case, f"a{a}x")], abs=tol)
        assert acc_nl[0, a] == acc[0, a]                                  # conductivity does not enter Eq. 3
        assert acc[1, a] == 0.0 and acc[2, a] == 0.0
        assert du_nl[a] == pytest.approx(g[(case, f"du{a}_noL")], abs=tol)
        assert du[a] - du_nl[a] == pytest.approx(g[(case, f"L{a}")], abs=tol)
        if (case, f"du{a}_P") in g:
            assert du_p[a] == pytest.approx(g[(case, f"du{a}_P")], abs=tol)
            assert du_nl[a] - du_p[a] == pytest.approx(g[(case, f"du{a}_AV")], abs=tol)
    if (case, "dt") in g:
        assert dt == pytest.approx(g[(case, "dt")], rel=1e-14)
    else:
        assert dt * dt * 16.0 / math.pi == pytest.approx(g[(case, "dt_sq_x16_over_pi")], rel=1e-14)


def test_pair_cases_discriminate():
    """The cases are chosen so that the plausible mistakes change a stored number: check that the numbers themselves
    differ in the ways the module docstring claims (a property of the golden file, not of the oracle)."""
    g = _gold()
    assert g[("A", "du0_AV")] > 0 and g[("A", "du0_AV")] != g[("A", "du0_P")]        # viscous magnitude is pinned
    assert g[("A", "L0")] < 0 < g[("A", "L1")]                                        # hot cools, cold warms
    assert g[("A", "dt")] < 0.3 * 1.0 / 4.0                                           # pair maximum of v_sig^dt decides
    h0, h1, r, m0, m1, _ = CASES["C"]
    assert math.sqrt(g[("C", "dt_sq_x16_over_pi")] * math.pi / 16.0) < 0.3 * h0 / 4.0  # force term decides
    assert g[("D", "a0x")] != g[("A", "a0x")] and g[("D", "du1_noL")] != g[("A", "du1_noL")]   # F(h_a) vs F(h_b)
    assert g[("E", "dt")] > g[("A", "dt")]                                            # outside 2 max(h): not in v_sig^dt
