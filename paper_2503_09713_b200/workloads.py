"""Seeded synthetic workload generators (inputs only; none of the method's arithmetic lives here, with one
stated exception: ``sedov`` shapes its injected-energy profile with the textbook M4 polynomial, "smoothed
by the kernel" -- an input profile, compared with nothing; neither side's kernels are used or checked through it).

Shared by the oracle-side tests and the CUDA-side tests/bench. NumPy only: this module imports neither
``oracle/`` nor the CUDA binding. Recipes follow SURVEY.md §8(d) / DESIGN.md "Input recipe": they stand in
for the paper's workloads (HCP Sedov lattice PAPER.md:354, Sod tube PAPER.md:229, circumbinary disc
PAPER.md:308-320) with the same shapes, sizes and value distributions; the paper's own initial-condition
files are not available.

RNG: counter-based and stateless. ``u(seed, particle, lane)`` is the SplitMix64 output function applied to
``seed + (4*particle + lane + 1) * G`` (G = SplitMix64 increment, wrap-around u64 arithmetic), mapped to [0,1)
by ``(x >> 11) * 2**-53``.
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

DEFAULT_SEED = 20250309
_G = np.uint64(0x9E3779B97F4A7C15)


def splitmix_u01(seed: int, particle: np.ndarray, lane: int) -> np.ndarray:
    """Uniform [0,1) doubles from the stateless counter-based generator described in the module docstring."""
    with np.errstate(over="ignore"):
        p = np.asarray(particle, dtype=np.uint64)
        z = np.uint64(seed) + (np.uint64(4) * p + np.uint64(lane + 1)) * _G
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        z = z ^ (z >> np.uint64(31))
    return (z >> np.uint64(11)).astype(np.float64) * (2.0 ** -53)


@dataclasses.dataclass
class Workload:
    """Initial conditions in SoA layout: ``pos``/``vel`` are float64 [3, N] (x row, y row, z row)."""

    name: str
    pos: np.ndarray
    vel: np.ndarray
    mass: np.ndarray
    u: np.ndarray
    h0: np.ndarray
    box_lo: tuple
    box_hi: tuple
    periodic: tuple
    gamma: float
    hfact: float = 1.2
    # optional physics switches (config C3 only)
    eos_isothermal: tuple | None = None  # (cs0, r0, q): cs = cs0 * (R / r0) ** -q
    point_mass: tuple | None = None  # (GM, softening, (cx, cy, cz))
    steps: int = 1
    cfl: tuple | None = None  # (C_cour, C_force) if not the defaults (Sedov blast)
    eps_v: float | None = None  # leapfrog corrector check G7; None / 0 = off
    kernel: int = 0  # SPH kernel: 0 = M4 (all BASELINE configs), 1 = M5, 2 = M6, 3/4/5 = Wendland C2/C4/C6
    morton_bits: int = 21  # grid bits per axis of the Morton code: 21, or 10 = the paper's 30-bit variant
    av_switch: int = 0  # 1 = shock-switch alpha evolution (G11-G13) instead of the constant alpha
    leaf_reduction: int = 0  # 0 = off; k >= 1: leaf groups from the paper's Alg. 1 with n_red = k - 1 passes

    @property
    def n(self) -> int:
        return int(self.pos.shape[1])


def cube(n_side: int, jitter: float = 0.1, seed: int = DEFAULT_SEED, vel_amp: float = 1e-4,
         gamma: float = 5.0 / 3.0, hfact: float = 1.2, steps: int = 5, name: str | None = None) -> Workload:
    """Uniform-density periodic unit cube: ``n_side**3`` sites at (i+1/2)/n_side, jitter = +-``jitter`` spacings
    per axis (lanes 0-2), total mass 1, u = 1, v_x = vel_amp*sin(2 pi x + phi), phi = 2 pi u(seed, 0, 3).
    C0 = cube(16, 0.05, vel_amp=0); C2 = cube(256, 0.1); C4 = the same recipe at 64..512."""
    n = n_side ** 3
    idx = np.arange(n, dtype=np.uint64)
    ix = (idx // np.uint64(n_side * n_side)).astype(np.float64)
    iy = ((idx // np.uint64(n_side)) % np.uint64(n_side)).astype(np.float64)
    iz = (idx % np.uint64(n_side)).astype(np.float64)
    d = 1.0 / n_side
    pos = np.empty((3, n), dtype=np.float64)
    for k, i in enumerate((ix, iy, iz)):
        p = (i + 0.5) * d
        if jitter != 0.0:
            p = p + (2.0 * splitmix_u01(seed, idx, k) - 1.0) * (jitter * d)
        pos[k] = p
    np.clip(pos, 0.0, np.nextafter(1.0, 0.0), out=pos)
    vel = np.zeros((3, n), dtype=np.float64)
    if vel_amp != 0.0:
        phi = 2.0 * math.pi * float(splitmix_u01(seed, np.array([0], dtype=np.uint64), 3)[0])
        vel[0] = vel_amp * np.sin(2.0 * math.pi * pos[0] + phi)
    mass = np.full(n, 1.0 / n, dtype=np.float64)
    u = np.ones(n, dtype=np.float64)
    h0 = np.full(n, hfact * d, dtype=np.float64)
    return Workload(name or f"cube{n_side}", pos, vel, mass, u, h0, (0.0, 0.0, 0.0), (1.0, 1.0, 1.0),
                    (1, 1, 1), gamma, hfact, steps=steps)


def sod(nx_left: int = 128, ny_left: int = 64, gamma: float = 1.4, hfact: float = 1.2, steps: int = 10,
        name: str | None = None) -> Workload:
    """3-D Sod tube (C1): periodic box [-1/2,1/2] x [-L/2,L/2]^2 with L = ny_left * D, D = 1/(2 nx_left).
    Left (x<0): nx_left x ny_left x ny_left cubic lattice, spacing D, rho = 1, P = 1. Right: half the counts at
    spacing 2D, rho = 1/8, P = 0.1. Equal masses m = D^3, v = 0, cell-centred sites, no jitter.
    Default = BASELINE config 1 (128x64x64 + 64x32x32 = 589,824 particles)."""
    D = 0.5 / nx_left
    Ly = ny_left * D

    def lattice(nx, ny, spacing, x0):
        i = np.arange(nx, dtype=np.float64)
        j = np.arange(ny, dtype=np.float64)
        X, Y, Z = np.meshgrid(x0 + (i + 0.5) * spacing, -0.5 * Ly + (j + 0.5) * spacing,
                              -0.5 * Ly + (j + 0.5) * spacing, indexing="ij")
        return np.stack([X.ravel(), Y.ravel(), Z.ravel()])

    pl = lattice(nx_left, ny_left, D, -0.5)
    pr = lattice(nx_left // 2, ny_left // 2, 2.0 * D, 0.0)
    pos = np.ascontiguousarray(np.concatenate([pl, pr], axis=1))
    nl, nr = pl.shape[1], pr.shape[1]
    n = nl + nr
    m = D ** 3
    mass = np.full(n, m, dtype=np.float64)
    u = np.concatenate([np.full(nl, 1.0 / ((gamma - 1.0) * 1.0)), np.full(nr, 0.1 / ((gamma - 1.0) * 0.125))])
    h0 = np.concatenate([np.full(nl, hfact * D), np.full(nr, hfact * 2.0 * D)])
    vel = np.zeros((3, n), dtype=np.float64)
    return Workload(name or f"sod{nx_left}x{ny_left}", pos, vel, mass, u, h0, (-0.5, -0.5 * Ly, -0.5 * Ly),
                    (0.5, 0.5 * Ly, 0.5 * Ly), (1, 1, 1), gamma, hfact, steps=steps)


def disc(n: int = 10_000_000, seed: int = DEFAULT_SEED, hfact: float = 1.2, steps: int = 5,
         name: str | None = None) -> Workload:
    """Locally isothermal disc (C3): R uniform on [2,10] (Sigma ~ 1/R), phi uniform, z ~ N(0,H) truncated at
    +-3H with H/R = 0.05 (R/2)^(1/4); c_s = 0.05 sqrt(1/2) (R/2)^(-1/4); v_phi from the softened point-mass
    potential (GM = 1, eps = 0.1); equal masses, M_disc = 0.01; open boundaries, key box = cube [-12,12]^3;
    h0 from the analytic rho(R, z)."""
    from scipy.special import ndtr, ndtri  # inverse normal CDF for the truncated Gaussian

    idx = np.arange(n, dtype=np.uint64)
    R = 2.0 + 8.0 * splitmix_u01(seed, idx, 0)
    phi = 2.0 * math.pi * splitmix_u01(seed, idx, 1)
    H = 0.05 * R * (R / 2.0) ** 0.25
    plo, phi_hi = ndtr(-3.0), ndtr(3.0)
    zeta = ndtri(plo + (phi_hi - plo) * splitmix_u01(seed, idx, 2))
    z = H * zeta
    pos = np.stack([R * np.cos(phi), R * np.sin(phi), z])
    GM, eps = 1.0, 0.1
    vphi = np.sqrt(GM * R * R / (R * R + eps * eps) ** 1.5)
    vel = np.stack([-vphi * np.sin(phi), vphi * np.cos(phi), np.zeros(n)])
    m_disc = 0.01
    mass = np.full(n, m_disc / n, dtype=np.float64)
    sigma = (m_disc / (16.0 * math.pi)) / R
    rho = sigma / (math.sqrt(2.0 * math.pi) * H * (phi_hi - plo)) * np.exp(-0.5 * zeta * zeta)
    h0 = hfact * (mass / rho) ** (1.0 / 3.0)
    cs0 = 0.05 * math.sqrt(0.5)
    u = np.zeros(n, dtype=np.float64)  # unused by the locally isothermal EOS
    return Workload(name or f"disc{n}", np.ascontiguousarray(pos), np.ascontiguousarray(vel), mass, u, h0,
                    (-12.0, -12.0, -12.0), (12.0, 12.0, 12.0), (0, 0, 0), 1.0, hfact,
                    eos_isothermal=(cs0, 2.0, 0.25), point_mass=(GM, eps, (0.0, 0.0, 0.0)), steps=steps)


def sedov(n_side: int = 128, E0: float = 1.0, cfl: float = 0.1, gamma: float = 5.0 / 3.0, hfact: float = 1.2,
          steps: int = 5, name: str | None = None) -> Workload:
    """Sedov-Taylor blast set-up, the paper's own performance benchmark (SURVEY.md 8(f)
    item 2): periodic box [-0.6, 0.6]^3, rho = 1, v = 0, particles on a close-packed (HCP) lattice with ``n_side``
    sites along x (row and layer counts rounded to even numbers and the y, z spacings stretched by a few per cent,
    less as n_side grows, so that the lattice is periodic), equal masses, and the energy E0 = 1 injected at the centre as u_a = E0 W(r_a, 2 h0)
    with the M4 kernel and h0 = hfact (m/rho)^(1/3) (the relaxed h of the lattice to 3e-4); u = 0 elsewhere.
    ``cfl`` sets both C_cour and C_force (0.1 for the physics run, 1e-3 for the paper's timing run); set
    ``eps_v`` on the result to switch on the leapfrog corrector re-cycle (G6-G10)."""
    L = 1.2
    nx = int(n_side)
    dx = L / nx
    ny = 2 * max(1, round(L / (dx * math.sqrt(3.0) / 2.0) / 2.0))
    nz = 2 * max(1, round(L / (dx * math.sqrt(6.0) / 3.0) / 2.0))
    dy, dz = L / ny, L / nz
    k, j, i = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    x = (i + 0.5 * (j % 2) + 0.5 * (k % 2) + 0.25) * dx
    y = (j + (k % 2) / 3.0 + 0.25) * dy
    z = (k + 0.25) * dz
    pos = np.stack([np.mod(x.ravel(), L), np.mod(y.ravel(), L), np.mod(z.ravel(), L)]) - 0.5 * L
    pos = np.ascontiguousarray(np.clip(pos, -0.5 * L, np.nextafter(0.5 * L, 0.0)))
    n = pos.shape[1]
    m = L ** 3 / n
    h0 = hfact * m ** (1.0 / 3.0)
    r = np.sqrt((pos * pos).sum(axis=0))
    hi = 2.0 * h0
    q = r / hi
    w = np.where(q < 1.0, 1.0 - 1.5 * q * q + 0.75 * q ** 3, np.where(q < 2.0, 0.25 * (2.0 - q) ** 3, 0.0)) / (math.pi * hi ** 3)
    u = E0 * w
    return Workload(name or f"sedov{n_side}", pos, np.zeros((3, n)), np.full(n, m), u, np.full(n, h0),
                    (-0.5 * L,) * 3, (0.5 * L,) * 3, (1, 1, 1), gamma, hfact, steps=steps, cfl=(cfl, cfl))


def random_cloud(n: int, seed: int = DEFAULT_SEED, periodic: bool = True, clustered: bool = True,
                 name: str | None = None) -> Workload:
    """Small non-uniform cloud for neighbour-search / tree tests (not a BASELINE config): positions are a
    mixture of uniform points and points concentrated towards one corner; h0 varies by a factor ~3."""
    idx = np.arange(n, dtype=np.uint64)
    pos = np.stack([splitmix_u01(seed, idx, k) for k in range(3)])
    if clustered:
        sel = splitmix_u01(seed + 1, idx, 0) < 0.5
        pos[:, sel] = pos[:, sel] ** 2.5
    np.clip(pos, 0.0, np.nextafter(1.0, 0.0), out=pos)
    h_mean = 1.2 * (1.0 / n) ** (1.0 / 3.0)
    h0 = h_mean * (0.6 + 1.2 * splitmix_u01(seed + 2, idx, 0))
    vel = np.stack([splitmix_u01(seed + 3, idx, k) - 0.5 for k in range(3)])
    mass = np.full(n, 1.0 / n)
    u = 0.5 + splitmix_u01(seed + 4, idx, 0)
    per = (1, 1, 1) if periodic else (0, 0, 0)
    return Workload(name or f"cloud{n}", np.ascontiguousarray(pos), np.ascontiguousarray(vel), mass, u, h0,
                    (0.0, 0.0, 0.0), (1.0, 1.0, 1.0), per, 5.0 / 3.0, 1.2)


def config(i: int) -> Workload:
    """BASELINE.json ``configs[i]`` for i in 0..3 (config 4 is ``cube(n)`` at n = 64, 128, 256, 384, 512)."""
    if i == 0:
        return cube(16, jitter=0.05, vel_amp=0.0, steps=0, name="C0_cube16")
    if i == 1:
        return sod(128, 64, steps=10, name="C1_sod")
    if i == 2:
        return cube(256, jitter=0.1, steps=5, name="C2_cube256")
    if i == 3:
        return disc(10_000_000, steps=5, name="C3_disc")
    raise ValueError("config index must be 0..3; config 4 is cube(n_side) for n_side in (64,128,256,384,512)")
