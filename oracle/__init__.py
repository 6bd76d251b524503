"""ctypes front-end of the CPU oracle (``oracle/sph_oracle.cpp``) -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may
import this package. It holds argument marshalling only; all arithmetic is in the C++ file, which restates
/root/reference/PAPER.md (citations there). It imports nothing from ``paper_2503_09713_b200``.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_DIR = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_DIR, "sph_oracle.cpp")
_LIB = os.path.join(_DIR, "libsph_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with g++ (-O2, no FMA contraction, single thread)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".{os.getpid()}.tmp"
        subprocess.check_call(["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fPIC", "-shared", "-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


class Box(C.Structure):
    _fields_ = [("lo", C.c_double * 3), ("hi", C.c_double * 3), ("periodic", C.c_int32 * 3)]


class Params(C.Structure):
    _fields_ = [("hfact", C.c_double), ("gamma", C.c_double), ("chi", C.c_double), ("lam", C.c_double),
                ("eps_h", C.c_double), ("alpha_av", C.c_double), ("beta_av", C.c_double), ("beta_u", C.c_double),
                ("c_cour", C.c_double), ("c_force", C.c_double), ("max_h_iter", C.c_int32),
                ("max_restarts", C.c_int32), ("eos", C.c_int32), ("newton_literal", C.c_int32),
                ("cs0", C.c_double), ("r0", C.c_double), ("q", C.c_double), ("GM", C.c_double), ("soft", C.c_double),
                ("centre", C.c_double * 3), ("eps_v", C.c_double), ("lambda_stiff", C.c_double),
                ("max_recycle", C.c_int32), ("kernel", C.c_int32), ("alpha_min", C.c_double), ("alpha_max", C.c_double),
                ("sigma_decay", C.c_double), ("av_switch", C.c_int32), ("pad_", C.c_int32)]


def make_box(lo, hi, periodic) -> Box:
    return Box((C.c_double * 3)(*lo), (C.c_double * 3)(*hi), (C.c_int32 * 3)(*[int(p) for p in periodic]))


def make_params(gamma=5.0 / 3.0, hfact=1.2, chi=1.1, lam=1.2, eps_h=1e-6, alpha_av=1.0, beta_av=2.0, beta_u=1.0,
                c_cour=0.3, c_force=0.25, max_h_iter=50, max_restarts=50, eos_isothermal=None, point_mass=None,
                newton_literal=0, eps_v=0.0, lambda_stiff=2.0, max_recycle=10, kernel=0, av_switch=0, alpha_min=0.0,
                alpha_max=1.0, sigma_decay=0.1) -> Params:
    p = Params()
    p.av_switch, p.alpha_min, p.alpha_max, p.sigma_decay = int(av_switch), alpha_min, alpha_max, sigma_decay
    p.hfact, p.gamma, p.chi, p.lam, p.eps_h = hfact, gamma, chi, lam, eps_h
    p.alpha_av, p.beta_av, p.beta_u, p.c_cour, p.c_force = alpha_av, beta_av, beta_u, c_cour, c_force
    p.max_h_iter, p.max_restarts, p.newton_literal = max_h_iter, max_restarts, newton_literal
    p.eps_v, p.lambda_stiff, p.max_recycle, p.kernel = eps_v, lambda_stiff, max_recycle, kernel
    p.eos = 0
    if eos_isothermal is not None:
        p.eos = 1
        p.cs0, p.r0, p.q = eos_isothermal
    if point_mass is not None:
        p.GM, p.soft = point_mass[0], point_mass[1]
        p.centre = (C.c_double * 3)(*point_mass[2])
    return p


def workload_box_params(w, **kw):
    """Box and Params for a ``workloads.Workload`` (duck-typed: the oracle does not import that module)."""
    cfl = getattr(w, "cfl", None)
    if cfl is not None:
        kw = dict(dict(c_cour=cfl[0], c_force=cfl[1]), **kw)
    if getattr(w, "eps_v", None):
        kw = dict(dict(eps_v=w.eps_v), **kw)
    if getattr(w, "kernel", 0):
        kw = dict(dict(kernel=w.kernel), **kw)
    if getattr(w, "av_switch", 0):
        kw = dict(dict(av_switch=1), **kw)
    return (make_box(w.box_lo, w.box_hi, w.periodic),
            make_params(gamma=w.gamma, hfact=w.hfact, eos_isothermal=w.eos_isothermal, point_mass=w.point_mass, **kw))


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        for name in ("orc_f", "orc_df"):
            getattr(_lib, name).restype = C.c_double
            getattr(_lib, name).argtypes = [C.c_double]
        for name in ("orc_W", "orc_F", "orc_dWdh"):
            getattr(_lib, name).restype = C.c_double
            getattr(_lib, name).argtypes = [C.c_double, C.c_double]
        _lib.orc_delta_beta.restype = C.c_int32
        _lib.orc_delta_beta.argtypes = [C.c_uint64, C.c_uint64, C.c_int32]
        _lib.orc_prefix_mask.restype = C.c_uint64
        _lib.orc_prefix_mask.argtypes = [C.c_uint64, C.c_uint64, C.c_int32]
        _lib.orc_neighbours_brute.restype = C.c_int64
        _lib.orc_neighbours_grid.restype = C.c_int64
        _lib.orc_density.restype = C.c_int64
        _lib.orc_forces.restype = C.c_double
        _lib.orc_evaluate.restype = C.c_int32
        _lib.orc_step.restype = C.c_int32
        _lib.orc_step2.restype = C.c_int32
        _lib.orc_step3.restype = C.c_int32
        _lib.orc_evaluate_alpha.restype = C.c_int32
        _lib.orc_alpha_update.restype = None
        _lib.orc_set_alpha.restype = None
    return _lib


def _p(a, dtype):
    assert a.dtype == dtype and a.flags["C_CONTIGUOUS"], (a.dtype, dtype)
    return a.ctypes.data_as(C.c_void_p)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


# ---- thin wrappers (marshalling only) ------------------------------------------------------------------------

def morton_keys(pos, box: Box, beta: int = 21) -> np.ndarray:
    """63-bit codes (beta = 21, the default) or the paper's shorter variant on a 2^beta grid (beta = 10: 30-bit codes)."""
    pos = _f64(pos)
    n = pos.shape[1]
    key = np.empty(n, dtype=np.uint64)
    if beta != 21:
        lib().orc_morton_keys_beta(C.c_int64(n), _p(pos, np.float64), C.byref(box), C.c_int32(int(beta)), _p(key, np.uint64))
        return key
    lib().orc_morton_keys(C.c_int64(n), _p(pos, np.float64), C.byref(box), _p(key, np.uint64))
    return key


def sort_keys(key):
    key = np.ascontiguousarray(key, dtype=np.uint64)
    n = key.shape[0]
    perm = np.empty(n, dtype=np.uint32)
    skey = np.empty(n, dtype=np.uint64)
    lib().orc_sort(C.c_int64(n), _p(key, np.uint64), _p(perm, np.uint32), _p(skey, np.uint64))
    return skey, perm


def leaf_reduction(skey, n_red: int):
    """Alg. 1 on sorted Morton codes: (xi mask u8[N], leaf codes u64[n_leaf], id map u32[n_leaf + 1])."""
    skey = np.ascontiguousarray(skey, dtype=np.uint64)
    n = skey.shape[0]
    xi = np.zeros(n, dtype=np.uint8)
    lib().orc_leaf_reduction(C.c_int64(n), _p(skey, np.uint64), C.c_int32(int(n_red)), _p(xi, np.uint8))
    codes = np.zeros(n, dtype=np.uint64)
    ids = np.zeros(n + 1, dtype=np.uint32)
    lib().orc_leaf_compact.restype = C.c_int64
    nl = lib().orc_leaf_compact(C.c_int64(n), _p(skey, np.uint64), _p(xi, np.uint8), _p(codes, np.uint64), _p(ids, np.uint32))
    return xi, codes[:nl].copy(), ids[:nl + 1].copy()


def tree(skey):
    """Radix-tree tables over sorted keys: dict(left, right, lflag, rflag, parent[2N-1], rlo, rhi)."""
    skey = np.ascontiguousarray(skey, dtype=np.uint64)
    n = skey.shape[0]
    ni = max(n - 1, 0)
    t = dict(left=np.zeros(ni, np.int32), right=np.zeros(ni, np.int32), lflag=np.zeros(ni, np.uint8),
             rflag=np.zeros(ni, np.uint8), parent=np.full(max(2 * n - 1, 0), -1, np.int32),
             rlo=np.zeros(ni, np.int32), rhi=np.zeros(ni, np.int32))
    lib().orc_tree(C.c_int64(n), _p(skey, np.uint64), _p(t["left"], np.int32), _p(t["right"], np.int32),
                   _p(t["lflag"], np.uint8), _p(t["rflag"], np.uint8), _p(t["parent"], np.int32),
                   _p(t["rlo"], np.int32), _p(t["rhi"], np.int32))
    return t


def aabb(t, pos_sorted, h_sorted):
    pos_sorted = _f64(pos_sorted)
    h_sorted = _f64(h_sorted)
    n = pos_sorted.shape[1]
    ni = max(n - 1, 0)
    box6 = np.zeros((ni, 6), np.float64)
    hmax = np.zeros(ni, np.float64)
    x, y, z = (np.ascontiguousarray(pos_sorted[k]) for k in range(3))
    lib().orc_aabb(C.c_int64(n), _p(t["left"], np.int32), _p(t["right"], np.int32), _p(t["lflag"], np.uint8),
                   _p(t["rflag"], np.uint8), _p(x, np.float64), _p(y, np.float64), _p(z, np.float64),
                   _p(h_sorted, np.float64), _p(box6, np.float64), _p(hmax, np.float64))
    return box6, hmax


def set_kernel(k: int = 0):
    """Select the SPH kernel of every later oracle call: 0 = M4, 1 = M5, 2 = M6, 3/4/5 = Wendland C2/C4/C6 (file-level selector in the C++)."""
    lib().orc_set_kernel(C.c_int32(int(k)))


def neighbours(pos, h, box: Box, chi=1.1, mode="brute", kernel=0):
    """CSR neighbour sets N(a) (self included, each list ascending): (offs u64[N+1], idx u32[total])."""
    pos = _f64(pos)
    h = _f64(h)
    n = pos.shape[1]
    set_kernel(kernel)
    fn = lib().orc_neighbours_brute if mode == "brute" else lib().orc_neighbours_grid
    offs = np.empty(n + 1, dtype=np.uint64)
    total = fn(C.c_int64(n), _p(pos, np.float64), _p(h, np.float64), C.byref(box), C.c_double(chi),
               _p(offs, np.uint64), None, C.c_int64(0))
    idx = np.empty(total, dtype=np.uint32)
    fn(C.c_int64(n), _p(pos, np.float64), _p(h, np.float64), C.byref(box), C.c_double(chi),
       _p(offs, np.uint64), _p(idx, np.uint32), C.c_int64(total))
    return offs, idx


def density(pos, m, hn, offs, idx, box: Box, p: Params):
    """One pass of Alg. 7's inner loop over a given cache. Returns dict(h, rho, omega, iters, exceeded, n_exceeded)."""
    pos, m, hn = _f64(pos), _f64(m), _f64(hn)
    n = pos.shape[1]
    out = dict(h=np.empty(n), rho=np.empty(n), omega=np.empty(n), iters=np.empty(n, np.int32),
               exceeded=np.empty(n, np.uint8))
    set_kernel(p.kernel)
    ne = lib().orc_density(C.c_int64(n), _p(pos, np.float64), _p(m, np.float64), _p(hn, np.float64),
                           _p(offs, np.uint64), _p(idx, np.uint32), C.byref(box), C.byref(p), _p(out["h"], np.float64),
                           _p(out["rho"], np.float64), _p(out["omega"], np.float64), _p(out["iters"], np.int32),
                           _p(out["exceeded"], np.uint8))
    out["n_exceeded"] = int(ne)
    return out


def h_bisect(pos, m, box: Box, hfact, h_lo, h_hi, kernel=0):
    pos, m, h_lo, h_hi = _f64(pos), _f64(m), _f64(h_lo), _f64(h_hi)
    n = pos.shape[1]
    out = np.empty(n)
    set_kernel(kernel)
    lib().orc_h_bisect(C.c_int64(n), _p(pos, np.float64), _p(m, np.float64), C.byref(box), C.c_double(hfact),
                       _p(h_lo, np.float64), _p(h_hi, np.float64), _p(out, np.float64))
    return out


def alpha_update(pos, vel, acc, m, h, rho, omega, u, offs, idx, box: Box, p: Params, dt, alpha):
    """G12-G13 with reading A18: dict(alpha, divv, curlv, alpha_loc)."""
    pos, vel, acc, m, h, rho, omega, u, alpha = (_f64(a) for a in (pos, vel, acc, m, h, rho, omega, u, alpha))
    n = pos.shape[1]
    out = dict(alpha=np.empty(n), divv=np.empty(n), curlv=np.empty(n), alpha_loc=np.empty(n))
    set_kernel(p.kernel)
    lib().orc_alpha_update(C.c_int64(n), _p(pos, np.float64), _p(vel, np.float64), _p(acc, np.float64), _p(m, np.float64),
                           _p(h, np.float64), _p(rho, np.float64), _p(omega, np.float64), _p(u, np.float64),
                           _p(offs, np.uint64), _p(idx, np.uint32), C.byref(box), C.byref(p), C.c_double(dt),
                           _p(alpha, np.float64), _p(out["alpha"], np.float64), _p(out["divv"], np.float64),
                           _p(out["curlv"], np.float64), _p(out["alpha_loc"], np.float64))
    return out


def forces(pos, vel, m, h, rho, omega, u, offs, idx, box: Box, p: Params, alpha=None):
    pos, vel, m, h, rho, omega, u = (_f64(a) for a in (pos, vel, m, h, rho, omega, u))
    n = pos.shape[1]
    acc = np.empty((3, n))
    dudt = np.empty(n)
    set_kernel(p.kernel)
    if alpha is not None:
        alpha = _f64(alpha)
        lib().orc_set_alpha(_p(alpha, np.float64))
    try:
        return _forces_call(pos, vel, m, h, rho, omega, u, offs, idx, box, p, acc, dudt, n)
    finally:
        lib().orc_set_alpha(None)


def _forces_call(pos, vel, m, h, rho, omega, u, offs, idx, box, p, acc, dudt, n):
    dt = lib().orc_forces(C.c_int64(n), _p(pos, np.float64), _p(vel, np.float64), _p(m, np.float64),
                          _p(h, np.float64), _p(rho, np.float64), _p(omega, np.float64), _p(u, np.float64),
                          _p(offs, np.uint64), _p(idx, np.uint32), C.byref(box), C.byref(p), _p(acc, np.float64),
                          _p(dudt, np.float64))
    return acc, dudt, float(dt)


_ERR = {-1: "h iteration did not converge within max_h_iter", -2: "more than max_restarts chi-restarts"}


def evaluate(pos, vel, m, u, h, box: Box, p: Params, mode="grid", alpha=None):
    """Neighbours -> h/rho/Omega with chi-restarts -> [shock switch] -> forces and dt, for a given state (h = h^n guess).
    With p.av_switch and `alpha` (the alpha^n array) the result carries the updated alpha (white step: a^n = 0, dt = 0)."""
    pos, vel, m, u = (_f64(a) for a in (pos, vel, m, u))
    h = np.array(h, dtype=np.float64, copy=True)
    n = pos.shape[1]
    out = dict(h=h, rho=np.empty(n), omega=np.empty(n), acc=np.empty((3, n)), dudt=np.empty(n))
    dt = C.c_double()
    nn = C.c_int64()
    set_kernel(p.kernel)
    args = [C.c_int64(n), _p(pos, np.float64), _p(vel, np.float64), _p(m, np.float64),
            _p(u, np.float64), _p(h, np.float64), C.byref(box), C.byref(p),
            C.c_int32(0 if mode == "brute" else 1), _p(out["rho"], np.float64),
            _p(out["omega"], np.float64), _p(out["acc"], np.float64), _p(out["dudt"], np.float64),
            C.byref(dt), C.byref(nn)]
    if alpha is not None:
        out["alpha"] = np.array(alpha, dtype=np.float64, copy=True)
        rc = lib().orc_evaluate_alpha(*args, _p(out["alpha"], np.float64))
    else:
        rc = lib().orc_evaluate(*args)
    if rc < 0:
        raise RuntimeError("oracle: " + _ERR.get(rc, str(rc)))
    out.update(dt=dt.value, restarts=int(rc), n_neigh=nn.value)
    return out


class State:
    """Mutable oracle-side simulation state (original particle order)."""

    def __init__(self, w, mode="grid", **param_kw):
        self.box, self.p = workload_box_params(w, **param_kw)
        self.mode = mode
        self.pos, self.vel, self.m, self.u = (np.array(a, dtype=np.float64, copy=True)
                                              for a in (w.pos, w.vel, w.mass, w.u))
        self.alpha = np.full(self.pos.shape[1], self.p.alpha_min) if self.p.av_switch else None
        ev = evaluate(self.pos, self.vel, self.m, self.u, w.h0, self.box, self.p, mode, alpha=self.alpha)   # "white" step
        self.h, self.rho, self.omega, self.acc, self.dudt = ev["h"], ev["rho"], ev["omega"], ev["acc"], ev["dudt"]
        if self.alpha is not None:
            self.alpha = ev["alpha"]
        self.dt = ev["dt"]
        self.restarts = ev["restarts"]
        self.t = 0.0

    def step(self, dt=None):
        """One leapfrog step (with the corrector re-cycle and CFL multiplier if the parameters set eps_v > 0)."""
        dt = self.dt if dt is None or dt <= 0 else dt
        n = self.pos.shape[1]
        dtn = C.c_double()
        mult = C.c_double(getattr(self, "cfl_mult", 1.0))
        nrec = C.c_int32()
        set_kernel(self.p.kernel)
        rc = lib().orc_step3(C.c_int64(n), _p(self.pos, np.float64), _p(self.vel, np.float64), _p(self.m, np.float64),
                             _p(self.u, np.float64), _p(self.h, np.float64), _p(self.acc, np.float64),
                             _p(self.dudt, np.float64), C.byref(self.box), C.byref(self.p),
                             C.c_int32(0 if self.mode == "brute" else 1), C.c_double(dt), _p(self.rho, np.float64),
                             _p(self.omega, np.float64), C.byref(dtn), C.byref(mult), C.byref(nrec),
                             _p(self.alpha, np.float64) if getattr(self, "alpha", None) is not None else None)
        if rc < 0:
            raise RuntimeError("oracle: " + _ERR.get(rc, str(rc)))
        self.restarts = int(rc)
        self.recycles = int(nrec.value)
        self.cfl_mult = float(mult.value)
        self.t += dt
        self.dt = dtn.value
        return dt
