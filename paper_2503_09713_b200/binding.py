"""Thin ctypes binding of libsph_b200 (include/sph_b200.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels behind the C ABI. PyTorch is used for device memory (the
library allocates through ``torch.empty`` via the allocator hooks), streams and host<->device tensors. There is
no CPU fallback: if the shared library is missing, or no sm_100 GPU is present, calls raise.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libsph_b200.so")
_lib = None

SPH_MEM_HOST, SPH_MEM_DEVICE = 0, 1
STATUS = {0: "SPH_OK", -1: "SPH_ERR_ARG", -2: "SPH_ERR_DEVICE", -3: "SPH_ERR_OOM", -4: "SPH_ERR_H_NOCONV",
          -5: "SPH_ERR_RESTARTS", -6: "SPH_ERR_PERIODIC_TOO_SMALL", -7: "SPH_ERR_ORDER", -8: "SPH_ERR_CAP"}

# every symbol include/sph_b200.h declares (tests check that the library exports all of them)
SYMBOLS = ["sph_default_params", "sph_init", "sph_init_ex", "sph_build_tree", "sph_compute_density",
           "sph_compute_forces", "sph_step_leapfrog", "sph_set_fields", "sph_get_fields", "sph_get_keys_perm",
           "sph_get_tree", "sph_get_neighbours", "sph_get_neighbours_range", "sph_get_leaves", "sph_get_alpha", "sph_get_stats", "sph_reset_timers", "sph_last_error", "sph_free",
           "sph_measure_fp64_peak", "sph_scan_u32_noalloc", "sph_scan_noalloc_max_items", "sph_noalloc_last_error"]


class SphError(RuntimeError):
    def __init__(self, code, msg=""):
        super().__init__(f"{STATUS.get(code, code)}: {msg}")
        self.code = code


class Box(C.Structure):
    _fields_ = [("lo", C.c_double * 3), ("hi", C.c_double * 3), ("periodic", C.c_int32 * 3)]


class Params(C.Structure):
    _fields_ = [("hfact", C.c_double), ("gamma", C.c_double), ("chi", C.c_double), ("lambda_", C.c_double),
                ("eps_h", C.c_double), ("alpha_av", C.c_double), ("beta_av", C.c_double), ("beta_u", C.c_double),
                ("c_cour", C.c_double), ("c_force", C.c_double), ("max_h_iter", C.c_int32),
                ("max_restarts", C.c_int32), ("eos", C.c_int32), ("kernel", C.c_int32), ("cs0", C.c_double),
                ("r0", C.c_double), ("q", C.c_double), ("GM", C.c_double), ("soft", C.c_double),
                ("centre", C.c_double * 3), ("eps_v", C.c_double), ("lambda_stiff", C.c_double),
                ("max_recycle", C.c_int32), ("group_max", C.c_int32), ("morton_bits", C.c_int32), ("leaf_reduction", C.c_int32), ("av_switch", C.c_int32),
                ("reserved4", C.c_int32), ("alpha_min", C.c_double), ("alpha_max", C.c_double), ("sigma_decay", C.c_double)]


ALLOC_FN = C.CFUNCTYPE(C.c_void_p, C.c_size_t, C.c_void_p)
FREE_FN = C.CFUNCTYPE(None, C.c_void_p, C.c_void_p)


class Allocator(C.Structure):
    _fields_ = [("alloc", ALLOC_FN), ("release", FREE_FN), ("user", C.c_void_p)]


class Stats(C.Structure):
    _fields_ = [(n, C.c_double) for n in ("ms_keys", "ms_sort", "ms_permute", "ms_tree", "ms_aabb", "ms_traverse",
                                          "ms_scan", "ms_density", "ms_forces", "ms_leapfrog", "ms_total")] + \
               [("n_particles", C.c_int64), ("n_groups", C.c_int64), ("n_neighbours", C.c_int64),
                ("nbr_min", C.c_int32), ("nbr_max", C.c_int32), ("nbr_mean", C.c_double), ("h_iter_max", C.c_int32),
                ("restarts", C.c_int32), ("steps", C.c_int64), ("kernel_launches", C.c_int64), ("dt", C.c_double),
                ("t", C.c_double), ("bytes_allocated", C.c_int64), ("cand_max", C.c_int32), ("groups_fallback", C.c_int32),
                ("chunks_shared", C.c_int32), ("share_chunk", C.c_int32), ("sort_passes", C.c_int32),
                ("sort_tie_max", C.c_int32), ("recycles", C.c_int32), ("reserved", C.c_int32), ("cfl_mult", C.c_double),
                ("density_sweeps", C.c_int64), ("n_inner", C.c_int64), ("n_grew", C.c_int64)]

    def as_dict(self):
        return {n: getattr(self, n) for n, _ in self._fields_}


def load():
    """Load the shared library (no GPU needed to load it). Raises if it has not been built."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_2503_09713_b200.build` "
                               "(there is no CPU fallback)")
        lib = C.CDLL(LIB_PATH)
        lib.sph_last_error.restype = C.c_char_p
        lib.sph_last_error.argtypes = [C.c_void_p]
        lib.sph_free.restype = None
        lib.sph_free.argtypes = [C.c_void_p]
        lib.sph_default_params.restype = None
        lib.sph_default_params.argtypes = [C.POINTER(Params)]
        vp, i64, dbl = C.c_void_p, C.c_int64, C.c_double
        lib.sph_init.argtypes = [C.POINTER(vp), i64, vp, vp, vp, vp, C.POINTER(Box), dbl, dbl]
        lib.sph_init_ex.argtypes = [C.POINTER(vp), i64, C.c_int, vp, vp, vp, vp, vp, C.POINTER(Box), C.POINTER(Params),
                                    vp, C.POINTER(Allocator), C.c_int]
        for name in ("sph_build_tree", "sph_compute_density", "sph_compute_forces", "sph_reset_timers"):
            getattr(lib, name).argtypes = [vp]
        lib.sph_step_leapfrog.argtypes = [vp, dbl, C.POINTER(dbl)]
        lib.sph_set_fields.argtypes = [vp, C.c_int] + [vp] * 6
        lib.sph_get_fields.argtypes = [vp, C.c_int] + [vp] * 8
        lib.sph_get_keys_perm.argtypes = [vp, C.c_int, vp, vp]
        lib.sph_get_tree.argtypes = [vp, C.c_int] + [vp] * 9
        lib.sph_get_neighbours.argtypes = [vp, C.c_int, vp, vp, C.c_uint64]
        lib.sph_get_neighbours_range.argtypes = [vp, C.c_int, i64, i64, vp, vp, C.c_uint64]
        lib.sph_get_leaves.argtypes = [vp, C.c_int, C.POINTER(C.c_int64), vp, vp]
        lib.sph_get_alpha.argtypes = [vp, C.c_int, vp]
        lib.sph_get_stats.argtypes = [vp, C.POINTER(Stats)]
        lib.sph_measure_fp64_peak.argtypes = [C.POINTER(dbl), vp]
        lib.sph_scan_u32_noalloc.argtypes = [vp, vp, i64, vp]
        lib.sph_scan_noalloc_max_items.restype = C.c_int64
        lib.sph_scan_noalloc_max_items.argtypes = []
        lib.sph_noalloc_last_error.restype = C.c_char_p
        lib.sph_noalloc_last_error.argtypes = []
        _lib = lib
    return _lib


def default_params(**kw) -> Params:
    p = Params()
    load().sph_default_params(C.byref(p))
    for k, v in kw.items():
        if k == "lambda":
            k = "lambda_"
        if k == "centre":
            v = (C.c_double * 3)(*v)
        if not hasattr(p, k):
            raise TypeError(f"unknown parameter {k}")
        setattr(p, k, v)
    return p


def params_for(w, **kw) -> Params:
    """Parameters for a ``workloads.Workload`` (gamma, hfact, EOS/point-mass switches) plus overrides."""
    extra = dict(gamma=w.gamma, hfact=w.hfact)
    if w.eos_isothermal is not None:
        extra.update(eos=1, cs0=w.eos_isothermal[0], r0=w.eos_isothermal[1], q=w.eos_isothermal[2])
    if w.point_mass is not None:
        extra.update(GM=w.point_mass[0], soft=w.point_mass[1], centre=w.point_mass[2])
    if getattr(w, "cfl", None) is not None:
        extra.update(c_cour=w.cfl[0], c_force=w.cfl[1])
    if getattr(w, "eps_v", None):
        extra.update(eps_v=w.eps_v)
    if getattr(w, "kernel", 0):
        extra.update(kernel=w.kernel)
    if getattr(w, "morton_bits", 21) != 21:
        extra.update(morton_bits=w.morton_bits)
    if getattr(w, "leaf_reduction", 0):
        extra.update(leaf_reduction=w.leaf_reduction)
    if getattr(w, "av_switch", 0):
        extra.update(av_switch=1)
    extra.update(kw)
    return default_params(**extra)


class _TorchAllocator:
    """Device memory for the library comes from PyTorch's caching allocator."""

    def __init__(self, device):
        import torch
        self.torch = torch
        self.device = device
        self.live = {}
        self._alloc = ALLOC_FN(self.alloc)
        self._free = FREE_FN(self.free)
        self.struct = Allocator(self._alloc, self._free, None)

    def alloc(self, nbytes, _user):
        try:
            t = self.torch.empty(int(nbytes), dtype=self.torch.uint8, device=self.device)
        except Exception:
            return None
        self.live[t.data_ptr()] = t
        return t.data_ptr()

    def free(self, ptr, _user):
        self.live.pop(ptr, None)


def _ptr(t):
    """Raw pointer of a torch tensor or numpy array (or None)."""
    if t is None:
        return None
    if isinstance(t, np.ndarray):
        assert t.flags["C_CONTIGUOUS"]
        return C.c_void_p(t.ctypes.data)
    assert t.is_contiguous()
    return C.c_void_p(t.data_ptr())


class Sim:
    """One simulation context on the current CUDA device. Fields cross the ABI in ORIGINAL particle order,
    SoA: ``pos``/``vel``/``acc`` are float64 [3, N]."""

    def __init__(self, pos, vel, mass, u, box_lo, box_hi, periodic, params: Params | None = None, h0=None,
                 white_step: bool = True, stream=None, use_torch_allocator: bool = True):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2503_09713_b200 needs a CUDA device (sm_100a); there is no CPU fallback")
        self.torch = torch
        self.lib = load()
        self.device = torch.device("cuda", torch.cuda.current_device())
        self.stream = stream if stream is not None else torch.cuda.current_stream()
        self.n = int(pos.shape[1])
        self.box = Box((C.c_double * 3)(*box_lo), (C.c_double * 3)(*box_hi), (C.c_int32 * 3)(*[int(x) for x in periodic]))
        self.params = params if params is not None else default_params()
        self._allocator = _TorchAllocator(self.device) if use_torch_allocator else None
        args = [self._as_input(a) for a in (pos, vel, mass, u, h0)]
        mems = {self._mem(a) for a in args if a is not None}
        assert len(mems) == 1, "all input buffers must live on the same side (host or device)"
        self.ctx = C.c_void_p()
        rc = self.lib.sph_init_ex(C.byref(self.ctx), self.n, mems.pop(), *[_ptr(a) for a in args], C.byref(self.box),
                                  C.byref(self.params), C.c_void_p(self.stream.cuda_stream),
                                  C.byref(self._allocator.struct) if self._allocator else None, int(white_step))
        self._check(rc)

    @classmethod
    def from_sph_init(cls, pos, vel, mass, u, box_lo, box_hi, periodic, gamma: float, hfact: float):
        """north_star's entry point ``sph_init``: device tensors, default parameters with the given gamma and hfact,
        the NULL stream, cudaMalloc, no initial smoothing lengths (fallback of reading A9); runs the white step."""
        import torch
        self = cls.__new__(cls)
        self.torch, self.lib = torch, load()
        self.device = torch.device("cuda", torch.cuda.current_device())
        self.stream = torch.cuda.default_stream()
        self.n = int(pos.shape[1])
        self.box = Box((C.c_double * 3)(*box_lo), (C.c_double * 3)(*box_hi), (C.c_int32 * 3)(*[int(x) for x in periodic]))
        self.params = default_params(gamma=gamma, hfact=hfact)
        self._allocator = None
        args = [a.contiguous() for a in (pos, vel, mass, u)]
        assert all(a.is_cuda and a.dtype == torch.float64 for a in args)
        torch.cuda.synchronize()          # the inputs were produced on torch's stream; sph_init works on the NULL stream
        self.ctx = C.c_void_p()
        self._check(self.lib.sph_init(C.byref(self.ctx), self.n, *[_ptr(a) for a in args], C.byref(self.box),
                                      float(gamma), float(hfact)))
        return self

    @classmethod
    def from_workload(cls, w, device_inputs: bool = True, **kw):
        import torch
        params = kw.pop("params", None) or params_for(w)
        arrs = [w.pos, w.vel, w.mass, w.u, w.h0]
        if device_inputs:
            arrs = [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in arrs]
        return cls(arrs[0], arrs[1], arrs[2], arrs[3], w.box_lo, w.box_hi, w.periodic, params=params, h0=arrs[4], **kw)

    # ---- helpers
    def _as_input(self, a):
        if a is None:
            return None
        if isinstance(a, np.ndarray):
            return np.ascontiguousarray(a, dtype=np.float64)
        assert a.dtype == self.torch.float64
        return a.contiguous()

    def _mem(self, a):
        if isinstance(a, np.ndarray) or not a.is_cuda:
            return SPH_MEM_HOST
        return SPH_MEM_DEVICE

    def _check(self, rc):
        if rc != 0:
            msg = self.lib.sph_last_error(self.ctx).decode() if self.ctx else ""
            raise SphError(rc, msg)

    def close(self):
        if getattr(self, "ctx", None):
            self.lib.sph_free(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- the hot path (names follow the C ABI)
    def build_tree(self):
        self._check(self.lib.sph_build_tree(self.ctx))

    def compute_density(self):
        self._check(self.lib.sph_compute_density(self.ctx))

    def compute_forces(self):
        self._check(self.lib.sph_compute_forces(self.ctx))

    def step_leapfrog(self, dt: float = 0.0, want_dt: bool = False):
        out = C.c_double()
        self._check(self.lib.sph_step_leapfrog(self.ctx, float(dt), C.byref(out) if want_dt else None))
        return out.value if want_dt else None

    # ---- field access
    def get_fields(self, names=("pos", "vel", "u", "h", "rho", "omega", "acc", "dudt"), host: bool = False, out=None):
        """Dict of fields in original order: device float64 tensors, or host (pinned) tensors if ``host``."""
        torch = self.torch
        order = ("pos", "vel", "u", "h", "rho", "omega", "acc", "dudt")
        res = {}
        for k in names:
            if out is not None and k in out:
                res[k] = out[k]
            else:
                shape = (3, self.n) if k in ("pos", "vel", "acc") else (self.n,)
                res[k] = torch.empty(shape, dtype=torch.float64, device="cpu" if host else self.device,
                                     pin_memory=host)
        with torch.cuda.stream(self.stream):
            self._check(self.lib.sph_get_fields(self.ctx, SPH_MEM_HOST if host else SPH_MEM_DEVICE,
                                                *[_ptr(res.get(k)) for k in order]))
        return res

    def set_fields(self, pos=None, vel=None, u=None, h=None, acc=None, dudt=None):
        args = [self._as_input(a) for a in (pos, vel, u, h, acc, dudt)]
        mems = {self._mem(a) for a in args if a is not None}
        assert len(mems) == 1
        self._check(self.lib.sph_set_fields(self.ctx, mems.pop(), *[_ptr(a) for a in args]))

    def get_keys_perm(self):
        keys = np.empty(self.n, dtype=np.uint64)
        perm = np.empty(self.n, dtype=np.uint32)
        self._check(self.lib.sph_get_keys_perm(self.ctx, SPH_MEM_HOST, _ptr(keys), _ptr(perm)))
        return keys, perm

    def get_tree(self):
        n, ni = self.n, max(self.n - 1, 0)
        t = dict(left=np.zeros(ni, np.int32), right=np.zeros(ni, np.int32), lflag=np.zeros(ni, np.uint8),
                 rflag=np.zeros(ni, np.uint8), parent=np.zeros(2 * n - 1, np.int32), rlo=np.zeros(ni, np.int32),
                 rhi=np.zeros(ni, np.int32), aabb=np.zeros((ni, 6), np.float64), hmax=np.zeros(ni, np.float64))
        self._check(self.lib.sph_get_tree(self.ctx, SPH_MEM_HOST, *[_ptr(t[k]) for k in
                                          ("left", "right", "lflag", "rflag", "parent", "rlo", "rhi", "aabb", "hmax")]))
        return t

    def get_neighbours(self):
        offs = np.empty(self.n + 1, dtype=np.uint64)
        self._check(self.lib.sph_get_neighbours(self.ctx, SPH_MEM_HOST, _ptr(offs), None, 0))
        idx = np.empty(int(offs[-1]), dtype=np.uint32)
        self._check(self.lib.sph_get_neighbours(self.ctx, SPH_MEM_HOST, _ptr(offs), _ptr(idx), idx.size))
        return offs, idx

    def get_neighbours_range(self, first: int, count: int):
        """Lists of the sorted slots [first, first + count): (offs relative to the first list, idx)."""
        offs = np.empty(count + 1, dtype=np.uint64)
        self._check(self.lib.sph_get_neighbours_range(self.ctx, SPH_MEM_HOST, first, count, _ptr(offs), None, 0))
        idx = np.empty(int(offs[-1] - offs[0]), dtype=np.uint32)
        self._check(self.lib.sph_get_neighbours_range(self.ctx, SPH_MEM_HOST, first, count, _ptr(offs), _ptr(idx), idx.size))
        return offs - offs[0], idx

    def get_alpha(self):
        """Shock-switch alpha_a in original order (av_switch = 1), as a numpy array."""
        out = np.empty(self.n, dtype=np.float64)
        self._check(self.lib.sph_get_alpha(self.ctx, SPH_MEM_HOST, _ptr(out)))
        return out

    def get_leaves(self):
        """Reduced leaves of Alg. 1 (leaf_reduction >= 1): (leaf codes u64[n_leaf], id map u32[n_leaf + 1])."""
        codes = np.empty(self.n, dtype=np.uint64)
        ids = np.empty(self.n + 1, dtype=np.uint32)
        nl = C.c_int64()
        self._check(self.lib.sph_get_leaves(self.ctx, SPH_MEM_HOST, C.byref(nl), _ptr(codes), _ptr(ids)))
        return codes[:nl.value].copy(), ids[:nl.value + 1].copy()

    def stats(self) -> dict:
        s = Stats()
        self._check(self.lib.sph_get_stats(self.ctx, C.byref(s)))
        return s.as_dict()

    def reset_timers(self):
        self._check(self.lib.sph_reset_timers(self.ctx))


def scan_u32_noalloc(counts, out=None, stream=None):
    """``sph_scan_u32_noalloc``: exclusive prefix sum of a CUDA uint32 tensor (as int32 storage is not accepted: pass
    ``torch.uint32`` or ``torch.int32`` holding non-negative counts) into an int64 tensor of n + 1 entries, without any
    device allocation inside the library (argument marshalling only; ``out`` may be passed to avoid torch's own)."""
    import torch
    assert counts.is_cuda and counts.is_contiguous() and counts.element_size() == 4
    n = counts.numel()
    if out is None:
        out = torch.empty(n + 1, dtype=torch.int64, device=counts.device)
    assert out.is_cuda and out.is_contiguous() and out.element_size() == 8 and out.numel() >= n + 1
    st = stream if stream is not None else torch.cuda.current_stream()
    rc = load().sph_scan_u32_noalloc(C.c_void_p(counts.data_ptr()), C.c_void_p(out.data_ptr()), n, C.c_void_p(st.cuda_stream))
    if rc != 0:
        raise SphError(rc, load().sph_noalloc_last_error().decode())
    return out


def measure_fp64_peak() -> float:
    import torch
    out = C.c_double()
    rc = load().sph_measure_fp64_peak(C.byref(out), C.c_void_p(torch.cuda.current_stream().cuda_stream))
    if rc != 0:
        raise SphError(rc, "sph_measure_fp64_peak")
    return out.value
