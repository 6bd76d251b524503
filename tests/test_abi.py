"""Host-side checks that need no GPU: the C-ABI library builds, loads and exports every symbol that
include/sph_b200.h declares; the binding's struct layouts match the header; without a device the entry points
fail loudly (no CPU fallback)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2503_09713_b200 import build, binding
    build.build()
    return binding.load()


def _declared_functions():
    text = open(os.path.join(ROOT, "include", "sph_b200.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(sph_[a-z0-9_]+)\s*\(", text)) - {"sph_alloc_fn", "sph_free_fn"})


def test_library_exports_every_declared_symbol(lib):
    from paper_2503_09713_b200 import binding
    names = _declared_functions()
    assert len(names) >= 20
    for n in names:
        assert hasattr(lib, n), f"{n} declared in sph_b200.h but not exported"
    assert sorted(binding.SYMBOLS) == names


def test_default_params_match_header_citations(lib):
    from paper_2503_09713_b200 import binding
    p = binding.default_params()
    assert (p.hfact, p.chi, p.lambda_, p.eps_h) == (1.2, 1.1, 1.2, 1e-6)
    assert (p.alpha_av, p.beta_av, p.beta_u, p.c_cour, p.c_force) == (1.0, 2.0, 1.0, 0.3, 0.25)
    assert p.gamma == pytest.approx(5.0 / 3.0) and p.max_h_iter == 50 and p.max_restarts == 50 and p.eos == 0
    assert (p.eps_v, p.lambda_stiff, p.max_recycle) == (0.0, 2.0, 10)      # corrector re-cycle off by default
    assert C.sizeof(binding.Params) == 10 * 8 + 4 * 4 + 5 * 8 + 3 * 8 + 2 * 8 + 4 * 4 + 2 * 4 + 3 * 8
    assert (p.av_switch, p.alpha_min, p.alpha_max, p.sigma_decay) == (0, 0.0, 1.0, 0.1)
    assert (p.group_max, p.morton_bits) == (32, 21)
    assert C.sizeof(binding.Box) == 6 * 8 + 3 * 4 + 4   # padded to 8


def test_argument_errors_and_no_cpu_fallback(lib):
    """Bad arguments are rejected before any device work; without a CUDA device sph_init* returns
    SPH_ERR_DEVICE instead of computing anything on the host."""
    from paper_2503_09713_b200 import binding
    ctx = C.c_void_p()
    box = binding.Box((C.c_double * 3)(0, 0, 0), (C.c_double * 3)(1, 1, 1), (C.c_int32 * 3)(1, 1, 1))
    x = np.zeros(3)
    assert lib.sph_init_ex(C.byref(ctx), 0, 0, x.ctypes.data, x.ctypes.data, x.ctypes.data, x.ctypes.data, None,
                           C.byref(box), None, None, None, 1) == -1
    assert lib.sph_init_ex(C.byref(ctx), 1, 0, None, x.ctypes.data, x.ctypes.data, x.ctypes.data, None,
                           C.byref(box), None, None, None, 1) == -1
    assert lib.sph_build_tree(None) == -1
    try:
        import torch
        has_gpu = torch.cuda.is_available()
    except Exception:
        has_gpu = False
    if not has_gpu:
        rc = lib.sph_init_ex(C.byref(ctx), 1, 0, x.ctypes.data, x.ctypes.data, x.ctypes.data, x.ctypes.data, None,
                             C.byref(box), None, None, None, 1)
        assert rc == -2
        from paper_2503_09713_b200 import workloads as W
        with pytest.raises(RuntimeError):
            binding.Sim.from_workload(W.config(0))


def test_product_does_not_import_oracle():
    """The product path must not route through the oracle (or any CPU fallback)."""
    pkg = os.path.join(ROOT, "paper_2503_09713_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text and "sph_oracle" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2503_09713_b200" not in text and "from paper_2503_09713_b200" not in text, f


def test_workload_generators_are_deterministic_and_shaped():
    from paper_2503_09713_b200 import workloads as W
    a, b = W.config(0), W.config(0)
    assert np.array_equal(a.pos, b.pos) and a.n == 4096
    assert np.all((a.pos >= 0) & (a.pos < 1)) and a.mass.sum() == pytest.approx(1.0)
    s = W.sod(16, 8)
    assert s.n == 16 * 8 * 8 + 8 * 4 * 4 and np.all(s.pos[0] >= -0.5) and np.all(s.pos[0] < 0.5)
    assert W.sod(32, 16).n == 589_824 // 64                  # C1 is sod(128, 64): 64 times as many sites
    d = W.disc(2000, seed=1)
    R = np.hypot(d.pos[0], d.pos[1])
    assert R.min() >= 2 and R.max() <= 10 and np.all(np.abs(d.pos[2]) <= 3 * 0.05 * R * (R / 2) ** 0.25 + 1e-12)
    u = W.splitmix_u01(1, np.arange(100000, dtype=np.uint64), 0)
    assert 0 <= u.min() and u.max() < 1 and abs(u.mean() - 0.5) < 0.01


def test_sedov_workload_recipe():
    """The Sedov-Taylor set-up: periodic HCP lattice (every site has 12 nearest neighbours at
    one distance, to the few-per-cent stretch), unit density, injected energy sum m u = E0 to the lattice quadrature error."""
    from paper_2503_09713_b200 import workloads as W
    w = W.sedov(24)
    assert w.n == 24 * 28 * 30 and w.cfl == (0.1, 0.1) and w.periodic == (1, 1, 1)
    assert abs(w.mass.sum() / 1.2 ** 3 - 1.0) < 1e-12
    assert abs((w.mass * w.u).sum() - 1.0) < 1e-3 and (w.u > 0).sum() < w.n // 4
    L = 1.2
    d = w.pos[:, :, None] - w.pos[:, None, :200]
    d -= L * np.round(d / L)
    r = np.sqrt((d * d).sum(axis=0))
    r[r == 0] = 9.0
    dx = L / 24
    assert np.all(((r > 0.95 * dx) & (r < 1.05 * dx)).sum(axis=0) == 12) and r.min() > 0.95 * dx
