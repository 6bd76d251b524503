"""`sph_scan_u32_noalloc`: the entry point that allocates nothing (static device scratch, fixed maximum size).

Collected last on purpose (file name): the suite runs with `pytest -x`, and a failure here must not hide other tests.
Checked against the EXISTING path -- the library's allocator-backed look-back scan, which produces the CSR offsets of
`sph_get_neighbours` -- on two calls in a row (integers: bit-exact, the bar of the other integer stages), then against
NumPy at the maximum size, the rejection beyond it, and that device memory in use does not grow across calls.
"""
import ctypes as C

import numpy as np
import pytest

from paper_2503_09713_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _offsets_existing_path(w):
    """CSR offsets of the neighbour cache from the existing path (sph_get_neighbours: k_scan over the list lengths)."""
    from paper_2503_09713_b200 import binding as B
    sim = B.Sim.from_workload(w, white_step=False)
    sim.build_tree()
    offs = np.empty(w.n + 1, dtype=np.uint64)
    sim._check(sim.lib.sph_get_neighbours(sim.ctx, B.SPH_MEM_HOST, B._ptr(offs), None, 0))
    sim.close()
    return offs


def test_noalloc_scan_matches_existing_path_two_calls_in_a_row():
    import torch
    from paper_2503_09713_b200 import binding as B
    lib = B.load()
    assert lib.sph_scan_noalloc_max_items() == 1 << 24

    cases = []
    for w in (W.random_cloud(5000, seed=3), W.cube(40, jitter=0.1, vel_amp=0.0, seed=2)):    # 3 tiles; 32 tiles, ragged tail
        offs = _offsets_existing_path(w)
        counts = np.diff(offs).astype(np.uint32)
        assert counts.min() >= 1 and int(counts.astype(np.uint64).sum()) == int(offs[-1])
        cases.append((torch.from_numpy(counts.view(np.int32)).cuda(), offs,
                      torch.empty(w.n + 1, dtype=torch.int64, device="cuda")))
    torch.cuda.synchronize()

    # two calls in a row on one stream (the second reuses the scratch the first left behind), then the first again
    order = [0, 1, 0]
    outs = [B.scan_u32_noalloc(cases[k][0], out=cases[k][2].clone()) for k in order]
    torch.cuda.synchronize()
    for k, out in zip(order, outs):
        assert np.array_equal(out.cpu().numpy().view(np.uint64), cases[k][1]), f"no-alloc scan differs from the existing path (case {k})"

    # device memory in use does not grow across further calls (outputs preallocated: nothing is allocated by anyone)
    free0, _ = torch.cuda.mem_get_info()
    for k in order:
        B.scan_u32_noalloc(cases[k][0], out=cases[k][2])
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 >= free0
    for k in (0, 1):
        assert np.array_equal(cases[k][2].cpu().numpy().view(np.uint64), cases[k][1])


def test_noalloc_scan_maximum_size_and_rejection():
    import torch
    from paper_2503_09713_b200 import binding as B
    lib = B.load()
    nmax = int(lib.sph_scan_noalloc_max_items())
    rng = np.random.default_rng(5)
    counts = rng.integers(0, 400, size=nmax, dtype=np.uint32)
    counts[::977] = 0xfffffff0                                  # large counts: the sums need all 64 bits of the output
    d = torch.from_numpy(counts.view(np.int32)).cuda()
    out = B.scan_u32_noalloc(d)
    small = B.scan_u32_noalloc(d[:2049].contiguous())           # right after: one tile + one item, stale status words beyond
    torch.cuda.synchronize()
    ref = np.concatenate([[0], np.cumsum(counts.astype(np.uint64))]).astype(np.uint64)
    assert np.array_equal(out.cpu().numpy().view(np.uint64), ref)
    assert np.array_equal(small.cpu().numpy().view(np.uint64), ref[:2050])
    # beyond the maximum: a clear error, nothing launched, nothing written
    before = out.clone()
    rc = lib.sph_scan_u32_noalloc(C.c_void_p(d.data_ptr()), C.c_void_p(out.data_ptr()), nmax + 1, None)
    assert rc == -8                                             # SPH_ERR_CAP
    msg = lib.sph_noalloc_last_error().decode()
    assert "exceeds the fixed maximum" in msg and str(nmax) in msg
    with pytest.raises(B.SphError) as e:
        B.scan_u32_noalloc(torch.zeros(nmax + 1, dtype=torch.int32, device="cuda"), out=torch.empty(nmax + 2, dtype=torch.int64, device="cuda"))
    assert e.value.code == -8
    assert lib.sph_scan_u32_noalloc(None, C.c_void_p(out.data_ptr()), 10, None) == -1      # SPH_ERR_ARG
    assert lib.sph_scan_u32_noalloc(C.c_void_p(d.data_ptr()), C.c_void_p(out.data_ptr()), 0, None) == -1
    torch.cuda.synchronize()
    assert torch.equal(out, before)
