"""Pins for the oracle's integer stages (Morton keys, sort, radix tree, node boxes) -- CPU only.

Each test checks ``oracle/`` against something other than itself: values printed in the paper
(tests/golden/*.txt with citations), brute force, or an independent characterisation written here.
"""
import os

import numpy as np
import pytest

import oracle as O
from paper_2503_09713_b200 import workloads as W

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _gold(name):
    rows = {}
    with open(os.path.join(GOLD, name)) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            k, *v = line.split()
            rows[k] = v
    return rows


def test_prefix_worked_example():
    """delta(0101,0111) = 2, mask 1100, prefix 0100."""
    g = _gold("prefix_example.txt")
    beta = int(g["beta"][0])
    m1, m2 = int(g["m1"][0], 2), int(g["m2"][0], 2)
    assert m1 ^ m2 == int(g["xor"][0], 2)
    assert O.lib().orc_delta_beta(m1, m2, beta) == int(g["delta"][0])
    mask = O.lib().orc_prefix_mask(m1, m2, beta)
    assert mask == int(g["mask"][0], 2)
    assert m2 & mask == int(g["prefix"][0], 2)


def test_table_b2():
    """PAPER.md:899-907 (Table B2): all five rows for the 12-leaf example."""
    g = _gold("table_b2.txt")
    keys = np.array([int(v) for v in g["keys"]], dtype=np.uint64)
    t = O.tree(keys)
    ids = np.arange(11)
    endrange = np.where(ids == t["rlo"], t["rhi"], t["rlo"])
    assert t["left"].tolist() == [int(v) for v in g["left-child-id"]]
    assert t["right"].tolist() == [int(v) for v in g["right-child-id"]]
    assert t["lflag"].tolist() == [int(v) for v in g["left-child-flag"]]
    assert t["rflag"].tolist() == [int(v) for v in g["right-child-flag"]]
    assert endrange.tolist() == [int(v) for v in g["endrange"]]
    # every node index is one end of its own range (Karras convention)
    assert np.all((ids == t["rlo"]) | (ids == t["rhi"]))


def _deinterleave(key):
    X = np.zeros((3, key.size), dtype=np.uint64)
    for j in range(21):
        for c in range(3):
            bit = (key >> np.uint64(62 - 3 * j - c)) & np.uint64(1)
            X[c] |= bit << np.uint64(20 - j)
    return X


def test_morton_roundtrip_and_halfspace():
    """integer grid coordinates, X0 Y0 Z0 X1 ... interleave, X0 = 1 <=> X >= 2^(beta-1)."""
    w = W.random_cloud(5000, seed=3)
    box = O.make_box(w.box_lo, w.box_hi, w.periodic)
    key = O.morton_keys(w.pos, box)
    X = _deinterleave(key)
    expect = np.minimum(np.floor(w.pos / 1.0 * 2097152.0), 2097151).astype(np.uint64)
    assert np.array_equal(X, expect)
    assert np.all(key >> np.uint64(63) == 0)
    top = (key >> np.uint64(62)) & np.uint64(1)
    assert np.array_equal(top == 1, w.pos[0] >= 0.5)
    # order-preserving within an octant path: equal (Y,Z) prefix and larger X => larger key
    a = np.array([[0.1, 0.2, 0.3], [0.3, 0.3, 0.3], [0.3, 0.3, 0.3]])
    k = O.morton_keys(a, box)
    assert k[0] < k[1] < k[2]


def test_morton_cube_embedding_and_clamp():
    """Reading A1: one scale L_c = max extent for all axes; out-of-box positions clamp to the edge cells."""
    box = O.make_box((-0.5, -0.125, -0.125), (0.5, 0.125, 0.125), (1, 1, 1))
    pos = np.array([[-0.5, 0.4999999, 0.0, 2.0, -3.0], [-0.125, 0.1249, 0.0, 0.0, 0.0], [0.0, 0.0, 0.0, 9.0, -9.0]])
    X = _deinterleave(O.morton_keys(pos, box))
    assert X[0, 0] == 0 and X[1, 0] == 0
    assert X[1].max() < 2 ** 19 + 1  # y spans a quarter of the cube
    assert X[0, 2] == 2 ** 20 and X[1, 2] == 2 ** 18
    assert X[0, 3] == 2 ** 21 - 1 and X[2, 3] == 2 ** 21 - 1 and X[0, 4] == 0 and X[2, 4] == 0


def test_keys_unique_and_sorted_on_c0():
    w = W.config(0)
    box = O.make_box(w.box_lo, w.box_hi, w.periodic)
    key = O.morton_keys(w.pos, box)
    assert np.unique(key).size == w.n
    skey, perm = O.sort_keys(key)
    assert np.all(skey[1:] > skey[:-1])
    assert np.array_equal(np.sort(perm), np.arange(w.n))
    assert np.array_equal(key[perm], skey)


def test_sort_is_stable():
    rng = np.random.default_rng(1)
    key = rng.integers(0, 50, size=4000).astype(np.uint64)
    skey, perm = O.sort_keys(key)
    ref = np.argsort(key, kind="stable")
    assert np.array_equal(perm, ref.astype(np.uint32))
    assert np.array_equal(skey, key[ref])


def _delta(keys, i, j):
    """Common-prefix length of the (key, index) 96-bit strings, written independently of the oracle."""
    a = (int(keys[i]) << 32) | i
    b = (int(keys[j]) << 32) | j
    return 96 - (a ^ b).bit_length()


def _brute_nodes(keys):
    """All internal nodes of the radix tree as maximal common-prefix ranges (independent characterisation):
    [i,j], i<j, is a node iff extending it by one key on either side shortens the common prefix."""
    n = len(keys)
    nodes = set()
    for i in range(n):
        for j in range(i + 1, n):
            d = _delta(keys, i, j)
            left_ok = i == 0 or _delta(keys, i - 1, j) < d
            right_ok = j == n - 1 or _delta(keys, i, j + 1) < d
            if left_ok and right_ok:
                nodes.add((i, j))
    return nodes


@pytest.mark.parametrize("seed,n,dups", [(0, 40, False), (1, 97, False), (2, 64, True), (3, 33, True)])
def test_tree_matches_bruteforce_ranges(seed, n, dups):
    rng = np.random.default_rng(seed)
    keys = np.sort(rng.integers(0, 2 ** 12 if dups else 2 ** 62, size=n).astype(np.uint64))
    if dups:
        keys[5:9] = keys[5]
        keys[20:22] = keys[20]
        keys = np.sort(keys)
    t = O.tree(keys)
    got = set(zip(t["rlo"].tolist(), t["rhi"].tolist()))
    assert len(got) == n - 1
    assert got == _brute_nodes(keys)
    ids = np.arange(n - 1)
    assert np.all((ids == t["rlo"]) | (ids == t["rhi"]))
    assert t["rlo"][0] == 0 and t["rhi"][0] == n - 1 and t["parent"][0] == -1
    for i in range(n - 1):
        l, r = t["left"][i], t["right"][i]
        assert r == l + 1
        llo = l if t["lflag"][i] else t["rlo"][l]
        lhi = l if t["lflag"][i] else t["rhi"][l]
        rlo = r if t["rflag"][i] else t["rlo"][r]
        rhi = r if t["rflag"][i] else t["rhi"][r]
        assert (llo, rhi) == (t["rlo"][i], t["rhi"][i]) and lhi == l and rlo == r
        assert t["parent"][(n - 1 + l) if t["lflag"][i] else l] == i
        assert t["parent"][(n - 1 + r) if t["rflag"][i] else r] == i
    # depth bound: <= key length (+32 with the tie-break)
    depth = np.zeros(n - 1, int)
    for i in sorted(range(1, n - 1), key=lambda i: t["rhi"][i] - t["rlo"][i], reverse=True):
        depth[i] = depth[t["parent"][i]] + 1
    assert depth.max() <= 96


def test_tree_tiny():
    assert O.tree(np.array([5], dtype=np.uint64))["parent"].tolist() == [-1]
    t = O.tree(np.array([5, 9], dtype=np.uint64))
    assert (t["left"][0], t["right"][0], t["lflag"][0], t["rflag"][0]) == (0, 1, 1, 1)


def test_aabb_hmax_against_range_minmax():
    w = W.random_cloud(300, seed=5)
    box = O.make_box(w.box_lo, w.box_hi, w.periodic)
    skey, perm = O.sort_keys(O.morton_keys(w.pos, box))
    ps, hs = w.pos[:, perm], w.h0[perm]
    t = O.tree(skey)
    box6, hmax = O.aabb(t, ps, hs)
    for i in range(w.n - 1):
        sl = slice(t["rlo"][i], t["rhi"][i] + 1)
        assert np.array_equal(box6[i, :3], ps[:, sl].min(axis=1))
        assert np.array_equal(box6[i, 3:], ps[:, sl].max(axis=1))
        assert hmax[i] == hs[sl].max()


def test_morton_30bit_variant():
    """The paper's 32-bit codes (2^10 cells per axis): grid coordinates floor(t 2^10), the same
    interleave; since floor(floor(t 2^21) / 2^11) = floor(t 2^10), the 30-bit code is the top 30 bits of the 63-bit one."""
    w = W.random_cloud(5000, seed=8)
    box = O.make_box(w.box_lo, w.box_hi, w.periodic)
    k30 = O.morton_keys(w.pos, box, beta=10)
    assert np.all(k30 < 2 ** 30)
    assert np.array_equal(k30, O.morton_keys(w.pos, box) >> np.uint64(33))
    X = np.zeros((3, w.n), dtype=np.uint64)
    for j in range(10):
        for c in range(3):
            X[c] |= ((k30 >> np.uint64(29 - 3 * j - c)) & np.uint64(1)) << np.uint64(9 - j)
    assert np.array_equal(X, np.minimum(np.floor(w.pos * 1024.0), 1023).astype(np.uint64))
    edge = np.array([[1.0, -0.5, 0.999999999], [7.0, 0.0, 0.5], [0.25, 0.25, 0.25]])
    ke = O.morton_keys(edge, box, beta=10)
    assert ke[0] >> np.uint64(29) == 1 and ke[1] < 2 ** 29          # clamp to the edge cells on both sides
    # the tree over coarse codes has ties: broken by the sorted index, every internal node still splits its range
    skey, perm = O.sort_keys(O.morton_keys(w.pos, box, beta=4))       # 4096 cells for 5000 particles
    assert np.unique(skey).size < w.n
    t = O.tree(skey)
    assert np.all(t["rhi"] > t["rlo"])


# ---------------------------------------------------------------- Alg. 1: duplicate removal and leaf reduction

def _leaf_gold():
    rows, extra = {}, {}
    for line in open(os.path.join(GOLD, "leaf_reduction.txt")):
        if line.startswith("#") or not line.strip():
            continue
        t = line.split()
        if t[0] in ("keys", "dupkeys", "dupmask", "dupids"):
            extra[t[0]] = [int(v) for v in t[1:]]
        else:
            vals = [int(v) for v in t[1:]]
            # kept keys, then the id map: the id map starts at the first 0 after a non-zero entry or is the tail
            # whose last element is 12; split by length: n kept keys followed by n + 1 ids
            n = (len(vals) - 1) // 2
            rows[int(t[0])] = (vals[:n], vals[n:])
    return rows, extra


def test_leaf_reduction_worked_example():
    """Alg. 1 on the Table B2 key list, every pass worked by hand in tests/golden/leaf_reduction.txt."""
    rows, extra = _leaf_gold()
    keys = np.array(extra["keys"], dtype=np.uint64)
    for n_red, (kept, ids) in rows.items():
        xi, codes, idmap = O.leaf_reduction(keys, n_red)
        assert list(codes) == kept and list(idmap) == ids, n_red
        assert list(np.nonzero(xi)[0]) == ids[:-1]
    xi, codes, idmap = O.leaf_reduction(np.array(extra["dupkeys"], dtype=np.uint64), 0)
    assert list(xi) == extra["dupmask"] and list(idmap) == extra["dupids"] and list(codes) == [0, 1, 2, 3]


@pytest.mark.parametrize("seed", [1, 2, 3])
def test_leaf_reduction_merges_exactly_the_two_leaf_parents(seed):
    """App. C2: a code is removable iff it is the second leaf of a parent whose two children are both
    leaves. Brute force through the radix tree of the codes kept before each pass (built by the recursive oracle
    builder, which knows nothing of Alg. 1): the codes a pass removes are exactly the right children of the internal
    nodes whose two children are leaves; leaves stay contiguous, sorted and non-empty."""
    rng = np.random.default_rng(seed)
    keys = np.sort(rng.integers(0, 1 << 20, size=3000, dtype=np.uint64) << np.uint64(43 - 7 * seed))
    keys[100:110] = keys[100]                                  # duplicates
    keys = np.sort(keys)
    prev_codes = np.unique(keys)
    xi0, codes0, ids0 = O.leaf_reduction(keys, 0)
    assert np.array_equal(codes0, prev_codes) and np.array_equal(keys[ids0[:-1]], codes0)
    for n_red in range(1, 8):
        xi, codes, ids = O.leaf_reduction(keys, n_red)
        t = O.tree(prev_codes)
        both = (t["lflag"] == 1) & (t["rflag"] == 1)
        expect_removed = set(prev_codes[t["right"][both]].tolist()) if prev_codes.size > 1 else set()
        removed = set(prev_codes.tolist()) - set(codes.tolist())
        assert removed == expect_removed and len(removed) > 0
        assert np.array_equal(keys[ids[:-1]], codes) and ids[0] == 0 and ids[-1] == keys.size
        assert np.all(np.diff(ids.astype(np.int64)) > 0) and np.all(np.diff(codes.astype(np.int64)) > 0)
        prev_codes = codes
    # every leaf of the reduced list is a prefix class: its objects share more leading bits with one another than with
    # either neighbouring leaf (the reduced tree "mirrors the initial one")
    for j in range(len(codes)):
        lo, hi = int(ids[j]), int(ids[j + 1]) - 1
        inner = 64 if lo == hi or keys[lo] == keys[hi] else 64 - int(keys[lo] ^ keys[hi]).bit_length()
        if lo > 0:
            assert 64 - int(keys[lo - 1] ^ keys[lo]).bit_length() < inner
        if hi + 1 < keys.size:
            assert 64 - int(keys[hi] ^ keys[hi + 1]).bit_length() < inner
