"""Pins for the oracle's position coder (no GPU).  Each check is independent of the oracle's own
formulae: the paper's printed values, brute-force set constructions, a recursive pointer octree
(PAPER.md:L97), closed forms and invariants."""
import os

import numpy as np
import pytest

from oracle import gsnfs_oracle as orc
from paper_2606_05650_b200 import synth

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _read_golden(name):
    rows = []
    with open(os.path.join(GOLD, name)) as f:
        for line in f:
            line = line.strip()
            if line and not line.startswith("#"):
                rows.append(line.split())
    return rows


# ------------------------------------------------------------------ Morton
def test_morton_paper_worked_values():
    for J, x, y, z, code in _read_golden("morton_examples.txt"):
        J, x, y, z = int(J), int(x), int(y), int(z)
        key = orc.morton_encode(np.array([[x, y, z]], dtype=np.uint64), J)[0]
        assert int(key) == int(code, 2)
        assert orc.morton_decode(np.array([key]), J)[0].tolist() == [x, y, z]
    # L142: parent of 100001 is 100; 5th child of node n is n*8 + 0b101
    assert (0b100001 >> 3) == 0b100
    assert orc.morton_encode(np.array([[1, 0, 2]], dtype=np.uint64), 2)[0] == 33
    assert orc.morton_encode(np.array([[1, 1, 2]], dtype=np.uint64), 2)[0] == 35


def test_morton_is_bit_interleave_bruteforce():
    # independent definition: build the bit string z_{J-1} y_{J-1} x_{J-1} ... z_0 y_0 x_0 as text
    rng = np.random.default_rng(0)
    for J in (1, 3, 7, 16, 21):
        v = rng.integers(0, 1 << J, (50, 3), dtype=np.uint64)
        keys = orc.morton_encode(v, J)
        for (x, y, z), k in zip(v.tolist(), keys.tolist()):
            s = "".join(f"{(z >> b) & 1}{(y >> b) & 1}{(x >> b) & 1}" for b in range(J - 1, -1, -1))
            assert k == int(s, 2)
            assert k < (1 << (3 * J))          # unused MSBs zero (L152)
        assert np.array_equal(orc.morton_decode(keys, J), v)


def test_morton_roundtrip_exhaustive_small():
    for J in (1, 2, 3, 4):
        g = np.arange(1 << J, dtype=np.uint64)
        v = np.stack(np.meshgrid(g, g, g, indexing="ij"), -1).reshape(-1, 3)
        keys = orc.morton_encode(v, J)
        assert sorted(keys.tolist()) == list(range(8 ** J))     # a bijection onto [0, 8^J)
        assert np.array_equal(orc.morton_decode(keys, J), v)


# ------------------------------------------------------------------ voxelise (L83-89, [O1][O2])
def test_voxelize_boundaries_and_exact_edges():
    J = 4
    lo, hi = np.zeros(3, np.float32), np.ones(3, np.float32)
    pts = np.array([[0.0, 0.0, 0.0], [1.0, 1.0, 1.0], [0.5, 0.25, 0.75],
                    [np.nextafter(np.float32(0.5), np.float32(0)), 0.0625, 0.9999999],
                    [-0.5, 2.0, 0.5]], dtype=np.float32)
    v = orc.voxelize(pts, lo, hi, J).tolist()
    assert v[0] == [0, 0, 0]
    assert v[1] == [15, 15, 15]                 # p = hi lands in the last voxel
    assert v[2] == [8, 4, 12]                   # exactly representable edges belong to the upper voxel
    assert v[3] == [7, 1, 15]
    assert v[4] == [0, 15, 8]                   # outside the bbox clamps
    # non-unit cuboid: per-axis scale (bounding *cuboid*, L83)
    lo2, hi2 = np.array([-1, 0, 2], np.float32), np.array([1, 4, 3], np.float32)
    v2 = orc.voxelize(np.array([[0.0, 1.0, 2.5]], np.float32), lo2, hi2, 3).tolist()
    assert v2 == [[4, 2, 4]]


def test_voxelize_matches_exact_rational_arithmetic():
    # for a unit cube and J <= 21, floor(p * 2^J) is exact in fp64, so python Fractions agree
    from fractions import Fraction
    rng = np.random.default_rng(1)
    p = rng.uniform(0, 1, (200, 3)).astype(np.float32)
    for J in (5, 16, 21):
        v = orc.voxelize(p, np.zeros(3, np.float32), np.ones(3, np.float32), J)
        for row, vr in zip(p.tolist(), v.tolist()):
            ref = [min(int(Fraction(c) * (1 << J)), (1 << J) - 1) for c in row]
            assert vr == ref


# ------------------------------------------------------------------ sort ([O8])
def test_sort_is_stable_and_matches_python_sorted():
    rng = np.random.default_rng(2)
    keys = rng.integers(0, 50, 2000, dtype=np.uint64)          # many ties
    perm = orc.sort_by_key(keys)
    ref = [i for _, i in sorted((int(k), i) for i, k in enumerate(keys.tolist()))]
    assert perm.tolist() == ref
    sk = keys[perm]
    assert np.all(sk[1:] >= sk[:-1])
    ties = sk[1:] == sk[:-1]
    assert np.all(perm[1:][ties] > perm[:-1][ties])


def test_unique_segments_and_merge_against_python_loops():
    rng = np.random.default_rng(3)
    keys = rng.integers(0, 40, 300, dtype=np.uint64)
    attr = rng.normal(0, 1, (300, 5)).astype(np.float32)
    perm = orc.sort_by_key(keys)
    vk, vs, w = orc.unique_segments(keys[perm])
    groups = {}
    for i, k in enumerate(keys.tolist()):
        groups.setdefault(k, []).append(i)
    ks = sorted(groups)
    assert vk.tolist() == ks
    assert w.tolist() == [len(groups[k]) for k in ks]
    assert int(w.sum()) == 300 and vs[-1] == 300
    merged = orc.merge_attributes(attr, perm, vs)
    for r, k in enumerate(ks):
        ref = np.mean(attr[groups[k]].astype(np.float64), axis=0)
        assert np.allclose(merged[r], ref, rtol=0, atol=1e-15)
        if len(groups[k]) == 1:                       # single Gaussian copied bit-exactly
            assert np.array_equal(merged[r].astype(np.float32), attr[groups[k][0]])


# ------------------------------------------------------------------ octree stream
def _bruteforce_stream(voxel_keys, J):
    """Independent of any sort: per-level python sets, then per parent test the 8 candidates."""
    leaf = set(int(k) for k in voxel_keys)
    levels = [None] * (J + 1)
    levels[J] = leaf
    for d in range(J - 1, -1, -1):
        levels[d] = set(c >> 3 for c in levels[d + 1])
    out = []
    for d in range(J):
        for p in sorted(levels[d]):
            byte = 0
            for i in range(8):
                if ((p << 3) + i) in levels[d + 1]:
                    byte |= 1 << i
            out.append(byte)
    return out, [len(levels[d]) for d in range(J + 1)]


class _Node:
    __slots__ = ("kids",)

    def __init__(self):
        self.kids = [None] * 8


def _recursive_level_order_stream(coords, J):
    """build a pointer octree top-down from integer coordinates, then emit occupancy
    bytes in one level-order (breadth-first) traversal visiting children 0..7 in order.  Child index
    = z y x bits at that depth (the Morton digit)."""
    root = _Node()
    for (x, y, z) in coords:
        n = root
        for b in range(J - 1, -1, -1):
            c = (((z >> b) & 1) << 2) | (((y >> b) & 1) << 1) | ((x >> b) & 1)
            if n.kids[c] is None:
                n.kids[c] = _Node()
            n = n.kids[c]
    out, frontier = [], [root]
    for _ in range(J):
        nxt = []
        for n in frontier:
            byte = 0
            for i in range(8):
                if n.kids[i] is not None:
                    byte |= 1 << i
                    nxt.append(n.kids[i])
            out.append(byte)
        frontier = nxt
    return out


def test_octree_fig2_example():
    rows = {r[0]: r[1:] for r in _read_golden("fig2_stream.txt")}
    vox = np.array([int(v) for v in rows["voxels"]], dtype=np.uint64)
    occ, sizes = orc.octree_encode(vox, 2)
    assert sizes.tolist() == [int(s) for s in rows["level_sizes"]]
    assert occ.tolist() == [int(b, 2) for b in rows["bytes"]]
    assert occ[0] == 0b00011000 and occ[1] == 0xFF                 # the paper's two printed bytes
    keys, coords, ok = orc.octree_decode(occ, sizes, 2)
    assert ok and keys.tolist() == vox.tolist()


@pytest.mark.parametrize("J,n,seed", [(1, 5, 0), (2, 11, 1), (3, 60, 2), (4, 300, 3), (6, 500, 4)])
def test_octree_stream_bruteforce_and_recursive(J, n, seed):
    rng = np.random.default_rng(seed)
    coords = rng.integers(0, 1 << J, (n, 3), dtype=np.uint64)
    keys = np.unique(orc.morton_encode(coords, J))
    occ, sizes = orc.octree_encode(keys, J)
    ref, ref_sizes = _bruteforce_stream(keys, J)
    assert occ.tolist() == ref
    assert sizes.tolist() == ref_sizes
    assert occ.tolist() == _recursive_level_order_stream(coords.tolist(), J)
    # invariants: no zero byte, sum popcount(level d) = |L_{d+1}|, |L_0| = 1, S = sum_{d<J} |L_d|
    assert np.all(occ != 0) and sizes[0] == 1 and occ.shape[0] == sizes[:-1].sum()
    ptr = 0
    for d in range(J):
        pc = sum(bin(b).count("1") for b in occ[ptr:ptr + sizes[d]].tolist())
        assert pc == sizes[d + 1]
        ptr += sizes[d]
    dk, dc, ok = orc.octree_decode(occ, sizes, J)
    assert ok and np.array_equal(dk, keys)
    assert sorted(map(tuple, dc.tolist())) == sorted(set(map(tuple, coords.tolist())))


def test_octree_full_cube_and_single_point():
    for J in (1, 2, 3):
        keys = np.arange(8 ** J, dtype=np.uint64)
        occ, sizes = orc.octree_encode(keys, J)
        assert occ.shape[0] == (8 ** J - 1) // 7 and np.all(occ == 0xFF)
        assert sizes.tolist() == [8 ** d for d in range(J + 1)]
    J = 7
    v = np.array([[5, 77, 100]], dtype=np.uint64)
    key = int(orc.morton_encode(v, J)[0])
    occ, sizes = orc.octree_encode(np.array([key], dtype=np.uint64), J)
    assert sizes.tolist() == [1] * (J + 1)
    # byte d = 1 << (d-th 3-bit digit of the code, most significant first)
    assert occ.tolist() == [1 << ((key >> (3 * (J - 1 - d))) & 7) for d in range(J)]


def test_octree_empty_and_corrupt():
    occ, sizes = orc.octree_encode(np.zeros(0, np.uint64), 5)
    assert occ.shape[0] == 0 and sizes.tolist() == [0] * 6
    k, c, ok = orc.octree_decode(occ, sizes, 5)
    assert ok and k.shape[0] == 0
    keys = np.array([1, 9, 300], dtype=np.uint64)
    occ, sizes = orc.octree_encode(keys, 3)
    bad = occ.copy()
    bad[1] = 0
    assert orc.octree_decode(bad, sizes, 3)[2] is False
    bad_sizes = sizes.copy()
    bad_sizes[3] += 1
    assert orc.octree_decode(occ, bad_sizes, 3)[2] is False


def test_position_encode_synthetic_config1():
    fr = synth.make_frame(1)
    pos = orc.position_encode(fr.xyz, fr.bbox_min, fr.bbox_max, fr.depth)
    assert sorted(pos["perm"].tolist()) == list(range(fr.n))
    assert int(pos["weights"].sum()) == fr.n
    dk, dc, ok = orc.octree_decode(pos["occ"], pos["level_sizes"], fr.depth)
    assert ok and np.array_equal(dk, pos["voxel_keys"])
    vox = orc.voxelize(fr.xyz, fr.bbox_min, fr.bbox_max, fr.depth)
    assert sorted(set(map(tuple, vox.tolist()))) == sorted(map(tuple, dc.tolist()))
    ref, ref_sizes = _bruteforce_stream(pos["voxel_keys"], fr.depth)
    assert pos["occ"].tolist() == ref and pos["level_sizes"].tolist() == ref_sizes
