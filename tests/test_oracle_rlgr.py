"""Pins for the RLGR oracle (oracle/rlgr_oracle.c; no GPU).  The paper names the coder and its block-parallel use
(Table A.5) but gives no rule, so the pins are: hand-computed streams (tests/golden), an independent
restatement of the rules with python bit lists, decode(encode(x)) = x, block independence, and size sanity."""
import os

import numpy as np
import pytest

from oracle import rlgr

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "rlgr_streams.txt")


def test_hand_computed_streams():
    n = 0
    for line in open(GOLD):
        if line.startswith("#") or "|" not in line:
            continue
        xs, hx = line.split("|")
        x = [int(t) for t in xs.split()]
        s, bits = rlgr.encode_block(x)
        assert s.hex() == hx.strip(), x
        assert bits == 4 * len(hx.strip())
        back, bad = rlgr.decode_block(s, len(x))
        assert not bad and back.tolist() == x
        n += 1
    assert n >= 7


# ------------------------------------------------------------------ independent restatement (python, bit lists)
def _fold(x):
    return 2 * x if x >= 0 else -2 * x - 1


def _gr(bits, u, st):
    kR = st["kRP"] >> 2
    p = u >> kR
    if p < 32:
        bits += [1] * p + [0] + [(u >> i) & 1 for i in range(kR - 1, -1, -1)]
    else:
        bits += [1] * 32 + [(u >> i) & 1 for i in range(31, -1, -1)]
    if p == 0:
        st["kRP"] = max(st["kRP"] - 2, 0)
    elif p > 1:
        st["kRP"] = min(st["kRP"] + min(p, 32) + 1, 127)


def _py_encode_block(xs):
    bits, st, kP, run = [], {"kRP": 8}, 0, 0
    for v in xs:
        k = kP >> 2
        if k == 0:
            _gr(bits, _fold(v), st)
            kP = min(kP + 3, 64) if v == 0 else max(kP - 1, 0)
        elif v == 0:
            run += 1
            if run == 1 << k:
                bits.append(0); run = 0; kP = min(kP + 2, 64)
        else:
            bits += [1] + [(run >> i) & 1 for i in range(k - 1, -1, -1)]
            run = 0
            _gr(bits, _fold(v) - 1, st)
            kP = max(kP - 3, 0)
    if run:
        bits.append(0)
    bits += [0] * (-len(bits) % 32)
    return bytes(int("".join(map(str, bits[i:i + 8])), 2) for i in range(0, len(bits), 8))


@pytest.mark.parametrize("kind", ["sparse", "dense", "laplace_fine", "zeros", "huge", "alternating", "ramp"])
def test_against_python_bit_lists_and_roundtrip(kind):
    rng = np.random.default_rng(hash(kind) % 1000)
    n = 3000
    x = {
        "sparse": lambda: (rng.random(n) < 0.05) * rng.integers(-4, 5, n),
        "dense": lambda: rng.integers(-40, 41, n),
        "laplace_fine": lambda: np.rint(rng.laplace(0, 300, n)).astype(np.int64),
        "zeros": lambda: np.zeros(n, np.int64),
        "huge": lambda: rng.integers(-2**31, 2**31, n),
        "alternating": lambda: np.tile([0, 0, 0, 1, 0, -1, 0, 0, 0, 0, 0, 0, 0, 0, 9], n // 15),
        "ramp": lambda: np.arange(n) - n // 2,
    }[kind]().astype(np.int32)
    s, bits = rlgr.encode_block(x)
    assert s == _py_encode_block([int(v) for v in x])
    back, bad = rlgr.decode_block(s, len(x))
    assert not bad and np.array_equal(back, x)
    if kind == "zeros":
        assert bits == 64 or bits == 32          # runs double: ~ log2(n) + a few bits for 3000 zeros
    if kind == "sparse":
        assert bits < 0.6 * n                    # well under one bit per coefficient at 5 % density


def test_extreme_values_and_long_runs():
    for x in ([-2**31], [2**31 - 1], [0] * 70000 + [1], [0] * 70000, [-2**31, 0, 2**31 - 1] * 5):
        s, bits = rlgr.encode_block(x)
        back, bad = rlgr.decode_block(s, len(x))
        assert not bad and back.tolist() == x
    s, bits = rlgr.encode_block([0] * 70000)
    assert bits == 64                             # k saturates at 16: 65536-zero runs


def test_truncated_stream_is_flagged():
    x = np.arange(-50, 50, dtype=np.int32)
    s, bits = rlgr.encode_block(x)
    back, bad = rlgr.decode_block(s[:4], len(x))
    assert bad


@pytest.mark.parametrize("n,C,B", [(1000, 3, 256), (2048, 8, 512), (777, 5, 8192), (1, 1, 256), (4097, 2, 4096)])
def test_tensor_layout_block_independence_roundtrip(n, C, B):
    rng = np.random.default_rng(n + C)
    q = (rng.laplace(0, 2.0, (n, C)) * (rng.random((n, C)) < 0.6)).round().astype(np.int32)
    bits, stream = rlgr.encode(q, B)
    nblk = (n + B - 1) // B
    assert bits.shape[0] == nblk * C and stream.size == int(bits.sum()) // 8 and np.all(bits % 32 == 0)
    # every block is the single-block stream of its rows of its channel, stored in the order b * C + c
    off = 0
    for b in range(nblk):
        for c in range(C):
            s, bl = rlgr.encode_block(q[b * B:(b + 1) * B, c])
            assert bl == bits[b * C + c] and stream[off:off + bl // 8].tobytes() == s
            off += bl // 8
    back, bad = rlgr.decode(stream, bits, n, C, B)
    assert not bad and np.array_equal(back, q)
    # independence: changing one coefficient changes the stream of its block only
    q2 = q.copy()
    q2[n // 2, C - 1] += 3
    bits2, stream2 = rlgr.encode(q2, B)
    changed = np.flatnonzero(bits != bits2).tolist()
    assert set(changed) <= {(n // 2 // B) * C + C - 1}


def test_smaller_blocks_cost_a_little_more():
    """Table A.5's trade-off: block size 512 costs on the order of a per cent more than 8192 (adaptation restarts)."""
    rng = np.random.default_rng(5)
    q = (rng.laplace(0, 1.5, (65536, 4)) * (rng.random((65536, 4)) < 0.5)).round().astype(np.int32)
    sizes = {B: rlgr.encode(q, B)[1].size for B in (256, 512, 2048, 8192)}
    assert sizes[256] >= sizes[512] >= sizes[2048] >= sizes[8192]
    assert sizes[512] <= 1.08 * sizes[8192]
