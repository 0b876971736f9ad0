"""Pins for the rANS oracle (oracle/rans_oracle.c; occupancy-byte entropy coding).  No GPU."""
import math
import os

import numpy as np
import pytest

from oracle import gsnfs_oracle as orc
from oracle import rans
from paper_2606_05650_b200 import synth

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "rans_stream.txt")


def test_hand_computed_block():
    line = [l for l in open(GOLD) if not l.startswith("#") and "|" in l][0]
    data, fs, words, hx = [t.strip() for t in line.split("|")]
    x = np.frombuffer(bytes.fromhex(data), dtype=np.uint8)
    f, nw, p = rans.encode(x)
    assert f[1] == 3072 and f[2] == 1024 and f.sum() == 4096 and nw.tolist() == [0]
    assert p.tobytes().hex() == hx
    back, bad = rans.decode(p, f, nw, len(x))
    assert not bad and np.array_equal(back, x)


def _py_model(x):
    hist = np.bincount(x, minlength=256).astype(object)
    S = len(x)
    f = [0 if h == 0 else max(1, h * 4096 // S) for h in hist]
    d = 4096 - sum(f)
    if d > 0:
        f[int(np.argmax(np.array(hist, dtype=np.int64)))] += d
    while d < 0:
        f[int(np.argmax(np.array(f)))] -= 1
        d += 1
    return f


def _py_decode_block(state, words, f, n):
    """Independent restatement of the decoder with python ints."""
    cum = np.concatenate([[0], np.cumsum(f)])
    x, w, out = state, 0, []
    for _ in range(n):
        slot = x & 4095
        s = int(np.searchsorted(cum, slot, side="right") - 1)
        out.append(s)
        x = f[s] * (x >> 12) + slot - int(cum[s])
        if x < 65536:
            x = (x << 16) | words[w]
            w += 1
    assert w == len(words) and x == 65536
    return out


@pytest.mark.parametrize("kind", ["occupancy", "skewed", "uniform255", "single", "two", "short"])
def test_model_roundtrip_python_decoder_and_entropy_bound(kind):
    rng = np.random.default_rng(len(kind))
    if kind == "occupancy":
        fr = synth.make_frame(1)
        x = orc.position_encode(fr.xyz, fr.bbox_min, fr.bbox_max, fr.depth)["occ"]
    elif kind == "skewed":
        x = rng.choice(np.arange(1, 256), size=20000, p=np.r_[0.7, np.full(254, 0.3 / 254)]).astype(np.uint8)
    elif kind == "uniform255":
        x = rng.integers(1, 256, 30000).astype(np.uint8)
    elif kind == "single":
        x = np.full(5000, 0xFF, np.uint8)
    elif kind == "two":
        x = np.array([1, 2] * 700 + [2], np.uint8)
    else:
        x = np.array([7], np.uint8)
    f, nw, p = rans.encode(x)
    assert f.tolist() == _py_model(x) and int(f.sum()) == 4096
    hist = np.bincount(x, minlength=256)
    assert np.all((f > 0) == (hist > 0))
    back, bad = rans.decode(p, f, nw, len(x))
    assert not bad and np.array_equal(back, x)
    # python decoder on every block
    off = 0
    for b, n_w in enumerate(nw.tolist()):
        state = int.from_bytes(p[off:off + 4].tobytes(), "little")
        words = [int.from_bytes(p[off + 4 + 2 * i:off + 6 + 2 * i].tobytes(), "little") for i in range(n_w)]
        blk = x[b * 1024:(b + 1) * 1024]
        assert _py_decode_block(state, words, [int(v) for v in f], len(blk)) == blk.tolist()
        off += 4 + 2 * n_w
    assert off == p.size
    # size: within the model's cross entropy + per-block flush (32-bit state + < 16 bits of slack)
    ideal = -sum(int(h) * math.log2(int(f[s]) / 4096.0) for s, h in enumerate(hist) if h)
    assert p.size * 8 <= ideal + 48 * len(nw) + 16
    assert p.size * 8 >= ideal - 1
    if kind == "occupancy":
        assert p.size < 0.85 * x.size            # occupancy bytes of surface data compress ("roughly halves")
    if kind == "single":
        assert p.size == 4 * len(nw)             # a one-symbol alphabet costs only the block states


def test_corruption_is_flagged_and_blocks_are_independent():
    rng = np.random.default_rng(2)
    x = rng.choice([0x18, 0xff, 0x01, 0x80, 0x11], size=5000, p=[.5, .2, .15, .1, .05]).astype(np.uint8)
    f, nw, p = rans.encode(x)
    assert rans.decode(p[:-2], f, nw, len(x))[1]
    q = p.copy(); q[10] ^= 0x40
    back, bad = rans.decode(q, f, nw, len(x))
    assert bad
    nblk = len(nw)
    off = np.concatenate([[0], np.cumsum(4 + 2 * nw.astype(np.int64))])
    blk = int(np.searchsorted(off, 10, side="right") - 1)
    for b in range(nblk):                          # only the damaged block can differ
        if b != blk:
            assert np.array_equal(back[b * 1024:(b + 1) * 1024], x[b * 1024:(b + 1) * 1024])
