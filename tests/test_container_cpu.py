"""The bitstream container (host-only entry points of the C ABI): pack / unpack round trip,
layout invariants and damage detection.  No GPU."""
import numpy as np
import pytest


@pytest.fixture(scope="module")
def B():
    from paper_2606_05650_b200 import build, binding
    build.build()
    binding.lib()
    return binding


def _desc(B, depth=12, channels=56, nv=1000, ob=4321):
    d = B.GsnfsFrameDesc()
    d.depth, d.channels, d.n_voxels, d.occ_bytes, d.rlgr_block, d.flags = depth, channels, nv, ob, 2048, 5
    d.bbox_min[:] = [0.0, -1.0, 2.5]
    d.bbox_max[:] = [1.0, 1.0, 3.0]
    d.dz_round, d.recon_bias = 1.0 / 3.0, 0.125
    return d


def test_roundtrip_and_layout(B):
    rng = np.random.default_rng(0)
    secs = {B.SEC_LEVEL_SIZES: np.arange(13, dtype=np.uint32), B.SEC_QSTEP: rng.random(56).astype(np.float32),
            B.SEC_OCC_RAW: rng.integers(1, 256, 4321).astype(np.uint8), B.SEC_WEIGHTS: np.ones(1000, np.uint32),
            B.SEC_COEF_BITS: rng.integers(0, 9999, 28).astype(np.uint32) * 32, B.SEC_COEF_STREAM: rng.integers(0, 256, 70001).astype(np.uint8),
            B.SEC_KLT: np.zeros(0, np.float32)}
    buf = B.container_pack(_desc(B), secs)
    assert buf[:4].tobytes() == b"GSNF" and buf.size % 8 == 0
    d, out = B.container_unpack(buf)
    assert (d.depth, d.channels, d.n_voxels, d.occ_bytes, d.rlgr_block, d.flags) == (12, 56, 1000, 4321, 2048, 5)
    assert list(d.bbox_min) == [0.0, -1.0, 2.5] and abs(d.recon_bias - 0.125) < 1e-9
    assert set(out) == set(secs)
    for k, a in secs.items():
        assert out[k].tobytes() == a.tobytes()
        if a.nbytes:
            assert (out[k].ctypes.data - buf.ctypes.data) % 8 == 0          # 8-byte aligned payloads, zero copy
    # overhead: header + table + padding only
    assert buf.size <= sum(a.nbytes for a in secs.values()) + 80 + 24 * len(secs) + 8 * len(secs) + 8


def test_damage_is_detected(B):
    secs = {B.SEC_LEVEL_SIZES: np.arange(5, dtype=np.uint32), B.SEC_OCC_RAW: np.arange(1, 200, dtype=np.uint8)}
    buf = B.container_pack(_desc(B, depth=4), secs)
    for pos in (0, 5, 20, 70, buf.size - 3, buf.size // 2):
        bad = buf.copy()
        bad[pos] ^= 0x01
        with pytest.raises(B.GsnfsError) as e:
            B.container_unpack(bad)
        assert e.value.status == B.GSNFS_E_CORRUPT_STREAM, pos
    with pytest.raises(B.GsnfsError):
        B.container_unpack(buf[:buf.size - 8])
    with pytest.raises(B.GsnfsError):
        B.container_unpack(buf[:10])
    d, out = B.container_unpack(np.concatenate([buf, np.zeros(64, np.uint8)]))      # trailing bytes are not part of the frame
    assert out[B.SEC_OCC_RAW].tobytes() == secs[B.SEC_OCC_RAW].tobytes()
    assert B.container_unpack(B.container_pack(_desc(B), {}))[1] == {}
