"""GPU parity for the occupancy-byte entropy coder: static order-0 rANS
through the C ABI against oracle/rans_oracle.c -- byte work: model, word counts and payload compared bit for bit."""
import numpy as np
import pytest
import torch

from oracle import gsnfs_oracle as orc
from oracle import rans as orn
from paper_2606_05650_b200 import synth

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


@pytest.fixture(scope="module")
def B():
    from paper_2606_05650_b200 import binding
    binding.lib()
    return binding


@pytest.fixture(scope="module")
def ctx(B):
    c = B.Context(max_points=1_000_000, max_channels=8, max_depth=16)
    yield c
    c.close()


def gpu_encode(B, ctx, x, counts=None, capacity=None, n=None):
    n = len(x) if n is None else n
    d_x = torch.from_numpy(np.ascontiguousarray(x, np.uint8)).to(DEV) if len(x) else torch.zeros(4, dtype=torch.uint8, device=DEV)
    nb = B.gsnfs_rans_blocks(n)
    d_f = torch.zeros(256, dtype=torch.int16, device=DEV)
    d_nw = torch.full((max(nb, 1),), -1, dtype=torch.int16, device=DEV)
    d_p = torch.zeros(max(B.gsnfs_rans_capacity(n) if capacity is None else capacity, 4), dtype=torch.uint8, device=DEV)
    d_info = torch.zeros(2, dtype=torch.int64, device=DEV)
    B.gsnfs_rans_encode(ctx, d_x, n, counts, d_f, d_nw, d_p, d_info)
    torch.cuda.synchronize()
    nbytes, nblocks, status = B.rlgr_info(d_info)
    return d_f, d_nw, d_p, nbytes, nblocks, status


def check(B, ctx, x):
    f, nw, p = orn.encode(x)
    d_f, d_nw, d_p, nbytes, nblocks, status = gpu_encode(B, ctx, x)
    assert status == 0 and nblocks == len(nw) and nbytes == p.size
    assert np.array_equal(d_f.cpu().numpy().view(np.uint16), f)
    assert np.array_equal(d_nw[:len(nw)].cpu().numpy().view(np.uint16), nw)
    assert np.array_equal(d_p[:nbytes].cpu().numpy(), p)
    d_out = torch.full((max(len(x), 1),), 9, dtype=torch.uint8, device=DEV)
    d_info = torch.zeros(2, dtype=torch.int64, device=DEV)
    B.gsnfs_rans_decode(ctx, d_p, nbytes, d_f, d_nw, len(x), d_out, d_info)
    torch.cuda.synchronize()
    assert B.rlgr_info(d_info)[2] == 0 and np.array_equal(d_out[:len(x)].cpu().numpy(), x)
    return nbytes


@pytest.mark.parametrize("kind", ["config1", "config2", "skewed", "uniform255", "single", "tiny", "edge1024", "edge1025", "edge32768"])
def test_payload_bit_exact(B, ctx, kind):
    rng = np.random.default_rng(len(kind))
    if kind in ("config1", "config2"):
        fr = synth.make_frame(int(kind[-1]))
        x = orc.position_encode(fr.xyz, fr.bbox_min, fr.bbox_max, fr.depth)["occ"]
    elif kind == "skewed":
        x = rng.choice(np.arange(1, 256), size=200_000, p=np.r_[0.7, np.full(254, 0.3 / 254)]).astype(np.uint8)
    elif kind == "uniform255":
        x = rng.integers(1, 256, 70_000).astype(np.uint8)
    elif kind == "single":
        x = np.full(5000, 0xFF, np.uint8)
    elif kind == "tiny":
        x = np.array([7], np.uint8)
    else:
        x = rng.choice([0x18, 0xff, 0x01, 0x80, 0x11, 0x00], size=int(kind[4:]), p=[.5, .2, .14, .1, .05, .01]).astype(np.uint8)
    check(B, ctx, x)


def test_config3_occupancy_stream_chained_on_the_device(B, ctx):
    """The headline frame's occupancy stream, with its length read on the device from the encoder's counts."""
    fr = synth.make_frame(3)
    buf = B.FrameBuffers(fr.n, 8, fr.depth, DEV)
    B.gsnfs_octree_encode(ctx, torch.from_numpy(fr.xyz).to(DEV), fr.n, fr.bbox_min, fr.bbox_max, fr.depth, buf.occ,
                          buf.level_sizes, buf.perm, buf.voxel_keys, buf.voxel_start, buf.counts)
    torch.cuda.synchronize()
    ob = int(buf.counts.cpu()[1])
    x = buf.occ[:ob].cpu().numpy()
    f, nw, p = orn.encode(x)
    cap = buf.occ.numel()
    nb = B.gsnfs_rans_blocks(cap)
    d_f = torch.zeros(256, dtype=torch.int16, device=DEV)
    d_nw = torch.zeros(nb, dtype=torch.int16, device=DEV)
    d_p = torch.zeros(B.gsnfs_rans_capacity(cap), dtype=torch.uint8, device=DEV)
    d_info = torch.zeros(2, dtype=torch.int64, device=DEV)
    B.gsnfs_rans_encode(ctx, buf.occ, cap, buf.counts, d_f, d_nw, d_p, d_info)
    torch.cuda.synchronize()
    nbytes, nblocks, status = B.rlgr_info(d_info)
    assert status == 0 and nblocks == len(nw) and nbytes == p.size
    assert np.array_equal(d_p[:nbytes].cpu().numpy(), p) and np.array_equal(d_f.cpu().numpy().view(np.uint16), f)
    assert nbytes < 0.8 * ob
    print(f"config3 occupancy: {ob} -> {nbytes} bytes ({ob / nbytes:.2f}x)")


def test_capacity_and_corruption(B, ctx):
    rng = np.random.default_rng(1)
    x = rng.choice([0x18, 0xff, 0x01, 0x80, 0x11], size=50_000, p=[.5, .2, .15, .1, .05]).astype(np.uint8)
    d_f, d_nw, d_p, nbytes, nblocks, status = gpu_encode(B, ctx, x, capacity=1000)
    assert status & 2 and bool((d_p == 0).all())
    d_f, d_nw, d_p, nbytes, nblocks, status = gpu_encode(B, ctx, x)
    d_out = torch.zeros(len(x), dtype=torch.uint8, device=DEV)
    d_info = torch.zeros(2, dtype=torch.int64, device=DEV)
    for mutate in ("truncate", "flip", "model", "words"):
        p2, f2, nw2, nb2 = d_p.clone(), d_f.clone(), d_nw.clone(), nbytes
        if mutate == "truncate":
            nb2 = nbytes // 2
        elif mutate == "flip":
            p2[100] ^= 0x10
        elif mutate == "model":
            f2[0x18] += 1
        else:
            nw2[3] -= 1
        B.gsnfs_rans_decode(ctx, p2, nb2, f2, nw2, len(x), d_out, d_info)
        torch.cuda.synchronize()
        assert B.rlgr_info(d_info)[2] & 1, mutate
    B.gsnfs_rans_decode(ctx, d_p, nbytes, d_f, d_nw, len(x), d_out, d_info)
    torch.cuda.synchronize()
    assert B.rlgr_info(d_info)[2] == 0 and np.array_equal(d_out.cpu().numpy(), x)
