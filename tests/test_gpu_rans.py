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


@pytest.mark.parametrize("shift_p,shift_o", [(0, 0), (1, 0), (2, 3), (4, 8), (6, 1), (8, 16)])
def test_decoder_accepts_any_buffer_alignment(B, ctx, shift_p, shift_o):
    """The decoder stages the payload with 16-byte copies and stores 16 output bytes at a time when the caller's buffers allow
    it; slices that start at other addresses (a section inside a larger buffer) take its byte-wise paths.  Same bytes out."""
    rng = np.random.default_rng(40 + shift_p)
    x = rng.choice([0x18, 0xff, 0x01, 0x80, 0x11, 0x22], size=100_000 + 333, p=[.5, .2, .14, .1, .05, .01]).astype(np.uint8)
    d_f, d_nw, d_p, nbytes, nblocks, status = gpu_encode(B, ctx, x)
    assert status == 0
    p_buf = torch.zeros(nbytes + 64, dtype=torch.uint8, device=DEV)
    p_view = p_buf[shift_p:shift_p + nbytes]
    p_view.copy_(d_p[:nbytes])
    o_buf = torch.full((len(x) + 64,), 9, dtype=torch.uint8, device=DEV)
    o_view = o_buf[shift_o:shift_o + len(x)]
    assert p_view.data_ptr() % 16 == shift_p % 16 and o_view.data_ptr() % 16 == shift_o % 16
    d_info = torch.full((2,), -1, dtype=torch.int64, device=DEV)
    B.gsnfs_rans_decode(ctx, p_view, nbytes, d_f, d_nw, len(x), o_view, d_info)
    torch.cuda.synchronize()
    assert B.rlgr_info(d_info)[2] == 0 and np.array_equal(o_view.cpu().numpy(), x)
    assert bool((o_buf[:shift_o] == 9).all()) and bool((o_buf[shift_o + len(x):] == 9).all())      # nothing outside the view
    d_info.fill_(-1)
    o_buf.fill_(9)
    B.gsnfs_rans_decode_static(p_view, nbytes, d_f, d_nw, len(x), o_view, d_info)
    torch.cuda.synchronize()
    assert B.rlgr_info(d_info)[2] == 0 and np.array_equal(o_view.cpu().numpy(), x)
    assert bool((o_buf[:shift_o] == 9).all()) and bool((o_buf[shift_o + len(x):] == 9).all())


def test_whole_frame_through_the_container(B):
    """A frame coded on the device (octree -> rANS, merge + RAHT + quantiser -> RLGR), framed by gsnfs_container_pack,
    parsed back, decoded on the device: voxels bit-exact, attributes as the raw-coefficient path gives them."""
    fr = synth.make_frame(2)
    n, C, J, blk = fr.n, fr.channels, fr.depth, 2048
    ctx = B.Context(max_points=n, max_channels=C, max_depth=J)
    try:
        buf = B.FrameBuffers(n, C, J, DEV)
        d_xyz, d_attr = torch.from_numpy(fr.xyz).to(DEV), torch.from_numpy(fr.attr).to(DEV)
        B.encode_frame(ctx, buf, d_xyz, d_attr, fr.bbox_min, fr.bbox_max, fr.qstep)
        cap = buf.occ.numel()
        d_f = torch.zeros(256, dtype=torch.int16, device=DEV)
        d_nw = torch.zeros(B.gsnfs_rans_blocks(cap), dtype=torch.int16, device=DEV)
        d_p = torch.zeros(B.gsnfs_rans_capacity(cap), dtype=torch.uint8, device=DEV)
        d_ri = torch.zeros(2, dtype=torch.int64, device=DEV)
        B.gsnfs_rans_encode(ctx, buf.occ, cap, buf.counts, d_f, d_nw, d_p, d_ri)
        d_bits = torch.zeros(B.gsnfs_rlgr_blocks(n, C, blk), dtype=torch.int32, device=DEV)
        d_stream = torch.zeros(B.gsnfs_rlgr_capacity(n, C, blk), dtype=torch.uint8, device=DEV)
        d_li = torch.zeros(2, dtype=torch.int64, device=DEV)
        B.gsnfs_rlgr_encode(ctx, buf.qcoeff, n, buf.counts, C, blk, d_bits, d_stream, d_li)
        torch.cuda.synchronize()
        cnt = buf.counts.cpu().numpy()
        nv, ob = int(cnt[0]), int(cnt[1])
        pbytes, pblocks, _ = B.rlgr_info(d_ri)
        sbytes, sblocks, _ = B.rlgr_info(d_li)
        desc = B.GsnfsFrameDesc()
        desc.depth, desc.channels, desc.n_voxels, desc.occ_bytes, desc.rlgr_block, desc.flags = J, C, nv, ob, blk, 0
        desc.bbox_min[:] = fr.bbox_min.tolist(); desc.bbox_max[:] = fr.bbox_max.tolist()
        desc.dz_round, desc.recon_bias = 1.0 / 3.0, 0.0
        file = B.container_pack(desc, {
            B.SEC_LEVEL_SIZES: buf.level_sizes.cpu().numpy(), B.SEC_QSTEP: fr.qstep,
            B.SEC_OCC_FREQ: d_f.cpu().numpy(), B.SEC_OCC_NWORDS: d_nw[:pblocks].cpu().numpy(), B.SEC_OCC_PAYLOAD: d_p[:pbytes].cpu().numpy(),
            B.SEC_WEIGHTS: buf.weights[:nv].cpu().numpy(),
            B.SEC_COEF_BITS: d_bits[:B.gsnfs_rlgr_blocks(nv, C, blk)].cpu().numpy(), B.SEC_COEF_STREAM: d_stream[:sbytes].cpu().numpy()})
        raw = n * 12 + n * C * 4
        print(f"container: {file.size} bytes for a {raw}-byte frame ({raw / file.size:.2f}x; occupancy {ob} -> {pbytes})")
        # ---- receiver
        d2, sec = B.container_unpack(file)
        J2, C2, nv2, ob2, blk2 = d2.depth, d2.channels, d2.n_voxels, d2.occ_bytes, d2.rlgr_block
        levels = sec[B.SEC_LEVEL_SIZES].view(np.uint32)
        qstep = sec[B.SEC_QSTEP].view(np.float32)
        dev = lambda a, dt: torch.from_numpy(np.ascontiguousarray(a).view(dt).copy()).to(DEV)
        r_occ = torch.zeros(max(ob2, 4), dtype=torch.uint8, device=DEV)
        info = torch.zeros(2, dtype=torch.int64, device=DEV)
        B.gsnfs_rans_decode(ctx, dev(sec[B.SEC_OCC_PAYLOAD], np.uint8), sec[B.SEC_OCC_PAYLOAD].size, dev(sec[B.SEC_OCC_FREQ], np.int16),
                            dev(sec[B.SEC_OCC_NWORDS], np.int16), ob2, r_occ, info)
        rbuf = B.FrameBuffers(nv2, C2, J2, DEV)
        B.gsnfs_octree_decode(ctx, r_occ, ob2, levels, J2, rbuf.dec_xyz, rbuf.dec_keys, rbuf.dec_counts)
        info2 = torch.zeros(2, dtype=torch.int64, device=DEV)
        B.gsnfs_rlgr_decode(ctx, dev(sec[B.SEC_COEF_STREAM], np.uint8), sec[B.SEC_COEF_STREAM].size,
                            dev(sec[B.SEC_COEF_BITS], np.int32), nv2, C2, blk2, rbuf.qcoeff, info2)
        B.gsnfs_raht_inverse(ctx, rbuf.dec_keys, dev(sec[B.SEC_WEIGHTS], np.int32), nv2, rbuf.dec_counts, J2, rbuf.qcoeff, None, C2,
                             qstep, (d2.dz_round, d2.recon_bias), rbuf.dec_attr)
        torch.cuda.synchronize()
        assert B.rlgr_info(info)[2] == 0 and B.rlgr_info(info2)[2] == 0 and int(rbuf.dec_counts.cpu()[2]) == 0
        assert torch.equal(r_occ[:ob2], buf.occ[:ob]) and torch.equal(rbuf.qcoeff[:nv2], buf.qcoeff[:nv])
        assert torch.equal(rbuf.dec_keys[:nv2], buf.voxel_keys[:nv])
        B.decode_frame(ctx, buf, buf.level_sizes.cpu().numpy(), ob, fr.qstep)
        torch.cuda.synchronize()
        assert torch.equal(rbuf.dec_attr[:nv2], buf.dec_attr[:nv]) and torch.equal(rbuf.dec_xyz[:nv2], buf.dec_xyz[:nv])
    finally:
        ctx.close()
