"""GPU parity for the block-parallel RLGR coder (Table A.5): the CUDA path
through the C ABI against oracle/rlgr_oracle.c -- integer work, so block sizes and stream bytes are compared bit for bit."""
import numpy as np
import pytest
import torch

from oracle import gsnfs_oracle as orc
from oracle import rlgr as orl
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
    c = B.Context(max_points=1_000_000, max_channels=64, max_depth=16)
    yield c
    c.close()


def gpu_encode(B, ctx, q, block, capacity=None, counts=None, n_rows=None):
    n, C = q.shape
    n_rows = n if n_rows is None else n_rows
    d_q = torch.from_numpy(np.ascontiguousarray(q, dtype=np.int32)).to(DEV)
    nb = B.gsnfs_rlgr_blocks(n_rows, C, block)
    cap = B.gsnfs_rlgr_capacity(n_rows, C, block) if capacity is None else capacity
    bits = torch.full((max(nb, 1),), -1, dtype=torch.int32, device=DEV)
    stream = torch.zeros(max(cap, 4), dtype=torch.uint8, device=DEV)
    info = torch.full((2,), -1, dtype=torch.int64, device=DEV)
    B.gsnfs_rlgr_encode(ctx, d_q if n else torch.zeros((1, C), dtype=torch.int32, device=DEV), n_rows, counts, C, block, bits,
                        stream, info)
    torch.cuda.synchronize()
    nbytes, nblocks, status = B.rlgr_info(info)
    return bits[:nb].cpu().numpy().view(np.uint32), stream, nbytes, nblocks, status, d_q


def gpu_decode(B, ctx, stream, nbytes, bits, n, C, block):
    d_bits = torch.from_numpy(np.ascontiguousarray(bits).view(np.int32)).to(DEV)
    out = torch.full((max(n, 1), C), 77, dtype=torch.int32, device=DEV)
    info = torch.zeros(2, dtype=torch.int64, device=DEV)
    B.gsnfs_rlgr_decode(ctx, stream, nbytes, d_bits, n, C, block, out, info)
    torch.cuda.synchronize()
    return out[:n].cpu().numpy(), B.rlgr_info(info)


def check_case(B, ctx, q, block, capacity=None):
    n, C = q.shape
    ref_bits, ref_stream = orl.encode(q, block)
    bits, stream, nbytes, nblocks, status, _ = gpu_encode(B, ctx, q, block, capacity)
    assert status == 0 and nblocks == ref_bits.size and nbytes == ref_stream.size
    assert np.array_equal(bits, ref_bits)
    assert np.array_equal(stream[:nbytes].cpu().numpy(), ref_stream)
    back, (_, _, st) = gpu_decode(B, ctx, stream, nbytes, bits, n, C, block)
    assert st == 0 and np.array_equal(back, q)
    return nbytes


@pytest.mark.parametrize("kind,n,C,block", [
    ("laplace", 5000, 56, 512), ("laplace", 4097, 56, 4096), ("sparse", 20000, 56, 2048), ("zeros", 3000, 8, 256),
    ("huge", 1500, 12, 256), ("dense", 777, 3, 8192), ("mixed", 1, 1, 64), ("mixed", 65, 7, 64), ("mixed", 33000, 35, 1024),
    ("laplace", 2000, 208, 512)])
def test_streams_bit_exact(B, kind, n, C, block):
    ctx = B.Context(max_points=max(n, 64), max_channels=max(C, 4), max_depth=8)
    try:
        rng = np.random.default_rng(n * 7 + C)
        q = {
            "laplace": lambda: np.rint(rng.laplace(0, 40, (n, C))),
            "sparse": lambda: (rng.random((n, C)) < 0.03) * rng.integers(-6, 7, (n, C)),
            "zeros": lambda: np.zeros((n, C)),
            "huge": lambda: rng.integers(-2**31, 2**31, (n, C)),
            "dense": lambda: rng.integers(-300, 301, (n, C)),
            "mixed": lambda: np.rint(rng.laplace(0, 3, (n, C))) * (rng.random((n, C)) < 0.5),
        }[kind]().astype(np.int32)
        # incompressible input expands (escape codes): the recommended capacity is the raw size, so give it room
        check_case(B, ctx, q, block, capacity=12 * n * C + 64 if kind == "huge" else None)
    finally:
        ctx.close()


def test_real_coefficients_all_table_a5_block_sizes(B, ctx):
    """Quantised RAHT coefficients of config 2 through every block size of Table A.5; the size ordering of the table
    (smaller blocks cost a little more) holds for the GPU streams too."""
    fr = synth.make_frame(2)
    ref = orc.encode_frame(fr.xyz, fr.attr, fr.bbox_min, fr.bbox_max, fr.depth, fr.qstep)
    q = ref["qcoeff"].astype(np.int32)
    sizes = {}
    for block in (256, 512, 1024, 2048, 4096, 8192):
        sizes[block] = check_case(B, ctx, q, block)
    assert sizes[256] >= sizes[512] >= sizes[2048] >= sizes[8192]
    assert sizes[512] <= 1.05 * sizes[8192]


@pytest.mark.parametrize("block", [512, 2048])
def test_config3_full_size_sampled_blocks_and_roundtrip(B, ctx, block):
    """BASELINE.json configs[2] at full size, at the block size bench.py times (RLGR_BLOCK = 512: 1954 CTAs) and at 2048
    (489 CTAs, a different occupancy regime): header compared in full with the oracle, decode(encode(q)) = q on the device,
    200 sampled block streams compared byte for byte."""
    rng = np.random.default_rng(11)
    n, C = 1_000_000, 56
    scale = np.concatenate([np.full(3, 60.0), np.full(4, 40.0), [30.0], np.full(3, 25.0), np.full(45, 6.0)])
    q = np.rint(rng.laplace(0, 1, (n, C)) * scale[None, :]).astype(np.int32)
    bits, stream, nbytes, nblocks, status, d_q = gpu_encode(B, ctx, q, block)
    assert status == 0
    ref_bits = np.zeros(nblocks, np.uint32)
    orl._L().rlgr_oracle_encode(q.ctypes.data, n, C, block, ref_bits.ctypes.data, None)
    assert np.array_equal(bits, ref_bits) and nbytes == int(ref_bits.astype(np.int64).sum()) // 8
    off = np.concatenate([[0], np.cumsum(ref_bits.astype(np.int64) // 8)])
    host = stream[:nbytes].cpu().numpy()
    for e in rng.integers(0, nblocks, 200).tolist():
        b, c = divmod(e, C)
        s, bl = orl.encode_block(q[b * block:(b + 1) * block, c])
        assert host[off[e]:off[e + 1]].tobytes() == s
    d_bits = torch.from_numpy(bits.view(np.int32)).to(DEV)
    out = torch.empty((n, C), dtype=torch.int32, device=DEV)
    info = torch.zeros(2, dtype=torch.int64, device=DEV)
    B.gsnfs_rlgr_decode(ctx, stream, nbytes, d_bits, n, C, block, out, info)
    torch.cuda.synchronize()
    assert B.rlgr_info(info)[2] == 0 and torch.equal(out, d_q)


def test_device_counts_chain_capacity_and_corruption(B, ctx):
    rng = np.random.default_rng(3)
    n, C, block = 10_000, 56, 512
    q = np.rint(rng.laplace(0, 20, (n, C))).astype(np.int32)
    # N_v read on the device: rows beyond it are not coded, their blocks have length 0
    counts = torch.tensor([7_000, 0, 0, 0], dtype=torch.int32, device=DEV)
    bits, stream, nbytes, nblocks, status, _ = gpu_encode(B, ctx, q, block, counts=counts)
    ref_bits, ref_stream = orl.encode(q[:7000], block)
    assert status == 0 and nbytes == ref_stream.size
    assert np.array_equal(bits[:ref_bits.size], ref_bits) and np.all(bits[ref_bits.size:] == 0)
    assert np.array_equal(stream[:nbytes].cpu().numpy(), ref_stream)
    # a stream buffer that is too small: reported, nothing written
    bits, stream, nbytes, nblocks, status, _ = gpu_encode(B, ctx, q, block, capacity=4096)
    assert status & 2 and nbytes > 4096 and bool((stream == 0).all())
    # corrupt / truncated streams are flagged, the call stays in bounds
    bits, stream, nbytes, nblocks, status, _ = gpu_encode(B, ctx, q, block)
    back, (_, _, st) = gpu_decode(B, ctx, stream, nbytes // 2, bits, n, C, block)
    assert st & 1
    bad_bits = bits.copy()
    bad_bits[5] -= 32                                     # a block shorter than what its coefficients need
    back, (_, _, st) = gpu_decode(B, ctx, stream, nbytes, bad_bits, n, C, block)
    assert st & 1
    # an entry damaged by a part of a word moves every later block of its row off a 4-byte boundary: flagged (status
    # bit 0), no misaligned load, the context stays usable
    for k, delta in ((5, 8), (5, 16), (0, 24), (C + 3, 8)):
        bad_bits = bits.copy()
        bad_bits[k] -= delta
        back, (_, _, st) = gpu_decode(B, ctx, stream, nbytes, bad_bits, n, C, block)
        assert st & 1, (k, delta)
    back, (_, _, st) = gpu_decode(B, ctx, stream, nbytes, bits, n, C, block)
    assert st == 0 and np.array_equal(back, q)
    # device-side N_v = 0 with a host bound > 0 (an empty frame, or one the decoder flagged): an empty stream, and the
    # info record is written (not left stale)
    zero = torch.zeros(4, dtype=torch.int32, device=DEV)
    ebits, _, nbytes0, nblocks0, status0, _ = gpu_encode(B, ctx, q, block, counts=zero)
    assert (nbytes0, status0) == (0, 0) and nblocks0 == ebits.size and np.all(ebits == 0)
    for bad_block in (32, 100_000):
        with pytest.raises(B.GsnfsError):
            gpu_encode(B, ctx, q, bad_block, capacity=1 << 20)


def test_packed_host_frame_calls(B):
    """gsnfs_frame_{encode,decode}_host_packed: the end-to-end path with RLGR bytes crossing PCIe instead of raw
    coefficients; stream and header bit-exact against the oracle chain, decoded attributes as in the raw-coefficient path."""
    fr = synth.make_frame(2)
    ref = orc.encode_frame(fr.xyz, fr.attr, fr.bbox_min, fr.bbox_max, fr.depth, fr.qstep)
    n, C, J, blk = fr.n, fr.channels, fr.depth, 2048
    ctx = B.Context(max_points=n, max_channels=C, max_depth=J)
    try:
        pin = lambda *s, dt: torch.empty(s, dtype=dt).pin_memory()
        h_xyz, h_attr = torch.from_numpy(fr.xyz).pin_memory(), torch.from_numpy(fr.attr).pin_memory()
        h_occ, h_lev = pin(B.gsnfs_occ_capacity(n, J), dt=torch.uint8), pin(J + 1, dt=torch.int32)
        h_w, h_cnt, h_info = pin(n, dt=torch.int32), pin(4, dt=torch.int32), pin(2, dt=torch.int64)
        h_bits = pin(B.gsnfs_rlgr_blocks(n, C, blk), dt=torch.int32)
        h_stream = pin(B.gsnfs_rlgr_capacity(n, C, blk), dt=torch.uint8)
        for _ in range(2):      # twice: the second call reuses the staging pool and the copy stream
            B.gsnfs_frame_encode_host_packed(ctx, h_xyz, h_attr, n, C, fr.bbox_min, fr.bbox_max, J, fr.qstep, None, blk,
                                             h_occ, h_lev, h_w, h_bits, h_stream, h_cnt, h_info)
        # an argument error that is only found after the attribute copy was queued (an empty bounding box is rejected by
        # the position coder): the call fails, returns with no DMA in flight on the caller's pinned buffers, and the
        # context serves the next frame
        with pytest.raises(B.GsnfsError):
            B.gsnfs_frame_encode_host_packed(ctx, h_xyz, h_attr, n, C, fr.bbox_min, fr.bbox_min, J, fr.qstep, None, blk,
                                             h_occ, h_lev, h_w, h_bits, h_stream, h_cnt, h_info)
        assert torch.cuda.current_stream().query()
        B.gsnfs_frame_encode_host_packed(ctx, h_xyz, h_attr, n, C, fr.bbox_min, fr.bbox_max, J, fr.qstep, None, blk,
                                         h_occ, h_lev, h_w, h_bits, h_stream, h_cnt, h_info)
        nv, ob = int(h_cnt[0]), int(h_cnt[1])
        nbytes = int(h_info.numpy().view(np.uint64)[0])
        assert nv == len(ref["voxel_keys"]) and np.array_equal(h_occ[:ob].numpy(), ref["occ"])
        # the GPU's quantised coefficients differ from the oracle's in <= 1e-4 of the entries (+-1), so the stream is
        # compared with the oracle coder applied to the GPU's own coefficients, which the raw-path call returns
        h_q = pin(n, C, dt=torch.int32)
        B.gsnfs_frame_encode_host(ctx, h_xyz, h_attr, n, C, fr.bbox_min, fr.bbox_max, J, fr.qstep, None,
                                  h_occ, h_lev, h_w, h_q, h_cnt)
        ref_bits, ref_stream = orl.encode(h_q[:nv].numpy(), blk)
        assert nbytes == ref_stream.size and np.array_equal(h_stream[:nbytes].numpy(), ref_stream)
        assert np.array_equal(h_bits[:ref_bits.size].numpy().view(np.uint32), ref_bits)
        assert nbytes < 0.5 * nv * C * 4                       # and it is worth shipping
        h_vx, h_out, h_cnt2 = pin(n, 3, dt=torch.int32), pin(n, C, dt=torch.float32), pin(4, dt=torch.int32)
        B.gsnfs_frame_decode_host_packed(ctx, h_occ, ob, h_lev.numpy(), J, h_w, h_bits, h_stream, nbytes, blk, C, fr.qstep,
                                         None, h_vx, h_out, h_cnt2)
        assert int(h_cnt2[2]) == 0
        h_out2 = pin(n, C, dt=torch.float32)
        B.gsnfs_frame_decode_host(ctx, h_occ, ob, h_lev.numpy(), J, h_w, h_q, C, fr.qstep, None, h_vx, h_out2, h_cnt2)
        assert torch.equal(h_out[:nv], h_out2[:nv])             # same coefficients in, same attributes out
        dk, dc, ok = orc.octree_decode(ref["occ"], ref["level_sizes"], J)
        assert np.array_equal(h_vx[:nv].numpy().astype(np.uint64), dc)
        # a damaged coefficient stream is reported as a corrupt frame
        bad = h_bits.clone().pin_memory()
        bad[3] -= 64
        B.gsnfs_frame_decode_host_packed(ctx, h_occ, ob, h_lev.numpy(), J, h_w, bad, h_stream, nbytes, blk, C, fr.qstep,
                                         None, h_vx, h_out, h_cnt2)
        assert int(h_cnt2[2]) & 1
        # so is a header entry damaged by part of a word (later blocks of the row would start off a 4-byte boundary): the
        # call reports status bit 0 instead of faulting, and the context still decodes the intact frame afterwards
        for delta in (8, 16):
            bad = h_bits.clone().pin_memory()
            bad[3] -= delta
            B.gsnfs_frame_decode_host_packed(ctx, h_occ, ob, h_lev.numpy(), J, h_w, bad, h_stream, nbytes, blk, C, fr.qstep,
                                             None, h_vx, h_out, h_cnt2)
            assert int(h_cnt2[2]) & 1, delta
        B.gsnfs_frame_decode_host_packed(ctx, h_occ, ob, h_lev.numpy(), J, h_w, h_bits, h_stream, nbytes, blk, C, fr.qstep,
                                         None, h_vx, h_out, h_cnt2)
        assert int(h_cnt2[2]) == 0 and torch.equal(h_out[:nv], h_out2[:nv])
    finally:
        ctx.close()
