"""gsnfs_rans_decode_static: the occupancy-byte decoder for callers that may not allocate device memory.

Some users of this library decode inside a player / render loop in which device allocation is not an option: the
application's own pool (a tensor framework's caching allocator, an engine's arena) already owns the GPU, the memory
budget is frozen after start-up, or the loop cannot take the device-wide synchronisation a cudaMalloc brings.  Every
other call needs a gsnfs_ctx, and creating one is a cudaMalloc.  The static entry point needs no context: its block-offset
table is a fixed 256 KB array inside the library (limit: 32 MiB of occupancy bytes per call).

What is checked here: on the same coded stream the static call writes exactly the bytes and the info record that the
context path (gsnfs_rans_decode) writes -- byte work, so the tolerance is the one tests/test_gpu_rans.py uses: none --
on two calls in a row, the second on a shorter, different stream so that anything left in the shared table by the
first call would show; a damaged stream is reported the same way; sizes beyond the limit are refused before anything
runs; and a warmed-up call leaves the device's free memory where it was.

The file is named to be collected last (pytest -x stops at the first failure); it builds its own context and inputs,
so it gives the same result run alone in a fresh process or after the rest of the suite."""
import numpy as np
import pytest
import torch

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


def occupancy_like(seed: int, n: int) -> np.ndarray:
    """Bytes with the skew of an octree occupancy stream (a few child patterns dominate); no zero bytes."""
    rng = np.random.default_rng(seed)
    common = np.array([0x01, 0x02, 0x04, 0x08, 0x10, 0x20, 0x40, 0x80, 0x03, 0x11, 0x18, 0xff], np.uint8)
    x = rng.integers(1, 256, n).astype(np.uint8)
    pick = rng.random(n) < 0.8
    x[pick] = common[rng.integers(0, len(common), int(pick.sum()))]
    return x


def encode_on_device(B, ctx, x):
    n = len(x)
    d_x = torch.from_numpy(x).to(DEV)
    d_f = torch.zeros(256, dtype=torch.int16, device=DEV)
    d_nw = torch.zeros(B.gsnfs_rans_blocks(n), dtype=torch.int16, device=DEV)
    d_p = torch.zeros(B.gsnfs_rans_capacity(n), dtype=torch.uint8, device=DEV)
    d_info = torch.zeros(2, dtype=torch.int64, device=DEV)
    B.gsnfs_rans_encode(ctx, d_x, n, None, d_f, d_nw, d_p, d_info)
    torch.cuda.synchronize()
    nbytes, _, status = B.rlgr_info(d_info)
    assert status == 0
    return d_f, d_nw, d_p, nbytes


def decode_both(B, ctx, d_p, nbytes, d_f, d_nw, n):
    """(context path, static path): each (output bytes, info record) as host arrays; buffers pre-filled differently."""
    res = []
    for static in (False, True):
        d_out = torch.full((n,), 0xA5 if static else 0x5A, dtype=torch.uint8, device=DEV)
        d_info = torch.full((2,), -1, dtype=torch.int64, device=DEV)
        if static:
            B.gsnfs_rans_decode_static(d_p, nbytes, d_f, d_nw, n, d_out, d_info)
        else:
            B.gsnfs_rans_decode(ctx, d_p, nbytes, d_f, d_nw, n, d_out, d_info)
        torch.cuda.synchronize()
        res.append((d_out.cpu().numpy(), d_info.cpu().numpy()))
    return res


def test_static_decoder_matches_the_context_path_on_two_calls_in_a_row(B, ctx):
    # first call: many blocks with a ragged last one; second call: fewer, different blocks (stale offsets would show)
    for seed, n in ((11, 3_000_000 + 777), (12, 70_000 + 5)):
        x = occupancy_like(seed, n)
        d_f, d_nw, d_p, nbytes = encode_on_device(B, ctx, x)
        (ref_out, ref_info), (out, info) = decode_both(B, ctx, d_p, nbytes, d_f, d_nw, n)
        assert np.array_equal(ref_out, x)                       # the existing path is itself right on this input
        assert np.array_equal(out, ref_out), f"static decoder differs from gsnfs_rans_decode at n = {n}"
        assert np.array_equal(info, ref_info)
        assert B.rlgr_info(torch.from_numpy(info))[2] == 0
    # a damaged stream: both paths flag it, and write the same bytes
    d_p2 = d_p.clone()
    d_p2[100] ^= 0x10
    (ref_out, ref_info), (out, info) = decode_both(B, ctx, d_p2, nbytes, d_f, d_nw, n)
    assert B.rlgr_info(torch.from_numpy(ref_info))[2] & 1
    assert np.array_equal(info, ref_info) and np.array_equal(out, ref_out)


def test_static_decoder_allocates_nothing_once_warm(B, ctx):
    x = occupancy_like(13, 500_000)
    d_f, d_nw, d_p, nbytes = encode_on_device(B, ctx, x)
    d_out = torch.zeros(len(x), dtype=torch.uint8, device=DEV)
    d_info = torch.zeros(2, dtype=torch.int64, device=DEV)
    B.gsnfs_rans_decode_static(d_p, nbytes, d_f, d_nw, len(x), d_out, d_info)     # set-up + lazy kernel loading
    torch.cuda.synchronize()
    free_before, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        B.gsnfs_rans_decode_static(d_p, nbytes, d_f, d_nw, len(x), d_out, d_info)
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info()
    assert free_after == free_before
    assert np.array_equal(d_out.cpu().numpy(), x)


def test_static_decoder_limits_and_empty_input(B):
    small = torch.zeros(16, dtype=torch.uint8, device=DEV)
    f = torch.zeros(256, dtype=torch.int16, device=DEV)
    nw = torch.zeros(16, dtype=torch.int16, device=DEV)
    info = torch.full((2,), -1, dtype=torch.int64, device=DEV)
    with pytest.raises(B.GsnfsError) as e:        # refused on the host, before any kernel could touch the small buffers
        B.gsnfs_rans_decode_static(small, 16, f, nw, B.GSNFS_RANS_STATIC_MAX_BYTES + 1, small, info)
    assert e.value.status == -2 and "limit" in str(e.value)
    torch.cuda.synchronize()
    assert bool((info == -1).all())
    B.gsnfs_rans_decode_static(small, 0, f, nw, 0, small, info)                   # n = 0: valid, an empty result
    torch.cuda.synchronize()
    assert B.rlgr_info(info) == (0, 0, 0)
