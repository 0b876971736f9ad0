"""Race / bounds evidence that does not need compute-sanitizer (closed on this GPU pool, see profiles/r2_sanitizer.md):
every ABI call of the hot path run repeatedly must give bit-identical outputs (a data race between CTAs or warps shows up
as run-to-run differences), and must not write a byte outside the extents gsnfs.h promises (guard bands around every
caller buffer)."""
import numpy as np
import pytest
import torch

from paper_2606_05650_b200 import synth

pytestmark = pytest.mark.gpu
DEV = "cuda:0"
GUARD = 1024          # elements of guard band on each side


@pytest.fixture(scope="module")
def B():
    from paper_2606_05650_b200 import binding
    binding.lib()
    return binding


class Guarded:
    """A tensor with a poisoned guard band in front of and behind the part handed to the library."""

    def __init__(self, n, dtype, shape=None):
        self.full = torch.empty(n + 2 * GUARD, dtype=dtype, device=DEV)
        self.poison = {torch.uint8: 0xA5, torch.int32: 0x5A5A5A5A, torch.int64: 0x5A5A5A5A5A5A5A5A, torch.float32: 12345.678,
                       torch.int16: 0x5A5A}[dtype]
        self.full.fill_(self.poison)
        self.t = self.full[GUARD:GUARD + n]
        if shape is not None:
            self.t = self.t.view(*shape)
        self.n = n

    def intact(self):
        p = torch.full((GUARD,), self.poison, dtype=self.full.dtype, device=DEV)
        return bool(torch.equal(self.full[:GUARD], p)) and bool(torch.equal(self.full[GUARD + self.n:], p))


def run_all(B, ctx, fr, g):
    n, C, J = fr.n, fr.channels, fr.depth
    blk = 512
    B.gsnfs_octree_encode(ctx, g["xyz"].t, n, fr.bbox_min, fr.bbox_max, J, g["occ"].t, g["levels"].t, g["perm"].t, g["vkeys"].t,
                          g["vstart"].t, g["counts"].t)
    B.gsnfs_voxel_merge(ctx, g["attr"].t, C, n, g["perm"].t, g["vstart"].t, g["counts"].t, g["merged"].t, g["w"].t)
    B.gsnfs_raht_forward(ctx, g["vkeys"].t, g["w"].t, n, g["counts"].t, J, g["merged"].t, C, fr.qstep, None, g["q"].t, g["coef"].t)
    B.gsnfs_merge_raht_forward(ctx, g["vkeys"].t, g["perm"].t, g["vstart"].t, n, g["counts"].t, J, g["attr"].t, C, fr.qstep, None,
                               g["w2"].t, g["q2"].t, None)
    B.gsnfs_quantize(ctx, g["coef"].t, n, g["counts"].t, C, fr.qstep, None, g["q3"].t)
    B.gsnfs_rlgr_encode(ctx, g["q"].t, n, g["counts"].t, C, blk, g["bits"].t, g["stream"].t, g["rinfo"].t)
    B.gsnfs_rans_encode(ctx, g["occ"].t, g["occ"].n, g["counts"].t, g["freq"].t, g["nw"].t, g["payload"].t, g["ainfo"].t)
    torch.cuda.synchronize()
    cnt = g["counts"].t.cpu().numpy()
    nv, ob = int(cnt[0]), int(cnt[1])
    levels = g["levels"].t.cpu().numpy()
    B.gsnfs_octree_decode(ctx, g["occ"].t, ob, levels, J, g["dxyz"].t, g["dkeys"].t, g["dcounts"].t)
    B.gsnfs_raht_inverse(ctx, g["dkeys"].t, g["w"].t, nv, None, J, g["q"].t, None, C, fr.qstep, None, g["dattr"].t)
    sb = B.rlgr_info(g["rinfo"].t)[0]
    B.gsnfs_rlgr_decode(ctx, g["stream"].t, sb, g["bits"].t, nv, C, blk, g["qback"].t, g["rinfo2"].t)
    pb = B.rlgr_info(g["ainfo"].t)[0]
    B.gsnfs_rans_decode(ctx, g["payload"].t, pb, g["freq"].t, g["nw"].t, ob, g["occback"].t, g["ainfo2"].t)
    if C >= 11 and (C - 11) % 3 == 0:
        B.gsnfs_klt_fit(ctx, g["attr"].t, n, None, C, g["klt"].t)
        B.gsnfs_color_forward(ctx, g["attr"].t, n, None, C, g["klt"].t, g["col"].t)
    torch.cuda.synchronize()
    return nv, ob, sb, pb


@pytest.mark.parametrize("maker", ["config1", "dense", "pointcloud_small", "long_runs"])
def test_repeatable_and_in_bounds(B, maker):
    fr = {"config1": lambda: synth.make_frame(1), "dense": lambda: synth.make_dense_frame(20_000, 5, 56, seed=9),
          "pointcloud_small": lambda: synth.make_pointcloud_frame(n=60_000, depth=8),
          "long_runs": lambda: synth.make_dense_frame(50_000, 2, 56, seed=11)}[maker]()     # chunk-wise merge pre-pass
    n, C, J = fr.n, fr.channels, fr.depth
    ctx = B.Context(max_points=n, max_channels=max(C, 4), max_depth=J)
    try:
        cap = B.gsnfs_occ_capacity(n, J)
        i32, u8, f32, i64, i16 = torch.int32, torch.uint8, torch.float32, torch.int64, torch.int16
        spec = {"xyz": (n * 3, f32, (n, 3)), "attr": (n * C, f32, (n, C)), "occ": (cap, u8, None), "levels": (J + 1, i32, None),
                "perm": (n, i32, None), "vkeys": (n, i64, None), "vstart": (n + 1, i32, None), "counts": (4, i32, None),
                "merged": (n * C, f32, (n, C)), "w": (n, i32, None), "w2": (n, i32, None), "q": (n * C, i32, (n, C)),
                "q2": (n * C, i32, (n, C)), "q3": (n * C, i32, (n, C)), "coef": (n * C, f32, (n, C)),
                "bits": (B.gsnfs_rlgr_blocks(n, C, 512), i32, None), "stream": (B.gsnfs_rlgr_capacity(n, C, 512), u8, None),
                "rinfo": (2, i64, None), "rinfo2": (2, i64, None), "ainfo": (2, i64, None), "ainfo2": (2, i64, None),
                "freq": (256, i16, None), "nw": (B.gsnfs_rans_blocks(cap), i16, None), "payload": (B.gsnfs_rans_capacity(cap), u8, None),
                "dxyz": (n * 3, i32, (n, 3)), "dkeys": (n, i64, None), "dcounts": (4, i32, None), "dattr": (n * C, f32, (n, C)),
                "qback": (n * C, i32, (n, C)), "occback": (cap, u8, None), "klt": (max(B.gsnfs_klt_floats(C), 4), f32, None),
                "col": (n * C, f32, (n, C))}
        g = {k: Guarded(*v) for k, v in spec.items()}
        g["xyz"].t.copy_(torch.from_numpy(fr.xyz))
        g["attr"].t.copy_(torch.from_numpy(fr.attr))
        first = None
        for rep in range(12):
            for k in ("q", "q2", "q3", "coef", "dattr", "occback", "qback", "stream", "payload"):
                g[k].t.zero_()
            nv, ob, sb, pb = run_all(B, ctx, fr, g)
            snap = {"occ": g["occ"].t[:ob].clone(), "perm": g["perm"].t.clone(), "vkeys": g["vkeys"].t[:nv].clone(),
                    "w": g["w"].t[:nv].clone(), "q": g["q"].t[:nv].clone(), "q2": g["q2"].t[:nv].clone(), "q3": g["q3"].t[:nv].clone(),
                    "coef": g["coef"].t[:nv].clone(), "stream": g["stream"].t[:sb].clone(), "payload": g["payload"].t[:pb].clone(),
                    "dxyz": g["dxyz"].t[:nv].clone(), "dattr": g["dattr"].t[:nv].clone(), "klt": g["klt"].t.clone(),
                    "col": g["col"].t.clone()}
            assert torch.equal(g["qback"].t[:nv], g["q"].t[:nv]) and torch.equal(g["occback"].t[:ob], g["occ"].t[:ob])
            assert torch.equal(g["q"].t[:nv], g["q2"].t[:nv]) and torch.equal(g["q"].t[:nv], g["q3"].t[:nv])
            if first is None:
                first = snap
            else:
                for k in first:
                    assert torch.equal(first[k], snap[k]), (maker, rep, k)
            for k, gb in g.items():
                assert gb.intact(), (maker, rep, k)
        assert ctx.poll_status() == B.GSNFS_OK
    finally:
        ctx.close()
