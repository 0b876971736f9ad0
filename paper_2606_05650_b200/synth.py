"""Seeded synthetic 3DGS frames (inputs only -- none of the codec's arithmetic lives here).

These frames stand in for the paper's datasets (HiFi4G, N3DV, 8i, CMU Panoptic, static scenes;
PAPER.md:L301-303, L434, L645), none of which is available offline.  They take the *shapes* of
those workloads: N Gaussians, C = 56 fp32 attribute channels at SH degree 3 (PAPER.md:L17-27,
Table 4), surface-like geometry, octree depth J.  The recipe is the one stated in
DESIGN.md "Input recipe" (from SURVEY.md section 8(d) / BASELINE.json configs).

Both the oracle tests and the CUDA path's tests/bench draw their inputs from this module; it
imports neither of them.  Everything is computed in fp64 with numpy ``default_rng(seed)`` (PCG64),
in the order written below, clipped to the unit cube and cast to fp32.
"""
from __future__ import annotations

import dataclasses

import numpy as np

N_CHANNELS = 56  # log-scale 3, rotation 4, opacity 1, SH DC 3, SH AC 45


@dataclasses.dataclass
class Frame:
    """One synthetic frame.  ``xyz``/``attr`` are C-contiguous fp32 host arrays."""

    name: str
    xyz: np.ndarray        # (N, 3) fp32 in [0, 1]^3
    attr: np.ndarray       # (N, C) fp32 row-major
    qstep: np.ndarray      # (C,) fp32, channel range / qdiv
    depth: int             # octree depth J
    qdiv: int              # D
    bbox_min: np.ndarray   # (3,) fp32
    bbox_max: np.ndarray   # (3,) fp32

    @property
    def n(self) -> int:
        return int(self.xyz.shape[0])

    @property
    def channels(self) -> int:
        return int(self.attr.shape[1])


# ----------------------------------------------------------------------------- geometry
def _unit_vectors(rng: np.random.Generator, n: int) -> np.ndarray:
    v = rng.standard_normal((n, 3))
    nrm = np.linalg.norm(v, axis=1, keepdims=True)
    nrm[nrm == 0.0] = 1.0
    return v / nrm


def _make_spheres(rng, k):
    return {"c": rng.uniform(0.3, 0.7, (k, 3)), "r": rng.uniform(0.1, 0.25, k)}


def _make_planes(rng, k):
    return {"axis": rng.integers(0, 3, k), "off": rng.uniform(0.1, 0.9, k)}


def _make_capsules(rng, k):
    return {
        "c": rng.uniform(0.2, 0.8, (k, 3)),
        "d": _unit_vectors(rng, k),
        "r": rng.uniform(0.02, 0.08, k),
        "len": rng.uniform(0.1, 0.4, k),
    }


def _sample_spheres(rng, sph, which, sigma):
    n = which.shape[0]
    u = _unit_vectors(rng, n)
    rad = sph["r"][which] + rng.normal(0.0, sigma, n)
    return sph["c"][which] + rad[:, None] * u


def _sample_planes(rng, pl, which, sigma):
    n = which.shape[0]
    p = rng.uniform(0.0, 1.0, (n, 3))
    ax = pl["axis"][which]
    p[np.arange(n), ax] = pl["off"][which] + rng.normal(0.0, sigma, n)
    return p


def _sample_capsules(rng, cap, which, sigma):
    n = which.shape[0]
    c, d, r, ln = cap["c"][which], cap["d"][which], cap["r"][which], cap["len"][which]
    on_side = rng.uniform(0.0, 1.0, n) < ln / (ln + 2.0 * r)
    axial = rng.uniform(-0.5, 0.5, n) * ln
    u = _unit_vectors(rng, n)
    # side: radial direction = component of u perpendicular to d, normalised
    perp = u - np.sum(u * d, axis=1, keepdims=True) * d
    pn = np.linalg.norm(perp, axis=1, keepdims=True)
    pn[pn == 0.0] = 1.0
    perp = perp / pn
    jit = rng.normal(0.0, sigma, n)
    side_pts = c + axial[:, None] * d + (r + jit)[:, None] * perp
    # cap: hemisphere chosen by the sign of u.d
    sgn = np.where(np.sum(u * d, axis=1) >= 0.0, 1.0, -1.0)
    cap_pts = c + (sgn * 0.5 * ln)[:, None] * d + (r + jit)[:, None] * u
    return np.where(on_side[:, None], side_pts, cap_pts)


def _positions(rng, n, surf_frac, n_spheres, n_planes, n_capsules, sigma):
    """Surface/uniform mixture; every surface point picks its surface uniformly at random."""
    sph = _make_spheres(rng, n_spheres) if n_spheres else None
    pl = _make_planes(rng, n_planes) if n_planes else None
    cap = _make_capsules(rng, n_capsules) if n_capsules else None
    n_surf = int(round(surf_frac * n))
    is_surf = np.zeros(n, dtype=bool)
    is_surf[rng.permutation(n)[:n_surf]] = True
    p = rng.uniform(0.0, 1.0, (n, 3))           # the uniform part (surface rows overwritten)
    k_tot = n_spheres + n_planes + n_capsules
    pick = rng.integers(0, k_tot, n)
    lo = 0
    for cnt, params, fn in ((n_spheres, sph, _sample_spheres), (n_planes, pl, _sample_planes),
                            (n_capsules, cap, _sample_capsules)):
        if cnt:
            m = is_surf & (pick >= lo) & (pick < lo + cnt)
            idx = np.flatnonzero(m)
            p[idx] = fn(rng, params, pick[idx] - lo, sigma)
            lo += cnt
    return np.clip(p, 0.0, 1.0), {"spheres": sph, "planes": pl, "capsules": cap, "pick": pick,
                                   "is_surf": is_surf}


# ----------------------------------------------------------------------------- attributes
def _attributes(rng, n):
    a = np.empty((n, N_CHANNELS), dtype=np.float64)
    a[:, 0:3] = rng.normal(-4.0, 0.5, (n, 3))            # log-scale
    q = rng.normal(0.0, 1.0, (n, 4))                      # rotation quaternion, normalised
    qn = np.linalg.norm(q, axis=1, keepdims=True)
    qn[qn == 0.0] = 1.0
    a[:, 3:7] = q / qn
    a[:, 7:8] = rng.normal(0.0, 2.0, (n, 1))              # opacity logit
    a[:, 8:11] = rng.normal(0.0, 0.5, (n, 3))             # SH DC
    a[:, 11:56] = rng.normal(0.0, 0.05, (n, 45))          # SH AC
    return a


def qstep_from_range(attr: np.ndarray, qdiv: int) -> np.ndarray:
    a64 = attr.astype(np.float64, copy=False)
    rng_c = a64.max(axis=0) - a64.min(axis=0) if a64.shape[0] else np.ones(a64.shape[1])
    rng_c = np.where(rng_c > 0.0, rng_c, 1.0)
    return (rng_c / float(qdiv)).astype(np.float32)


_CONFIGS = {
    # id: (seed, N, surf_frac, spheres, planes, capsules, sigma, depth J, qdiv D)
    1: (0, 10_000, 0.70, 3, 0, 0, 1e-3, 10, 256),
    2: (1, 100_000, 0.70, 8, 4, 0, 1e-3, 12, 256),
    3: (2, 1_000_000, 1.00, 0, 0, 20, 5e-4, 16, 256),
    4: (3, 3_000_000, 0.85, 0, 4, 20, 5e-4, 18, 1024),
    5: (4, 1_000_000, 1.00, 0, 0, 20, 5e-4, 16, 256),   # frame 0 of the dynamic sequence
}

LADDER_QDIVS = (64, 256, 1024, 4096)   # config-5 bitrate ladder


def make_frame(config: int, n_override: int | None = None) -> Frame:
    """BASELINE.json configs[config-1]; ``n_override`` shrinks N (same recipe) for tests."""
    seed, n, frac, ns, npl, nc, sigma, depth, qdiv = _CONFIGS[config]
    if n_override is not None:
        n = int(n_override)
    rng = np.random.default_rng(seed)
    pos, _ = _positions(rng, n, frac, ns, npl, nc, sigma)
    attr = _attributes(rng, n)
    xyz32 = np.ascontiguousarray(pos, dtype=np.float32)
    attr32 = np.ascontiguousarray(attr, dtype=np.float32)
    return Frame(name=f"config{config}" + (f"_n{n}" if n_override else ""), xyz=xyz32, attr=attr32,
                 qstep=qstep_from_range(attr32, qdiv), depth=depth, qdiv=qdiv,
                 bbox_min=np.zeros(3, np.float32), bbox_max=np.ones(3, np.float32))


def make_dense_frame(n: int = 20_000, depth: int = 5, channels: int = N_CHANNELS, seed: int = 7,
                     qdiv: int = 256) -> Frame:
    """Duplicate-heavy cloud (config-2 geometry voxelised at a coarse depth): exercises the merge,
    which the timed configs barely do (SURVEY.md section 8(d) note)."""
    rng = np.random.default_rng(seed)
    pos, _ = _positions(rng, n, 0.70, 8, 4, 0, 1e-3)
    attr = _attributes(rng, n)
    if channels != N_CHANNELS:
        reps = -(-channels // N_CHANNELS)
        attr = np.tile(attr, (1, reps))[:, :channels] + rng.normal(0, 0.01, (n, channels))
    xyz32 = np.ascontiguousarray(pos, dtype=np.float32)
    attr32 = np.ascontiguousarray(attr, dtype=np.float32)
    return Frame(name=f"dense_n{n}_J{depth}_C{channels}", xyz=xyz32, attr=attr32,
                 qstep=qstep_from_range(attr32, qdiv), depth=depth, qdiv=qdiv,
                 bbox_min=np.zeros(3, np.float32), bbox_max=np.ones(3, np.float32))


def make_uniform_frame(n: int, depth: int, channels: int, seed: int, qdiv: int = 256) -> Frame:
    """Small i.i.d.-uniform cloud with an arbitrary channel count (edge-case tests)."""
    rng = np.random.default_rng(seed)
    xyz32 = np.ascontiguousarray(rng.uniform(0.0, 1.0, (n, 3)), dtype=np.float32)
    attr32 = np.ascontiguousarray(rng.normal(0.0, 1.0, (n, channels)), dtype=np.float32)
    return Frame(name=f"uniform_n{n}_J{depth}_C{channels}", xyz=xyz32, attr=attr32,
                 qstep=qstep_from_range(attr32, qdiv) if n else np.ones(channels, np.float32),
                 depth=depth, qdiv=qdiv,
                 bbox_min=np.zeros(3, np.float32), bbox_max=np.ones(3, np.float32))


def make_pointcloud_frame(n: int = 1_000_000, depth: int = 10, seed: int = 5) -> Frame:
    """Point-cloud mode (Table A.4: 8i / CMU Panoptic frames of ~0.7-1M points voxelised at depth
    J = 10, colour only, quantisation step 0.1): the config-3 surface recipe (20 capsules, sigma = 5e-4) voxelised at
    depth 10 -- about 0.8 occupied voxels per point, i.e. a fifth of the points are merged as duplicates -- with three
    colour channels in [0, 1]: a smooth function of position plus N(0, 0.03) noise, clipped.  qstep = 0.1 per channel."""
    rng = np.random.default_rng(seed)
    pos, _ = _positions(rng, n, 1.0, 0, 0, 20, 5e-4)
    phase = rng.uniform(0.0, 2.0 * np.pi, (3, 3))
    freq = rng.uniform(2.0, 9.0, (3, 3))
    col = np.empty((n, 3), dtype=np.float64)
    for c in range(3):
        col[:, c] = 0.5 + 0.5 * np.prod(np.sin(freq[c][None, :] * pos + phase[c][None, :]), axis=1)
    col = np.clip(col + rng.normal(0.0, 0.03, (n, 3)), 0.0, 1.0)
    xyz32 = np.ascontiguousarray(pos, dtype=np.float32)
    attr32 = np.ascontiguousarray(col, dtype=np.float32)
    return Frame(name=f"pointcloud_n{n}_J{depth}", xyz=xyz32, attr=attr32, qstep=np.full(3, 0.1, np.float32), depth=depth,
                 qdiv=10, bbox_min=np.zeros(3, np.float32), bbox_max=np.ones(3, np.float32))


class DynamicSequence:
    """Config 5: frame t = frame-0 positions + smooth per-capsule deformation + jitter; attributes
    random-walk.  Frames are produced one at a time (300 x 236 MB cannot be pre-stored)."""

    def __init__(self, n_override: int | None = None):
        seed, n, frac, ns, npl, nc, sigma, depth, qdiv = _CONFIGS[5]
        if n_override is not None:
            n = int(n_override)
        rng = np.random.default_rng(seed)
        pos, info = _positions(rng, n, frac, ns, npl, nc, sigma)
        self.p0 = pos
        self.attr = _attributes(rng, n)
        self.k = _unit_vectors(rng, nc)[info["pick"]]       # k_c: one unit vector per capsule
        self.rng = rng
        self.depth = depth
        self.t = 0
        self.qsteps = {d: qstep_from_range(self.attr.astype(np.float32), d) for d in LADDER_QDIVS}

    def next_frame(self) -> Frame:
        t = self.t
        if t == 0:
            pos = self.p0
        else:
            phase = 2.0 * np.pi * (0.5 * t / 30.0 + np.sum(self.k * self.p0, axis=1))
            pos = self.p0 + 0.01 * np.sin(phase)[:, None] * self.k \
                + self.rng.normal(0.0, 1e-4, self.p0.shape)
            pos = np.clip(pos, 0.0, 1.0)
            self.attr = self.attr + self.rng.normal(0.0, 0.01, self.attr.shape)
        self.t += 1
        xyz32 = np.ascontiguousarray(pos, dtype=np.float32)
        attr32 = np.ascontiguousarray(self.attr, dtype=np.float32)
        return Frame(name=f"config5_t{t}", xyz=xyz32, attr=attr32, qstep=self.qsteps[256],
                     depth=self.depth, qdiv=256,
                     bbox_min=np.zeros(3, np.float32), bbox_max=np.ones(3, np.float32))


class DynamicSequenceDevice:
    """Config 5 generated on the device (300 x 236 MB cannot be pre-stored, and 300 numpy steps of
    56M normal draws would take minutes).  Frame 0 is ``DynamicSequence``'s (numpy, seed 4); frames t >= 1 use the
    same formulas in fp64 with a seeded ``torch.Generator`` on the device: positions from frame 0 directly,
    attributes by a random walk, one N(0, 0.01) step per frame on all channels.  ``frame(t)`` returns the fp32
    device tensors; ``host_frame(t)`` copies them into a ``Frame`` so a CPU checker sees the very same arrays."""

    def __init__(self, device="cuda:0", n_override: int | None = None):
        import torch
        self.torch = torch
        base = DynamicSequence(n_override)
        self.depth = base.depth
        self.qsteps = base.qsteps                       # from frame 0's channel ranges, one per ladder rung
        self.device = device
        self.p0 = torch.from_numpy(base.p0).to(device)                   # fp64
        self.k = torch.from_numpy(np.ascontiguousarray(base.k)).to(device)
        self.attr = torch.from_numpy(base.attr).to(device)               # fp64 random-walk state
        self.proj = (self.k * self.p0).sum(dim=1)
        self.gen = torch.Generator(device=device)
        self.gen.manual_seed(_CONFIGS[5][0])
        self.t = 0
        self.n, self.channels = int(self.p0.shape[0]), int(self.attr.shape[1])
        self._xyz = self.p0.to(torch.float32).contiguous()
        self._attr = self.attr.to(torch.float32).contiguous()

    def _step(self):
        torch = self.torch
        self.t += 1
        t = self.t
        phase = 2.0 * np.pi * (0.5 * t / 30.0 + self.proj)
        jit = torch.randn(self.p0.shape, generator=self.gen, device=self.device, dtype=torch.float64) * 1e-4
        pos = (self.p0 + 0.01 * torch.sin(phase)[:, None] * self.k + jit).clamp_(0.0, 1.0)
        self.attr += torch.randn(self.attr.shape, generator=self.gen, device=self.device, dtype=torch.float64) * 0.01
        self._xyz = pos.to(torch.float32).contiguous()
        self._attr = self.attr.to(torch.float32).contiguous()

    def frame(self, t: int):
        """Device tensors (xyz N x 3, attr N x C, fp32) of frame t; frames are visited in increasing order."""
        if t < self.t:
            raise ValueError("frames must be requested in increasing order")
        while self.t < t:
            self._step()
        return self._xyz, self._attr

    def host_frame(self, t: int, qdiv: int = 256) -> Frame:
        xyz, attr = self.frame(t)
        return Frame(name=f"config5_t{t}_D{qdiv}", xyz=xyz.cpu().numpy(), attr=attr.cpu().numpy(),
                     qstep=self.qsteps[qdiv], depth=self.depth, qdiv=qdiv,
                     bbox_min=np.zeros(3, np.float32), bbox_max=np.ones(3, np.float32))
