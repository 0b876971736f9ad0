#!/usr/bin/env python
"""bench.py -- encode + decode of one synthetic 3DGS frame (octree + RAHT hot path) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--impl ours|reference]

A "step" is one pass of the whole hot path over one frame: gsnfs_octree_encode -> gsnfs_merge_raht_forward (duplicate
merge fused into the forward transform + quantiser) on the encoder side, the decoder's header read-back, then
gsnfs_octree_decode -> gsnfs_raht_inverse.  `value` is whole-job Mgaussians/s with inputs resident in HBM; `e2e` is the
same metric through the *_host_packed ABI calls with pinned host buffers (H2D/D2H inside the timed region; the
coefficients cross PCIe as RLGR bytes), one frame at a time on one context (the round-1 protocol); `e2e_pipelined` is the
same calls on a back-to-back frame stream (an encoder thread and a decoder thread, one context each: pipeline throughput, not
frame latency); `e2e_raw` goes through the *_host calls (raw int32 coefficients, one frame at a time).  `entropy` times
the RLGR coder on the frame's quantised coefficients, outside the step.  `--config pc` is the
point-cloud shaped workload (NEXT-4: 1M points, depth 10, 3 colour channels).
Multi-GPU: frames are independent (intra-only codec) => replicas only, one frame stream per
rank, no collective on the data path ("scaling": "weak").  `--impl reference` times the fp64 oracle on the
host cores (a deliberately slow baseline, not the target).  At N = 1 the line also carries `ladder`: the 300-frame
dynamic sequence of BASELINE.json configs[4] encoded + decoded at 4 qstep rungs per frame (`--ladder-frames 0` skips it).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "encode+decode Mgaussians/s per frame (octree+RAHT)"
UNIT = "Mgaussians/s"


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.gpu = gpu_index
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.gpu), "-lms", "100"], stdout=subprocess.PIPE, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[1]))
                mx.append(float(r[2]))
                for k, nm in enumerate(names):
                    if r[5 + k].lower().startswith("active"):
                        reasons.add(nm)
            except Exception:
                continue
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def load_frame(synth, args):
    if args.config == "pc":
        return synth.make_pointcloud_frame()
    return synth.make_frame(int(args.config), n_override=args.n_override)


def workload_name(args, fr):
    if args.config == "pc":
        return (f"point-cloud mode (PAPER.md L434-436 shape; SURVEY 8(f) NEXT-4): N={fr.n} points, C={fr.channels} colour "
                f"channels, octree depth {fr.depth}, qstep 0.1, synth.make_pointcloud_frame()")
    return (f"BASELINE.json configs[{int(args.config) - 1}]{' recipe with N overridden' if args.n_override else ''}: N={fr.n} "
            f"Gaussians, C={fr.channels} fp32 channels, octree depth {fr.depth}, qstep=range/{fr.qdiv}, seed per "
            f"synth.make_frame({args.config})")


# ------------------------------------------------------------------------------------------------
def algorithmic_bytes(n, nv, s_occ, channels, depth):
    """SURVEY.md section 8(d) / DESIGN.md 'Algorithmic bytes': what each kernel must move, per launch."""
    k = 4 if 3 * depth <= 32 else 8
    passes = (3 * depth + 7) // 8
    c4 = 4 * channels
    return {
        "voxelize_morton_hist": 12 * n + k * n,
        "onesweep_pass": 2 * (k + 4) * n,
        "octree_count": k * n,
        "octree_emit": k * n + 12 * nv + s_occ,
        "merge": 4 * n + 8 * nv + c4 * n + c4 * nv + 4 * nv,
        "raht_schedule": (k + 4) * nv + 16 * nv,                # codes + weights in, <= 16 B/voxel of schedule out
        "raht_forward": 4 * n + c4 * n + c4 * nv,               # fused merge + forward: perm + the N input rows in, N_v rows out
        "raht_inverse": c4 * nv + c4 * nv,                      # 4C*N_v read + 4C*N_v write
        "rlgr_count": c4 * nv, "rlgr_write": c4 * nv, "rlgr_decode": c4 * nv,
        "scan_reduce": None, "scan_sums": None, "scan_down": None,   # used twice with different inputs
        "octree_decode": s_occ + 20 * nv,                       # stream in, leaf codes + coordinates out
        "quantize": 8 * channels * nv,
        "radix_sort": k * n + passes * 2 * (k + 4) * n,         # histogram read + P passes of (key, index) in and out
        "_sort_total": k * n + passes * 2 * (k + 4) * n, "_passes": passes,
    }


def run_ladder(B, synth, torch, ctx, buf, dev, n_frames):
    """BASELINE.json configs[4]: the dynamic sequence, every frame encoded + decoded at the 4 qstep rungs back to
    back on one stream through the public calls.  Frames are generated on the device outside the timed region;
    per frame the 4 rungs are bracketed by CUDA events.  Two variants: "independent" = 4 full encode+decode passes;
    "shared" = one sort/octree/transform + 4 gsnfs_quantize, one octree decode + one schedule + 4 inverse transforms."""
    seq = synth.DynamicSequenceDevice(dev)
    n, C, J = seq.n, seq.channels, seq.depth
    lo, hi = np.zeros(3, np.float32), np.ones(3, np.float32)
    stream = torch.cuda.current_stream()
    h_hdr = torch.empty(J + 1 + 4, dtype=torch.int32).pin_memory()
    coeff = torch.empty((n, C), dtype=torch.float32, device=dev)
    qrung = [torch.empty((n, C), dtype=torch.int32, device=dev) for _ in synth.LADDER_QDIVS]
    e0, e1, e2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))

    def header():
        h_hdr[:J + 1].copy_(buf.level_sizes, non_blocking=True)
        h_hdr[J + 1:].copy_(buf.counts, non_blocking=True)
        stream.synchronize()
        return h_hdr[:J + 1].numpy(), int(h_hdr[J + 2])

    def independent(xyz, attr):
        for d in synth.LADDER_QDIVS:
            B.encode_frame(ctx, buf, xyz, attr, lo, hi, seq.qsteps[d])
            levels, occ_bytes = header()
            B.decode_frame(ctx, buf, levels, occ_bytes, seq.qsteps[d])

    def shared(xyz, attr):
        B.gsnfs_octree_encode(ctx, xyz, n, lo, hi, J, buf.occ, buf.level_sizes, buf.perm, buf.voxel_keys,
                              buf.voxel_start, buf.counts)
        B.gsnfs_merge_raht_forward(ctx, buf.voxel_keys, buf.perm, buf.voxel_start, n, buf.counts, J, attr, C, None, None,
                                   buf.weights, None, coeff)
        for i, d in enumerate(synth.LADDER_QDIVS):
            B.gsnfs_quantize(ctx, coeff, n, buf.counts, C, seq.qsteps[d], None, qrung[i])
        levels, occ_bytes = header()
        nv = int(levels[J])
        B.gsnfs_octree_decode(ctx, buf.occ, occ_bytes, levels, J, buf.dec_xyz, buf.dec_keys, buf.dec_counts)
        for i, d in enumerate(synth.LADDER_QDIVS):        # rungs 2.. reuse the first rung's schedule (keys = None)
            B.gsnfs_raht_inverse(ctx, buf.dec_keys if i == 0 else None, buf.weights, nv, None, J, qrung[i], None, C,
                                 seq.qsteps[d], None, buf.dec_attr)

    xyz, attr = seq.frame(0)
    for _ in range(3):
        independent(xyz, attr)
        shared(xyz, attr)
    torch.cuda.synchronize()
    ms_ind = ms_sh = 0.0
    for t in range(n_frames):
        xyz, attr = seq.frame(t)
        torch.cuda.synchronize()
        e0.record(stream)
        independent(xyz, attr)
        e1.record(stream)
        shared(xyz, attr)
        e2.record(stream)
        torch.cuda.synchronize()
        ms_ind += e0.elapsed_time(e1)
        ms_sh += e1.elapsed_time(e2)
    r = len(synth.LADDER_QDIVS)
    return {"workload": f"BASELINE.json configs[4]: {n_frames} frames x {r} rungs (qstep = range/{list(synth.LADDER_QDIVS)}), "
                        f"N={n}, C={C}, depth {J}, frames generated on the device (synth.DynamicSequenceDevice)",
            "frames": n_frames, "rungs": r, "target_fps": 30.0,
            "independent": {"frames_per_s": round(n_frames / (ms_ind * 1e-3), 1),
                            "frame_rungs_per_s": round(n_frames * r / (ms_ind * 1e-3), 1),
                            "ms_per_frame": round(ms_ind / n_frames, 4)},
            "shared_geometry_and_transform": {"frames_per_s": round(n_frames / (ms_sh * 1e-3), 1),
                                              "frame_rungs_per_s": round(n_frames * r / (ms_sh * 1e-3), 1),
                                              "ms_per_frame": round(ms_sh / n_frames, 4)}}


def other_config_kernels(B, synth, torch, cfg, dev, device_index, peak, steps=10):
    """Per-kernel live timings of one more workload (the 3M-Gaussian and point-cloud fractions were
    builder-run only): the same step as the headline loop, 3 warm-up + `steps` profiled passes, own context and buffers."""
    fr = synth.make_pointcloud_frame() if cfg == "pc" else synth.make_frame(int(cfg))
    n, C, J = fr.n, fr.channels, fr.depth
    ctx = B.Context(max_points=n, max_channels=C, max_depth=J, device=device_index)
    try:
        buf = B.FrameBuffers(n, C, J, dev)
        d_xyz, d_attr = torch.from_numpy(fr.xyz).to(dev), torch.from_numpy(fr.attr).to(dev)
        B.encode_frame(ctx, buf, d_xyz, d_attr, fr.bbox_min, fr.bbox_max, fr.qstep)
        torch.cuda.synchronize()
        levels, cnt = buf.level_sizes.cpu().numpy(), buf.counts.cpu().numpy()
        nv, s_occ = int(cnt[0]), int(cnt[1])

        def step():
            B.encode_frame(ctx, buf, d_xyz, d_attr, fr.bbox_min, fr.bbox_max, fr.qstep)
            B.decode_frame(ctx, buf, levels, s_occ, fr.qstep)

        for _ in range(3):
            step()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(torch.cuda.current_stream())
        for _ in range(steps):
            step()
        e1.record(torch.cuda.current_stream())
        torch.cuda.synchronize()
        ms_step = e0.elapsed_time(e1) / steps
        ctx.profile_start(4096)
        for _ in range(steps):
            step()
        prof = ctx.profile_stop()
        ab = algorithmic_bytes(n, nv, s_occ, C, J)
        ks = {}
        for name, (c, tot_ms) in prof.items():
            avg_us = tot_ms / c * 1e3
            b = ab.get(name)
            ks[name] = {"avg_us": round(avg_us, 2), "launches_per_step": c / steps,
                        "frac_of_peak": round(b / (avg_us * 1e-6) / 1e9 / peak, 4) if b else None}
        return {"workload": f"config {cfg}: N={n}, C={C}, depth {J}", "n_voxels": nv, "occ_bytes": s_occ,
                "ms_per_step": round(ms_step, 4), "Mgaussians_per_s": round(n / (ms_step * 1e-3) / 1e6, 1), "steps": steps,
                "note": "header read back once before the loop (no per-step host read); inputs resident in HBM",
                "kernels": ks}
    finally:
        ctx.close()


def run_ours(args, rank, world, local_rank):
    import torch
    import torch.distributed as dist
    from paper_2606_05650_b200 import binding as B, dist as gdist, synth

    torch.cuda.set_device(local_rank)
    dev = f"cuda:{local_rank}"
    fr = load_frame(synth, args)
    n, C, J = fr.n, fr.channels, fr.depth
    ctx = B.Context(max_points=n, max_channels=C, max_depth=J, device=local_rank)
    buf = B.FrameBuffers(n, C, J, dev)
    d_xyz = torch.from_numpy(fr.xyz).to(dev)
    d_attr = torch.from_numpy(fr.attr).to(dev)
    h_hdr = torch.empty(J + 1 + 4, dtype=torch.int32).pin_memory()
    stream = torch.cuda.current_stream()

    hdr_ready = torch.cuda.Event()

    def step():
        B.gsnfs_octree_encode(ctx, d_xyz, n, fr.bbox_min, fr.bbox_max, J, buf.occ, buf.level_sizes, buf.perm,
                              buf.voxel_keys, buf.voxel_start, buf.counts)
        # the decoder needs the stream header (level sizes) on the host, like a receiver would: copy it out as soon
        # as the position coder is done, so the host can enqueue the decode while the GPU runs the attribute coder
        h_hdr[:J + 1].copy_(buf.level_sizes, non_blocking=True)
        h_hdr[J + 1:].copy_(buf.counts, non_blocking=True)
        hdr_ready.record(stream)
        B.gsnfs_merge_raht_forward(ctx, buf.voxel_keys, buf.perm, buf.voxel_start, n, buf.counts, J, d_attr, C,
                                   fr.qstep, None, buf.weights, buf.qcoeff, None)
        hdr_ready.synchronize()
        levels = h_hdr[:J + 1].numpy()
        B.decode_frame(ctx, buf, levels, int(h_hdr[J + 2]), fr.qstep)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    nv, s_occ = int(h_hdr[J + 1]), int(h_hdr[J + 2])

    sampler = ClockSampler(local_rank)
    sampler.start()
    l0 = ctx.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record(stream)
    for _ in range(args.steps):
        step()
    e1.record(stream)
    barrier()
    ms_total = e0.elapsed_time(e1)
    launches = ctx.launch_count() - l0
    clocks = sampler.stop()
    ms_total = gdist.max_over_ranks(ms_total, dev)          # replicas: the job is as slow as its slowest rank
    ms_step = ms_total / args.steps
    value = world * n / (ms_step * 1e-3) / 1e6

    # ---- stage split (encode / decode) and per-kernel durations, live, on the same stream
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
    enc_ms, dec_ms = [], []
    for _ in range(args.steps):
        ev[0].record(stream)
        B.encode_frame(ctx, buf, d_xyz, d_attr, fr.bbox_min, fr.bbox_max, fr.qstep)
        ev[1].record(stream)
        B.decode_frame(ctx, buf, h_hdr[:J + 1].numpy(), s_occ, fr.qstep)
        ev[2].record(stream)
        torch.cuda.synchronize()
        enc_ms.append(ev[0].elapsed_time(ev[1]))
        dec_ms.append(ev[1].elapsed_time(ev[2]))
    ctx.profile_start(8192)
    for _ in range(args.steps):
        step()
    prof = ctx.profile_stop()

    peak, peak_src = load_peaks()
    ab = algorithmic_bytes(n, nv, s_occ, C, J)
    kernels = {}
    for name, (cnt, tot_ms) in prof.items():
        avg_us = tot_ms / cnt * 1e3
        b = ab.get(name)
        kernels[name] = {"launches_per_step": cnt / args.steps, "avg_us": round(avg_us, 2),
                         "ms_per_step": round(tot_ms / args.steps, 4),
                         "alg_GBps": round(b / (avg_us * 1e-6) / 1e9, 1) if b else None}
    dom = max((k for k in kernels if ab.get(k)), key=lambda k: kernels[k]["ms_per_step"])
    traffic = None
    tpath = os.path.join(ROOT, "profiles", "r2_dram_traffic.csv")       # ncu dram bytes per launch (profiles/r2_dram_traffic.md)
    if os.path.exists(tpath):
        try:
            for line in open(tpath).read().splitlines()[1:]:
                cfg, kname, nbytes = line.split(",")
                if cfg == f"config{args.config}" and kname == dom and args.n_override is None:     # same workload only
                    traffic = int(nbytes)
        except Exception:
            traffic = None
    roofline = {"bound": "hbm", "kernel": dom, "achieved": kernels[dom]["alg_GBps"], "peak": peak, "unit": "GB/s",
                "frac": round(kernels[dom]["alg_GBps"] / peak, 4), "traffic": traffic, "peak_source": peak_src,
                "alg_bytes_per_launch": ab[dom]}
    sort_ms = kernels.get("radix_sort", {}).get("ms_per_step", 0.0)
    sort_frac = (ab["_sort_total"] / (sort_ms * 1e-3) / 1e9 / peak) if sort_ms else None

    # ---- end to end through the host-buffer ABI calls (pinned host memory, copies inside the timed region)
    RLGR_BLOCK = 512                       # Table A.5's fastest block size (here too: profiles/r2_stages.md, RLGR block sweep)
    e2e = e2e_raw = e2e_pipelined = entropy = None
    if rank == 0 or world > 1:
        cap = B.gsnfs_occ_capacity(n, J)
        pin = lambda *s, dt: torch.empty(s, dtype=dt).pin_memory()
        h_xyz, h_attr = torch.from_numpy(fr.xyz).pin_memory(), torch.from_numpy(fr.attr).pin_memory()
        h_occ, h_lev = pin(cap, dt=torch.uint8), pin(J + 1, dt=torch.int32)
        h_w, h_q, h_cnt = pin(n, dt=torch.int32), pin(n, C, dt=torch.int32), pin(4, dt=torch.int32)
        h_vx, h_out, h_cnt2 = pin(n, 3, dt=torch.int32), pin(n, C, dt=torch.float32), pin(4, dt=torch.int32)
        h_bits = pin(B.gsnfs_rlgr_blocks(n, C, RLGR_BLOCK), dt=torch.int32)
        h_stream, h_info = pin(n * C * 4, dt=torch.uint8), pin(2, dt=torch.int64)

        def raw_step():
            B.gsnfs_frame_encode_host(ctx, h_xyz, h_attr, n, C, fr.bbox_min, fr.bbox_max, J, fr.qstep, None,
                                      h_occ, h_lev, h_w, h_q, h_cnt)
            B.gsnfs_frame_decode_host(ctx, h_occ, int(h_cnt[1]), h_lev.numpy(), J, h_w, h_q, C, fr.qstep, None,
                                      h_vx, h_out, h_cnt2)

        def packed_step():
            B.gsnfs_frame_encode_host_packed(ctx, h_xyz, h_attr, n, C, fr.bbox_min, fr.bbox_max, J, fr.qstep, None,
                                             RLGR_BLOCK, h_occ, h_lev, h_w, h_bits, h_stream, h_cnt, h_info)
            B.gsnfs_frame_decode_host_packed(ctx, h_occ, int(h_cnt[1]), h_lev.numpy(), J, h_w, h_bits, h_stream,
                                             int(h_info[0]), RLGR_BLOCK, C, fr.qstep, None, h_vx, h_out, h_cnt2)

        def time_e2e(fn):
            for _ in range(2):
                fn()
            barrier()
            ks = max(2, min(args.steps, 10))
            e0.record(stream)
            for _ in range(ks):
                fn()
            e1.record(stream)
            barrier()
            return gdist.max_over_ranks(e0.elapsed_time(e1), dev) / ks, ks

        ms_p, ks = time_e2e(packed_step)
        nv_e, ob_e, sb = int(h_cnt[0]), int(h_cnt[1]), int(h_info[0])
        nbits4 = 4 * B.gsnfs_rlgr_blocks(n, C, RLGR_BLOCK)
        side = ob_e + nv_e * 4 + nbits4 + sb                      # occupancy bytes, weights, block header, block streams
        e2e = {"value": round(world * n / (ms_p * 1e-3) / 1e6, 3), "unit": UNIT, "ms_per_step": round(ms_p, 4),
               "h2d_bytes_per_step": n * 12 + n * C * 4 + side,
               "d2h_bytes_per_step": 16 + 4 * (J + 1) + 16 + side + 16 + 16 + nv_e * 12 + nv_e * C * 4, "steps": ks,
               "api": "gsnfs_frame_encode_host_packed + gsnfs_frame_decode_host_packed (coefficients as RLGR bytes, "
                      f"block {RLGR_BLOCK})", "coefficient_stream_bytes": sb}
        # the same packed calls as a two-stage pipeline: a second context decodes frame t on its own stream (a second host
        # thread) while this one encodes frame t + 1, so the two PCIe directions are busy at the same time -- the
        # back-to-back streaming use-case; encoder and decoder share nothing but the host buffers
        if world == 1:
            import queue
            ctx2 = B.Context(max_points=n, max_channels=C, max_depth=J, device=local_rank)
            s_enc, s_dec = torch.cuda.Stream(), torch.cuda.Stream()
            sets = []
            for _ in range(3):      # three sets: with two the encoder waits for the decoder to hand a set back (10.2 vs 7.2 ms / frame)
                sets.append(dict(occ=pin(cap, dt=torch.uint8), lev=pin(J + 1, dt=torch.int32), w=pin(n, dt=torch.int32),
                                 bits=pin(B.gsnfs_rlgr_blocks(n, C, RLGR_BLOCK), dt=torch.int32),
                                 stream=pin(n * C * 4, dt=torch.uint8), cnt=pin(4, dt=torch.int32), info=pin(2, dt=torch.int64)))
            h_out2, h_vx2, h_cnt3 = pin(n, C, dt=torch.float32), pin(n, 3, dt=torch.int32), pin(4, dt=torch.int32)
            ready, free = queue.Queue(), queue.Queue()
            kp = max(4, min(args.steps, 12))

            def producer():
                for i in range(kp + 2):
                    b = free.get()
                    B.gsnfs_frame_encode_host_packed(ctx, h_xyz, h_attr, n, C, fr.bbox_min, fr.bbox_max, J, fr.qstep, None,
                                                     RLGR_BLOCK, b["occ"], b["lev"], b["w"], b["bits"], b["stream"],
                                                     b["cnt"], b["info"], stream=s_enc)
                    ready.put(b)

            def consumer(times):
                for i in range(kp + 2):
                    b = ready.get()
                    if i == 2:
                        times.append(time.perf_counter())          # two frames of warm-up, then kp timed frames
                    B.gsnfs_frame_decode_host_packed(ctx2, b["occ"], int(b["cnt"][1]), b["lev"].numpy(), J, b["w"], b["bits"],
                                                     b["stream"], int(b["info"][0]), RLGR_BLOCK, C, fr.qstep, None, h_vx2,
                                                     h_out2, h_cnt3, stream=s_dec)
                    free.put(b)
                times.append(time.perf_counter())

            for b in sets:
                free.put(b)
            times = []
            ta, tb = threading.Thread(target=producer), threading.Thread(target=consumer, args=(times,))
            torch.cuda.synchronize()
            ta.start(); tb.start(); ta.join(); tb.join()
            torch.cuda.synchronize()
            ms_pp = (times[1] - times[0]) * 1e3 / kp
            ok_pp = bool(torch.equal(h_out2[:nv_e], h_out[:nv_e]))
            # `e2e` stays what it was in round 1: one frame at a time (encode, then decode) through the blocking host calls
            # on ONE context, timed with CUDA events -- comparable across rounds.  The back-to-back frame stream (the
            # codec's use-case, config 5 / PAPER.md L45-49) is a different protocol and is reported beside it.
            e2e["how"] = "encode then decode of one frame at a time on one context: the two PCIe directions never overlap"
            e2e_pipelined = {
                "value": round(n / (ms_pp * 1e-3) / 1e6, 3), "unit": UNIT, "ms_per_step": round(ms_pp, 4), "steps": kp,
                "h2d_bytes_per_step": e2e["h2d_bytes_per_step"], "d2h_bytes_per_step": e2e["d2h_bytes_per_step"],
                "same_output_as_serial": ok_pp, "api": e2e["api"],
                "how": "back-to-back frames: an encoder thread and a decoder thread, one context and stream each, three sets "
                       "of pinned host buffers in rotation, every frame's inputs copied host -> device and its results "
                       "device -> host inside the timed region; host wall clock over the timed frames (all calls are "
                       "blocking).  Throughput of a pipeline, not the latency of a frame"}
            ctx2.close()
        ms_r, ks = time_e2e(raw_step)
        e2e_raw = {"value": round(world * n / (ms_r * 1e-3) / 1e6, 3), "unit": UNIT, "ms_per_step": round(ms_r, 4),
                   "h2d_bytes_per_step": n * 12 + n * C * 4 + ob_e + nv_e * 4 + nv_e * C * 4,
                   "d2h_bytes_per_step": 16 + 4 * (J + 1) + ob_e + nv_e * 4 + nv_e * C * 4 + 16 + nv_e * 12 + nv_e * C * 4,
                   "steps": ks, "api": "gsnfs_frame_encode_host + gsnfs_frame_decode_host (raw int32 coefficients)"}

    # ---- entropy coder, on the device, on this frame's quantised coefficients
    if rank == 0 and world == 1:
        B.encode_frame(ctx, buf, d_xyz, d_attr, fr.bbox_min, fr.bbox_max, fr.qstep)
        d_bits = torch.empty(B.gsnfs_rlgr_blocks(n, C, RLGR_BLOCK), dtype=torch.int32, device=dev)
        d_stream = torch.empty(n * C * 4, dtype=torch.uint8, device=dev)
        d_info = torch.zeros(2, dtype=torch.int64, device=dev)
        d_back = torch.empty((n, C), dtype=torch.int32, device=dev)
        ev3 = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
        enc_t, dec_t = [], []
        for it in range(8):
            ev3[0].record(stream)
            B.gsnfs_rlgr_encode(ctx, buf.qcoeff, n, buf.counts, C, RLGR_BLOCK, d_bits, d_stream, d_info)
            ev3[1].record(stream)
            torch.cuda.synchronize()
            sbytes, _, st = B.rlgr_info(d_info)
            B.gsnfs_rlgr_decode(ctx, d_stream, sbytes, d_bits, nv, C, RLGR_BLOCK, d_back, d_info)
            ev3[2].record(stream)
            torch.cuda.synchronize()
            if it >= 3:
                enc_t.append(ev3[0].elapsed_time(ev3[1]))
                dec_t.append(ev3[1].elapsed_time(ev3[2]))
        ok = bool(torch.equal(d_back[:nv], buf.qcoeff[:nv])) and B.rlgr_info(d_info)[2] == 0
        sweep = None
        if args.rlgr_sweep:                                   # Table A.5's axis: block size vs latency and size
            sweep = []
            for blk in (256, 512, 1024, 2048, 4096, 8192):
                sb_bits = torch.empty(B.gsnfs_rlgr_blocks(n, C, blk), dtype=torch.int32, device=dev)
                te, td = [], []
                for it in range(6):
                    ev3[0].record(stream)
                    B.gsnfs_rlgr_encode(ctx, buf.qcoeff, n, buf.counts, C, blk, sb_bits, d_stream, d_info)
                    ev3[1].record(stream)
                    torch.cuda.synchronize()
                    sb_bytes = B.rlgr_info(d_info)[0]
                    B.gsnfs_rlgr_decode(ctx, d_stream, sb_bytes, sb_bits, nv, C, blk, d_back, d_info)
                    ev3[2].record(stream)
                    torch.cuda.synchronize()
                    if it >= 2:
                        te.append(ev3[0].elapsed_time(ev3[1])); td.append(ev3[1].elapsed_time(ev3[2]))
                sweep.append({"block": blk, "encode_ms": round(float(np.median(te)), 4), "decode_ms": round(float(np.median(td)), 4),
                              "stream_bytes": sb_bytes})
        # the other stages around the path: occupancy bytes through rANS (NEXT-3), colour decorrelation (NEXT-2)
        cap_o = buf.occ.numel()
        a_f = torch.zeros(256, dtype=torch.int16, device=dev)
        a_nw = torch.zeros(B.gsnfs_rans_blocks(cap_o), dtype=torch.int16, device=dev)
        a_p = torch.zeros(B.gsnfs_rans_capacity(cap_o), dtype=torch.uint8, device=dev)
        a_back = torch.zeros(cap_o, dtype=torch.uint8, device=dev)
        others = {}
        t_a, t_b = [], []
        for it in range(6):
            ev3[0].record(stream)
            B.gsnfs_rans_encode(ctx, buf.occ, cap_o, buf.counts, a_f, a_nw, a_p, d_info)
            ev3[1].record(stream)
            torch.cuda.synchronize()
            pb = B.rlgr_info(d_info)[0]
            B.gsnfs_rans_decode(ctx, a_p, pb, a_f, a_nw, s_occ, a_back, d_info)
            ev3[2].record(stream)
            torch.cuda.synchronize()
            if it >= 2:
                t_a.append(ev3[0].elapsed_time(ev3[1])); t_b.append(ev3[1].elapsed_time(ev3[2]))
        others["occupancy_rans"] = {"encode_ms": round(float(np.median(t_a)), 4), "decode_ms": round(float(np.median(t_b)), 4),
                                    "bytes_in": s_occ, "bytes_out": pb, "ratio": round(s_occ / max(pb, 1), 3),
                                    "roundtrip_exact": bool(torch.equal(a_back[:s_occ], buf.occ[:s_occ]))}
        if B.gsnfs_klt_floats(C):
            d_klt = torch.zeros(B.gsnfs_klt_floats(C), dtype=torch.float32, device=dev)
            t_a, t_b, t_c = [], [], []
            ev4 = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
            for it in range(6):
                ev4[0].record(stream)
                B.gsnfs_klt_fit(ctx, d_attr, n, None, C, d_klt)
                ev4[1].record(stream)
                B.gsnfs_color_forward(ctx, d_attr, n, None, C, d_klt, buf.merged)
                ev4[2].record(stream)
                B.gsnfs_color_inverse(ctx, buf.merged, n, None, C, d_klt, buf.merged)
                ev4[3].record(stream)
                torch.cuda.synchronize()
                if it >= 2:
                    t_a.append(ev4[0].elapsed_time(ev4[1])); t_b.append(ev4[1].elapsed_time(ev4[2])); t_c.append(ev4[2].elapsed_time(ev4[3]))
            others["colour_decorrelation"] = {"klt_fit_ms": round(float(np.median(t_a)), 4), "forward_ms": round(float(np.median(t_b)), 4),
                                              "inverse_ms": round(float(np.median(t_c)), 4),
                                              "max_abs_roundtrip_error": float((buf.merged[:n] - d_attr).abs().max())}
        entropy = {"coder": f"block-parallel RLGR, block {RLGR_BLOCK} (PAPER.md L257, L803)", "encode_ms": round(float(np.median(enc_t)), 4),
                   "decode_ms": round(float(np.median(dec_t)), 4), "stream_bytes": sbytes, "raw_bytes": nv * C * 4,
                   "ratio": round(nv * C * 4 / max(sbytes, 1), 3), "roundtrip_exact": ok,
                   "note": "synthetic attributes are i.i.d. (SURVEY 8(d)): the ratio is not a compression claim",
                   "block_sweep": sweep, "other_stages": others}

    ladder = None
    if rank == 0 and world == 1 and args.ladder_frames > 0 and args.config == "3" and args.n_override is None:
        ladder = run_ladder(B, synth, torch, ctx, buf, dev, args.ladder_frames)
    others_cfg = None
    if rank == 0 and world == 1 and args.other_configs and args.config == "3" and args.n_override is None:
        del d_attr, d_xyz                      # the 3M frame needs the room
        others_cfg = {c: other_config_kernels(B, synth, torch, c, dev, local_rank, peak)
                      for c in args.other_configs.split(",") if c}
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu = oracle_time(fr, sample_n=min(fr.n, 1_000_000))
        cpu["all_cores"] = oracle_all_cores(args)
    ctx.close()
    if rank != 0:
        return
    out = {
        "metric": METRIC, "value": round(value, 3), "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": round(ms_step, 4), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": workload_name(args, fr),
                   "n_gaussians": n, "n_voxels": nv, "occ_bytes": s_occ, "channels": C, "depth": J,
                   "replicas": world, "l2_policy": "inputs larger than L2 (236 MB frame vs 126 MB L2); "
                   "intermediates stay wherever the pipeline leaves them"},
        "encode_ms": round(float(np.median(enc_ms)), 4), "decode_ms": round(float(np.median(dec_ms)), 4),
        "clocks": clocks, "e2e": e2e, "e2e_pipelined": e2e_pipelined, "e2e_raw": e2e_raw, "entropy": entropy, "gpu_launches": int(launches),
        "gpu_launches_per_step": launches / args.steps,
        "roofline": roofline,
        "sort": {"alg_bytes": ab["_sort_total"], "ms_per_step": sort_ms, "passes": ab["_passes"],
                 "frac_of_peak": round(sort_frac, 4) if sort_frac else None},
        "kernels": kernels, "other_configs": others_cfg, "ladder": ladder, "cpu_baseline": cpu,
    }
    print(json.dumps(out))


# ------------------------------------------------------------------------------------------------
def oracle_time(fr, sample_n=None, steps=1):
    """Times the fp64 oracle, as it stands, on this box's host cores (single thread: numpy)."""
    from oracle import gsnfs_oracle as orc
    xyz, attr = fr.xyz, fr.attr
    if sample_n is not None and sample_n < fr.n:
        xyz, attr = xyz[:sample_n], attr[:sample_n]
    n = xyz.shape[0]
    t0 = time.perf_counter()
    for _ in range(steps):
        enc = orc.encode_frame(xyz, attr, fr.bbox_min, fr.bbox_max, fr.depth, fr.qstep)
        dec = orc.decode_frame(enc["occ"], enc["level_sizes"], fr.depth, enc["qcoeff"], fr.qstep, enc["weights"])
    dt = (time.perf_counter() - t0) / steps
    assert dec["ok"]
    return {"value": round(n / dt / 1e6, 5), "unit": UNIT, "cores": 1, "kind": "oracle",
            "sample": f"first {n} of {fr.n} Gaussians of the same frame, encode+decode, {steps} step(s), "
                      f"{dt:.2f} s/step", "ms_per_step": round(dt * 1e3, 2)}


def _oracle_worker(config):
    from paper_2606_05650_b200 import synth

    class A:
        pass
    a = A()
    a.config, a.n_override = config, None
    fr = load_frame(synth, a)
    t0 = time.perf_counter()
    oracle_time(fr)
    return fr.n, time.perf_counter() - t0


def oracle_all_cores(args):
    """The oracle on all host cores: one independent frame per core (frames are the codec's independent unit; the oracle
    itself is single-threaded numpy and is not tuned for this)."""
    import multiprocessing as mp
    cores = len(os.sched_getaffinity(0))
    workers = max(1, min(cores, 16))
    t0 = time.perf_counter()
    with mp.get_context("spawn").Pool(workers) as pool:
        res = pool.map(_oracle_worker, [args.config] * workers)
    wall = time.perf_counter() - t0
    longest = max(r[1] for r in res)
    n_tot = sum(r[0] for r in res)
    return {"value": round(n_tot / longest / 1e6, 5), "unit": UNIT, "cores": workers, "kind": "oracle, one frame per core",
            "sample": f"{workers} whole frames in parallel, slowest {longest:.2f} s (wall incl. process start {wall:.1f} s)"}


def run_reference(args, rank, world):
    if rank != 0:
        return
    from paper_2606_05650_b200 import synth
    fr = load_frame(synth, args)
    # the whole frame, every step (config 3: ~7 s per step on one core; the driver allows 30 minutes)
    sample_n = fr.n
    for _ in range(args.warmup):
        oracle_time(fr, sample_n)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        r = oracle_time(fr, sample_n)
    dt = (time.perf_counter() - t0) / args.steps
    val = round(sample_n / dt / 1e6, 5)
    cpu = {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": r["sample"]}
    out = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": round(dt * 1e3, 3), "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": workload_name(args, fr), "n_gaussians": sample_n, "channels": fr.channels,
                      "depth": fr.depth},
           "cpu_baseline": cpu,
           "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(out))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="3", choices=["1", "2", "3", "4", "pc"],
                    help="BASELINE.json config (1-based); 3 = headline 1M frame; pc = point-cloud shaped frame (NEXT-4)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--other-configs", default="4,pc",
                    help="also report per-kernel timings at these workloads (comma list of 4, pc, 1, 2; '' to skip)")
    ap.add_argument("--rlgr-sweep", action="store_true", help="also time the RLGR coder at Table A.5's block sizes")
    ap.add_argument("--n-override", type=int, default=None,
                    help="same recipe with another N (e.g. 16000000: key arrays no longer fit the 126 MB L2); not the headline")
    ap.add_argument("--ladder-frames", type=int, default=300,
                    help="frames of the config-5 dynamic sequence to run at 4 rungs each (0 = skip; N=1, config 3 only)")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
        return
    if world > 1:
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl")
    run_ours(args, rank, world, local_rank)
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
