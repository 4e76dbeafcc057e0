#!/usr/bin/env python
"""bench.py — throughput of the Oblique-MERF render hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 1]

A *step* is one pass of the whole hot path (S2..S9: ray generation, clip, occupancy-plane march,
gathers, activations, compositing, deferred MLP, outputs) over one batch = the camera(s) of
BASELINE.json configs[1] (one 1920x1080 view of the 1000x1000x100 m scene).  Inputs are seeded
synthetic stand-ins for the paper's baked scenes.

value   = Mpixels/s, whole job (all ranks), scene resident in HBM, device-timed with CUDA events on the
          launching stream; L2 is flushed between timed steps (the flush is outside the event pairs).
e2e     = the same through omerf_render_host: cameras from host memory, rgb + counts copied back to pinned
          host memory inside the timed region.
roofline= march kernel against the BINDING ceiling of SURVEY 8(d) ("the smallest ceiling is the roofline"): the gather
          rate calibrated live by omerf_gather_probe on the same frame and layout (requested texel bytes per second);
gather_vs_hbm = algorithmic bytes (168 B per sample + 16 B per pixel) / launch duration against the measured
          HBM copy rate in MEASURED_PEAKS.json; issue = executed lane-operations (ncu capture, cited) against the issue peak.
parity  = element-wise comparison of the timed frame with the oracle's render of the same run (outside the timed region).
cpu_baseline = the CPU oracle as it stands on this box's host cores, on a bounded sample of the same frame.
--gpus N starts N ranks itself (torchrun) when it is not already running under one; N > 1 adds "strong": the batch
          partitioned across the ranks by samples (paper_2404_09531_b200/partition.py), beside the weak-scaling replicas.
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

import synth  # noqa: E402

BYTES_PER_SAMPLE = 168   # 20 distinct texels x 8 B (64 B grid + 96 B planes) + one (z_min, z_max) pair of 8 B
BYTES_PER_PIXEL = 16     # 12 B rgb + 4 B sample count written
ORACLE_BLOCK = 128            # rows per oracle call of the cpu_baseline sample (the oracle runs its rows in parallel)
TEXEL_BYTES_PER_SAMPLE = 160   # the distinct texels a sample needs: 20 x 8 B (fetched as 10 entries of 16 B)
# Figures of ONE march-kernel launch on configs[1] from the committed `ncu --set full` capture (profiles/r03_march_kernel.md,
# which names the command and the commit it was taken at); cited constants, not measured by this run:
NCU_CAPTURE = {"profile": "profiles/r03_march_kernel.md", "commit": "9ea54f3",
               "csrc_sha16": "bbd2ed3859f8b911",            # csrc_sha16() of the kernel sources that were captured
               "dram_bytes": 177942272 + 19446528,          # dram__bytes_read.sum + dram__bytes_write.sum
               "warp_instructions": 344585510,              # smsp__inst_executed.sum
               "lanes_per_instruction": 28.23}              # smsp__thread_inst_executed_per_inst_executed.ratio


MARCH_KERNEL_SOURCES = ("omerf_device.cuh", "omerf_mlp.cuh", "omerf_render.cu")   # everything omerf_march_kernel is compiled from


def csrc_sha16() -> str:
    """First 16 hex digits of the SHA-256 over the sources of the march kernel (MARCH_KERNEL_SOURCES under csrc/; the host
    glue of omerf_api.cu and the scene-build kernels do not enter the captured launch).  The cited ncu figures above
    describe one build of that kernel: when its sources differ from the captured ones the bench line carries null
    instead of a stale figure."""
    import hashlib
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2404_09531_b200", "csrc")
    for name in MARCH_KERNEL_SOURCES:
        h.update(name.encode() + b"\0" + open(os.path.join(d, name), "rb").read() + b"\0")
    return h.hexdigest()[:16]


def workload_name(cfg: int) -> str:
    return {0: "configs[0] tiny 128x128", 1: "configs[1] 1080p oblique frame, 1000x1000x100 m scene",
            2: "configs[2] 16 x 1080p views", 3: "configs[3] 8 x 2160p views, 4000x4000x200 m scene",
            4: "configs[4] sampling ablation (config-1 scene+camera)",
            5: "SURVEY 8(f).4 low-altitude cameras: 4 x 1080p views inside the config-1 box"}[cfg]


class ClockSampler:
    """nvidia-smi clocks + throttle reasons during the timed region (B200_PROFILING.md 'clocks' line)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                mx.append(float(r[1]))
                for nm, val in zip(names, r[3:7]):
                    if val.lower().startswith("active"):
                        reasons.add(nm)
            except (ValueError, IndexError):
                pass
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def oracle_bounded(scene, cams, W, H, sampler=0, budget_s=15.0, soft_eps=0.0, count_sectors=False):
    """Time the oracle (clipped loop, OpenMP over image rows) on view 0: the whole frame if it fits `budget_s`, else
    evenly spaced blocks of ORACLE_BLOCK consecutive rows.  The oracle parallelises over the rows of one call, so it is
    called with blocks of rows, never row by row (a one-row call runs on one thread whatever `cores` says)."""
    import oracle
    O = oracle.OracleScene(scene, sampler=sampler, soft_eps=soft_eps)
    B = min(ORACLE_BLOCK, H)
    t0 = time.perf_counter()
    r = O.render(cams[:1], W, H, mode="clipped", rows=((H - B) // 2, (H - B) // 2 + B))     # probe: one block at mid-height
    per_row = (time.perf_counter() - t0) / B
    n_rows = int(budget_s / max(per_row, 1e-9))
    if n_rows >= H:
        blocks = [(0, H)]
    else:
        nb = max(n_rows // B, 1)
        blocks = [(int(round(i * (H - B) / max(nb - 1, 1))),) for i in range(nb)] if nb > 1 else [((H - B) // 2,)]
        blocks = [(b0[0], b0[0] + B) for b0 in blocks]
    rows = [v for b0, b1 in blocks for v in range(b0, b1)]
    t0 = time.perf_counter()
    samples = 0
    threads = 1
    ref_n = np.zeros((len(rows), W), dtype=np.uint32)
    ref_rgb = np.zeros((len(rows), W, 3), dtype=np.float64)
    at = 0
    for b0, b1 in blocks:
        r = O.render(cams[:1], W, H, mode="clipped", rows=(b0, b1))
        samples += int(r["nsamples"][0, b0:b1].sum())
        threads = r["threads"]
        ref_n[at:at + b1 - b0], ref_rgb[at:at + b1 - b0] = r["nsamples"][0, b0:b1], r["rgb"][0, b0:b1]
        at += b1 - b0
    dt = time.perf_counter() - t0
    px = len(rows) * W
    stride = 1 if len(rows) == H else 0
    what = f"all {H} rows of view 0 in one call" if len(rows) == H else \
        f"{len(rows)} of {H} rows of view 0 ({len(blocks)} evenly spaced blocks of {B} consecutive rows)"
    out = {"mpix_s": px / dt / 1e6, "msamples_s": samples / dt / 1e6, "seconds": dt, "pixels": px, "samples": samples,
           "cores": threads, "sample": what + ", clipped loop",
           "rows": rows, "ref_n": ref_n, "ref_rgb": ref_rgb}
    if count_sectors and stride == 1:
        # distinct 32-byte sectors the frame's samples touch (untimed second pass over the same rows)
        with oracle.SectorMaps(O) as M:
            O.render(cams[:1], W, H, mode="clipped")
        out["compulsory_bytes"] = M.compulsory_bytes()
        out["sectors"] = M.sectors()
    return out


def run_reference(args):
    """--impl reference: the CPU oracle as it stands, timed on the host cores (rank 0 only)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = args.config
    scene = synth.make_scene(cfg)
    cams = synth.make_cameras(cfg)
    W, H = synth.config_resolution(cfg)
    budget = 120.0 / max(args.steps + args.warmup, 1)
    times, res = [], None
    for i in range(args.warmup + args.steps):
        res = oracle_bounded(scene, cams, W, H, sampler=1 if args.sampler == "grid" else 0, budget_s=min(budget, 20.0), soft_eps=args.soft_eps)
        if i >= args.warmup:
            times.append(res)
    mp = float(np.mean([r["mpix_s"] for r in times]))
    line = {
        "impl": "reference", "metric": "Mpixels/s", "value": mp, "unit": "Mpixels/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": float(np.mean([r["seconds"] for r in times]) * 1e3),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32 decisions / f64 colour",
        "data": "synthetic", "config": {"workload": workload_name(cfg), "sample_per_step": res["sample"]},
        "gsamples_s": float(np.mean([r["msamples_s"] for r in times]) / 1e3),
        "cpu_baseline": {"value": mp, "unit": "Mpixels/s", "cores": res["cores"], "kind": "oracle", "sample": res["sample"]},
        "e2e": {"value": mp, "unit": "Mpixels/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def max_over_ranks(values, world: int, device: str):
    """Element-wise max over all ranks (the slowest rank defines the job's time)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values), device=device, dtype=torch.float64)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t.tolist()]


def aggregate_throughput(units_per_rank_step: float, steps: int, world: int, max_total_ms: float) -> float:
    """Whole-job units per second: every rank processed units_per_rank_step per step (weak scaling)."""
    return world * units_per_rank_step * steps / (max_total_ms / 1e3)


def gather_shares(plans, rank, my_rgb, my_n, n_views, H, W, device):
    """Optional last step of SURVEY 8(e): every rank's share is sent to rank 0 (peer copy over NVLink under NCCL, plain
    sockets under gloo), which assembles the batch.  my_rgb / my_n: this rank's share as torch tensors on `device` -
    mode "views": [len(views)][H][W][3] and [len(views)][H][W]; mode "rows": [rows][W][3] and [rows][W] for the flattened
    pixel rows of its band.  Returns (rgb, nsamples) on rank 0, None elsewhere."""
    import torch
    import torch.distributed as dist

    from paper_2404_09531_b200 import partition
    if rank != 0:
        if my_n.numel():
            dist.send(my_rgb.contiguous(), 0)
            dist.send(my_n.contiguous(), 0)
        return None
    rgb = torch.zeros((n_views, H, W, 3), dtype=my_rgb.dtype, device=device)
    ns = torch.zeros((n_views, H, W), dtype=my_n.dtype, device=device)
    seen = np.zeros(n_views * H, dtype=np.int32)
    for plan in plans:
        if plan.mode == "views":
            shape_rgb, shape_n = (len(plan.views), H, W, 3), (len(plan.views), H, W)
        else:
            r0, r1 = partition.pixel_row_range(plan, H)
            shape_rgb, shape_n = (r1 - r0, W, 3), (r1 - r0, W)
        if plan.rank == 0:
            p_rgb, p_n = my_rgb, my_n
        else:
            p_rgb = torch.empty(shape_rgb, dtype=my_rgb.dtype, device=device)
            p_n = torch.empty(shape_n, dtype=my_n.dtype, device=device)
            if p_n.numel():
                dist.recv(p_rgb, plan.rank)
                dist.recv(p_n, plan.rank)
        if plan.mode == "views":
            for i, v in enumerate(plan.views):
                rgb[v], ns[v] = p_rgb[i], p_n[i]
                seen[v * H:(v + 1) * H] += 1
        else:
            rgb.view(n_views * H, W, 3)[r0:r1] = p_rgb
            ns.view(n_views * H, W)[r0:r1] = p_n
            seen[r0:r1] += 1
    assert np.all(seen == 1), "every pixel row must be rendered by exactly one rank"
    return rgb, ns


def run_partitioned(omerf, h, cams, W, H, prev_n, world, rank, steps, timed, barrier, stream, comm_device="cuda"):
    """Strong scaling: the batch partitioned across the ranks by the previous frame's sample counts, timed
    like the main region (L2 flushed, CUDA events, max over ranks); then the shares are gathered on rank 0 and compared
    bit for bit with this rank's own full render.  comm_device: where the tensors that torch.distributed moves live -
    "cuda" under NCCL (one rank per GPU), "cpu" under gloo (shares staged through host memory; lets several ranks share
    one GPU, tests/test_gpu_partition.py)."""
    import torch

    from paper_2404_09531_b200 import partition
    n_views = cams.shape[0]
    prev = prev_n.cpu().numpy().view(np.uint32)
    plans = partition.make_plans(prev, world)
    plan = plans[rank]
    full_rgb = torch.empty((n_views, H, W, 3), dtype=torch.float32, device="cuda")
    full_n = torch.zeros((n_views, H, W), dtype=torch.int32, device="cuda")
    if plan.mode == "views":
        my_cams = cams[plan.views]
        my_rgb = torch.empty((len(plan.views), H, W, 3), dtype=torch.float32, device="cuda")
        my_n = torch.empty((len(plan.views), H, W), dtype=torch.int32, device="cuda")

        def step():
            if len(plan.views):
                omerf.render(h, my_cams, W, H, my_rgb, my_n, stream=stream)
    else:
        def step():
            omerf.render_tiles(h, cams, W, H, full_rgb, full_n, plan.tile_first, plan.tile_end, stream=stream)
    for _ in range(3):
        step()
    barrier()
    ms = timed(steps, True, step)
    barrier()
    if plan.mode == "rows":
        r0, r1 = partition.pixel_row_range(plan, H)
        my_rgb, my_n = full_rgb.view(n_views * H, W, 3)[r0:r1], full_n.view(n_views * H, W)[r0:r1]
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    if comm_device != "cuda":
        torch.cuda.synchronize()
        my_rgb, my_n = my_rgb.to(comm_device), my_n.to(comm_device)
    got = gather_shares(plans, rank, my_rgb, my_n, n_views, H, W, comm_device)
    e1.record(stream)
    barrier()
    total = max_over_ranks([float(np.sum(ms))], world, comm_device)[0]
    out = {"scaling": "strong", "mode": plan.mode, "ms_per_step": total / steps, "frames_per_s": n_views * steps / (total / 1e3),
           "mpixels_s": n_views * W * H * steps / (total / 1e3) / 1e6, "cost_imbalance": plan.imbalance,
           "sample_imbalance": plan.sample_imbalance, "samples_per_rank": [p.samples for p in plans],
           "gather_to_rank0_ms": e0.elapsed_time(e1), "parallelism": f"scene replicated x{world}, batch partitioned by {plan.mode}"}
    if rank == 0:
        ref_rgb = torch.empty(got[0].shape, dtype=got[0].dtype, device="cuda")
        ref_n = torch.empty(got[1].shape, dtype=got[1].dtype, device="cuda")
        omerf.render(h, cams, W, H, ref_rgb, ref_n, stream=stream)
        torch.cuda.synchronize()
        out["stitched_equals_single_rank"] = bool(torch.equal(got[1], ref_n.to(comm_device)) and torch.equal(got[0], ref_rgb.to(comm_device)))
    return out


def run_ours(args):
    import torch
    import torch.distributed as dist

    import paper_2404_09531_b200 as omerf

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the renderer has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    cfg = args.config
    scene = synth.make_scene(cfg)
    cams = synth.make_cameras(cfg)
    W, H = synth.config_resolution(cfg)
    n_views = cams.shape[0]
    sampler = omerf.SAMPLER_GRID if args.sampler == "grid" else omerf.SAMPLER_PLANE
    h = omerf.scene_create(scene, sampler=sampler, soft_eps=args.soft_eps, grid_block=args.grid_block, lowz_bake=args.lowz)
    info = omerf.scene_info(h)
    out_rgb = torch.empty((n_views, H, W, 3), dtype=torch.float32, device="cuda")
    out_n = torch.empty((n_views, H, W), dtype=torch.int32, device="cuda")
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")           # > 126 MB L2
    stream = torch.cuda.current_stream()
    pixels = n_views * W * H

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    def timed(n_steps, do_flush, fn):
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n_steps)]
        for a, b in evs:
            if do_flush:
                flush.fill_(1)
            a.record(stream)
            fn()
            b.record(stream)
        torch.cuda.synchronize()
        return [a.elapsed_time(b) for a, b in evs]

    def dev_step():
        omerf.render(h, cams, W, H, out_rgb, out_n, stream=stream)

    for _ in range(max(args.warmup, 3)):
        dev_step()
    barrier()
    clocks = ClockSampler(local)
    if rank == 0:
        clocks.start()
    ms = timed(args.steps, True, dev_step)                                     # the timed region: K steps
    barrier()
    launches_per_step = omerf.last_launch_count(h)
    ms_warm = timed(args.steps, False, dev_step)                               # extra: L2-warm static camera
    barrier()
    # extra (SURVEY 8(d) second regime): a yaw orbit, a new view every frame, no flush
    ms_orbit = None
    if n_views == 1 and cfg in (0, 1, 3, 4):
        orbit = synth.orbit_cameras(cfg, 64)
        it = iter(range(10 ** 9))

        def orbit_step():
            omerf.render(h, orbit[next(it) % 64:][:1], W, H, out_rgb, out_n, stream=stream)

        for _ in range(3):
            orbit_step()
        ms_orbit = timed(max(args.steps, 64), False, orbit_step)
        omerf.render(h, cams, W, H, out_rgb, out_n, stream=stream)              # restore the workload's own frame
        barrier()
    clk = clocks.stop() if rank == 0 else None
    total_ms = float(np.sum(ms))
    samples = int(out_n.sum(dtype=torch.int64).item())
    per_view = [int(x) for x in out_n.view(n_views, -1).sum(dim=1, dtype=torch.int64).tolist()]
    hist = torch.bincount(out_n.view(-1).clamp(max=63).to(torch.int64), minlength=64).tolist()   # samples/ray, last bin = 63+

    # N > 1: the SAME batch partitioned across the ranks: by views or by bands of tile rows, balanced by the
    # previous frame's sample counts; scene replicated, no collective on the data path; shares gathered on rank 0 afterwards
    strong = None
    if world > 1:
        strong = run_partitioned(omerf, h, cams, W, H, out_n, world, rank, args.steps, timed, barrier, stream)

    # configs[4]: the same frame through the other sampler (binary occupancy grid + DDA), timed the same way
    ablation = None
    if cfg == 4 and rank == 0:
        other = omerf.SAMPLER_PLANE if sampler == omerf.SAMPLER_GRID else omerf.SAMPLER_GRID
        h2 = omerf.scene_create(scene, sampler=other)
        n2 = torch.empty_like(out_n)
        rgb2 = torch.empty_like(out_rgb)

        def other_step():
            omerf.render(h2, cams, W, H, rgb2, n2, stream=stream)

        for _ in range(3):
            other_step()
        ms2 = float(np.mean(timed(args.steps, True, other_step)))
        s2 = int(n2.sum(dtype=torch.int64).item())
        name = {omerf.SAMPLER_PLANE: "plane", omerf.SAMPLER_GRID: "grid"}
        ablation = {name[sampler]: {"ms_per_frame": total_ms / args.steps, "frames_per_s": 1e3 / (total_ms / args.steps),
                                    "samples_per_ray": samples / pixels, "gsamples_s": samples / (total_ms / args.steps) / 1e6},
                    name[other]: {"ms_per_frame": ms2, "frames_per_s": 1e3 / ms2, "samples_per_ray": s2 / pixels,
                                  "gsamples_s": s2 / ms2 / 1e6, "occ_bits_set": omerf.scene_info(h2)["occ_bits_set"] or None},
                    "pixels_where_counts_differ": int((n2 != out_n).sum().item())}
        omerf.scene_destroy(h2)

    # gather calibration: the same frame's 10 entry loads per sample replayed with no arithmetic
    probe = omerf.gather_probe(h, cams[0], W, H, repeats=10, flush_l2=True) if rank == 0 else None

    # e2e through the C-ABI with HOST buffers (pinned), copies inside the timed region
    h_rgb = torch.empty((n_views, H, W, 3), dtype=torch.float32).pin_memory()
    h_n = torch.empty((n_views, H, W), dtype=torch.int32).pin_memory()

    def e2e_step():
        omerf.render_host(h, cams, W, H, h_rgb, h_n, stream=stream)

    for _ in range(3):
        e2e_step()
    barrier()
    t0 = time.perf_counter()
    ms_e2e = timed(args.steps, True, e2e_step)
    barrier()
    wall_e2e = time.perf_counter() - t0
    assert int(h_n.sum(dtype=torch.int64).item()) == samples, "host and device outputs disagree"

    # e2e, pipelined (the call a frame loop makes): K frames through omerf_render_host_async, two pinned host buffer sets in
    # turn, one omerf_wait at the end - frame N's copy-back overlaps frame N+1's render; every copy is inside the timed region
    h_sets = [(h_rgb, h_n), (torch.empty_like(h_rgb).pin_memory(), torch.empty_like(h_n).pin_memory())]

    def pipelined(n_frames):
        for i in range(n_frames):
            omerf.render_host_async(h, cams, W, H, *h_sets[i & 1], stream=stream)
        omerf.wait(h)

    pipelined(3)
    barrier()
    pa, pb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0 = time.perf_counter()
    pa.record(stream)
    pipelined(args.steps)
    pb.record(stream)                       # issued after omerf_wait returned: every host buffer has been delivered
    torch.cuda.synchronize()
    wall_pipe = time.perf_counter() - t0
    ms_pipe = pa.elapsed_time(pb)
    barrier()
    for hs in h_sets[:min(args.steps, 2)]:
        assert int(hs[1].sum(dtype=torch.int64).item()) == samples, "pipelined host outputs disagree with the device path"

    # max over ranks of the device time
    total_ms, total_e2e_ms, total_warm_ms, total_pipe_ms = max_over_ranks(
        [total_ms, float(np.sum(ms_e2e)), float(np.sum(ms_warm)), float(ms_pipe)], world, "cuda")

    if rank == 0:
        peaks = {}
        pk = os.path.join(ROOT, "MEASURED_PEAKS.json")
        if os.path.exists(pk):
            peaks = json.load(open(pk))
        hbm = float(peaks.get("hbm_gbs", 6650.0))
        k = args.steps
        secs = total_ms / 1e3
        march_ms = total_ms / k                                  # one launch per step: the fused march kernel
        alg_bytes = samples * BYTES_PER_SAMPLE + pixels * BYTES_PER_PIXEL
        achieved = alg_bytes / (march_ms / 1e3) / 1e9
        cpu = None
        if not args.no_cpu_baseline:
            cpu = oracle_bounded(scene, cams, W, H, sampler=1 if args.sampler == "grid" else 0, budget_s=15.0, soft_eps=args.soft_eps, count_sectors=True)
        # figures of the committed ncu capture apply to the workload that was captured only
        # and to the kernel sources that were captured: a later kernel change turns them into null, not into a stale figure
        sha = csrc_sha16()
        captured = (cfg == 1 and args.sampler == "plane" and not (args.soft_eps or args.grid_block or args.lowz)
                    and sha == NCU_CAPTURE["csrc_sha16"])
        props = torch.cuda.get_device_properties(local)
        issue_peak = props.multi_processor_count * 128 * float(peaks.get("sm_max_mhz", 1965.0)) * 1e6 / 1e12   # Tlane-op/s
        host_feature_bytes = int(sum(np.asarray(getattr(scene, nm)).nbytes for nm in ("grid", "plane_xy", "plane_xz", "plane_yz")))
        line = {
            "metric": "Mpixels/s", "value": aggregate_throughput(pixels, k, world, total_ms) / 1e6, "unit": "Mpixels/s", "n_gpus": world,
            "steps": k, "warmup": max(args.warmup, 3), "ms_per_step": total_ms / k, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32 (u8 features, integer interpolation)",
            "data": "synthetic",
            "config": {"workload": workload_name(cfg), "views": n_views, "W": W, "H": H, "sampler": args.sampler, "soft_eps": args.soft_eps, "grid_block": args.grid_block,
                       "lowz_bake": bool(args.lowz), "plane_bytes": info["plane_bytes"], "xz_band": info["xz_band"], "yz_band": info["yz_band"],
                       "grid_bytes": info["grid_bytes"], "grid_blocks": [info["grid_blocks_allocated"], info["grid_blocks_total"]],
                       "scene_device_bytes": info["device_bytes"],
                       # VRAM against the plain 8-byte-texel arrays of the host scene (the paired 16-byte entries double
                       # every stored texel; sparse blocks and the low-z bake store fewer texels)
                       "scene_host_feature_bytes": host_feature_bytes,
                       "device_over_host_feature_bytes": info["device_bytes"] / host_feature_bytes, "l2": "flushed between timed steps (256 MiB fill, "
                       "outside the event pairs); scene 296 MiB > L2", "parallelism": f"replicated scene x{world}"},
            "frames_per_s": world * n_views * k / secs,
            "gsamples_s": world * samples * k / secs / 1e9,
            "samples_per_step": samples, "samples_per_ray": samples / pixels,
            "per_view_samples": per_view, "samples_per_ray_hist": hist,
            "l2_warm": {"ms_per_step": total_warm_ms / k, "mpixels_s": world * pixels * k / (total_warm_ms / 1e3) / 1e6},
            "orbit": ({"ms_per_step_median": float(np.median(ms_orbit)), "ms_per_step_mean": float(np.mean(ms_orbit)),
                       "mpixels_s": pixels / (float(np.median(ms_orbit)) / 1e3) / 1e6, "views": 64} if ms_orbit else None),
            "ms_per_step_median": float(np.median(ms)),
            "e2e": {"value": world * pixels * k / (total_pipe_ms / 1e3) / 1e6, "unit": "Mpixels/s",
                    "h2d_bytes_per_step": int(cams.nbytes), "d2h_bytes_per_step": pixels * BYTES_PER_PIXEL,
                    "ms_per_step": total_pipe_ms / k, "wall_ms_per_step": wall_pipe * 1e3 / k,
                    "mode": "pipelined: K x omerf_render_host_async (cameras from host memory, outputs into two pinned host "
                            "buffer sets in turn) + one omerf_wait, all inside one CUDA-event pair; frame N's copy-back overlaps "
                            "frame N+1's render",
                    "l2": "not flushed between frames: the resident scene and the 16 B per pixel of output stream through L2 "
                          "(inputs larger than L2); the flushed one-call-at-a-time figure is `sync`",
                    "sync": {"value": world * pixels * k / (total_e2e_ms / 1e3) / 1e6, "ms_per_step": total_e2e_ms / k,
                             "wall_ms_per_step": wall_e2e * 1e3 / k,
                             "mode": "K x omerf_render_host, each call synchronised before the next; L2 flushed between calls"}},
            "gpu_launches": launches_per_step * k,
            # filled in below: the binding ceiling is the gather rate calibrated live on this frame
            "roofline": None,
            "gather_vs_hbm": {"bound": "hbm", "achieved": achieved, "peak": hbm, "unit": "GB/s", "frac": achieved / hbm,
                              "peak_source": "MEASURED_PEAKS.json hbm_gbs (of measured)" if peaks else "fallback 6650 (of fallback)",
                              "algorithmic_bytes_per_launch": alg_bytes, "launch_ms": march_ms,
                              "traffic": NCU_CAPTURE["dram_bytes"] if captured else None, "traffic_source": NCU_CAPTURE["profile"]},
            "clocks": clk,
        }
        if probe and probe["samples"]:
            ceil_gs = probe["samples"] / probe["ms_frame_order"] / 1e6           # Gsamples/s, gather only, frame order
            view0 = probe["samples"] / (march_ms / n_views) / 1e6 if n_views == 1 else samples * k / secs / 1e9
            # "the smallest ceiling is the roofline" - the L2/L1 gather rate, calibrated on this frame, this
            # layout, this GPU, in this run: requested texel bytes per second of the march kernel against the gather-only replay
            line["roofline"] = {
                "bound": "gather (L2/L1 gather rate, SURVEY 8(d); calibrated live, not HBM)", "kernel": "omerf_march_kernel",
                "achieved": view0 * TEXEL_BYTES_PER_SAMPLE, "peak": ceil_gs * TEXEL_BYTES_PER_SAMPLE, "unit": "GB/s",
                "unit_note": "requested texel bytes (samples x 160 B, served by L1/L2), NOT DRAM traffic: that is `traffic`",
                "peak_kind": "calibrated gather replay",
                "frac": view0 / ceil_gs, "traffic": NCU_CAPTURE["dram_bytes"] if captured else None,
                "traffic_source": NCU_CAPTURE["profile"] if captured else
                f"none: kernel sources {sha} are not the captured ones ({NCU_CAPTURE['csrc_sha16']}) or another workload",
                # the same launch against the measured HBM copy rate, in SURVEY 8(d)'s algorithmic bytes (168 B per sample
                # + 16 B per pixel): the figure that does not move with the calibration
                "hbm_frac": achieved / hbm, "hbm_achieved_gbs": achieved, "hbm_peak_gbs": hbm,
                "hbm_peak_source": "MEASURED_PEAKS.json hbm_gbs" if peaks else "fallback 6650",
                "algorithmic_bytes_per_launch": alg_bytes, "compulsory_bytes_oracle": None,
                "peak_source": "omerf_gather_probe in this run: the frame's texel loads replayed with no arithmetic, one sample "
                               "per thread, frame order, L2 flushed",
                "march_gsamples_s": view0, "ceiling_gsamples_s": ceil_gs, "launch_ms": march_ms,
                "scattered_gsamples_s": probe["samples"] / probe["ms_scattered"] / 1e6}
            line["gather_calibrated"] = {"frac": view0 / ceil_gs, "ceiling_gsamples_s": ceil_gs, "march_gsamples_s": view0}
        if captured and NCU_CAPTURE["warp_instructions"]:
            lane_ops = NCU_CAPTURE["warp_instructions"] * NCU_CAPTURE["lanes_per_instruction"]
            line["issue"] = {"bound": "alu", "achieved": lane_ops / (march_ms / 1e3) / 1e12, "peak": issue_peak, "unit": "Tlane-op/s",
                             "frac": lane_ops / (march_ms / 1e3) / 1e12 / issue_peak,
                             "what": "executed lane-operations of one launch (smsp__inst_executed.sum x lanes per instruction, "
                                     "ncu capture) / this run's launch time, against SMs x 128 lanes x max SM clock of this device",
                             "source": NCU_CAPTURE["profile"], "commit": NCU_CAPTURE["commit"]}
        if strong is not None:
            line["strong"] = strong
        if ablation is not None:
            line["ablation"] = ablation
        if cpu is not None:
            # element-wise parity of the rows the oracle just rendered (the whole frame when it fits the time budget)
            # against the device outputs of the timed workload; outside every timed region
            got_n = out_n[0].cpu().numpy().view(np.uint32)[cpu["rows"]]
            got_rgb = out_rgb[0].cpu().numpy()[cpu["rows"]].astype(np.float64)
            line["parity"] = {"pixels_compared": int(got_n.size), "of_pixels_in_view0": W * H,
                              "count_mismatches": int((got_n != cpu["ref_n"]).sum()),
                              "max_abs_drgb": float(np.abs(got_rgb - cpu["ref_rgb"]).max()), "rgb_tol": 2e-3,
                              "against": "oracle (clipped loop), same run"}
            line["cpu_baseline"] = {"value": cpu["mpix_s"], "unit": "Mpixels/s", "cores": cpu["cores"], "kind": "oracle",
                                    "sample": cpu["sample"], "msamples_s": cpu["msamples_s"], "seconds": cpu["seconds"]}
            if "compulsory_bytes" in cpu:     # the HBM ceiling of SURVEY 8(d): bytes an unbounded cache would still fetch
                line["gather_vs_hbm"]["compulsory_bytes_oracle"] = cpu["compulsory_bytes"]
                line["gather_vs_hbm"]["compulsory_sectors_oracle"] = cpu["sectors"]
                line["gather_vs_hbm"]["compulsory_ms_at_peak"] = cpu["compulsory_bytes"] / (hbm * 1e9) * 1e3
                if line["roofline"] is not None:
                    line["roofline"]["compulsory_bytes_oracle"] = cpu["compulsory_bytes"]
        print(json.dumps(line))
    omerf.scene_destroy(h)
    if world > 1:
        dist.destroy_process_group()


def run_smoothness(args):
    """--workload smoothness: Eq. 9-10 forward over 2^20 directions x 15 perturbations on the
    config-1 scene's MLP.  Secondary line: same JSON shape, metric = MLP evaluations per second."""
    import torch

    import paper_2404_09531_b200 as omerf
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    n, S = 1 << 20, 15
    scene = synth.make_scene(0)                  # the MLP is all this workload uses; weights are Xavier as everywhere
    F, d, delta = synth.smoothness_batch(7, n, S)
    h = omerf.scene_create(scene)
    tF, td, tdl = (torch.from_numpy(a).cuda() for a in (F, d, delta))
    out = torch.empty(n, dtype=torch.float32, device="cuda")
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    stream = torch.cuda.current_stream()
    for _ in range(max(args.warmup, 3)):
        omerf.mlp_smoothness(h, tF, td, tdl, out_loss=out)
    torch.cuda.synchronize()
    ms = []
    for _ in range(args.steps):
        flush.fill_(1)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        omerf.mlp_smoothness(h, tF, td, tdl, out_loss=out)
        b.record(stream)
        torch.cuda.synchronize()
        ms.append(a.elapsed_time(b))
    evals = n * (S + 1)
    t = float(np.mean(ms)) / 1e3
    peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json"))) if os.path.exists(os.path.join(ROOT, "MEASURED_PEAKS.json")) else {}
    hbm = float(peaks.get("hbm_gbs", 6650.0))
    alg_bytes = n * (7 + 3 + 3 * S + 1) * 4
    tflops = evals * 2 * 883 / t / 1e12
    tf32_peak = float(peaks.get("bf16_tflops", 2250.0)) * 0.5
    import oracle
    m = 4096
    t0 = time.perf_counter()
    oracle.mlp_smoothness(oracle.OracleScene(scene), F[:m], d[:m], delta[:m])
    cpu_s = time.perf_counter() - t0
    line = {"metric": "MLP evaluations/s", "value": evals / t, "unit": "eval/s", "n_gpus": 1, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": t * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32 (3xTF32 tensor-core products)", "data": "synthetic",
            "config": {"workload": "SURVEY 8(f).3 smoothness term, 2^20 directions x 15 perturbations", "n": n, "S": S,
                       "l2": "flushed between timed steps"},
            "gpu_launches": args.steps, "mean_loss": float(out.mean().item()),
            # a dense contraction (883 MACs per evaluation) on tensor cores: tf32 peak = measured bf16 peak x 1/2 (guide's
            # nominal ratio); the kernel issues 3 tf32 products per algorithmic product (hi/lo split for fp32 accuracy)
            "roofline": {"bound": "tensor", "achieved": tflops, "peak": tf32_peak, "unit": "TFLOP/s", "frac": tflops / tf32_peak,
                         "traffic": None, "algorithmic_flops_per_launch": evals * 2 * 883, "executed_mma_tflops": 3 * tflops,
                         "peak_source": "MEASURED_PEAKS.json bf16_tflops x 0.5 (tf32)" if peaks else "fallback 2250 x 0.5",
                         "hbm_gbs_algorithmic": alg_bytes / t / 1e9, "hbm_peak": hbm},
            "cpu_baseline": {"value": m * (S + 1) / cpu_s, "unit": "eval/s", "cores": os.cpu_count(), "kind": "oracle",
                             "sample": f"first {m} directions"}}
    print(json.dumps(line))
    omerf.scene_destroy(h)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=1, choices=[0, 1, 2, 3, 4, 5])
    ap.add_argument("--sampler", default="plane", choices=["plane", "grid"])
    ap.add_argument("--soft-eps", type=float, default=0.0, help="SURVEY 8(f).2: soft occupancy (Eq. 6-8) buffer height; 0 = binary mask")
    ap.add_argument("--grid-block", type=int, default=0, help="SURVEY 8(f).1: store V as sparse blocks of this edge (0 = dense)")
    ap.add_argument("--lowz", action="store_true", help="SURVEY 8(f).1: low-z bake of the xz / yz planes (PAPER.md:186)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--workload", default="render", choices=["render", "smoothness"])
    args = ap.parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ and args.impl == "ours":
        # not under a launcher yet: start one rank per GPU ourselves (same command line), NCCL over NVLink for the barriers
        import socket
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__), *sys.argv[1:]]
        raise SystemExit(subprocess.call(cmd))
    if args.workload == "smoothness" and args.impl == "ours":
        run_smoothness(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
