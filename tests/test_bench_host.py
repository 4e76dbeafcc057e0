"""Host-side logic of bench.py for N > 1, on CPU with the gloo backend (world_size 2)."""
import json
import os
import socket
import subprocess
import sys

import pytest
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    local = [10.0 + 5.0 * rank, 3.0 - rank, 7.0]          # per-rank device times (ms)
    got = bench.max_over_ranks(local, world, "cpu")
    val = bench.aggregate_throughput(1920 * 1080, 4, world, got[0])
    out.put((rank, got, val))
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_and_aggregate_world2():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = [q.get(timeout=120) for _ in procs]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, got, val in res:
        assert got == [15.0, 3.0, 7.0]                     # slowest rank per entry
        assert val == pytest.approx(2 * 1920 * 1080 * 4 / 15e-3)


def _partition_worker(rank, world, port, out):
    """One rank of the partitioned render on CPU: the oracle stands in for the GPU renderer, gloo for NCCL;
    partitioner, share bookkeeping and the gather onto rank 0 are the code bench.py runs."""
    import numpy as np
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    import oracle
    import synth
    from paper_2404_09531_b200 import partition
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    sc = synth.make_scene(0)
    O = oracle.OracleScene(sc)
    res = {}
    for name, cams, W, H in (("rows", synth.make_cameras(0), 64, 98),                      # one view, ragged height
                             ("views", synth.orbit_cameras(0, 6), 40, 32)):                # six views on two ranks
        full = O.render(cams, W, H, mode="clipped")                                        # "previous frame" = single-rank render
        plans = partition.make_plans(full["nsamples"], world)
        plan = plans[rank]
        assert plan.mode == name
        if plan.mode == "views":
            r = O.render(cams[plan.views], W, H, mode="clipped")
            my_rgb, my_n = torch.from_numpy(r["rgb"]), torch.from_numpy(r["nsamples"].astype(np.int64))
        else:
            r0, r1 = partition.pixel_row_range(plan, H)
            assert (r0, r1) == (min(plan.row_first * 4, H), min(plan.row_end * 4, H))
            assert plan.tile_first == plan.row_first * 8 and plan.tile_end == plan.row_end * 8   # 64 / 8 tiles per row
            r = O.render(cams, W, H, mode="clipped", rows=(r0, r1))
            my_rgb, my_n = torch.from_numpy(r["rgb"][0, r0:r1]), torch.from_numpy(r["nsamples"][0, r0:r1].astype(np.int64))
        got = bench.gather_shares(plans, rank, my_rgb, my_n, cams.shape[0], H, W, "cpu")
        if rank == 0:
            same = bool(np.array_equal(got[1].numpy(), full["nsamples"]) and np.array_equal(got[0].numpy(), full["rgb"]))
            if name == "views":
                covered = sorted(v for p in plans for v in p.views) == list(range(cams.shape[0]))
            else:
                covered = plans[0].tile_first == 0 and plans[-1].tile_end == 8 * 25 and all(
                    a.tile_end == b.tile_first for a, b in zip(plans, plans[1:]))
            res[name] = (same, covered, plan.imbalance, [p.samples for p in plans], int(full["nsamples"].sum()))
    out.put((rank, res))
    dist.barrier()
    dist.destroy_process_group()


def test_partitioned_render_world2_every_tile_once_balanced_and_bit_identical():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_partition_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = dict(q.get(timeout=300) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for name in ("rows", "views"):
        same, covered, imb, per_rank, total = res[0][name]
        assert same, f"{name}: the stitched batch differs from the single-rank render"
        assert covered, f"{name}: some tile or view is not rendered exactly once"
        assert sum(per_rank) == total
        assert imb <= 0.10, f"{name}: cost imbalance {imb}"


def test_partitioner_properties():
    """Contiguous bands: optimal bottleneck on small cases (brute force); views: every view once; one rank = everything."""
    import itertools

    import numpy as np
    sys.path.insert(0, ROOT)
    from paper_2404_09531_b200 import partition
    rng = np.random.default_rng(3)
    for _ in range(30):
        n, world = int(rng.integers(3, 9)), int(rng.integers(1, 4))
        c = rng.integers(0, 50, n).astype(np.float64)
        b = partition.split_rows(c, world)
        assert b[0] == 0 and b[-1] == n and np.all(np.diff(b) >= 0) and len(b) == world + 1
        got = max(c[b[i]:b[i + 1]].sum() for i in range(world))
        best = min(max(c[x:y].sum() for x, y in zip((0, *cut), (*cut, n)))
                   for cut in itertools.combinations_with_replacement(range(n + 1), world - 1))
        assert got <= best + 1e-9
    ns = rng.integers(0, 30, (7, 20, 24))
    parts = partition.assign_views(partition.view_costs(ns), 3)
    assert sorted(v for p in parts for v in p) == list(range(7))
    plans = partition.make_plans(ns[:1], 1)
    assert plans[0].mode == "views" and plans[0].views == [0]
    plans = partition.make_plans(ns[:1], 3)          # fewer views than ranks: bands of tile rows
    assert plans[0].mode == "rows" and plans[0].tile_first == 0 and plans[-1].tile_end == 3 * 5
    # balanced by samples, not pixels: an empty (sky) upper half pushes the boundary down
    ns2 = np.zeros((1, 64, 64), dtype=np.int64)
    ns2[0, 32:] = 40
    p2 = partition.make_plans(ns2, 2)
    assert p2[0].row_end > 8 and p2[0].imbalance < 0.1


def test_reference_arm_prints_one_json_line():
    """--impl reference runs the oracle on a bounded sample (tiny config here) and prints the contract keys."""
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "0",
                          "--steps", "1", "--warmup", "0"], capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "Mpixels/s" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["gpu_launches"] == 0


def test_reference_arm_other_ranks_exit_quietly():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "0",
                          "--steps", "1", "--warmup", "0", "--gpus", "2"], capture_output=True, text=True, timeout=120,
                         cwd=ROOT, env=env)
    assert out.returncode == 0 and out.stdout.strip() == ""


def test_cited_ncu_figures_are_keyed_on_the_kernel_sources():
    """bench.NCU_CAPTURE (DRAM traffic, instruction counts of one committed ncu capture) names the hash of the kernel
    sources it was taken at; bench.py prints the figures only while csrc_sha16() equals it and null otherwise, so a
    kernel change can never be reported beside a stale capture.  The hash is over content: stable across calls, 16 hex
    digits, and the profile it cites exists."""
    import bench
    h = bench.csrc_sha16()
    assert h == bench.csrc_sha16() and len(h) == 16 and int(h, 16) >= 0
    assert len(bench.NCU_CAPTURE["csrc_sha16"]) == 16
    assert os.path.exists(os.path.join(bench.ROOT, bench.NCU_CAPTURE["profile"]))
