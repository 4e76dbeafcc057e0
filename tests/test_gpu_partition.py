"""SURVEY 8(e) on the GPU (-m gpu): every rank's share of a partitioned batch, rendered through omerf_render_tiles /
omerf_render on one device, stitches to the single-rank render bit for bit - first with all shares rendered by one
process, then end to end: two rank PROCESSES that share GPU 0 run bench.run_partitioned (the code of `bench.py --gpus N`)
with the real library, each with its own scene, and rank 0 assembles the batch.  The ranks talk over gloo with the
shares staged through host memory, because NCCL refuses two ranks on one GPU; the NCCL transport of the same gather has
not run on hardware (no multi-GPU box in this project), which DESIGN.md sec. 6 states."""
import os
import socket
import sys

import numpy as np
import pytest

import synth

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _two_ranks_worker(rank, world, port, out):
    """One rank of the end-to-end test: own process, own CUDA context on GPU 0, own omerf scene."""
    sys.path.insert(0, ROOT)
    import torch
    import torch.distributed as dist

    import bench
    import paper_2404_09531_b200 as omerf
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    torch.cuda.set_device(0)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    stream = torch.cuda.current_stream()

    def barrier():
        torch.cuda.synchronize()
        dist.barrier()

    def timed(n_steps, do_flush, fn):
        ms = []
        for _ in range(n_steps):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            fn()
            e1.record(stream)
            e1.synchronize()
            ms.append(e0.elapsed_time(e1))
        return ms

    res = {}
    with omerf.scene_create(synth.make_scene(0)) as h:
        for name, cams, W, H in (("rows", synth.make_cameras(0), 130, 99),         # one view on two ranks: bands of tile rows
                                 ("views", synth.orbit_cameras(0, 6), 64, 48)):    # six views on two ranks
            _, ns = omerf.render(h, cams, W, H)                                    # "previous frame": balances the shares
            torch.cuda.synchronize()
            r = bench.run_partitioned(omerf, h, cams, W, H, ns, world, rank, 2, timed, barrier, stream, comm_device="cpu")
            res[name] = {k: r.get(k) for k in ("mode", "stitched_equals_single_rank", "samples_per_rank", "ms_per_step")}
            res[name]["total"] = int(ns.sum(dtype=torch.int64).item())
    out.put((rank, res))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_processes_on_one_gpu_run_the_partitioned_bench_path():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import torch.multiprocessing as mp
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_two_ranks_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    try:
        res = dict(q.get(timeout=600) for _ in procs)
    finally:
        for p in procs:
            p.join(timeout=120)
            if p.is_alive():
                p.kill()
    assert all(p.exitcode == 0 for p in procs)
    for name in ("rows", "views"):
        r0 = res[0][name]
        assert r0["mode"] == name == res[1][name]["mode"]
        assert r0["stitched_equals_single_rank"] is True, f"{name}: rank 0's assembled batch differs from its own full render"
        assert res[1][name]["stitched_equals_single_rank"] is None            # only rank 0 assembles
        assert sum(r0["samples_per_rank"]) == r0["total"] and min(r0["samples_per_rank"]) > 0
        assert r0["ms_per_step"] > 0


@pytest.fixture(scope="module")
def omerf():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2404_09531_b200 as m
    m.load_library()
    return m


@pytest.mark.parametrize("world", [2, 3, 8])
def test_shares_stitch_to_the_single_rank_render(omerf, world):
    import torch

    from paper_2404_09531_b200 import partition
    sc = synth.make_scene(0)
    for cams, W, H in ((synth.make_cameras(0), 130, 99),               # one view: bands of tile rows, ragged sizes
                       (synth.orbit_cameras(0, 16), 64, 48)):          # 16 views: whole views, longest first
        n_views = cams.shape[0]
        with omerf.scene_create(sc) as h:
            rgb, ns = omerf.render(h, cams, W, H)
            torch.cuda.synchronize()
            full_rgb, full_n = rgb.cpu().numpy(), ns.cpu().numpy()
            plans = partition.make_plans(full_n.view(np.uint32), world)          # previous frame's counts
            parts = []
            for plan in plans:
                if plan.mode == "views":
                    r, n = omerf.render(h, cams[plan.views], W, H)
                    torch.cuda.synchronize()
                    parts.append((r.cpu().numpy(), n.cpu().numpy()))
                else:
                    r = torch.full((n_views, H, W, 3), -7.0, dtype=torch.float32, device="cuda")
                    n = torch.full((n_views, H, W), -7, dtype=torch.int32, device="cuda")
                    omerf.render_tiles(h, cams, W, H, r, n, plan.tile_first, plan.tile_end)
                    torch.cuda.synchronize()
                    r0, r1 = partition.pixel_row_range(plan, H)
                    rr, nn = r.cpu().numpy().reshape(n_views * H, W, 3), n.cpu().numpy().reshape(n_views * H, W)
                    assert np.all(nn[:r0] == -7) and np.all(nn[r1:] == -7) and np.all(rr[:r0] == -7.0)   # nothing else is written
                    parts.append((rr[r0:r1], nn[r0:r1]))
        got_rgb, got_n = partition.stitch(plans, parts, n_views, H, W)
        assert np.array_equal(got_n, full_n) and np.array_equal(got_rgb, full_rgb)
        assert sum(p.samples for p in plans) == int(full_n.view(np.uint32).sum())


def test_render_tiles_argument_checks(omerf):
    import torch
    sc, cams = synth.make_scene(0), synth.make_cameras(0)
    W, H = 64, 48
    tiles = 8 * 12
    with omerf.scene_create(sc) as h:
        r = torch.zeros((1, H, W, 3), dtype=torch.float32, device="cuda")
        n = torch.zeros((1, H, W), dtype=torch.int32, device="cuda")
        omerf.render_tiles(h, cams, W, H, r, n, 5, 5)                  # empty range: no-op
        torch.cuda.synchronize()
        assert omerf.last_launch_count(h) == 0 and int(n.abs().sum().item()) == 0
        for first, end in ((3, 2), (0, tiles + 1)):
            with pytest.raises(omerf.OmerfError):
                omerf.render_tiles(h, cams, W, H, r, n, first, end)
        omerf.render_tiles(h, cams, W, H, r, n, 0, tiles)
        ref_r, ref_n = omerf.render(h, cams, W, H)
        torch.cuda.synchronize()
        assert torch.equal(n, ref_n) and torch.equal(r, ref_r)
