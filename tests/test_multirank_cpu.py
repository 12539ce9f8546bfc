"""world_size-2 gloo test (CPU) of bench.py's multi-rank host logic: every rank gets its own scan
batch (no data-path collective) and the job time is the max over ranks."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    from paper_2607_02236_b200 import workloads as W
    wl = bench.shard_workload(W.make_workload(2, nframes=8), rank)
    t = bench.max_over_ranks(10.0 + 5.0 * rank, dist, torch.device("cpu"))
    dist.barrier()
    q.put((rank, wl.probes_xy.copy(), wl.slice_steps, t))
    dist.destroy_process_group()


def test_two_rank_sharding_and_max_time():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + (os.getpid() % 2000)
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted([q.get(timeout=120) for _ in procs], key=lambda x: x[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, xy0, n0, t0), (r1, xy1, n1, t1) = res
    assert n0 == n1                                   # weak scaling: same work per rank
    assert np.allclose(xy1 - xy0, 0.1)                # a different scan batch per rank
    assert t0 == t1 == 15.0                           # max over ranks


def test_reference_arm_rank_gating(monkeypatch, capsys):
    """--impl reference: only rank 0 runs and prints (ranks > 0 return without work)."""
    sys.path.insert(0, ROOT)
    import bench
    monkeypatch.setenv("RANK", "1")

    class A:
        ref_frames, warmup, steps, gpus = 1, 0, 1, 2
    bench.run_reference(A, None, 1)
    assert capsys.readouterr().out == ""


def test_oracle_plan_is_bounded_for_every_config():
    """The oracle sample of bench.py (cpu_baseline / --impl reference) stays a bounded piece of the same workload: at most 4
    probes, whole frames for the small configs, one frame of a z-thinned sample with the same lateral cell, grid and atoms per
    slice for the large ones."""
    sys.path.insert(0, ROOT)
    import bench
    from paper_2607_02236_b200 import workloads as W

    class A:
        ref_frames = None
    for cfg in (1, 2, 3, 4, 5):
        wl = W.make_workload(cfg, nprobes=128 if cfg == 5 else None)
        wls, nf, cells = bench.oracle_plan(A, wl)
        assert wls.nprobes <= 4 and nf >= 1 and (wls.nx, wls.ny, wls.lx) == (wl.nx, wl.ny, wl.lx)
        assert wls.natoms / wls.nslices_total == wl.natoms / wl.nslices_total
        if cfg <= 2:
            assert cells is None and wls.nslices_total == wl.nslices_total
        if cfg == 5:
            assert cells is not None and wls.nslices_total < wl.nslices_total
