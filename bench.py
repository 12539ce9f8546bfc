#!/usr/bin/env python
"""bench.py -- TACAW hot path on B200: slice-steps/s and fraction of the HBM roofline.

One "step" = one pass of the whole hot path over one batch of the workload (default configs[1] of
BASELINE.json: rutile 8x8x20, 256^2 grid, 4 probes x 256 frames x 40 slices):
  tacaw_build_slices for every frame -> tacaw_propagate (all probes x frames x slices) ->
  tacaw_accumulate (q-ROI gather) -> tacaw_spectrum.
`value`  : slice-steps/s with the inputs (atom positions of every frame) resident in HBM.
`e2e`    : the same metric through the C ABI with HOST buffers (positions copied H2D inside the
           timed region through tacaw_build_slices_host, the spectrum I(q,E) copied back D2H).
`roofline`: the fused slice-step kernel pair (k_row + k_col), algorithmic bytes
           B_step = 16 N^2 + 8 N^2/R per wave and slice over the CUDA-event time of the
           tacaw_propagate calls inside the timed region.
`cpu_baseline`: the fp64 oracle, as it stands, on a bounded sample of the same workload.
`--impl reference` times the oracle alone (this tier's reference arm).
Multi-GPU (`--gpus N` under torchrun): every rank runs its own scan batch of the same size (the
paper's independent computational batches) -- no data-path collective; weak scaling.
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

METRIC = "multislice slice-steps/s (probe x frame x slice)"
UNIT = "slice-steps/s"


def load_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            d = json.load(open(p))
            return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def workload_config(wl, extra=None):
    c = {"workload": f"BASELINE.json configs[{int(wl.name[1]) - 1}] ({wl.name}): rutile TiO2, {wl.nx}x{wl.ny} grid, "
                     f"{wl.nprobes} probes x {wl.nframes} frames x {wl.nslices_total} slices",
         "grid": [wl.nx, wl.ny], "probes": wl.nprobes, "frames": wl.nframes, "slices": wl.nslices_total,
         "atoms": wl.natoms, "roi_pixels": None, "slice_steps_per_step": wl.slice_steps,
         "l2": "inputs larger than L2 (transmissions + waves of one step >> 126 MB); no flush needed"}
    if extra:
        c.update(extra)
    return c


def shard_workload(wl, rank: int):
    """Rank r works on its own scan batch: the same raster shifted by 0.1 A * r (independent unit)."""
    if rank > 0:
        wl.probes_xy = wl.probes_xy + 0.1 * rank
    return wl


def max_over_ranks(value_ms: float, dist, device):
    """Timing contract: the step time of the job is the slowest rank's."""
    if dist is None:
        return value_ms
    import torch
    t = torch.tensor([value_ms], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 50 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows = []
        self.proc = None
        self.index = index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "50"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([s.strip() for s in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
                for n, v in zip(names, r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                continue
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def oracle_sample(wl, nframes_sample: int):
    """Time the oracle, as it stands, on `nframes_sample` frames x all probes x all slices."""
    import oracle
    from oracle import pipeline as OP
    oracle.build()
    t0 = time.perf_counter()
    OP.exit_waves(wl, list(range(nframes_sample)), output_space=1, pot_mode=1)
    dt = time.perf_counter() - t0
    steps = wl.nprobes * wl.nslices_total * nframes_sample
    return steps / dt, dt, oracle.num_threads()


def oracle_plan(args, wl):
    """Bounded oracle sample: <= 4 probes and as many frames as give roughly 15 s of host work (--ref-frames overrides).
    The estimate scales a measured 280 slice-steps/s (16 cores, 256^2) by the N^2 log N cost of a slice step."""
    from paper_2607_02236_b200 import workloads as W
    import math
    npr = min(wl.nprobes, 4)
    wls = wl if npr == wl.nprobes else W.make_workload(args.config, nframes=wl.nframes, nprobes=npr)
    if args.ref_frames is not None:
        nf = max(1, args.ref_frames)
    else:
        cores = max(1, min(16, len(os.sched_getaffinity(0))))
        rate = 280.0 * (cores / 16.0) * (256.0 * 256.0 * 16.0) / (wl.nx * wl.ny * math.log2(wl.nx * wl.ny))
        nf = int(max(1, min(wl.nframes, round(15.0 * rate / (npr * wl.nslices_total)))))
    return wls, nf


def run_reference(args, wl):
    """--impl reference: the fp64 oracle on host cores, bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    wl, nf = oracle_plan(args, wl)
    for _ in range(args.warmup):
        oracle_sample(wl, 1)
    vals, times = [], []
    for _ in range(args.steps):
        v, dt, cores = oracle_sample(wl, nf)
        vals.append(v); times.append(dt)
    value = float(np.sum([wl.nprobes * wl.nslices_total * nf] * len(times)) / np.sum(times))
    sample = f"{nf} frame(s) x {wl.nprobes} probes x {wl.nslices_total} slices of {wl.name} per step (build + propagate)"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * float(np.mean(times)), "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "complex128", "data": "synthetic",
            "config": workload_config(wl, {"sample": sample}),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="tacaw", choices=["tacaw", "reference"])
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config number 1..5 (default 2 = configs[1])")
    ap.add_argument("--frames", type=int, default=None, help="truncate the workload to its first FRAMES frames")
    ap.add_argument("--probes", type=int, default=None, help="truncate the workload to its first PROBES probes")
    ap.add_argument("--ref-frames", type=int, default=None, help="frames per step of the oracle sample (default: ~15 s of host work)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    args = ap.parse_args()

    from paper_2607_02236_b200 import workloads as W
    wl = W.make_workload(args.config, nframes=args.frames, nprobes=args.probes)
    if args.impl == "reference":
        run_reference(args, wl)
        return

    import torch
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the TACAW path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local_rank}"))
    shard_workload(wl, rank)          # every rank = its own scan batch of the same size

    from paper_2607_02236_b200 import build as _build
    _build.build_lib()                # no-op when libtacaw.so matches the sources; never a fallback: it raises if nvcc fails
    from paper_2607_02236_b200.pipeline import Runner
    r = Runner(wl, device=local_rank)
    r.alloc_buffer()
    dev = r.dev
    # inputs resident in HBM: positions of every frame and segment
    pos_h = [seg.frames(0, wl.nframes, wl.dt_fs) for seg in wl.segments]
    pos_d = [torch.from_numpy(p).to(dev) for p in pos_h]
    spec_h = [np.ascontiguousarray(s.species, dtype=np.int32) for s in wl.segments]
    R = r.P
    npix = wl.nx * wl.ny
    b_step = 16 * npix + 8 * npix / R

    prop_events = []

    def one_step(timed: bool):
        for f0 in range(0, wl.nframes, r.fpb):
            nf = min(r.fpb, wl.nframes - f0)
            r.build_block([p[f0:f0 + nf] for p in pos_d], nf)
            if timed:
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
            _, wp, wf = r.propagate_block(nf, 1)
            if timed:
                e1.record()
                prop_events.append((e0, e1, nf * R * wl.nslices_total))
            r.gather_block(nf, f0, wp, wf)
        return r.spectrum()

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        one_step(False)
    barrier()
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    l0 = r.tc.launches
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record()
    for _ in range(args.steps):
        I, E = one_step(True)
    ev1.record()
    barrier()
    elapsed_ms = ev0.elapsed_time(ev1)
    launches = r.tc.launches - l0
    clocks = sampler.stop() if rank == 0 else None
    elapsed_ms = max_over_ranks(elapsed_ms, dist, dev)
    total_steps = wl.slice_steps * args.steps * world
    value = total_steps / (elapsed_ms * 1e-3)

    prop_ms = sum(a.elapsed_time(b) for a, b, _ in prop_events)
    prop_units = sum(n for _, _, n in prop_events)
    peak, peak_src = load_peak()
    achieved = prop_units * b_step / (prop_ms * 1e-3) / 1e9
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": None,
                "kernel": "fused slice-step pair k_row<N,MID> + k_col<N,MID> (one slice step of every wave in a launch)",
                "bytes_per_slice_step": b_step, "peak_source": peak_src,
                "propagate_share_of_step": prop_ms / elapsed_ms,
                "propagate_slice_steps_per_s": prop_units / (prop_ms * 1e-3)}
    # dram__bytes_read.sum + dram__bytes_write.sum of the pair from the committed ncu --set full capture, per slice
    # step like `bytes_per_slice_step`, times the slice steps one tacaw_propagate launch pair covers
    tr = os.path.join(ROOT, "profiles", "r1_traffic.csv")
    if os.path.exists(tr):
        try:
            import csv
            for row in csv.DictReader(open(tr)):
                if row["workload"] == wl.name:
                    roofline["traffic"] = float(row["dram_bytes_per_slice_step"])
                    roofline["traffic_note"] = "bytes per slice step (one wave, row + column kernel), cold-cache ncu capture"
        except Exception:
            pass

    # ---- end to end through the C ABI with host buffers ------------------------------------
    e2e = None
    if not args.no_e2e:
        I_host = torch.empty(I.shape, dtype=I.dtype).pin_memory()
        # the step's inputs live in pinned host memory (numpy views of pinned tensors)
        pos_pin = [torch.from_numpy(p).pin_memory() for p in pos_h]
        pos_hp = [t.numpy() for t in pos_pin]
        h2d = sum(p.nbytes for p in pos_h) + sum(s.nbytes for s in spec_h) * ((wl.nframes + r.fpb - 1) // r.fpb)
        d2h = I_host.numel() * 4

        def e2e_step():
            for f0 in range(0, wl.nframes, r.fpb):
                nf = min(r.fpb, wl.nframes - f0)
                r.build_block_host(pos_hp, f0, nf)
                _, wp, wf = r.propagate_block(nf, 1)
                r.gather_block(nf, f0, wp, wf)
            Ie, _ = r.spectrum()
            I_host.copy_(Ie, non_blocking=True)
            torch.cuda.synchronize()

        e2e_step()
        barrier()
        t0 = time.perf_counter()
        nrep = max(1, min(args.steps, 3))
        for _ in range(nrep):
            e2e_step()
        barrier()
        e_ms = (time.perf_counter() - t0) * 1e3
        e_ms = max_over_ranks(e_ms, dist, dev)
        e2e = {"value": wl.slice_steps * nrep * world / (e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": int(h2d),
               "d2h_bytes_per_step": int(d2h), "steps": nrep}

    # Welch average over half-length chunks (nu = 2) of the resident time-ordered buffer
    welch = None
    if wl.nframes >= 16:
        Lc = 1 << ((wl.nframes // 2).bit_length() - 1)
        r.spectrum_welch(Lc, 2)
        w0, w1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        w0.record()
        for _ in range(5):
            _, _, nch = r.spectrum_welch(Lc, 2)
        w1.record()
        torch.cuda.synchronize()
        w_ms = w0.elapsed_time(w1) / 5
        in_bytes = nch * Lc * wl.nprobes * int(r.roi.numel()) * 8
        welch = {"chunk_len": Lc, "chunk_overlap": 2, "nchunks": int(nch), "window": "hann", "ms": w_ms,
                 "spectra_per_s": wl.nprobes * int(r.roi.numel()) / (w_ms * 1e-3), "read_GBps": in_bytes / (w_ms * 1e-3) / 1e9}

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        wls, nfs = oracle_plan(args, wl)
        v, dt, cores = oracle_sample(wls, nfs)
        cpu = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"{nfs} frame(s) x {wls.nprobes} probes x {wl.nslices_total} slices of {wl.name} "
                         f"(build + propagate), {dt:.1f} s"}

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": elapsed_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "complex64", "data": "synthetic",
                "config": workload_config(wl, {"roi_pixels": int(r.roi.numel()), "frames_per_block": r.fpb,
                                               "parallelism": f"replicas x{world} (independent scan batches, no collective)"}),
                "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline, "cpu_baseline": cpu,
                "spectra_per_s": wl.nprobes * int(r.roi.numel()) * args.steps * world / (elapsed_ms * 1e-3), "welch": welch}
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
