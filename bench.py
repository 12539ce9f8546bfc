#!/usr/bin/env python
"""bench.py -- TACAW hot path on B200: slice-steps/s and fraction of the HBM roofline.

Default workload (N = 1): the largest single-GPU configuration of BASELINE.json, configs[4] (c5: rutile 24x24x60 with a planar
fault, 2048^2 grid, 120 slices), as ONE scan sub-batch of 128 probes (rows 0-3 of the 32x32 raster, `scanning_batch_shape`
4x32, Listing 1 :428).  One "step" = one pass of the whole hot path over a block of 16 consecutive MD frames of
that batch:
  tacaw_build_slices (16 frames x 120 slices) -> tacaw_propagate_accumulate (128 probes x 16 frames x 120 slices, the
  annular q-ROI gathered by the last column kernel) -> tacaw_spectrum (window, time FFT, |.|^2, Bose factor, E-ROI).
Consecutive steps take consecutive frame blocks, so the default 4 timed steps cover 64 consecutive frames.
`value`  : slice-steps/s of the whole step with the inputs (atom positions of every frame) resident in HBM.
`e2e`    : the same metric through the C ABI with HOST buffers (positions copied H2D from pinned memory inside the timed
           region through tacaw_build_slices_host, the spectrum I(q,E) copied back D2H).
`roofline`: the fused slice-step kernel pair (k_row + k_col), algorithmic bytes B_step = 16 N^2 + 8 N^2/R per wave and slice
            over the CUDA-event time of the tacaw_propagate_accumulate calls inside the timed region.
`roofline_by_grid`: the same fraction measured in the same run on short samples of configs[2] (512^2) and configs[3] (1024^2),
           and on the paper's own 1680^2 grid (mixed-radix path).
`comparison`: cuFFT plan-many and torch.fft.fft2 slice loops on the same grid (library baselines, not the product).
`cpu_baseline`: the fp64 oracle, as it stands, on a bounded sample of the same workload.
`--impl reference` times the oracle alone (this tier's reference arm).
Multi-GPU (`--gpus N` under torchrun): every rank runs its own scan sub-batch of the same size (the paper's independent
computational batches) -- no data-path collective; weak scaling.
"""
from __future__ import annotations

import argparse
import json
import math
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
DEFAULTS = {1: dict(probes=None, fps=None), 2: dict(probes=None, fps=None), 3: dict(probes=None, fps=8),
            4: dict(probes=None, fps=8), 5: dict(probes=128, fps=16)}


def load_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            d = json.load(open(p))
            return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def workload_config(wl, fps, extra=None):
    c = {"workload": f"BASELINE.json configs[{int(wl.name[1]) - 1}] ({wl.name}): rutile TiO2, {wl.nx}x{wl.ny} grid, one scan "
                     f"sub-batch of {wl.nprobes} probes x {fps} consecutive frames per step x {wl.nslices_total} slices",
         "grid": [wl.nx, wl.ny], "probes": wl.nprobes, "frames_per_step": fps, "slices": wl.nslices_total,
         "atoms": wl.natoms, "roi_pixels": None, "slice_steps_per_step": wl.nprobes * fps * wl.nslices_total,
         "l2": "inputs larger than L2 (transmissions + waves of one step >> 126 MB); no flush needed"}
    if extra:
        c.update(extra)
    return c


def shard_workload(wl, rank: int):
    """Rank r works on its own scan sub-batch: the same raster shifted by 0.1 A * r (independent unit)."""
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
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
                for n, v in zip(names, r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                continue
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_median": float(np.median(pw)) if pw else None, "reasons": sorted(reasons), "samples": len(sm)}


# ------------------------------------------------------------------------------------------------- oracle legs
def oracle_plan(args, wl):
    """Bounded oracle sample of the workload, about 15 s of host work (--ref-frames overrides the frame count): at most 4
    probes, whole frames while they fit, otherwise ONE frame of a sample thinned along z (same lateral cell, grid, atoms per
    slice, probes; fewer cells along the beam -- the per-slice-step cost is the workload's).  The estimate scales a measured
    280 slice-steps/s (16 cores, 256^2) by the N^2 log N cost of a slice step and adds the potential of a slice
    (atoms x in-band pixels at ~1.2e9 terms/s on 16 cores)."""
    from paper_2607_02236_b200 import workloads as W
    cfg = int(wl.name[1])
    npr = min(wl.nprobes, 4)
    cores = max(1, min(16, len(os.sched_getaffinity(0))))
    step_s = (wl.nx * wl.ny * math.log2(wl.nx * wl.ny)) / (256.0 * 256.0 * 16.0) / (280.0 * cores / 16.0)
    atoms_per_slice = wl.natoms / wl.nslices_total
    slice_s = atoms_per_slice * (math.pi / 9.0) * wl.nx * wl.ny / (1.2e9 * cores / 16.0)
    frame_s = wl.nslices_total * (npr * step_s + slice_s)
    if args.ref_frames is not None or frame_s <= 20.0:
        nf = max(1, args.ref_frames) if args.ref_frames is not None else int(max(1, min(wl.nframes, round(15.0 / frame_s))))
        return W.make_workload(cfg, nframes=wl.nframes, nprobes=npr), nf, None
    nseg = len(wl.segments)
    cells = max(1, int(round(15.0 / (2 * nseg * (npr * step_s + slice_s)))))
    return W.make_workload(cfg, nframes=wl.nframes, nprobes=npr, ncz=cells), 1, cells


def oracle_sample(wl, nframes_sample: int):
    """Time the oracle, as it stands, on `nframes_sample` frames x all probes x all slices of `wl`."""
    import oracle
    from oracle import pipeline as OP
    oracle.build()
    t0 = time.perf_counter()
    OP.exit_waves(wl, list(range(nframes_sample)), output_space=1, pot_mode=1)
    dt = time.perf_counter() - t0
    steps = wl.nprobes * wl.nslices_total * nframes_sample
    return steps / dt, dt, oracle.num_threads()


def sample_text(wls, nf, cells, dt=None):
    thin = f" thinned to {cells} cell(s) per z-segment ({wls.nslices_total} slices; same lateral cell, grid and atoms per slice)" if cells else ""
    tail = f", {dt:.1f} s" if dt is not None else ""
    return f"{nf} frame(s) x {wls.nprobes} probes x {wls.nslices_total} slices of {wls.name}{thin} (build + propagate){tail}"


def run_reference(args, wl, fps):
    """--impl reference: the fp64 oracle on host cores, bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    wls, nf, cells = oracle_plan(args, wl)
    for _ in range(args.warmup):
        oracle_sample(wls, nf)
    vals, times = [], []
    for _ in range(args.steps):
        v, dt, cores = oracle_sample(wls, nf)
        vals.append(v); times.append(dt)
    value = float(wls.nprobes * wls.nslices_total * nf * len(times) / np.sum(times))
    sample = sample_text(wls, nf, cells) + " per step"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * float(np.mean(times)), "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "complex128", "data": "synthetic",
            "config": workload_config(wl, fps, {"sample": sample}),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


# --------------------------------------------------------------------------------------- library comparison arms
def comparison_arms(torch, dev, n, nwaves, nslices, b_step, peak):
    """SURVEY.md 8(d) protocol: the same slice step psi <- IFFT2{P FFT2{t psi}} as (a) torch.fft.fft2 / ifft2 calls and (b) one
    cuFFT plan-many C2C plan (ctypes on the libcufft torch ships) plus torch elementwise multiplies, timed in this run on
    this grid: nwaves waves sharing each transmission, nslices slices, CUDA events.  Baselines, not the product."""
    out = {}
    g = torch.Generator(device=dev).manual_seed(7)
    t = torch.polar(torch.ones((nslices, n, n), device=dev), torch.rand((nslices, n, n), device=dev, generator=g)).to(torch.complex64)
    P = torch.polar(torch.ones((n, n), device=dev), torch.rand((n, n), device=dev, generator=g)).to(torch.complex64) / (n * n)
    psi0 = torch.randn((nwaves, n, n), dtype=torch.complex64, device=dev, generator=g)

    def timed(fn, reps=3):
        fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(reps):
            fn()
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / reps
        rate = nwaves * nslices / (ms * 1e-3)
        return {"slice_steps_per_s": rate, "frac_of_hbm_roofline": rate * b_step / 1e9 / peak, "ms": ms,
                "waves": nwaves, "slices": nslices}

    psi = psi0.clone()

    def torch_loop():
        x = psi
        for s in range(nslices):
            x = torch.fft.ifft2(torch.fft.fft2(x * t[s]) * P, norm="forward")
        return x
    try:
        out["torch_fft"] = timed(torch_loop)
    except Exception as ex:  # pragma: no cover
        out["torch_fft"] = {"error": str(ex)[:200]}
    try:
        import ctypes as C
        import glob
        cands = glob.glob(os.path.join(os.path.dirname(torch.__file__), "..", "nvidia", "cufft", "lib", "libcufft.so*")) + \
            glob.glob("/usr/local/cuda/lib64/libcufft.so*")
        lib = C.CDLL(sorted(cands)[0])
        plan = C.c_int(0)
        dims = (C.c_int * 2)(n, n)
        CUFFT_C2C = 0x29
        rc = lib.cufftPlanMany(C.byref(plan), 2, dims, None, 1, 0, None, 1, 0, CUFFT_C2C, nwaves)
        if rc != 0:
            raise RuntimeError(f"cufftPlanMany failed ({rc})")
        lib.cufftSetStream(plan, C.c_void_p(torch.cuda.current_stream().cuda_stream))
        buf = psi0.clone()
        ptr = C.c_void_p(buf.data_ptr())

        def cufft_loop():
            for s in range(nslices):
                buf.mul_(t[s])
                lib.cufftExecC2C(plan, ptr, ptr, -1)
                buf.mul_(P)
                lib.cufftExecC2C(plan, ptr, ptr, 1)
        out["cufft_plan_many"] = timed(cufft_loop)
        lib.cufftDestroy(plan)
    except Exception as ex:  # pragma: no cover
        out["cufft_plan_many"] = {"error": str(ex)[:200]}
    return out


def propagate_only(torch, cfg, nframes, reps, peak):
    """roofline_by_grid: build `nframes` frames of configs[cfg-1], then time tacaw_propagate alone (all probes, all slices)."""
    from paper_2607_02236_b200 import workloads as W
    from paper_2607_02236_b200.pipeline import Runner
    wl = W.make_workload(cfg, nframes=max(8, nframes))
    r = Runner(wl, frames_per_block=nframes)
    pos_d = r.upload_positions(0, nframes)
    r.build_block(pos_d, nframes)
    r.propagate_block(nframes, 1)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(reps):
        r.propagate_block(nframes, 1)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / reps
    units = nframes * r.P * wl.nslices_total
    b = 16 * wl.nx * wl.ny + 8 * wl.nx * wl.ny / r.P
    rate = units / (ms * 1e-3)
    r.close()
    return {"workload": f"{wl.name}: {wl.nx}x{wl.ny}, {r.P} probes x {nframes} frame(s) x {wl.nslices_total} slices (tacaw_propagate only)",
            "propagate_slice_steps_per_s": rate, "bytes_per_slice_step": b, "achieved_GBps": rate * b / 1e9, "frac": rate * b / 1e9 / peak,
            "ms": ms}


def generic_grid_sample(torch, n, nwaves, nslices, reps, peak):
    """roofline_by_grid: the paper's own grid edge, 1680 = 2^4 3 5 7, which runs on the plain mixed-radix kernels
    of csrc/generic.cu: `nwaves` random unit-norm waves of one frame through `nslices` random unit-modulus transmissions."""
    from paper_2607_02236_b200 import binding as B
    tc = B.Tacaw(n, n, 93.0, 93.0, 0.0487, 9.2e-4, 1)
    g = torch.Generator(device="cuda").manual_seed(1680)
    t = torch.polar(torch.ones((nslices, n, n), device="cuda"), torch.randn((nslices, n, n), device="cuda", generator=g)).to(torch.complex64)
    w = torch.randn((nwaves, n, n), dtype=torch.complex64, device="cuda", generator=g)
    w /= torch.linalg.vector_norm(w, dim=(1, 2), keepdim=True)
    wf = np.zeros(nwaves, np.int32)
    tc.propagate(w, wf, [[t]], 1.5, 1)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(reps):
        tc.propagate(w, wf, [[t]], 1.5, 1)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / reps
    rate = nwaves * nslices / (ms * 1e-3)
    b = 16 * n * n + 8 * n * n / nwaves
    tc.close()
    return {"workload": f"{n}x{n} (the paper's grid; mixed-radix path of csrc/generic.cu, not tuned), {nwaves} waves x {nslices} random slices "
                        "(tacaw_propagate only)",
            "propagate_slice_steps_per_s": rate, "bytes_per_slice_step": b, "achieved_GBps": rate * b / 1e9, "frac": rate * b / 1e9 / peak,
            "ms": ms}


def measured_traffic(wl_name):
    """dram__bytes_read.sum + dram__bytes_write.sum of the slice-step pair per wave and slice, from the committed ncu --set full
    capture -- used only if that capture was taken at exactly the kernel sources this run was built from."""
    from paper_2607_02236_b200 import build as _build
    path = os.path.join(ROOT, "profiles", "r2_traffic.csv")
    if not os.path.exists(path):
        return None, "no ncu capture committed"
    import csv
    h = _build._source_hash()
    for row in csv.DictReader(open(path)):
        if row["workload"] == wl_name:
            if row["source_hash"] == h:
                return float(row["dram_bytes_per_slice_step"]), "ncu --set full at this source hash (profiles/r2_traffic.csv), cold cache"
            return None, "committed ncu capture is from other kernel sources (hash mismatch): not reported"
    return None, "no ncu capture for this workload"


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None, help="timed steps (default 4; 20 for configs 1-2)")
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="tacaw", choices=["tacaw", "reference"])
    ap.add_argument("--config", type=int, default=5, help="BASELINE.json config number 1..5 (default 5 = configs[4], the largest)")
    ap.add_argument("--frames", type=int, default=None, help="frames per step (default: 16 for c5, 8 for c3/c4, all for c1/c2)")
    ap.add_argument("--probes", type=int, default=None, help="probes of the scan sub-batch (default: 128 for c5, all otherwise)")
    ap.add_argument("--ref-frames", type=int, default=None, help="frames per step of the oracle sample (default: ~15 s of host work)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-extras", action="store_true", help="skip roofline_by_grid and the cuFFT / torch.fft comparison arms")
    args = ap.parse_args()
    if args.steps is None:
        args.steps = 20 if args.config <= 2 else 4

    from paper_2607_02236_b200 import workloads as W
    d = DEFAULTS[args.config]
    nprobes = args.probes if args.probes is not None else d["probes"]
    wl = W.make_workload(args.config, nprobes=nprobes)
    fps = args.frames if args.frames is not None else (d["fps"] or wl.nframes)
    fps = min(fps, wl.nframes)
    if args.impl == "reference":
        run_reference(args, wl, fps)
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
    shard_workload(wl, rank)          # every rank = its own scan sub-batch of the same size

    from paper_2607_02236_b200 import build as _build
    _build.build_lib()                # no-op when libtacaw.so matches the sources; never a fallback: it raises if nvcc fails
    from paper_2607_02236_b200.pipeline import Runner
    wl.nframes_total = wl.nframes
    nblocks = max(1, min(wl.nframes // fps, args.steps))          # distinct consecutive frame blocks the steps rotate over
    wl_step = W.make_workload(args.config, nprobes=nprobes, nframes=fps)
    shard_workload(wl_step, rank)
    dev = torch.device(f"cuda:{local_rank}")
    # inputs resident in HBM: positions of every frame block and segment (uploaded first, so that the batch plan below is
    # sized from the HBM that is really left)
    # (generated with the workload recipe on the device: the numpy path needs minutes per thousand frames of a 200 000-atom cell)
    pos_d = [W.frames_on_device(seg, 0, nblocks * fps, wl.dt_fs, dev) for seg in wl.segments]
    r = Runner(wl_step, device=local_rank)                        # frames per block from the free-HBM budget (plan_memory)
    r.alloc_buffer(fps)
    spec_h = [np.ascontiguousarray(s.species, dtype=np.int32) for s in wl.segments]
    R = r.P
    npix = wl.nx * wl.ny
    b_step = 16 * npix + 8 * npix / R
    units_per_step = R * fps * wl.nslices_total
    prop_events = []
    host_issue = [0.0, 0]      # host wall time inside the asynchronous propagate calls, launches they issued

    def one_step(blk: int, timed: bool):
        base = (blk % nblocks) * fps
        for f0 in range(0, fps, r.fpb):
            nf = min(r.fpb, fps - f0)
            r.build_block([p[base + f0: base + f0 + nf] for p in pos_d], nf)
            if timed:
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                h0, n0 = time.perf_counter(), r.tc.launches
            r.propagate_gather_block(nf, f0)          # tacaw_propagate_accumulate: the last column kernel gathers the q-ROI
            if timed:
                host_issue[0] += time.perf_counter() - h0
                host_issue[1] += r.tc.launches - n0
                e1.record()
                prop_events.append((e0, e1, nf * R * wl.nslices_total))
        return r.spectrum()

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for i in range(args.warmup):
        one_step(i, False)
    barrier()
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    l0 = r.tc.launches
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record()
    for i in range(args.steps):
        I, E = one_step(i, True)
    ev1.record()
    barrier()
    elapsed_ms = ev0.elapsed_time(ev1)
    launches = r.tc.launches - l0
    clocks = sampler.stop() if rank == 0 else None
    elapsed_ms = max_over_ranks(elapsed_ms, dist, dev)
    total_steps = units_per_step * args.steps * world
    value = total_steps / (elapsed_ms * 1e-3)
    peak_alloc = torch.cuda.max_memory_allocated(dev)

    prop_ms = sum(a.elapsed_time(b) for a, b, _ in prop_events)
    prop_units = sum(n for _, _, n in prop_events)
    peak, peak_src = load_peak()
    achieved = prop_units * b_step / (prop_ms * 1e-3) / 1e9
    traffic, traffic_note = measured_traffic(wl.name)
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": traffic,
                "traffic_note": traffic_note,
                "kernel": "fused slice-step pair k_row<N,MID> + k_col<N,MID> (one slice step of every wave of an L2 group per launch pair)",
                "bytes_per_slice_step": b_step, "frac_is": "ALGORITHMIC bytes per slice step / measured HBM copy bandwidth; the waves of a "
                "group stay in L2 between the two kernels, so DRAM traffic is below the algorithmic bytes and the binding units are the "
                "fp32 pipe and L1TEX (DESIGN.md section 9)",
                "peak_source": peak_src, "propagate_share_of_step": prop_ms / elapsed_ms,
                "propagate_slice_steps_per_s": prop_units / (prop_ms * 1e-3)}
    if host_issue[1] > 0:
        # the call returns without synchronising: below ~1000 launches per call (the depth of the driver's launch queue) this is
        # the host's issue cost per launch; beyond that the host blocks on the queue and the figure tends to the GPU time
        roofline["host_issue_us_per_launch"] = host_issue[0] * 1e6 / host_issue[1]
        roofline["gpu_us_per_launch"] = prop_ms * 1e3 / host_issue[1]
        roofline["launches_per_propagate_call"] = host_issue[1] / max(1, len(prop_events))
    if traffic is not None:
        roofline["dram_frac"] = traffic * (prop_units / (prop_ms * 1e-3)) / 1e9 / peak

    # ---- end to end through the C ABI with host buffers ------------------------------------
    e2e = None
    if not args.no_e2e:
        I_host = torch.empty(I.shape, dtype=I.dtype).pin_memory()
        # the step's inputs live in pinned host memory (numpy views of pinned tensors): the frame blocks the e2e steps use
        nrep = max(1, min(args.steps, 2 if args.config >= 3 else 3))
        ne2e = min(nblocks, nrep) * fps
        pos_pin = [p[:ne2e].cpu().pin_memory() for p in pos_d]
        pos_hp = [t.numpy() for t in pos_pin]
        h2d = sum(p[:fps].numel() * 8 for p in pos_pin) + sum(s.nbytes for s in spec_h) * ((fps + r.fpb - 1) // r.fpb)
        d2h = I_host.numel() * 4

        def e2e_step(blk: int):
            base = (blk % min(nblocks, nrep)) * fps
            for f0 in range(0, fps, r.fpb):
                nf = min(r.fpb, fps - f0)
                r.build_block_host(pos_hp, base + f0, nf)
                r.propagate_gather_block(nf, f0)
            Ie, _ = r.spectrum()
            I_host.copy_(Ie, non_blocking=True)
            torch.cuda.synchronize()

        e2e_step(0)
        barrier()
        t0 = time.perf_counter()
        for i in range(nrep):
            e2e_step(i)
        barrier()
        e_ms = (time.perf_counter() - t0) * 1e3
        e_ms = max_over_ranks(e_ms, dist, dev)
        e2e = {"value": units_per_step * nrep * world / (e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": int(h2d),
               "d2h_bytes_per_step": int(d2h), "steps": nrep}

    # Welch average over half-length chunks (nu = 2) of the resident time-ordered buffer
    welch = None
    if 16 <= fps <= 512:
        Lc = 1 << ((fps // 2).bit_length() - 1)
        r.spectrum_welch(Lc, 2)
        w0, w1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        w0.record()
        for _ in range(5):
            _, _, nch = r.spectrum_welch(Lc, 2)
        w1.record()
        torch.cuda.synchronize()
        w_ms = w0.elapsed_time(w1) / 5
        in_bytes = nch * Lc * R * int(r.roi.numel()) * 8
        welch = {"chunk_len": Lc, "chunk_overlap": 2, "nchunks": int(nch), "window": "hann", "ms": w_ms,
                 "spectra_per_s": R * int(r.roi.numel()) / (w_ms * 1e-3), "read_GBps": in_bytes / (w_ms * 1e-3) / 1e9}
    roi_pixels = int(r.roi.numel())
    fpb = r.fpb
    plan = r.plan
    r.close()
    del r, pos_d, I
    torch.cuda.empty_cache()

    by_grid, comparison = None, None
    if rank == 0 and world == 1 and not args.no_extras:
        by_grid = {}
        for cfg, nf in ((3, 2), (4, 1)):
            try:
                by_grid[f"c{cfg}"] = propagate_only(torch, cfg, nf, 3, peak)
            except Exception as ex:  # pragma: no cover
                by_grid[f"c{cfg}"] = {"error": str(ex)[:200]}
            torch.cuda.empty_cache()
        try:
            by_grid["paper_1680"] = generic_grid_sample(torch, 1680, 16, 8, 3, peak)
        except Exception as ex:  # pragma: no cover
            by_grid["paper_1680"] = {"error": str(ex)[:200]}
        torch.cuda.empty_cache()
        nw_c = {2048: 16, 1024: 64}.get(wl.nx, 128)
        comparison = comparison_arms(torch, dev, wl.nx, min(nw_c, max(R, 1)) if wl.nx >= 1024 else nw_c, 8, b_step, peak)
        comparison["note"] = ("library baselines on this grid, same byte model; each slice step = 2 batched 2D FFT calls + 2 elementwise passes "
                              "(4 HBM round trips per wave), every wave shares each transmission")

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        wls, nfs, cells = oracle_plan(args, wl)
        v, dt, cores = oracle_sample(wls, nfs)
        cpu = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample_text(wls, nfs, cells, dt),
               "note": "plain fp64 radix-2 oracle, never tuned: a reported baseline, not a comparator"}

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": elapsed_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "complex64", "data": "synthetic",
                "config": workload_config(wl, fps, {"roi_pixels": roi_pixels, "frames_per_block": fpb,
                                                    "frames_covered": f"steps rotate over {nblocks} consecutive blocks of {fps} frames "
                                                                      f"(frames 0..{nblocks * fps - 1})",
                                                    "hbm_peak_allocated_bytes": int(peak_alloc),
                                                    "memory_plan_bytes": {"buffer": plan.buffer, "spectrum": plan.spectrum, "probes": plan.probes,
                                                                          "per_frame": plan.per_frame, "total": plan.total},
                                                    "parallelism": f"replicas x{world} (independent scan sub-batches, no collective)"}),
                "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline, "roofline_by_grid": by_grid,
                "comparison": comparison, "cpu_baseline": cpu,
                "spectra_per_s": R * roi_pixels * args.steps * world / (elapsed_ms * 1e-3), "welch": welch}
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
