"""Workload driver on top of the C ABI: which frames / probes go into which call, nothing else.

One "batch" = (scan sub-batch of probes) x (the trajectory), the paper's computational batch (PAPER.md:131,
:122; Listing 1 :426-428 `scanning_batch_shape`): for every block of frames build the transmission functions,
propagate every probe of the sub-batch through them, gather the q-ROI into the time-ordered buffer; after the
last block, one spectrum call.  Block and sub-batch sizes come from a byte budget (`plan_memory`, the paper's
memory rule Eq.(B2), :501-505: the exit-wave ROI buffer plus the transmission functions dominate).
All arithmetic happens inside libtacaw's kernels; this module only marshals arrays and sizes buffers.
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import Callable, Dict, Iterator, List, Optional, Sequence, Tuple

import numpy as np

from .binding import ROI_MODES, Tacaw, make_roi, make_window, scan_batch


@dataclass
class MemoryPlan:
    """Bytes of one computational batch (Eq.(B2) of the paper restated for this data layout, complex64 / float32)."""
    nprobes: int
    frames_per_block: int
    buffer: int          # time-ordered exit-wave buffer  P * T * Q * 8   (the paper's s_x s_y k_x k_y c term; no x2: in-place FFT)
    spectrum: int        # I(q, E) of the batch           P * nE * Q * 4
    probes: int          # entrance probes                P * N^2 * 8
    per_frame: int       # transmissions + waves + positions of one in-flight frame
    workspace: int

    @property
    def total(self) -> int:
        return self.buffer + self.spectrum + self.probes + self.frames_per_block * self.per_frame + self.workspace


def n_energy_bins(wl, nframes: Optional[int] = None) -> int:
    """Bins of the ascending energy axis inside the workload's E-ROI (all of them without one)."""
    T = wl.nframes if nframes is None else nframes
    if wl.e_roi_meV is None:
        return T
    from .workloads import H_MEV_FS
    e = H_MEV_FS * (np.arange(T) - T // 2) / (T * wl.dt_fs)
    return int(np.count_nonzero((e >= wl.e_roi_meV[0] - 1e-9) & (e <= wl.e_roi_meV[1] + 1e-9)))


def plan_memory(wl, nprobes: int, nroi: int, budget_bytes: float, nframes: Optional[int] = None,
                max_frames_per_block: Optional[int] = None) -> MemoryPlan:
    """Frames per block that fill `budget_bytes` once the batch-sized allocations are paid (at least one frame)."""
    T = wl.nframes if nframes is None else nframes
    npix = wl.nx * wl.ny
    buffer = nprobes * T * nroi * 8
    spectrum = nprobes * n_energy_bins(wl, T) * nroi * 4
    probes = nprobes * npix * 8
    per_frame = 8 * npix * (wl.nslices_total + nprobes) + 24 * wl.natoms
    workspace = 64 << 20
    left = budget_bytes - (buffer + spectrum + probes + workspace)
    fpb = int(max(1, min(T, left // per_frame)))
    if max_frames_per_block is not None:
        fpb = max(1, min(fpb, int(max_frames_per_block)))
    return MemoryPlan(nprobes, fpb, buffer, spectrum, probes, per_frame, workspace)


class Runner:
    """Holds the device-resident state of one computational batch: context, probes, ROI, buffers."""

    def __init__(self, wl, device: int = 0, frames_per_block: Optional[int] = None, probes: Optional[Sequence[int]] = None,
                 budget_bytes: Optional[float] = None, fused_gather: bool = True):
        import torch
        self.torch = torch
        self.wl = wl
        self.dev = torch.device(f"cuda:{device}")
        self.tc = Tacaw(wl.nx, wl.ny, wl.lx, wl.ly, wl.lam, wl.sigma, wl.bandlimit, device)
        self.probe_ids = list(range(wl.nprobes)) if probes is None else list(probes)
        self.P = len(self.probe_ids)
        self.roi_h = make_roi(wl.nx, wl.ny, wl.lx, wl.ly, wl.lam, wl.roi_mode, [p * 1e-3 for p in wl.roi_params_mrad])
        self.roi = torch.from_numpy(self.roi_h).to(self.dev)
        self.fused_gather = fused_gather       # run_block: tacaw_propagate_accumulate instead of the unfused pair
        self.roi_inv = self.tc.make_roi_inverse(self.roi) if fused_gather else None
        self.nseg = len(wl.segments)
        self.nsl = [s.nslices for s in wl.segments]
        if budget_bytes is None:
            # what the device has free now, minus head-room for the allocator and the CUDA context
            free, _ = torch.cuda.mem_get_info(self.dev)
            budget_bytes = 0.90 * free
        self.plan = plan_memory(wl, self.P, int(self.roi.numel()), budget_bytes, max_frames_per_block=frames_per_block)
        self.fpb = self.plan.frames_per_block
        # caller-owned workspace for the largest calls of this batch (the library itself never allocates)
        self.tc.reserve(natoms=max(s.pos0.shape[0] for s in wl.segments), nframes=self.fpb, nslices=max(self.nsl),
                        nsegments=self.nseg, nwaves=self.fpb * self.P, nprobes=self.P, host_staging=1)
        self.probes = self.tc.make_probes(wl.probes_xy[self.probe_ids], wl.alpha_mrad * 1e-3)
        # one [fpb][S_k][ny][nx] tensor per z-segment (tacaw_build_slices is batched over frames);
        # trans[f][k] are views of it
        self.trans_seg = [torch.empty((self.fpb, s, wl.ny, wl.nx), dtype=torch.complex64, device=self.dev) for s in self.nsl]
        self.trans = [[self.trans_seg[k][f] for k in range(self.nseg)] for f in range(self.fpb)]
        self.waves = torch.empty((self.fpb * self.P, wl.ny, wl.nx), dtype=torch.complex64, device=self.dev)
        self.species_h = [np.ascontiguousarray(s.species, dtype=np.int32) for s in wl.segments]
        self.species_d = [torch.from_numpy(s).to(self.dev) for s in self.species_h]
        self.buf = None

    def set_probes(self, probe_ids: Sequence[int]):
        """Switch to another scan sub-batch of the same size (probes regenerated in place)."""
        assert len(probe_ids) == self.P
        self.probe_ids = list(probe_ids)
        self.tc.make_probes(self.wl.probes_xy[self.probe_ids], self.wl.alpha_mrad * 1e-3, out=self.probes)

    def alloc_buffer(self, nframes: Optional[int] = None):
        T = self.wl.nframes if nframes is None else nframes
        if self.buf is None or self.buf.shape[1] != T:
            self.buf = None
            self.buf = self.torch.empty((self.P, T, self.roi.numel()), dtype=self.torch.complex64, device=self.dev)
        self.buf.zero_()
        return self.buf

    def upload_positions(self, f0: int, f1: int):
        """Positions of frames [f0, f1) for every segment as CUDA float64 tensors [F][Na][3]."""
        return [self.torch.from_numpy(seg.frames(f0, f1, self.wl.dt_fs)).to(self.dev) for seg in self.wl.segments]

    def build_block(self, pos_d, nf: int):
        for k, seg in enumerate(self.wl.segments):
            self.tc.build_slices(pos_d[k][:nf], self.species_d[k], self.wl.a, self.wl.b, self.wl.dz, seg.nslices, 0.0,
                                 out=self.trans_seg[k][:nf])

    def build_block_host(self, pos_h, f0: int, nf: int):
        """Same from HOST position arrays [T][Na][3] (tacaw_build_slices_host, asynchronous)."""
        for k, seg in enumerate(self.wl.segments):
            self.tc.build_slices_host(pos_h[k][f0:f0 + nf], self.species_h[k], self.wl.a, self.wl.b, self.wl.dz,
                                      seg.nslices, 0.0, self.trans_seg[k][:nf], want_clamped=False)

    def propagate_block(self, nf: int, output_space: int = 1):
        nw = nf * self.P
        wave_frame = np.repeat(np.arange(nf, dtype=np.int32), self.P)
        wave_probe = np.tile(np.arange(self.P, dtype=np.int32), nf)
        self.tc.propagate(self.waves[:nw], wave_frame, self.trans[:nf], self.wl.dz, output_space, probes=self.probes,
                          wave_probe=wave_probe)
        return self.waves[:nw], wave_probe, wave_frame

    def gather_block(self, nf: int, f0: int, wave_probe, wave_frame):
        self.tc.accumulate(self.waves[: nf * self.P], wave_probe, wave_frame + f0, self.roi, self.buf)

    def propagate_gather_block(self, nf: int, f0: int):
        """tacaw_propagate_accumulate: the last column kernel writes the ROI pixels into the time-ordered buffer."""
        nw = nf * self.P
        wave_frame = np.repeat(np.arange(nf, dtype=np.int32), self.P)
        wave_probe = np.tile(np.arange(self.P, dtype=np.int32), nf)
        self.tc.propagate_accumulate(self.waves[:nw], wave_probe, wave_frame, wave_frame + f0, self.trans[:nf], self.wl.dz,
                                     self.roi_inv, int(self.roi.numel()), self.buf, probes=self.probes)

    def run_block(self, pos_d, f0: int, nf: int):
        self.build_block(pos_d, nf)
        if self.fused_gather:
            self.propagate_gather_block(nf, f0)
        else:
            _, wp, wf = self.propagate_block(nf, 1)
            self.gather_block(nf, f0, wp, wf)

    def spectrum(self, out=None):
        wl = self.wl
        emin, emax = wl.e_roi_meV if wl.e_roi_meV is not None else (-np.inf, np.inf)
        return self.tc.spectrum(self.buf, wl.dt_fs, wl.window, wl.temperature_K, emin, emax, out=out)

    def spectrum_welch(self, chunk_len: int, chunk_overlap: int = 2, window: str = "hann", param: float = 0.0,
                       skip_init: int = 0, stride: int = 1):
        """Welch average over trajectory chunks of the time-ordered buffer (Eq.(2)): (I, E, nchunks)."""
        wl = self.wl
        emin, emax = wl.e_roi_meV if wl.e_roi_meV is not None else (-np.inf, np.inf)
        w = make_window(window, chunk_len, param)
        return self.tc.spectrum_welch(self.buf, chunk_len, chunk_overlap, wl.dt_fs, w, wl.temperature_K, emin, emax,
                                      skip_init=skip_init, stride=stride)

    def run(self, nframes: Optional[int] = None, on_block: Optional[Callable[[int, int], None]] = None) -> Dict[str, object]:
        """Whole path over the workload's frames for the current probes: returns dict(I, E, roi, buf)."""
        wl = self.wl
        T = wl.nframes if nframes is None else nframes
        self.alloc_buffer(T)
        for f0 in range(0, T, self.fpb):
            nf = min(self.fpb, T - f0)
            pos_d = self.upload_positions(f0, f0 + nf)
            self.run_block(pos_d, f0, nf)
            if on_block is not None:
                on_block(f0, nf)
        I, E = self.spectrum()
        return dict(I=I, E=E, roi=self.roi_h, buf=self.buf)

    def exit_waves(self, frames: Sequence[int], output_space: int = 1):
        """Exit waves [len(frames)][P][ny][nx] for the given frame indices (sampled parity)."""
        out = []
        for f in frames:
            pos_d = self.upload_positions(f, f + 1)
            self.build_block(pos_d, 1)
            w, _, _ = self.propagate_block(1, output_space)
            out.append(w.clone())
        return self.torch.stack(out)

    def close(self):
        self.tc.close()


def scan_batches(scan_shape: Sequence[int], batch_shape: Sequence[int]) -> List[np.ndarray]:
    """Scan rows of every sub-batch (tacaw_scan_batch; Listing 1 :428)."""
    _, nb = scan_batch(scan_shape, batch_shape, 0)
    return [scan_batch(scan_shape, batch_shape, b)[0] for b in range(nb)]


def run_scan(wl, scan_shape: Sequence[int], batch_shape: Sequence[int], device: int = 0,
             budget_bytes: Optional[float] = None, nframes: Optional[int] = None,
             batches: Optional[Sequence[int]] = None) -> Iterator[Tuple[int, np.ndarray, object, np.ndarray, "Runner"]]:
    """The paper's batch loop over a scan: every scan sub-batch makes its own pass over the trajectory
    (transmissions are rebuilt per pass) and yields (batch index, scan rows, I [P_b][nE][Q] on the device, E, runner).
    Sub-batches of equal size reuse one Runner (buffers sized once from the byte budget); ragged edge batches get
    their own.  The caller consumes I (copy out, or reduce with tacaw_detect) before the next batch overwrites it."""
    tiles = scan_batches(scan_shape, batch_shape)
    which = range(len(tiles)) if batches is None else batches
    runner = None
    try:
        for b in which:
            ids = tiles[b]
            if runner is None or runner.P != len(ids):
                if runner is not None:
                    runner.close()
                    runner = None
                runner = Runner(wl, device=device, probes=ids, budget_bytes=budget_bytes)
            else:
                runner.set_probes(ids)
            out = runner.run(nframes)
            yield b, ids, out["I"], out["E"], runner
    finally:
        if runner is not None:
            runner.close()


def run_reassembled(wl, offsets: np.ndarray, chunk_len: int, device: int = 0, probes: Optional[Sequence[int]] = None):
    """Segment re-assembly per averaging chunk: every z-segment of the stack follows ONE trajectory (segment 0 of
    the workload); for chunk i, stack position k shows that trajectory from snapshot offsets[i][k] on (offsets drawn by the
    seeded input generator), so chunk frame f is built from trajectory frames offsets[i][k] + f.  Only the pointer table of
    tacaw_propagate changes: d_trans[f*nsegments + k] points at the transmissions of snapshot offsets[i][k] + f.
    Returns the time-ordered buffers [nchunks][P][chunk_len][Q] on the device."""
    import torch
    r = Runner(wl, device=device, frames_per_block=1, probes=probes)
    seg = wl.segments[0]
    nch, nstack = offsets.shape
    Q = int(r.roi.numel())
    out = torch.zeros((nch, r.P, chunk_len, Q), dtype=torch.complex64, device=r.dev)
    # transmissions of every snapshot any (chunk, frame, position) needs, built once
    need = sorted({int(offsets[i, k]) + f for i in range(nch) for k in range(nstack) for f in range(chunk_len)})
    slot = {t: j for j, t in enumerate(need)}
    pos = torch.from_numpy(np.concatenate([seg.frames(t, t + 1, wl.dt_fs) for t in need])).to(r.dev)
    trans = torch.empty((len(need), seg.nslices, wl.ny, wl.nx), dtype=torch.complex64, device=r.dev)
    for j0 in range(0, len(need), 16):
        j1 = min(len(need), j0 + 16)
        r.tc.build_slices(pos[j0:j1], r.species_d[0], wl.a, wl.b, wl.dz, seg.nslices, 0.0, out=trans[j0:j1])
    wp = np.arange(r.P, dtype=np.int32)
    for i in range(nch):
        waves = torch.empty((chunk_len * r.P, wl.ny, wl.nx), dtype=torch.complex64, device=r.dev)
        table = [[trans[slot[int(offsets[i, k]) + f]] for k in range(nstack)] for f in range(chunk_len)]
        wave_frame = np.repeat(np.arange(chunk_len, dtype=np.int32), r.P)
        wave_probe = np.tile(wp, chunk_len)
        r.tc.propagate(waves, wave_frame, table, wl.dz, 1, probes=r.probes, wave_probe=wave_probe)
        r.tc.accumulate(waves, wave_probe, wave_frame, r.roi, out[i])
    r.close()
    return out
