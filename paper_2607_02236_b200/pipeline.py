"""Workload driver on top of the C ABI: which frames / probes go into which call, nothing else.

One "batch" = (probe set) x (block of frames), the paper's computational batch (PAPER.md:131,
:122): build the transmission functions of each frame in the block, propagate every probe through
them, gather the q-ROI into the time-ordered buffer; after the last block, one spectrum call.
All arithmetic happens inside libtacaw's kernels; this module only marshals arrays.
"""
from __future__ import annotations

from typing import Dict, List, Optional, Sequence

import numpy as np

from .binding import ROI_MODES, Tacaw, make_roi, make_window


class Runner:
    """Holds the device-resident state of one workload: context, probes, ROI, buffers."""

    def __init__(self, wl, device: int = 0, frames_per_block: Optional[int] = None, probes: Optional[Sequence[int]] = None):
        import torch
        self.torch = torch
        self.wl = wl
        self.dev = torch.device(f"cuda:{device}")
        self.tc = Tacaw(wl.nx, wl.ny, wl.lx, wl.ly, wl.lam, wl.sigma, wl.bandlimit, device)
        self.probe_ids = list(range(wl.nprobes)) if probes is None else list(probes)
        self.P = len(self.probe_ids)
        self.roi_h = make_roi(wl.nx, wl.ny, wl.lx, wl.ly, wl.lam, wl.roi_mode, [p * 1e-3 for p in wl.roi_params_mrad])
        self.roi = torch.from_numpy(self.roi_h).to(self.dev)
        self.probes = self.tc.make_probes(wl.probes_xy[self.probe_ids], wl.alpha_mrad * 1e-3)
        self.nseg = len(wl.segments)
        self.nsl = [s.nslices for s in wl.segments]
        npix = wl.nx * wl.ny
        if frames_per_block is None:
            # transmissions of a block + its waves within ~8 GB, at least one frame
            per_frame = 8 * npix * (sum(self.nsl) + self.P)
            frames_per_block = max(1, min(wl.nframes, int(8e9 // per_frame)))
        self.fpb = int(frames_per_block)
        # one [fpb][S_k][ny][nx] tensor per z-segment (tacaw_build_slices is batched over frames);
        # trans[f][k] are views of it
        self.trans_seg = [torch.empty((self.fpb, s, wl.ny, wl.nx), dtype=torch.complex64, device=self.dev) for s in self.nsl]
        self.trans = [[self.trans_seg[k][f] for k in range(self.nseg)] for f in range(self.fpb)]
        self.waves = torch.empty((self.fpb * self.P, wl.ny, wl.nx), dtype=torch.complex64, device=self.dev)
        self.species_h = [np.ascontiguousarray(s.species, dtype=np.int32) for s in wl.segments]
        self.species_d = [torch.from_numpy(s).to(self.dev) for s in self.species_h]
        self.buf = None

    def alloc_buffer(self, nframes: Optional[int] = None):
        T = self.wl.nframes if nframes is None else nframes
        self.buf = self.torch.zeros((self.P, T, self.roi.numel()), dtype=self.torch.complex64, device=self.dev)
        return self.buf

    def upload_positions(self, f0: int, f1: int):
        """Positions of frames [f0, f1) for every segment as CUDA float64 tensors [F][Na][3]."""
        return [self.torch.from_numpy(seg.frames(f0, f1, self.wl.dt_fs)).to(self.dev) for seg in self.wl.segments]

    def build_block(self, pos_d, nf: int):
        for k, seg in enumerate(self.wl.segments):
            self.tc.build_slices(pos_d[k][:nf], self.species_d[k], self.wl.a, self.wl.b, self.wl.dz, seg.nslices, 0.0,
                                 out=self.trans_seg[k][:nf])

    def build_block_host(self, pos_h, f0: int, nf: int):
        """Same from HOST position arrays [T][Na][3] (tacaw_build_slices_host)."""
        for k, seg in enumerate(self.wl.segments):
            self.tc.build_slices_host(pos_h[k][f0:f0 + nf], self.species_h[k], self.wl.a, self.wl.b, self.wl.dz,
                                      seg.nslices, 0.0, self.trans_seg[k][:nf])

    def propagate_block(self, nf: int, output_space: int = 1):
        nw = nf * self.P
        wave_frame = np.repeat(np.arange(nf, dtype=np.int32), self.P)
        wave_probe = np.tile(np.arange(self.P, dtype=np.int32), nf)
        self.tc.propagate(self.waves[:nw], wave_frame, self.trans[:nf], self.wl.dz, output_space, probes=self.probes,
                          wave_probe=wave_probe)
        return self.waves[:nw], wave_probe, wave_frame

    def gather_block(self, nf: int, f0: int, wave_probe, wave_frame):
        self.tc.accumulate(self.waves[: nf * self.P], wave_probe, wave_frame + f0, self.roi, self.buf)

    def run_block(self, pos_d, f0: int, nf: int):
        self.build_block(pos_d, nf)
        _, wp, wf = self.propagate_block(nf, 1)
        self.gather_block(nf, f0, wp, wf)

    def spectrum(self):
        wl = self.wl
        emin, emax = wl.e_roi_meV if wl.e_roi_meV is not None else (-np.inf, np.inf)
        return self.tc.spectrum(self.buf, wl.dt_fs, wl.window, wl.temperature_K, emin, emax)

    def spectrum_welch(self, chunk_len: int, chunk_overlap: int = 2, window: str = "hann", param: float = 0.0):
        """Welch average over trajectory chunks of the time-ordered buffer (Eq.(2)): (I, E, nchunks)."""
        wl = self.wl
        emin, emax = wl.e_roi_meV if wl.e_roi_meV is not None else (-np.inf, np.inf)
        w = make_window(window, chunk_len, param)
        return self.tc.spectrum_welch(self.buf, chunk_len, chunk_overlap, wl.dt_fs, w, wl.temperature_K, emin, emax)

    def run(self) -> Dict[str, object]:
        """Whole path over the workload's frames: returns dict(I, E, roi, buf)."""
        wl = self.wl
        self.alloc_buffer()
        for f0 in range(0, wl.nframes, self.fpb):
            nf = min(self.fpb, wl.nframes - f0)
            pos_d = self.upload_positions(f0, f0 + nf)
            self.run_block(pos_d, f0, nf)
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
