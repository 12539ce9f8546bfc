"""Oracle-side driver: run a Workload through O1-O10 frame by frame.  TEST INFRASTRUCTURE.

Follows PAPER.md:122 ("In each batch the Calculator performs the multislice calculation on each
snapshot ... collects the time-consecutive exit wave functions from the defined ROI ... FFT from
the time to the energy domain ... squared modulus ... quantum statistics correction factor").
Imports only numpy, the oracle C front end and the workload *input* generators.
"""
from __future__ import annotations

from typing import Dict, Optional, Sequence

import numpy as np

from . import (accumulate, build_slices, make_probes, make_roi, propagate, spectrum)


def roi_for(wl) -> np.ndarray:
    params = [p * 1e-3 for p in wl.roi_params_mrad]
    return make_roi(wl.nx, wl.ny, wl.lx, wl.ly, wl.lam, wl.roi_mode, params)


def frame_transmissions(wl, f: int, pot_mode: int = 1):
    """Transmission functions of frame f for every z-segment: list of c128 [S_k][ny][nx]."""
    out = []
    for seg in wl.segments:
        pos = seg.frames(f, f + 1, wl.dt_fs)[0]
        r = build_slices(wl.nx, wl.ny, wl.lx, wl.ly, pos, seg.species, wl.a, wl.b, wl.dz, seg.nslices, 0.0,
                         wl.sigma, bandlimit=wl.bandlimit, pot_mode=pot_mode)
        out.append(r["trans"])
    return out


def exit_waves(wl, frames: Sequence[int], probes: Optional[Sequence[int]] = None, output_space: int = 1,
               pot_mode: int = 1) -> np.ndarray:
    """[len(frames)][len(probes)][ny][nx] c128 exit waves (q-space unnormalised by default)."""
    pr = list(range(wl.nprobes)) if probes is None else list(probes)
    psi0 = make_probes(wl.nx, wl.ny, wl.lx, wl.ly, wl.lam, wl.probes_xy[pr], wl.alpha_mrad * 1e-3)
    out = np.empty((len(frames), len(pr), wl.ny, wl.nx), dtype=np.complex128)
    for i, f in enumerate(frames):
        tr = frame_transmissions(wl, f, pot_mode)
        out[i] = propagate(wl.lx, wl.ly, wl.lam, wl.bandlimit, psi0, None, [tr], wl.dz, output_space)
    return out


def run(wl, probes: Optional[Sequence[int]] = None, pot_mode: int = 1) -> Dict[str, np.ndarray]:
    """Whole path for the workload's nframes: returns dict(I [P][nE][Q], E, roi, buf)."""
    pr = list(range(wl.nprobes)) if probes is None else list(probes)
    roi = roi_for(wl)
    buf = np.zeros((len(pr), wl.nframes, roi.size), dtype=np.complex128)
    psi0 = make_probes(wl.nx, wl.ny, wl.lx, wl.ly, wl.lam, wl.probes_xy[pr], wl.alpha_mrad * 1e-3)
    for f in range(wl.nframes):
        tr = frame_transmissions(wl, f, pot_mode)
        q = propagate(wl.lx, wl.ly, wl.lam, wl.bandlimit, psi0, None, [tr], wl.dz, 1)
        accumulate(q, np.arange(len(pr)), np.full(len(pr), f), roi, buf)
    emin, emax = wl.e_roi_meV if wl.e_roi_meV is not None else (-np.inf, np.inf)
    I, E = spectrum(buf, wl.dt_fs, wl.window, wl.temperature_K, emin, emax)
    return dict(I=I, E=E, roi=roi, buf=buf)


def run_reassembled(wl, offsets: np.ndarray, chunk_len: int, probes: Optional[Sequence[int]] = None,
                    pot_mode: int = 1) -> np.ndarray:
    """'one may perform a single longer MD trajectory and, for each averaging chunk in the TACAW
    calculation, construct the stacked supercell from randomly selected segments of that trajectory.'
    The workload's z-segments all follow segment 0's trajectory; for chunk i, stack position k shows that trajectory from
    snapshot offsets[i][k] on, so chunk frame f is built from trajectory frames offsets[i][k] + f (the offsets are drawn
    by the seeded input generator, never here).  Returns the time-ordered buffers [nchunks][P][chunk_len][Q] (c128)."""
    pr = list(range(wl.nprobes)) if probes is None else list(probes)
    roi = roi_for(wl)
    nch, nstack = offsets.shape
    seg = wl.segments[0]
    psi0 = make_probes(wl.nx, wl.ny, wl.lx, wl.ly, wl.lam, wl.probes_xy[pr], wl.alpha_mrad * 1e-3)
    out = np.zeros((nch, len(pr), chunk_len, roi.size), dtype=np.complex128)
    for i in range(nch):
        for f in range(chunk_len):
            tr = []
            for k in range(nstack):
                t = int(offsets[i, k]) + f
                pos = seg.frames(t, t + 1, wl.dt_fs)[0]
                tr.append(build_slices(wl.nx, wl.ny, wl.lx, wl.ly, pos, seg.species, wl.a, wl.b, wl.dz, seg.nslices, 0.0,
                                       wl.sigma, bandlimit=wl.bandlimit, pot_mode=pot_mode)["trans"])
            q = propagate(wl.lx, wl.ly, wl.lam, wl.bandlimit, psi0, None, [tr], wl.dz, 1)
            accumulate(q, np.arange(len(pr)), np.full(len(pr), f), roi, out[i])
    return out
