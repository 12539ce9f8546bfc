"""Seeded synthetic TACAW workloads (inputs only; none of the method's arithmetic lives here).

The paper's inputs are ORB-MLIP molecular-dynamics trajectories of rutile TiO2 (PAPER.md:58-84,
:162, :225, :245) which are not available; these generators stand in for them with the shapes
`BASELINE.json:configs` names.  Both the fp64 oracle (`oracle/`) and the CUDA library consume the
arrays produced here, so no random number is ever drawn inside either implementation.

Everything is numpy/fp64.  What is produced: atom positions per frame [F][Na][3] (Angstrom),
species ids [Na], the two-species 4-Gaussian scattering-factor table, probe positions, the beam
constants (lambda, sigma) and the plain numbers of each config (grid, slices, dt, T, ROI radii).

Readings of under-specified points are restated in DESIGN.md.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Sequence, Tuple

import numpy as np

# ---------------------------------------------------------------------------------------------
# physical constants (CODATA 2018) -- input-side only: lambda and sigma are *inputs* to both
# libraries, computed once here.
H_JS = 6.62607015e-34
C_MS = 299792458.0
E_C = 1.602176634e-19
M0_KG = 9.1093837015e-31
KB_EV_K = 8.617333262e-5
H_MEV_FS = 4135.667696
AMU_KG = 1.66053906660e-27

SEED_BASE = 26070223600

RUTILE_A = 4.594
RUTILE_C = 2.959
RUTILE_U = 0.305
MASS_U = (47.867, 15.999)  # Ti, O


def electron_wavelength_A(kv: float) -> float:
    """Relativistic de Broglie wavelength in Angstrom for an accelerating voltage in kV."""
    eu = E_C * kv * 1e3
    lam_m = H_JS * C_MS / np.sqrt(eu * (2.0 * M0_KG * C_MS ** 2 + eu))
    return float(lam_m * 1e10)


def interaction_sigma(kv: float) -> float:
    """Interaction constant sigma in rad/(V*Angstrom)."""
    eu = E_C * kv * 1e3
    m0c2 = M0_KG * C_MS ** 2
    lam = electron_wavelength_A(kv)
    u_volt = kv * 1e3
    return float(2.0 * np.pi / (lam * u_volt) * (m0c2 + eu) / (2.0 * m0c2 + eu))


def species_table(seed: int) -> Tuple[np.ndarray, np.ndarray]:
    """Two species (0 = Ti, 1 = O) x 4 Gaussians.  a in V*A^3 (= 100 * U(0.1, 2), reading G5),
    b in A^2 (U(0.1, 10), crystallographic q, reading G6)."""
    rng = np.random.default_rng(seed)
    a = 100.0 * rng.uniform(0.1, 2.0, size=(2, 4))
    b = rng.uniform(0.1, 10.0, size=(2, 4))
    return a, b


def rutile_supercell(ncx: int, ncy: int, ncz: int, a: float = RUTILE_A, c: float = RUTILE_C,
                     u: float = RUTILE_U) -> Tuple[np.ndarray, np.ndarray]:
    """Equilibrium positions [Na][3] (A) and species [Na] of an ncx x ncy x ncz rutile block.

    Basis (reading G20): Ti (0,0,0), (1/2,1/2,1/2); O +-(u,u,0), (1/2+-u, 1/2-+u, 1/2); every z is
    then offset by c/4 so the atomic planes sit at c/4 and 3c/4 of each cell."""
    basis = np.array([
        [0.0, 0.0, 0.0],
        [0.5, 0.5, 0.5],
        [u, u, 0.0],
        [1.0 - u, 1.0 - u, 0.0],
        [0.5 + u, 0.5 - u, 0.5],
        [0.5 - u, 0.5 + u, 0.5],
    ])
    spec = np.array([0, 0, 1, 1, 1, 1], dtype=np.int32)
    iz, iy, ix = np.meshgrid(np.arange(ncz), np.arange(ncy), np.arange(ncx), indexing="ij")
    cells = np.stack([ix.ravel(), iy.ravel(), iz.ravel()], axis=1).astype(np.float64)
    frac = cells[:, None, :] + basis[None, :, :]
    pos = frac.reshape(-1, 3) * np.array([a, a, c])
    pos[:, 2] += 0.25 * c
    species = np.tile(spec, cells.shape[0]).astype(np.int32)
    return pos, species


# ---------------------------------------------------------------------------------------------
@dataclass
class ModeSet:
    """A set of M plane-wave harmonic modes (reading G15)."""
    kappa: np.ndarray      # [M][3] 1/A
    evec: np.ndarray       # [M][3] unit vectors
    energy_meV: np.ndarray  # [M]
    phase: np.ndarray      # [M]
    amp: np.ndarray        # [M][nspecies] A


@dataclass
class Segment:
    """One z-segment of the sample: its own periodic cell and its own trajectory."""
    pos0: np.ndarray       # [Na][3] equilibrium positions, z relative to the segment
    species: np.ndarray    # [Na] int32
    lz: float
    nslices: int
    kind: str              # "einstein" or "modes"
    modes: ModeSet | None = None
    einstein_energy_meV: np.ndarray | None = None   # [3]
    einstein_phase: np.ndarray | None = None        # [Na][3 modes][3 cart]
    einstein_amp: float = 0.0

    def frames(self, f0: int, f1: int, dt_fs: float) -> np.ndarray:
        """Positions [f1-f0][Na][3] at t_f = f*dt, f in [f0, f1)."""
        t = np.arange(f0, f1, dtype=np.float64) * dt_fs
        out = np.repeat(self.pos0[None, :, :], len(t), axis=0)
        if self.kind == "static":
            return out
        if self.kind == "einstein":
            for m in range(len(self.einstein_energy_meV)):
                w = 2.0 * np.pi * self.einstein_energy_meV[m] / H_MEV_FS  # rad/fs
                out += self.einstein_amp * np.cos(w * t[:, None, None] + self.einstein_phase[None, :, m, :])
            return out
        ms = self.modes
        for m in range(len(ms.energy_meV)):
            w = 2.0 * np.pi * ms.energy_meV[m] / H_MEV_FS
            arg = 2.0 * np.pi * (self.pos0 @ ms.kappa[m])[None, :] - w * t[:, None] + ms.phase[m]
            amp = ms.amp[m][self.species]                       # [Na]
            out += (amp[None, :] * np.cos(arg))[:, :, None] * ms.evec[m][None, None, :]
        return out


def frames_on_device(seg: "Segment", f0: int, f1: int, dt_fs: float, device, chunk: int = 32):
    """The same positions as Segment.frames, evaluated with torch float64 on `device` in chunks of frames (same formula; the
    last bit of a cosine may differ from numpy's).  For benchmarks that keep thousands of frames of a 200 000-atom cell resident:
    the numpy path needs minutes of host time per thousand frames there.  Parity tests use Segment.frames for both sides."""
    import torch
    t_all = torch.arange(f0, f1, dtype=torch.float64, device=device) * dt_fs
    pos0 = torch.from_numpy(seg.pos0).to(device)
    out = pos0.unsqueeze(0).repeat(f1 - f0, 1, 1)
    if seg.kind == "static":
        return out
    for c0 in range(0, f1 - f0, chunk):
        t = t_all[c0:c0 + chunk]
        o = out[c0:c0 + chunk]
        if seg.kind == "einstein":
            ph = torch.from_numpy(seg.einstein_phase).to(device)
            for m in range(len(seg.einstein_energy_meV)):
                w = 2.0 * np.pi * float(seg.einstein_energy_meV[m]) / H_MEV_FS
                o += seg.einstein_amp * torch.cos(w * t[:, None, None] + ph[None, :, m, :])
            continue
        ms = seg.modes
        species = torch.from_numpy(seg.species.astype(np.int64)).to(device)
        for m in range(len(ms.energy_meV)):
            w = 2.0 * np.pi * float(ms.energy_meV[m]) / H_MEV_FS
            kap = torch.from_numpy(ms.kappa[m]).to(device)
            arg = 2.0 * np.pi * (pos0 @ kap)[None, :] - w * t[:, None] + float(ms.phase[m])
            amp = torch.from_numpy(ms.amp[m]).to(device)[species]
            o += (amp[None, :] * torch.cos(arg))[:, :, None] * torch.from_numpy(ms.evec[m]).to(device)[None, None, :]
    return out


@dataclass
class Workload:
    name: str
    nx: int
    ny: int
    lx: float
    ly: float
    kv: float
    lam: float
    sigma: float
    alpha_mrad: float            # 0 -> plane wave
    probes_xy: np.ndarray        # [P][2] A
    nframes: int
    dt_fs: float
    temperature_K: float
    dz: float
    segments: List[Segment]
    roi_mode: str                # "full" | "disc" | "annulus"
    roi_params_mrad: Tuple[float, ...]
    a: np.ndarray
    b: np.ndarray
    window: int = 1              # 1 Hann, 0 rect
    e_roi_meV: Tuple[float, float] | None = None
    bandlimit: int = 1
    notes: str = ""
    extra: dict = field(default_factory=dict)

    @property
    def nprobes(self) -> int:
        return int(self.probes_xy.shape[0])

    @property
    def nslices_total(self) -> int:
        return int(sum(s.nslices for s in self.segments))

    @property
    def natoms(self) -> int:
        return int(sum(s.pos0.shape[0] for s in self.segments))

    @property
    def slice_steps(self) -> int:
        return self.nprobes * self.nframes * self.nslices_total


def _mode_set(rng: np.random.Generator, nmodes: int, e_lo: float, e_hi: float, lx: float, ly: float,
              lz: float, amp_kind: str, temperature_K: float, rms_A: float = 0.07,
              on_bins: Tuple[int, float] | None = None) -> ModeSet:
    ijl = np.stack([rng.integers(-4, 5, size=nmodes), rng.integers(-4, 5, size=nmodes),
                    rng.integers(-8, 9, size=nmodes)], axis=1).astype(np.float64)
    kappa = ijl / np.array([lx, ly, lz])
    v = rng.normal(size=(nmodes, 3))
    evec = v / np.linalg.norm(v, axis=1, keepdims=True)
    lo = max(e_lo, 5.0)
    energy = lo + (e_hi - lo) * (1.0 - rng.uniform(0.0, 1.0, size=nmodes))   # (lo, e_hi]
    if on_bins is not None:   # snap mode energies onto exact FFT bins (test workloads only)
        nfr, dt = on_bins
        de = H_MEV_FS / (nfr * dt)
        energy = np.maximum(1, np.round(energy / de)) * de
    phase = rng.uniform(0.0, 2.0 * np.pi, size=nmodes)
    if amp_kind == "gaussian":
        g = rng.normal(size=nmodes)
        amp = (rms_A * np.sqrt(2.0 / nmodes) * g)[:, None] * np.ones((1, 2))
    else:  # "thermal": A = sqrt(2 kB T / (M_s w^2 M))
        w = 2.0 * np.pi * energy / H_MEV_FS * 1e15          # rad/s
        kbt = KB_EV_K * temperature_K * E_C                 # J
        amp = np.empty((nmodes, 2))
        for s in range(2):
            amp[:, s] = np.sqrt(2.0 * kbt / (MASS_U[s] * AMU_KG * w ** 2 * nmodes)) * 1e10
    return ModeSet(kappa=kappa, evec=evec, energy_meV=energy, phase=phase, amp=amp)


def _raster(x0: float, y0: float, wx: float, wy: float, npx: int, npy: int) -> np.ndarray:
    """Raster with the end point excluded, x fastest."""
    xs = x0 + wx * np.arange(npx) / npx
    ys = y0 + wy * np.arange(npy) / npy
    yy, xx = np.meshgrid(ys, xs, indexing="ij")
    return np.stack([xx.ravel(), yy.ravel()], axis=1)


def make_workload(cfg: int, *, nframes: int | None = None, nprobes: int | None = None,
                  ncz: int | None = None) -> Workload:
    """configs[cfg-1] of BASELINE.json (cfg = 1..5).  `nframes` / `nprobes` only *truncate* the
    workload (first frames / first probes) for sampled parity and bounded benchmarks; `ncz`
    (cells along z, per segment) makes a thinner sample of the same lateral size and grid for
    parity cases the fp64 oracle can finish."""
    a0, c0 = RUTILE_A, RUTILE_C
    dz = 0.5 * c0
    kv = 100.0
    lam, sig = electron_wavelength_A(kv), interaction_sigma(kv)
    sa, sb = species_table(SEED_BASE + 7)
    temp = 300.0
    if cfg == 1:
        ncx, ncy, ncz, n, T, dt = 3, 3, 4, 64, 32, 5.0
        pos0, spec = rutile_supercell(ncx, ncy, ncz)
        rng = np.random.default_rng(SEED_BASE + 100 * cfg)
        seg = Segment(pos0=pos0, species=spec, lz=ncz * c0, nslices=2 * ncz, kind="einstein",
                      einstein_energy_meV=np.array([20.0, 45.0, 80.0]),
                      einstein_phase=rng.uniform(0, 2 * np.pi, size=(pos0.shape[0], 3, 3)),
                      einstein_amp=0.05)
        wl = Workload("c1", n, n, ncx * a0, ncy * a0, kv, lam, sig, 0.0, np.zeros((1, 2)), T, dt, temp, dz,
                      [seg], "full", (), sa, sb,
                      notes="216 atoms (6 per rutile cell; configs[0] prints 108, reading G14)")
    elif cfg == 2:
        ncx, ncy, ncz, n, T, dt = 8, 8, 20, 256, 256, 5.0
        pos0, spec = rutile_supercell(ncx, ncy, ncz)
        rng = np.random.default_rng(SEED_BASE + 100 * cfg)
        ms = _mode_set(rng, 12, 5.0, 100.0, ncx * a0, ncy * a0, ncz * c0, "gaussian", temp)
        seg = Segment(pos0, spec, ncz * c0, 2 * ncz, "modes", modes=ms)
        u = RUTILE_U
        probes = (np.array([[4.0, 4.0], [4.0 + u, 4.0 + u], [4.5, 4.0], [4.25, 4.0]]) * a0)
        wl = Workload("c2", n, n, ncx * a0, ncy * a0, kv, lam, sig, 30.0, probes, T, dt, temp, dz,
                      [seg], "disc", (60.0,), sa, sb)
    elif cfg == 3:
        ncx, ncy, ncz, n, T, dt = 10, 10, (ncz or 100), 512, 1024, 5.0
        pos0, spec = rutile_supercell(ncx, ncy, ncz)
        rng = np.random.default_rng(SEED_BASE + 100 * cfg)
        ms = _mode_set(rng, 64, 0.0, 110.0, ncx * a0, ncy * a0, ncz * c0, "thermal", temp)
        seg = Segment(pos0, spec, ncz * c0, 2 * ncz, "modes", modes=ms)
        probes = _raster(5 * a0, 5 * a0, a0, a0, 16, 16)
        wl = Workload("c3", n, n, ncx * a0, ncy * a0, kv, lam, sig, 30.0, probes, T, dt, temp, dz,
                      [seg], "disc", (40.0,), sa, sb)
    elif cfg == 4:
        ncx, ncy, ncz_seg, nseg, n, T, dt = 12, 12, (ncz or 85), 4, 1024, 1024, 5.0
        segs = []
        for k in range(nseg):
            pos0, spec = rutile_supercell(ncx, ncy, ncz_seg)
            rng = np.random.default_rng(SEED_BASE + 100 * cfg + k)
            ms = _mode_set(rng, 64, 0.0, 110.0, ncx * a0, ncy * a0, ncz_seg * c0, "thermal", temp)
            segs.append(Segment(pos0, spec, ncz_seg * c0, 2 * ncz_seg, "modes", modes=ms))
        probes = _raster(6 * a0, 6 * a0, a0, a0, 8, 8)
        wl = Workload("c4", n, n, ncx * a0, ncy * a0, kv, lam, sig, 30.0, probes, T, dt, temp, dz,
                      segs, "disc", (50.0,), sa, sb)
    elif cfg == 5:
        ncx, ncy, ncz, n, T, dt = 24, 24, (ncz or 60), 2048, 2048, 4.0
        pos0, spec = rutile_supercell(ncx, ncy, ncz)
        lx = ncx * a0
        shift = pos0[:, 0] >= 0.5 * lx           # planar fault across (100), reading G16
        pos0[shift, 1] = np.mod(pos0[shift, 1] + 0.5, ncy * a0)
        rng = np.random.default_rng(SEED_BASE + 100 * cfg)
        ms = _mode_set(rng, 128, 0.0, 120.0, lx, ncy * a0, ncz * c0, "thermal", temp)
        seg = Segment(pos0, spec, ncz * c0, 2 * ncz, "modes", modes=ms)
        probes = _raster(0.5 * lx - a0, 12 * a0 - a0, 2 * a0, 2 * a0, 32, 32)
        wl = Workload("c5", n, n, lx, ncy * a0, kv, lam, sig, 30.0, probes, T, dt, temp, dz,
                      [seg], "annulus", (30.0, 55.0), sa, sb, e_roi_meV=(-120.0, 120.0),
                      notes="annulus 30-55 mrad (reading G12); probe batches of 128 (R4)")
    else:
        raise ValueError(f"config {cfg} not in 1..5")
    if nframes is not None:
        wl.nframes = int(nframes)
    if nprobes is not None:
        wl.probes_xy = wl.probes_xy[: int(nprobes)].copy()
    return wl


def tiny_workload(n: int = 16, ncell: Tuple[int, int, int] = (1, 1, 2), nframes: int = 8,
                  dt_fs: float = 5.0, seed: int = 1, alpha_mrad: float = 0.0,
                  mode_bins: Sequence[int] | None = None, amp_A: float = 0.05) -> Workload:
    """Small test workload; with `mode_bins` the Einstein energies sit exactly on FFT bins."""
    a0, c0 = RUTILE_A, RUTILE_C
    kv = 100.0
    pos0, spec = rutile_supercell(*ncell)
    rng = np.random.default_rng(seed)
    if mode_bins is None:
        energies = np.array([20.0, 45.0, 80.0])
    else:
        energies = np.asarray(mode_bins, dtype=np.float64) * H_MEV_FS / (nframes * dt_fs)
    seg = Segment(pos0, spec, ncell[2] * c0, 2 * ncell[2], "einstein",
                  einstein_energy_meV=energies,
                  einstein_phase=rng.uniform(0, 2 * np.pi, size=(pos0.shape[0], len(energies), 3)),
                  einstein_amp=amp_A)
    sa, sb = species_table(SEED_BASE + 7)
    probes = np.array([[0.37 * ncell[0] * a0, 0.61 * ncell[1] * a0]])
    return Workload("tiny", n, n, ncell[0] * a0, ncell[1] * a0, kv, electron_wavelength_A(kv),
                    interaction_sigma(kv), alpha_mrad, probes, nframes, dt_fs, 300.0, 0.5 * c0, [seg],
                    "full", (), sa, sb)


def segment_offsets(seed: int, nchunks: int, nstack: int, ntraj: int, chunk_len: int) -> np.ndarray:
    """Random start snapshots for re-assembling a stack from one trajectory: offsets[i][k] uniform in
    [0, ntraj - chunk_len], one per (averaging chunk, stack position).  Input generator only: both implementations take the
    table as an input."""
    rng = np.random.default_rng(seed)
    return rng.integers(0, ntraj - chunk_len + 1, size=(nchunks, nstack)).astype(np.int64)
