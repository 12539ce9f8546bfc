"""ctypes front end of the fp64 CPU oracle (oracle/tacaw_oracle.c).  TEST INFRASTRUCTURE, NOT PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package.  It never imports paper_2607_02236_b200's CUDA binding and shares no code with it.
Functions up to `spectrum` are marshalling shims around the C routine of the same name; the arithmetic and
the paper citations live in the C file's header.  The Welch / window additions at the end are
plain numpy on top of oracle_spectrum_table, each citing the passage it follows.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import List, Optional, Sequence, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "tacaw_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile liboracle.so with gcc (OpenMP over independent slices / waves / series)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-std=c11", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(_LIB)
        _lib.oracle_bose.restype = C.c_double
        _lib.oracle_bose.argtypes = [C.c_double]
    return _lib


def _p(a: np.ndarray):
    return a.ctypes.data_as(C.c_void_p)


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def set_num_threads(n: int) -> None:
    lib().oracle_set_num_threads(C.c_int(n))


def set_fft_mode(mode: int) -> None:
    """0 auto (naive DFT for n<=64, radix-2 above), 1 force naive DFT, 2 force radix-2."""
    lib().oracle_set_fft_mode(C.c_int(mode))


def dft_naive(x: np.ndarray, sign: int) -> np.ndarray:
    x = np.ascontiguousarray(x, dtype=np.complex128)
    out = np.empty_like(x)
    lib().oracle_dft_naive(C.c_int(x.size), _p(x), _p(out), C.c_int(sign))
    return out


def fft_radix2(x: np.ndarray, sign: int) -> np.ndarray:
    x = np.array(x, dtype=np.complex128, order="C")
    lib().oracle_fft_radix2(C.c_int(x.size), _p(x), C.c_int(sign))
    return x


def fft2(a: np.ndarray, sign: int) -> np.ndarray:
    """sign=-1 forward (unscaled), +1 inverse (1/(nx ny))."""
    a = np.array(a, dtype=np.complex128, order="C")
    ny, nx = a.shape
    lib().oracle_fft2(C.c_int(ny), C.c_int(nx), _p(a), C.c_int(sign))
    return a


def build_slices(nx: int, ny: int, lx: float, ly: float, pos: np.ndarray, species: np.ndarray,
                 a: np.ndarray, b: np.ndarray, dz: float, nslices: int, z0: float, sigma: float,
                 bandlimit: int = 1, pot_mode: int = 1, want_v: bool = False, want_vq: bool = False):
    """Returns dict(trans [S][ny][nx] c128, n_clamped, max_imag[, v][, vq])."""
    pos = np.ascontiguousarray(pos, dtype=np.float64)
    species = np.ascontiguousarray(species, dtype=np.int32)
    a = np.ascontiguousarray(a, dtype=np.float64)
    b = np.ascontiguousarray(b, dtype=np.float64)
    trans = np.empty((nslices, ny, nx), dtype=np.complex128)
    v = np.empty((nslices, ny, nx), dtype=np.float64) if want_v else None
    vq = np.empty((nslices, ny, nx), dtype=np.complex128) if want_vq else None
    ncl = C.c_int(0)
    mi = C.c_double(0.0)
    rc = lib().oracle_build_slices(
        C.c_int(nx), C.c_int(ny), C.c_double(lx), C.c_double(ly), _p(pos), _p(species),
        C.c_int(pos.shape[0]), C.c_int(a.shape[0]), _p(a), _p(b), C.c_double(dz), C.c_int(nslices),
        C.c_double(z0), C.c_double(sigma), C.c_int(bandlimit), C.c_int(pot_mode), _p(trans),
        _p(v) if want_v else None, _p(vq) if want_vq else None, C.byref(ncl), C.byref(mi))
    if rc != 0:
        raise RuntimeError(f"oracle_build_slices failed: {rc}")
    out = dict(trans=trans, n_clamped=int(ncl.value), max_imag=float(mi.value))
    if want_v:
        out["v"] = v
    if want_vq:
        out["vq"] = vq
    return out


def make_probes(nx: int, ny: int, lx: float, ly: float, lam: float, probe_xy: np.ndarray,
                alpha_rad: float) -> np.ndarray:
    probe_xy = np.ascontiguousarray(probe_xy, dtype=np.float64).reshape(-1, 2)
    waves = np.empty((probe_xy.shape[0], ny, nx), dtype=np.complex128)
    rc = lib().oracle_make_probes(C.c_int(nx), C.c_int(ny), C.c_double(lx), C.c_double(ly), C.c_double(lam),
                                  _p(probe_xy), C.c_int(probe_xy.shape[0]), C.c_double(alpha_rad), _p(waves))
    if rc != 0:
        raise RuntimeError(f"oracle_make_probes failed: {rc}")
    return waves


def propagate(lx: float, ly: float, lam: float, bandlimit: int, waves: np.ndarray,
              wave_frame: Optional[Sequence[int]], trans: Sequence[Sequence[np.ndarray]], dz: float,
              output_space: int = 0, want_norms: bool = False):
    """waves [nw][ny][nx] c128 (copied).  trans[f][k] = c128 [S_k][ny][nx] for in-flight frame f and
    z-segment k.  Returns the propagated waves (and norms [nw][S+1] if asked)."""
    waves = np.array(waves, dtype=np.complex128, order="C")
    nw, ny, nx = waves.shape
    nframes = len(trans)
    nseg = len(trans[0])
    keep = [[np.ascontiguousarray(t, dtype=np.complex128) for t in fr] for fr in trans]
    nsl = np.array([t.shape[0] for t in keep[0]], dtype=np.int32)
    ptrs = (C.c_void_p * (nframes * nseg))()
    for f in range(nframes):
        assert len(keep[f]) == nseg
        for k in range(nseg):
            assert keep[f][k].shape == (nsl[k], ny, nx)
            ptrs[f * nseg + k] = keep[f][k].ctypes.data
    wf = np.ascontiguousarray(wave_frame if wave_frame is not None else np.zeros(nw), dtype=np.int32)
    total = int(nsl.sum())
    norms = np.empty((nw, total + 1), dtype=np.float64) if want_norms else None
    rc = lib().oracle_propagate(C.c_int(nx), C.c_int(ny), C.c_double(lx), C.c_double(ly), C.c_double(lam),
                                C.c_int(bandlimit), _p(waves), _p(wf), C.c_int(nw), ptrs, C.c_int(nframes),
                                _p(nsl), C.c_int(nseg), C.c_double(dz), C.c_int(output_space),
                                _p(norms) if want_norms else None)
    if rc != 0:
        raise RuntimeError(f"oracle_propagate failed: {rc}")
    return (waves, norms) if want_norms else waves


ROI_MODES = {"full": 0, "disc": 1, "annulus": 2, "rect": 3}


def make_roi(nx: int, ny: int, lx: float, ly: float, lam: float, mode: str, params_rad: Sequence[float]) -> np.ndarray:
    params = np.ascontiguousarray(list(params_rad) + [0.0] * 4, dtype=np.float64)
    cnt = C.c_int64(0)
    args = [C.c_int(nx), C.c_int(ny), C.c_double(lx), C.c_double(ly), C.c_double(lam), C.c_int(ROI_MODES[mode]), _p(params)]
    rc = lib().oracle_make_roi(*args, None, C.byref(cnt))
    if rc != 0:
        raise RuntimeError(f"oracle_make_roi failed: {rc}")
    idx = np.empty(cnt.value, dtype=np.int32)
    lib().oracle_make_roi(*args, _p(idx), C.byref(cnt))
    return idx


def accumulate(qwaves: np.ndarray, wave_probe: Sequence[int], wave_frame: Sequence[int], roi_idx: np.ndarray,
               buf: np.ndarray) -> None:
    """buf [nprobes][nframes][nroi] c128, updated in place."""
    qwaves = np.ascontiguousarray(qwaves, dtype=np.complex128)
    nw, ny, nx = qwaves.shape
    wp = np.ascontiguousarray(wave_probe, dtype=np.int32)
    wf = np.ascontiguousarray(wave_frame, dtype=np.int32)
    roi_idx = np.ascontiguousarray(roi_idx, dtype=np.int32)
    assert buf.dtype == np.complex128 and buf.flags.c_contiguous and buf.shape[2] == roi_idx.size
    rc = lib().oracle_accumulate(C.c_int(nx), C.c_int(ny), _p(qwaves), C.c_int(nw), _p(wp), _p(wf), _p(roi_idx),
                                 C.c_int64(roi_idx.size), _p(buf), C.c_int(buf.shape[0]), C.c_int(buf.shape[1]))
    if rc != 0:
        raise RuntimeError(f"oracle_accumulate failed: {rc}")


def bose(x: float) -> float:
    return float(lib().oracle_bose(C.c_double(x)))


def window(kind: int, nframes: int) -> np.ndarray:
    w = np.empty(nframes, dtype=np.float64)
    lib().oracle_window(C.c_int(kind), C.c_int(nframes), _p(w))
    return w


def energy_axis(nframes: int, dt_fs: float, emin: float = -np.inf, emax: float = np.inf) -> Tuple[np.ndarray, np.ndarray]:
    E = np.empty(nframes, dtype=np.float64)
    bins = np.empty(nframes, dtype=np.int32)
    lib().oracle_energy_axis.restype = C.c_int
    n = lib().oracle_energy_axis(C.c_int(nframes), C.c_double(dt_fs), C.c_double(emin), C.c_double(emax), _p(E), _p(bins))
    return E[:n].copy(), bins[:n].copy()


def spectrum(buf: np.ndarray, dt_fs: float, window_kind: int, temperature_K: float,
             emin: float = -np.inf, emax: float = np.inf) -> Tuple[np.ndarray, np.ndarray]:
    """buf [P][T][Q] c128 -> (I [P][nE][Q] f64, E [nE] meV ascending)."""
    buf = np.ascontiguousarray(buf, dtype=np.complex128)
    P, T, Q = buf.shape
    E, _ = energy_axis(T, dt_fs, emin, emax)
    I = np.empty((P, E.size, Q), dtype=np.float64)
    Eo = np.empty(E.size, dtype=np.float64)
    nE = C.c_int(0)
    rc = lib().oracle_spectrum(_p(buf), C.c_int(P), C.c_int64(Q), C.c_int(T), C.c_double(dt_fs), C.c_int(window_kind),
                               C.c_double(temperature_K), C.c_double(emin), C.c_double(emax), _p(I), _p(Eo), C.byref(nE))
    if rc != 0:
        raise RuntimeError(f"oracle_spectrum failed: {rc}")
    assert nE.value == E.size
    return I, Eo


# ---------------------------------------------------------------------------------------------
# Welch chunks with Eq.(2) averaging, further window functions.

def window_table(kind: str, n: int, param: float = 0.0) -> np.ndarray:
    """Window functions of PAPER.md:170-182 / Appendix A in the periodic form x = f/n (reading G9: the periodic Hann is
    the variant for which the zero-loss peak does not leak, :182).  'tukey': param = alpha, the summed fractional width of
    the two cosine tapers; alpha = 1 is Hann, alpha = 0 is rectangular (:170).  'blackman_harris': 4-term cosine sum.
    'kaiser': param = beta, I0(beta sqrt(1 - (2x-1)^2))/I0(beta) (numpy.i0 is the library Bessel routine)."""
    x = np.arange(n, dtype=np.float64) / n
    if kind == "rect":
        return np.ones(n)
    if kind == "hann":
        return 0.5 - 0.5 * np.cos(2 * np.pi * x)
    if kind == "tukey":
        a = float(param)
        if a == 0.0:
            return np.ones(n)
        w = np.ones(n)
        up = x < a / 2
        dn = x > 1 - a / 2
        w[up] = 0.5 * (1 - np.cos(2 * np.pi * x[up] / a))
        w[dn] = 0.5 * (1 - np.cos(2 * np.pi * (1 - x[dn]) / a))
        return w
    if kind == "blackman_harris":
        return 0.35875 - 0.48829 * np.cos(2 * np.pi * x) + 0.14128 * np.cos(4 * np.pi * x) - 0.01168 * np.cos(6 * np.pi * x)
    if kind == "kaiser":
        u = 2 * x - 1
        return np.i0(param * np.sqrt(np.maximum(0.0, 1 - u * u))) / np.i0(param)
    if kind == "dolph_chebyshev":
        return dolph_chebyshev(n, float(param))
    raise ValueError(kind)


def dolph_chebyshev(n: int, attenuation_db: float) -> np.ndarray:
    """'the Dolph-Chebyshev window with attenuation 100 dB' (Appendix A; the paper points to scipy [59] for
    the definition).  Definition written out: the window of M points whose discrete-time Fourier transform is the
    Chebyshev polynomial of order M-1 in x0 cos(theta/2), all side lobes `attenuation_db` below the main lobe:
        W(theta) = T_{M-1}(x0 cos(theta/2)),   x0 = cosh(acosh(10^(att/20)) / (M-1)),
        w[j] = (1/M) sum_{k=0}^{M-1} W(2 pi k/M) cos(2 pi k (j - (M-1)/2) / M),   normalised to max w = 1
    (the sum is the inverse DFT of the M samples of W, centred on the window's midpoint; T_m(x) = cos(m acos x) for
    |x| <= 1, cosh(m acosh x) for x > 1, (-1)^m cosh(m acosh(-x)) for x < -1).  Periodic form (reading G9): the symmetric
    window of M = n + 1 points without its last sample.  Plain O(M^2) loops, no FFT."""
    M = n + 1
    if M < 2:
        return np.ones(n)
    m = M - 1
    x0 = np.cosh(np.arccosh(10.0 ** (abs(attenuation_db) / 20.0)) / m)

    def cheb(x: float) -> float:
        if x > 1.0:
            return float(np.cosh(m * np.arccosh(x)))
        if x < -1.0:
            return float((1.0 if m % 2 == 0 else -1.0) * np.cosh(m * np.arccosh(-x)))
        return float(np.cos(m * np.arccos(x)))

    W = np.array([cheb(x0 * np.cos(np.pi * k / M)) for k in range(M)])      # W(theta_k), theta_k = 2 pi k / M
    w = np.zeros(M)
    for j in range(M):
        acc = 0.0
        for k in range(M):
            acc += W[k] * np.cos(2.0 * np.pi * k * (j - 0.5 * m) / M)
        w[j] = acc / M
    w = w / w.max()
    return w[:n].copy()


def chunk_starts(nframes_total: int, chunk_len: int, chunk_overlap: int, skip_init: int = 0, stride: int = 1):
    """'If a chunk indexed by n starts at snapshot s_n, then the next chunk starts at
    s_{n+1} = s_n + L/nu, using remainder-less division'; only complete chunks are used.
    skip_init: the first `skip_init` snapshots are discarded (Listing 1 :443 `trajectory_chunks_skip_init = 200`: the
    3 ps thermalisation period of :164 at 15 fs).  stride: 'a stride for snapshot reading' (:140) -- chunk n holds the L
    snapshots s_n, s_n + stride, ..., and s counts in units of the stored snapshots, so the next chunk starts
    (L/nu) * stride stored snapshots later (reading G24)."""
    step = (chunk_len // chunk_overlap) * stride
    out, s = [], skip_init
    while s + (chunk_len - 1) * stride + 1 <= nframes_total:
        out.append(s)
        s += step
    return out


def spectrum_table(buf: np.ndarray, frame0: int, nframes: int, dt_fs: float, w: np.ndarray, temperature_K: float,
                   emin: float = -np.inf, emax: float = np.inf) -> Tuple[np.ndarray, np.ndarray]:
    """O9 on frames [frame0, frame0+nframes) of buf [P][Ttot][Q] with the window table w[nframes]."""
    buf = np.ascontiguousarray(buf, dtype=np.complex128)
    w = np.ascontiguousarray(w, dtype=np.float64)
    P, Ttot, Q = buf.shape
    E, _ = energy_axis(nframes, dt_fs, emin, emax)
    I = np.empty((P, E.size, Q), dtype=np.float64)
    Eo = np.empty(E.size, dtype=np.float64)
    nE = C.c_int(0)
    rc = lib().oracle_spectrum_table(_p(buf), C.c_int(P), C.c_int64(Q), C.c_int(Ttot), C.c_int(frame0), C.c_int(nframes),
                                     C.c_double(dt_fs), _p(w), C.c_double(temperature_K), C.c_double(emin), C.c_double(emax),
                                     _p(I), _p(Eo), C.byref(nE))
    if rc != 0:
        raise RuntimeError(f"oracle_spectrum_table failed: {rc}")
    return I, Eo


def spectrum_welch(buf: np.ndarray, chunk_len: int, chunk_overlap: int, dt_fs: float, w: np.ndarray, temperature_K: float,
                   emin: float = -np.inf, emax: float = np.inf, skip_init: int = 0, stride: int = 1):
    """Eq.(2): the average over the N trajectory chunks of I_i(q,E), each chunk windowed, transformed,
    squared and Bose-corrected as in O9 (:142).  With a snapshot stride the chunk's time step is stride * dt.
    Returns (I [P][nE][Q], E [nE], N)."""
    starts = chunk_starts(buf.shape[1], chunk_len, chunk_overlap, skip_init, stride)
    acc, E = None, None
    for s in starts:
        sub = np.ascontiguousarray(buf[:, s: s + (chunk_len - 1) * stride + 1: stride])     # the chunk's L snapshots
        I, E = spectrum_table(sub, 0, chunk_len, dt_fs * stride, w, temperature_K, emin, emax)
        acc = I / len(starts) if acc is None else acc + I / len(starts)
    if E is None:
        E, _ = energy_axis(chunk_len, dt_fs * stride, emin, emax)
    return acc, E, len(starts)


# DetectorSet.

def detector_weights(nx: int, ny: int, lx: float, ly: float, lam: float, kind: str, center_rad, radii_rad,
                     roi_idx: np.ndarray) -> np.ndarray:
    """'circular and annular -- with arbitrary center and radii' (:114): pixel (h,k) of the ROI is on the detector iff
    its scattering angle theta = lambda q, measured from the detector centre, lies inside the (inclusive) radii."""
    idx = np.asarray(roi_idx, dtype=np.int64)
    ix, iy = idx % nx, idx // nx
    h = np.where(ix < nx // 2, ix, ix - nx).astype(np.float64)
    k = np.where(iy < ny // 2, iy, iy - ny).astype(np.float64)
    tx = lam * h / lx - center_rad[0]
    ty = lam * k / ly - center_rad[1]
    t2 = tx * tx + ty * ty
    on = t2 <= radii_rad[1] * radii_rad[1]
    if kind == "annular":
        on &= t2 >= radii_rad[0] * radii_rad[0]
    elif kind != "circular":
        raise ValueError(kind)
    return on.astype(np.float64)


def detect(I: np.ndarray, weights: np.ndarray) -> np.ndarray:
    """Energy-filtered STEM signal: out[d][e][p] = sum_r weights[d][r] I[p][e][r]; axes [detector][energy][scan] (:150)."""
    return np.einsum("dr,per->dep", np.asarray(weights, dtype=np.float64), np.asarray(I, dtype=np.float64))


# SURVEY.md 8(f) item 4 (workload variants): scan grids (Listing 1 :416-428).

def scan_positions(mode: str, shape: Sequence[int], origin: Sequence[float], a: Sequence[float],
                   b: Optional[Sequence[float]] = None, cell: Optional[Sequence[float]] = None) -> np.ndarray:
    """The four scanning modes (:378).  'the scanning is performed over a two dimensional grid with grid shape ...
    defined by the user explicitly.  Note that the end point is by design "not included" -- for example, 5 scan
    points on interval [0.0, 1.0) would result in points {0.0, 0.2, 0.4, 0.6, 0.8}' (:378-380).
    Point (i, j), i < shape[0], j < shape[1], row p = i*shape[1] + j (reading G23):
      'box'           r = origin + (i/n0 (a_x - o_x), j/n1 (a_y - o_y));   a = scanning_box_end [A]  (:419-424)
      'box_relative'  the same with origin and a given as fractions of the simulation cell (cell = lx, ly [A])
      'unitcell'      box from origin over one unit cell with edges a = (a_uc, b_uc) [A]
      'parallelogram' r = origin + (i/n0) a + (j/n1) b;   a, b edge vectors [A]
    Plain loops, no vectorisation."""
    n0, n1 = int(shape[0]), int(shape[1])
    out = np.zeros((n0 * n1, 2), dtype=np.float64)
    for i in range(n0):
        for j in range(n1):
            fi, fj = i / n0, j / n1
            if mode == "box":
                x = origin[0] + fi * (a[0] - origin[0])
                y = origin[1] + fj * (a[1] - origin[1])
            elif mode == "box_relative":
                x = (origin[0] + fi * (a[0] - origin[0])) * cell[0]
                y = (origin[1] + fj * (a[1] - origin[1])) * cell[1]
            elif mode == "unitcell":
                x = origin[0] + fi * a[0]
                y = origin[1] + fj * a[1]
            elif mode == "parallelogram":
                x = origin[0] + fi * a[0] + fj * b[0]
                y = origin[1] + fi * a[1] + fj * b[1]
            else:
                raise ValueError(mode)
            out[i * n1 + j] = (x, y)
    return out


def scan_batches(shape: Sequence[int], batch_shape: Sequence[int]) -> List[np.ndarray]:
    """Scan sub-batches (:131 'scan sub-batch', Listing 1 :428 scanning_batch_shape = [4, 8] for a 16 x 16 scan): the
    scan grid is cut into tiles of batch_shape[0] x batch_shape[1] points (ragged at the far edges); tiles are numbered
    row-major over the tile grid and each lists its scan rows p = i*shape[1] + j in ascending (i, j)."""
    n0, n1 = int(shape[0]), int(shape[1])
    b0, b1 = int(batch_shape[0]), int(batch_shape[1])
    tiles = []
    for ti in range(0, n0, b0):
        for tj in range(0, n1, b1):
            tiles.append(np.array([i * n1 + j for i in range(ti, min(ti + b0, n0)) for j in range(tj, min(tj + b1, n1))],
                                  dtype=np.int32))
    return tiles
