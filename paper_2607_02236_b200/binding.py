"""Thin Python binding of libtacaw.so (include/tacaw.h): argument marshalling only.

Every step of the path runs in the library's CUDA kernels; PyTorch is used for device memory and
streams.  There is no CPU fallback: if the shared library is missing or there is no CUDA device the
calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import List, Optional, Sequence, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libtacaw.so")

EXPORTS = ["tacaw_version", "tacaw_create", "tacaw_destroy", "tacaw_last_error", "tacaw_launch_count",
           "tacaw_workspace_bytes", "tacaw_set_workspace", "tacaw_device_status",
           "tacaw_build_slices", "tacaw_build_slices_host", "tacaw_make_probes", "tacaw_propagate",
           "tacaw_make_roi", "tacaw_accumulate", "tacaw_make_roi_inverse", "tacaw_propagate_accumulate", "tacaw_spectrum", "tacaw_make_window", "tacaw_spectrum_welch",
           "tacaw_make_detector", "tacaw_detect", "tacaw_make_scan", "tacaw_scan_batch", "tacaw_build_slices_static"]

STATIC_SCRATCH_BYTES = 4 << 20     # TACAW_STATIC_SCRATCH_BYTES of include/tacaw.h

DETECTORS = {"circular": 0, "annular": 1}

SCAN_MODES = {"box": 0, "box_relative": 1, "unitcell": 2, "parallelogram": 3}

WINDOWS = {"rect": 0, "hann": 1, "tukey": 2, "blackman_harris": 3, "kaiser": 4, "dolph_chebyshev": 5}

ROI_MODES = {"full": 0, "disc": 1, "annulus": 2, "rect": 3}


class TacawError(RuntimeError):
    pass


class _Grid(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("lx_A", C.c_double), ("ly_A", C.c_double)]


class _Beam(C.Structure):
    _fields_ = [("lambda_A", C.c_double), ("sigma_rad_per_VA", C.c_double), ("bandlimit", C.c_int)]


class _Species(C.Structure):
    _fields_ = [("nspecies", C.c_int), ("a", C.c_void_p), ("b", C.c_void_p)]


class _Sizes(C.Structure):
    _fields_ = [("natoms", C.c_int), ("nframes", C.c_int), ("nslices", C.c_int), ("nsegments", C.c_int),
                ("nwaves", C.c_int), ("nprobes", C.c_int), ("host_staging", C.c_int)]

SIZE_KEYS = ("natoms", "nframes", "nslices", "nsegments", "nwaves", "nprobes", "host_staging")


_lib = None


def load_library():
    """dlopen libtacaw.so; raises TacawError if it has not been built (no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise TacawError(f"{LIB_PATH} not found: build it with `python -m paper_2607_02236_b200.build` "
                             "(or __graft_entry__.build()); there is no CPU fallback")
        lib = C.CDLL(LIB_PATH)
        lib.tacaw_version.restype = C.c_char_p
        lib.tacaw_last_error.restype = C.c_char_p
        lib.tacaw_last_error.argtypes = [C.c_void_p]
        lib.tacaw_launch_count.restype = C.c_int64
        lib.tacaw_launch_count.argtypes = [C.c_void_p]
        lib.tacaw_workspace_bytes.restype = C.c_size_t
        lib.tacaw_workspace_bytes.argtypes = [C.c_void_p, C.c_void_p]
        _lib = lib
    return _lib


def make_roi(nx: int, ny: int, lx: float, ly: float, lam: float, mode: str, params_rad: Sequence[float]) -> np.ndarray:
    """tacaw_make_roi (host, exact): int32 flat FFT indices in ascending (k, h) order."""
    lib = load_library()
    g = _Grid(nx, ny, lx, ly)
    params = (C.c_double * 4)(*(list(params_rad) + [0.0] * 4)[:4])
    cnt = C.c_int64(0)
    rc = lib.tacaw_make_roi(C.byref(g), C.c_double(lam), C.c_int(ROI_MODES[mode]), params, None, C.byref(cnt))
    if rc != 0:
        raise TacawError(f"tacaw_make_roi failed ({rc})")
    idx = np.empty(cnt.value, dtype=np.int32)
    rc = lib.tacaw_make_roi(C.byref(g), C.c_double(lam), C.c_int(ROI_MODES[mode]), params,
                            idx.ctypes.data_as(C.c_void_p), C.byref(cnt))
    if rc != 0:
        raise TacawError(f"tacaw_make_roi failed ({rc})")
    return idx


def _i32(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.int32)


class Tacaw:
    """One context = one grid + beam on one CUDA device (tacaw_create / tacaw_destroy)."""

    def __init__(self, nx: int, ny: int, lx: float, ly: float, lam: float, sigma: float, bandlimit: int = 1,
                 device: int = 0):
        import torch
        self.torch = torch
        if not torch.cuda.is_available():
            raise TacawError("no CUDA device: the TACAW path has no CPU fallback")
        self.lib = load_library()
        self.nx, self.ny, self.lx, self.ly, self.lam, self.sigma = nx, ny, lx, ly, lam, sigma
        self.device = device
        self._ctx = C.c_void_p()
        g, b = _Grid(nx, ny, lx, ly), _Beam(lam, sigma, bandlimit)
        rc = self.lib.tacaw_create(C.byref(self._ctx), C.byref(g), C.byref(b), C.c_int(device))
        if rc != 0:
            raise TacawError(f"tacaw_create failed ({rc})")
        self._ws = None                                  # the caller-owned workspace tensor (torch owns the memory)
        self._ws_sizes = dict.fromkeys(SIZE_KEYS, 0)

    # ------------------------------------------------------------------------------------------
    def workspace_bytes(self, **sizes) -> int:
        """tacaw_workspace_bytes for the given largest call sizes (keys: SIZE_KEYS)."""
        z = _Sizes(*[int(sizes.get(k, 0)) for k in SIZE_KEYS])
        return int(self.lib.tacaw_workspace_bytes(self._ctx, C.byref(z)))

    def set_workspace(self, tensor, **sizes):
        """tacaw_set_workspace: hand the library a caller-owned CUDA uint8 tensor (kept alive by this object)."""
        z = _Sizes(*[int(sizes.get(k, 0)) for k in SIZE_KEYS])
        nbytes = tensor.numel() * tensor.element_size() if tensor is not None else 0
        rc = self.lib.tacaw_set_workspace(self._ctx, C.c_void_p(tensor.data_ptr()) if tensor is not None else None,
                                          C.c_size_t(nbytes), C.byref(z))
        self._check(rc, "tacaw_set_workspace")
        self._ws = tensor
        self._ws_sizes = {k: int(sizes.get(k, 0)) for k in SIZE_KEYS}

    def reserve(self, **sizes):
        """Caller-side convenience: make sure the workspace covers calls of these sizes (grow-only; the library itself
        never allocates).  Growing allocates a new torch tensor on the current stream and hands it over; work already
        queued against the old one is ordered before the next call because a context is driven from one stream."""
        if all(int(sizes.get(k, 0)) <= self._ws_sizes[k] for k in SIZE_KEYS) and self._ws is not None:
            return
        new = {k: max(int(sizes.get(k, 0)), self._ws_sizes[k]) for k in SIZE_KEYS}
        nbytes = self.workspace_bytes(**new)
        t = self.torch.empty(nbytes + 256, dtype=self.torch.uint8, device=f"cuda:{self.device}")
        off = (-t.data_ptr()) % 256
        self.set_workspace(t[off:off + nbytes], **new)
        self._ws_base = t

    def device_status(self):
        """tacaw_device_status: synchronises the current stream; raises if a kernel flagged bad input."""
        self._check(self.lib.tacaw_device_status(self._ctx, self._stream()), "tacaw_device_status")

    def close(self):
        if getattr(self, "_ctx", None) is not None and self._ctx.value:
            self.lib.tacaw_destroy(self._ctx)
            self._ctx = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ------------------------------------------------------------------------------------------
    def _check(self, rc: int, what: str):
        if rc != 0:
            msg = self.lib.tacaw_last_error(self._ctx)
            raise TacawError(f"{what} failed ({rc}): {msg.decode() if msg else ''}")

    def _stream(self) -> C.c_void_p:
        return C.c_void_p(self.torch.cuda.current_stream(self.device).cuda_stream)

    def _dev(self, t, dtype, what):
        if not (t.is_cuda and t.dtype == dtype and t.is_contiguous()):
            raise TacawError(f"{what}: need a contiguous CUDA tensor of dtype {dtype}")
        return C.c_void_p(t.data_ptr())

    @property
    def launches(self) -> int:
        return int(self.lib.tacaw_launch_count(self._ctx))

    def _species(self, a, b):
        a = np.ascontiguousarray(a, dtype=np.float64)
        b = np.ascontiguousarray(b, dtype=np.float64)
        return _Species(a.shape[0], a.ctypes.data, b.ctypes.data), (a, b)

    # ------------------------------------------------------------------------------------------
    def build_slices(self, pos, species, a, b, dz: float, nslices: int, z0: float = 0.0, out=None,
                     want_clamped: bool = False):
        """tacaw_build_slices, batched over frames.  pos: CUDA float64 [F][Na][3] (or [Na][3] for one frame);
        species: CUDA int32 [Na].  Returns (trans complex64 [F][S][ny][nx] (or [S][ny][nx]), n_clamped or None)."""
        torch = self.torch
        single = pos.dim() == 2
        nframes = 1 if single else int(pos.shape[0])
        natoms = int(pos.shape[-2])
        if out is None:
            shape = (nslices, self.ny, self.nx) if single else (nframes, nslices, self.ny, self.nx)
            out = torch.empty(shape, dtype=torch.complex64, device=pos.device)
        if out.numel() != nframes * nslices * self.ny * self.nx:
            raise TacawError("build_slices: output tensor has the wrong size")
        sp, keep = self._species(a, b)
        ncl = C.c_int(0)
        self.reserve(natoms=natoms, nframes=nframes, nslices=nslices)
        rc = self.lib.tacaw_build_slices(self._ctx, self._dev(pos, torch.float64, "pos"),
                                         self._dev(species, torch.int32, "species"), C.c_int(natoms), C.c_int(nframes),
                                         C.byref(sp), C.c_double(dz), C.c_int(nslices), C.c_double(z0),
                                         self._dev(out, torch.complex64, "trans"),
                                         C.byref(ncl) if want_clamped else None, self._stream())
        self._check(rc, "tacaw_build_slices")
        return out, (int(ncl.value) if want_clamped else None)

    def build_slices_static(self, pos, species, a, b, dz: float, nslices: int, z0: float, out):
        """tacaw_build_slices_static: same result as build_slices with the scratch in the library's static device array.
        Allocates nothing (the caller passes `out`) and needs no workspace; sizes beyond STATIC_SCRATCH_BYTES raise."""
        torch = self.torch
        nframes = 1 if pos.dim() == 2 else int(pos.shape[0])
        natoms = int(pos.shape[-2])
        if out.numel() != nframes * nslices * self.ny * self.nx:
            raise TacawError("build_slices_static: output tensor has the wrong size")
        sp, keep = self._species(a, b)
        rc = self.lib.tacaw_build_slices_static(self._ctx, self._dev(pos, torch.float64, "pos"),
                                                self._dev(species, torch.int32, "species"), C.c_int(natoms),
                                                C.c_int(nframes), C.byref(sp), C.c_double(dz), C.c_int(nslices),
                                                C.c_double(z0), self._dev(out, torch.complex64, "trans"), self._stream())
        self._check(rc, "tacaw_build_slices_static")
        return out

    def build_slices_host(self, pos_h: np.ndarray, species_h: np.ndarray, a, b, dz: float, nslices: int,
                          z0: float, out, want_clamped: bool = True):
        """tacaw_build_slices_host: positions [F][Na][3] / species are HOST arrays (H2D inside the call)."""
        torch = self.torch
        pos_h = np.ascontiguousarray(pos_h, dtype=np.float64)
        species_h = np.ascontiguousarray(species_h, dtype=np.int32)
        nframes = 1 if pos_h.ndim == 2 else int(pos_h.shape[0])
        natoms = int(pos_h.shape[-2])
        if out.numel() != nframes * nslices * self.ny * self.nx:
            raise TacawError("build_slices_host: output tensor has the wrong size")
        sp, keep = self._species(a, b)
        ncl = C.c_int(0)
        self.reserve(natoms=natoms, nframes=nframes, nslices=nslices, host_staging=1)
        rc = self.lib.tacaw_build_slices_host(self._ctx, pos_h.ctypes.data_as(C.c_void_p),
                                              species_h.ctypes.data_as(C.c_void_p), C.c_int(natoms), C.c_int(nframes),
                                              C.byref(sp), C.c_double(dz), C.c_int(nslices), C.c_double(z0),
                                              self._dev(out, torch.complex64, "trans"),
                                              C.byref(ncl) if want_clamped else None, self._stream())
        self._check(rc, "tacaw_build_slices_host")
        return out, (int(ncl.value) if want_clamped else None)

    def make_probes(self, probe_xy: np.ndarray, alpha_rad: float, out=None):
        torch = self.torch
        xy = np.ascontiguousarray(probe_xy, dtype=np.float64).reshape(-1, 2)
        if out is None:
            out = torch.empty((xy.shape[0], self.ny, self.nx), dtype=torch.complex64, device=f"cuda:{self.device}")
        self.reserve(nprobes=xy.shape[0])
        rc = self.lib.tacaw_make_probes(self._ctx, xy.ctypes.data_as(C.c_void_p), C.c_int(xy.shape[0]),
                                        C.c_double(alpha_rad), self._dev(out, torch.complex64, "waves"), self._stream())
        self._check(rc, "tacaw_make_probes")
        return out

    def propagate(self, waves, wave_frame, trans: Sequence[Sequence], dz: float, output_space: int = 1,
                  probes=None, wave_probe=None):
        """tacaw_propagate, in place on `waves` (CUDA complex64 [nw][ny][nx]).
        trans[f][k]: CUDA complex64 [S_k][ny][nx] for in-flight frame f and z-segment k."""
        torch = self.torch
        nw = waves.shape[0]
        nframes, nseg = len(trans), len(trans[0])
        ptrs = (C.c_void_p * (nframes * nseg))()
        nsl = np.array([int(t.shape[0]) for t in trans[0]], dtype=np.int32)
        for f in range(nframes):
            if len(trans[f]) != nseg:
                raise TacawError("every frame needs the same number of segments")
            for k in range(nseg):
                t = trans[f][k]
                if tuple(t.shape) != (int(nsl[k]), self.ny, self.nx):
                    raise TacawError("transmission tensor has the wrong shape")
                ptrs[f * nseg + k] = self._dev(t, torch.complex64, "trans").value
        wf = _i32(wave_frame)
        wp = _i32(wave_probe) if wave_probe is not None else None
        if wf.size != nw or (wp is not None and wp.size != nw):
            raise TacawError("wave_frame / wave_probe length mismatch")
        self.reserve(nwaves=nw, nframes=nframes, nsegments=nseg)
        rc = self.lib.tacaw_propagate(self._ctx, self._dev(waves, torch.complex64, "waves"),
                                      self._dev(probes, torch.complex64, "probes") if probes is not None else None,
                                      C.c_int(int(probes.shape[0]) if probes is not None else 0),
                                      wp.ctypes.data_as(C.c_void_p) if wp is not None else None,
                                      wf.ctypes.data_as(C.c_void_p), C.c_int(nw), ptrs, C.c_int(nframes),
                                      nsl.ctypes.data_as(C.c_void_p), C.c_int(nseg), C.c_double(dz), C.c_int(output_space),
                                      self._stream())
        self._check(rc, "tacaw_propagate")
        return waves

    def _trans_table(self, trans):
        torch = self.torch
        nframes, nseg = len(trans), len(trans[0])
        ptrs = (C.c_void_p * (nframes * nseg))()
        nsl = np.array([int(t.shape[0]) for t in trans[0]], dtype=np.int32)
        for f in range(nframes):
            if len(trans[f]) != nseg:
                raise TacawError("every frame needs the same number of segments")
            for k in range(nseg):
                t = trans[f][k]
                if tuple(t.shape) != (int(nsl[k]), self.ny, self.nx):
                    raise TacawError("transmission tensor has the wrong shape")
                ptrs[f * nseg + k] = self._dev(t, torch.complex64, "trans").value
        return ptrs, nsl, nframes, nseg

    def make_roi_inverse(self, roi_idx, out=None):
        """tacaw_make_roi_inverse: CUDA int32 [ny][nx], position of each pixel in the ROI list or -1."""
        torch = self.torch
        if out is None:
            out = torch.empty((self.ny, self.nx), dtype=torch.int32, device=roi_idx.device)
        rc = self.lib.tacaw_make_roi_inverse(self._ctx, self._dev(roi_idx, torch.int32, "roi_idx"), C.c_int64(roi_idx.numel()),
                                             self._dev(out, torch.int32, "roi_inv"), self._stream())
        self._check(rc, "tacaw_make_roi_inverse")
        return out

    def propagate_accumulate(self, waves, wave_probe, wave_frame, wave_time, trans, dz: float, roi_inv, nroi: int, buf, probes=None):
        """tacaw_propagate_accumulate: multislice + fused ROI gather into buf (CUDA complex64 [P][T][Q]); `waves` is scratch."""
        torch = self.torch
        nw = waves.shape[0]
        ptrs, nsl, nframes, nseg = self._trans_table(trans)
        wp, wf, wt = _i32(wave_probe), _i32(wave_frame), _i32(wave_time)
        if wp.size != nw or wf.size != nw or wt.size != nw:
            raise TacawError("wave_probe / wave_frame / wave_time length mismatch")
        self.reserve(nwaves=nw, nframes=nframes, nsegments=nseg)
        rc = self.lib.tacaw_propagate_accumulate(
            self._ctx, self._dev(waves, torch.complex64, "waves"),
            self._dev(probes, torch.complex64, "probes") if probes is not None else None,
            C.c_int(int(probes.shape[0]) if probes is not None else 0), wp.ctypes.data_as(C.c_void_p),
            wf.ctypes.data_as(C.c_void_p), wt.ctypes.data_as(C.c_void_p), C.c_int(nw), ptrs, C.c_int(nframes),
            nsl.ctypes.data_as(C.c_void_p), C.c_int(nseg), C.c_double(dz), self._dev(roi_inv, torch.int32, "roi_inv"),
            C.c_int64(nroi), self._dev(buf, torch.complex64, "buf"), C.c_int(buf.shape[0]), C.c_int(buf.shape[1]), self._stream())
        self._check(rc, "tacaw_propagate_accumulate")
        return buf

    def accumulate(self, qwaves, wave_probe, wave_frame, roi_idx, buf):
        """tacaw_accumulate: buf (CUDA complex64 [P][T][Q]) updated in place."""
        torch = self.torch
        wp, wf = _i32(wave_probe), _i32(wave_frame)
        self.reserve(nwaves=qwaves.shape[0])
        rc = self.lib.tacaw_accumulate(self._ctx, self._dev(qwaves, torch.complex64, "qwaves"), C.c_int(qwaves.shape[0]),
                                       wp.ctypes.data_as(C.c_void_p), wf.ctypes.data_as(C.c_void_p),
                                       self._dev(roi_idx, torch.int32, "roi_idx"), C.c_int64(roi_idx.numel()),
                                       self._dev(buf, torch.complex64, "buf"), C.c_int(buf.shape[0]), C.c_int(buf.shape[1]),
                                       self._stream())
        self._check(rc, "tacaw_accumulate")
        return buf

    def spectrum(self, buf, dt_fs: float, window: int, temperature_K: float, emin: float = -np.inf,
                 emax: float = np.inf, out=None):
        """tacaw_spectrum: returns (I float32 CUDA [P][nE][Q], E float64 numpy [nE])."""
        torch = self.torch
        P, T, Q = buf.shape
        nE = C.c_int(0)
        E = np.empty(T, dtype=np.float64)
        args = [C.c_int(P), C.c_int64(Q), C.c_int(T), C.c_double(dt_fs), C.c_int(window), C.c_double(temperature_K),
                C.c_double(emin), C.c_double(emax)]
        self.reserve()
        rc = self.lib.tacaw_spectrum(self._ctx, None, *args, None, E.ctypes.data_as(C.c_void_p), C.byref(nE), self._stream())
        self._check(rc, "tacaw_spectrum")
        if out is None:
            out = torch.empty((P, nE.value, Q), dtype=torch.float32, device=buf.device)
        rc = self.lib.tacaw_spectrum(self._ctx, self._dev(buf, torch.complex64, "buf"), *args,
                                     self._dev(out, torch.float32, "I"), E.ctypes.data_as(C.c_void_p), C.byref(nE),
                                     self._stream())
        self._check(rc, "tacaw_spectrum")
        return out, E[: nE.value].copy()

    def spectrum_welch(self, buf, chunk_len: int, chunk_overlap: int, dt_fs: float, window_table, temperature_K: float,
                       emin: float = -np.inf, emax: float = np.inf, out=None, skip_init: int = 0, stride: int = 1):
        """tacaw_spectrum_welch: returns (I float32 CUDA [P][nE][Q] averaged over the chunks, E float64 numpy [nE], nchunks)."""
        torch = self.torch
        P, Ttot, Q = buf.shape
        w = np.ascontiguousarray(window_table, dtype=np.float64)
        if w.shape != (chunk_len,):
            raise ValueError("window_table must have chunk_len entries")
        nE, nch = C.c_int(0), C.c_int(0)
        E = np.empty(chunk_len, dtype=np.float64)
        args = [C.c_int(P), C.c_int64(Q), C.c_int(Ttot), C.c_int(chunk_len), C.c_int(chunk_overlap), C.c_int(skip_init),
                C.c_int(stride), C.c_double(dt_fs),
                w.ctypes.data_as(C.c_void_p), C.c_double(temperature_K), C.c_double(emin), C.c_double(emax)]
        self.reserve()
        rc = self.lib.tacaw_spectrum_welch(self._ctx, None, *args, None, E.ctypes.data_as(C.c_void_p), C.byref(nE), C.byref(nch),
                                           self._stream())
        self._check(rc, "tacaw_spectrum_welch")
        if out is None:
            out = torch.zeros((P, nE.value, Q), dtype=torch.float32, device=buf.device)
        rc = self.lib.tacaw_spectrum_welch(self._ctx, self._dev(buf, torch.complex64, "buf"), *args,
                                           self._dev(out, torch.float32, "I"), E.ctypes.data_as(C.c_void_p), C.byref(nE),
                                           C.byref(nch), self._stream())
        self._check(rc, "tacaw_spectrum_welch")
        return out, E[: nE.value].copy(), nch.value

    def detect(self, I, weights, out=None):
        """tacaw_detect: I float32 CUDA [P][nE][Q], weights float32 CUDA [D][Q] -> out float32 CUDA [D][nE][P]."""
        torch = self.torch
        P, nE, Q = I.shape
        D = weights.shape[0]
        if weights.shape != (D, Q):
            raise ValueError("weights must be [ndet][nroi]")
        if out is None:
            out = torch.empty((D, nE, P), dtype=torch.float32, device=I.device)
        for d0 in range(0, D, 8):
            d1 = min(D, d0 + 8)
            rc = self.lib.tacaw_detect(self._ctx, self._dev(I, torch.float32, "I"), C.c_int(P), C.c_int(nE), C.c_int64(Q),
                                       self._dev(weights[d0:d1], torch.float32, "weights"), C.c_int(d1 - d0),
                                       self._dev(out[d0:d1], torch.float32, "out"), self._stream())
            self._check(rc, "tacaw_detect")
        return out


def make_detector(nx: int, ny: int, lx: float, ly: float, lam: float, kind: str, center_rad: Sequence[float],
                  radii_rad: Sequence[float], roi_idx: np.ndarray) -> np.ndarray:
    """tacaw_make_detector (host, exact): float32 0/1 weights over the ROI pixels for a circular (radii = (_, r)) or
    annular (radii = (r_in, r_out)) detector centred at center_rad."""
    lib = load_library()
    g = _Grid(nx, ny, lx, ly)
    idx = np.ascontiguousarray(roi_idx, dtype=np.int32)
    c = (C.c_double * 2)(*center_rad)
    r = (C.c_double * 2)(*radii_rad)
    w = np.empty(idx.size, dtype=np.float32)
    rc = lib.tacaw_make_detector(C.byref(g), C.c_double(lam), C.c_int(DETECTORS[kind]), c, r, idx.ctypes.data_as(C.c_void_p),
                                 C.c_int64(idx.size), w.ctypes.data_as(C.c_void_p))
    if rc != 0:
        raise TacawError(f"tacaw_make_detector failed ({rc})")
    return w


def make_window(kind: str, n: int, param: float = 0.0) -> np.ndarray:
    """tacaw_make_window (host): fp64 table of a periodic window ('rect', 'hann', 'tukey', 'blackman_harris', 'kaiser', 'dolph_chebyshev')."""
    lib = load_library()
    w = np.empty(n, dtype=np.float64)
    rc = lib.tacaw_make_window(C.c_int(WINDOWS[kind]), C.c_int(n), C.c_double(param), w.ctypes.data_as(C.c_void_p))
    if rc != 0:
        raise TacawError(f"tacaw_make_window failed ({rc})")
    return w


def make_scan(mode: str, shape: Sequence[int], origin: Sequence[float], a: Sequence[float],
              b: Optional[Sequence[float]] = None, cell: Optional[Sequence[float]] = None) -> np.ndarray:
    """tacaw_make_scan (host): scan positions [shape[0]*shape[1]][2] in Angstrom, end point excluded."""
    lib = load_library()
    sh = (C.c_int32 * 2)(*[int(v) for v in shape])
    d2 = lambda v: None if v is None else (C.c_double * 2)(*[float(x) for x in v])
    n = max(int(shape[0]), 0) * max(int(shape[1]), 0)
    xy = np.empty((n, 2), dtype=np.float64)
    rc = lib.tacaw_make_scan(C.c_int(SCAN_MODES[mode]), sh, d2(origin), d2(a), d2(b), d2(cell), xy.ctypes.data_as(C.c_void_p))
    if rc != 0:
        raise TacawError(f"tacaw_make_scan failed ({rc})")
    return xy


def scan_batch(shape: Sequence[int], batch_shape: Sequence[int], batch: int) -> Tuple[np.ndarray, int]:
    """tacaw_scan_batch (host): scan rows of sub-batch `batch` and the number of sub-batches."""
    lib = load_library()
    sh = (C.c_int32 * 2)(*[int(v) for v in shape])
    bs = (C.c_int32 * 2)(*[int(v) for v in batch_shape])
    cnt, nb = C.c_int32(0), C.c_int32(0)
    rc = lib.tacaw_scan_batch(sh, bs, C.c_int(batch), None, C.byref(cnt), C.byref(nb))
    if rc != 0:
        raise TacawError(f"tacaw_scan_batch failed ({rc})")
    idx = np.empty(cnt.value, dtype=np.int32)
    rc = lib.tacaw_scan_batch(sh, bs, C.c_int(batch), idx.ctypes.data_as(C.c_void_p), C.byref(cnt), C.byref(nb))
    if rc != 0:
        raise TacawError(f"tacaw_scan_batch failed ({rc})")
    return idx, nb.value
