"""CPU-side checks of libtacaw: it builds/loads, exports every symbol include/tacaw.h declares, fails
loudly without a GPU, and its host-side ROI map is bit-exact against the oracle.  No GPU compute."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_2607_02236_b200 import binding, workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2607_02236_b200 import build
    build.build_lib()
    return binding.load_library()


def test_header_symbols_exported(lib):
    hdr = open(os.path.join(ROOT, "include", "tacaw.h")).read()
    declared = set(re.findall(r"\b(tacaw_[a-z_]+)\s*\(", hdr))
    assert declared == set(binding.EXPORTS)
    for name in declared:
        assert getattr(lib, name) is not None
    assert b"sm_100a" in lib.tacaw_version()


def test_create_fails_loudly_without_gpu(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    ctx = C.c_void_p()
    g, b = binding._Grid(64, 64, 10.0, 10.0), binding._Beam(0.037, 9e-4, 1)
    assert lib.tacaw_create(C.byref(ctx), C.byref(g), C.byref(b), 0) == -4      # TACAW_E_CUDA, no fallback
    assert not ctx.value
    with pytest.raises(binding.TacawError):
        binding.Tacaw(64, 64, 10.0, 10.0, 0.037, 9e-4)


def test_create_rejects_unsupported_grids(lib):
    ctx = C.c_void_p()
    b = binding._Beam(0.037, 9e-4, 1)
    # supported: powers of two in [16, 2048] and other even sizes in that range with prime factors 2, 3, 5, 7 only
    for nx, ny in ((46, 64), (63, 64), (8, 64), (64, 4096), (64, 2046), (0, 0)):
        g = binding._Grid(nx, ny, 10.0, 10.0)
        assert lib.tacaw_create(C.byref(ctx), C.byref(g), C.byref(b), 0) == -2  # TACAW_E_UNSUPPORTED


def test_create_accepts_the_papers_1680_grid_and_other_2357_sizes(lib):
    """Even sizes in [16, 2048] whose prime factors are 2, 3, 5, 7 pass the size check (1680 = 2^4 3 5 7): without
    a GPU the call then fails with TACAW_E_CUDA (-4), never with TACAW_E_UNSUPPORTED (-2)."""
    b = binding._Beam(0.037, 9e-4, 1)
    for nx, ny in ((1680, 1680), (210, 256), (48, 16), (2048, 1680), (1260, 420)):
        ctx = C.c_void_p()
        g = binding._Grid(nx, ny, 10.0, 10.0)
        rc = lib.tacaw_create(C.byref(ctx), C.byref(g), C.byref(b), 0)
        assert rc in (0, -4), (nx, ny, rc)
        if rc == 0:
            lib.tacaw_destroy(ctx)


@pytest.mark.parametrize("cfg", [1, 2, 3, 4, 5])
def test_roi_map_bit_exact_all_configs(lib, oracle, cfg):
    wl = W.make_workload(cfg, nframes=1, nprobes=1, ncz=1 if cfg >= 3 else None)
    params = [p * 1e-3 for p in wl.roi_params_mrad]
    ours = binding.make_roi(wl.nx, wl.ny, wl.lx, wl.ly, wl.lam, wl.roi_mode, params)
    ref = oracle.make_roi(wl.nx, wl.ny, wl.lx, wl.ly, wl.lam, wl.roi_mode, params)
    assert ours.dtype == np.int32 and np.array_equal(ours, ref)
    expect = {1: 4096, 2: 11165, 3: 7721, 4: 17449}
    if cfg in expect:
        assert ours.size == expect[cfg]
    else:
        assert 55000 < ours.size < 65000


def test_roi_edge_cases(lib, oracle):
    for mode, params in (("rect", [-0.01, 0.02, -0.005, 0.0]), ("disc", [0.0]), ("annulus", [0.5, 0.6]),
                         ("full", [])):
        ours = binding.make_roi(32, 64, 9.0, 17.0, 0.037, mode, params)       # rectangular cell
        ref = oracle.make_roi(32, 64, 9.0, 17.0, 0.037, mode, params)
        assert np.array_equal(ours, ref)
    assert binding.make_roi(32, 32, 9.0, 9.0, 0.037, "disc", [0.0]).tolist() == [0]
    assert binding.make_roi(32, 32, 9.0, 9.0, 0.037, "annulus", [0.5, 0.6]).size == 0
