"""tacaw_build_slices_static: the allocation-free variant of tacaw_build_slices (scratch in a static device array inside the
library, include/tacaw.h) against the workspace path on the same inputs.

Collected last on purpose (file name): the run uses `pytest -x`.  Passes alone in a fresh process and after
the other GPU tests (it uses its own contexts and the static array, nothing from earlier tests).
"""
import numpy as np
import pytest

from paper_2607_02236_b200 import workloads as W
from util import rel_l2

pytestmark = pytest.mark.gpu

TOL_TRANS = 1e-5          # the bound tests/test_gpu_parity.py uses for transmission functions


def test_build_slices_static_matches_workspace_path_on_consecutive_calls():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (no CPU fallback exists)")
    from paper_2607_02236_b200 import binding as B, build
    build.build_lib()
    B.load_library()

    wl = W.make_workload(2)                       # 256^2 grid, 7680 atoms, 40 slices, 2 species
    seg = wl.segments[0]
    sp = torch.from_numpy(np.ascontiguousarray(seg.species, dtype=np.int32)).cuda()
    ref_ctx = B.Tacaw(wl.nx, wl.ny, wl.lx, wl.ly, wl.lam, wl.sigma, wl.bandlimit)     # existing path: caller-owned workspace
    tc = B.Tacaw(wl.nx, wl.ny, wl.lx, wl.ly, wl.lam, wl.sigma, wl.bandlimit)          # never given a workspace

    # consecutive calls of different sizes on one stream: the second is smaller, so the array still holds the first
    # call's keys and counts beyond what the second one clears and rewrites; the third repeats the first
    first = None
    for f0, f1 in ((0, 8), (11, 14), (0, 8)):
        nf = f1 - f0
        pos = torch.from_numpy(seg.frames(f0, f1, wl.dt_fs)).cuda()
        want, _ = ref_ctx.build_slices(pos, sp, wl.a, wl.b, wl.dz, seg.nslices, 0.0)
        out = torch.full((nf, seg.nslices, wl.ny, wl.nx), float("nan"), dtype=torch.complex64, device="cuda")
        tc.build_slices_static(pos, sp, wl.a, wl.b, wl.dz, seg.nslices, 0.0, out)
        torch.cuda.synchronize()
        assert tc._ws is None                     # the static path never asked for a workspace
        got, ref = out.cpu().numpy(), want.cpu().numpy()
        assert np.all(np.isfinite(got.view(np.float32)))
        assert np.max(np.abs(np.abs(got) - 1.0)) <= 1e-6
        for f in range(nf):
            assert rel_l2(got[f], ref[f]) <= TOL_TRANS, (f0, f)
        if first is None:
            first = got
        elif (f0, f1) == (0, 8):
            assert np.array_equal(got, first)     # same input, same kernels: nothing of the call in between leaked
    tc.device_status()

    # sizes beyond the static array are refused with a clear error before any work is queued
    nf_big = 32                                   # 32 x 7680 atom-frames need 4.9 MB > 4 MiB
    assert 256 + 4 * (5 * nf_big * seg.pos0.shape[0] + 2 * nf_big * seg.nslices * 2 + 2) > B.STATIC_SCRATCH_BYTES
    pos_big = torch.zeros((nf_big, seg.pos0.shape[0], 3), dtype=torch.float64, device="cuda")
    out_big = torch.empty((nf_big, seg.nslices, wl.ny, wl.nx), dtype=torch.complex64, device="cuda")
    launches = tc.launches
    with pytest.raises(B.TacawError, match="static array holds"):
        tc.build_slices_static(pos_big, sp, wl.a, wl.b, wl.dz, seg.nslices, 0.0, out_big)
    assert tc.launches == launches
    tc.close()
    ref_ctx.close()
