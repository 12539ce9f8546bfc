"""Grids that are not powers of two ("1680 x 1680" = 2^4 3 5 7): the mixed-radix
path of csrc/generic.cu against the fp64 oracle (whose transforms of such lengths are its plain O(N^2) DFT, pinned against
numpy in tests/test_oracle_pins.py P8).  Same tolerances as tests/test_gpu_parity.py."""
import numpy as np
import pytest

from paper_2607_02236_b200 import workloads as W
from util import rel_l2

pytestmark = pytest.mark.gpu

TOL_WAVE = 2e-4
TOL_SPEC = 1e-3


@pytest.fixture(scope="module")
def torch():
    import torch as t
    if not t.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (no CPU fallback exists)")
    return t


@pytest.fixture(scope="module")
def B(torch):
    from paper_2607_02236_b200 import binding, build
    build.build_lib()
    binding.load_library()
    return binding


def dev(torch, a, dtype=None):
    t = torch.from_numpy(np.ascontiguousarray(a)).cuda()
    return t if dtype is None else t.to(dtype)


@pytest.mark.parametrize("nx,ny,bandlimit", [(48, 48, 1), (48, 48, 0), (210, 210, 1), (240, 210, 1), (210, 256, 1), (210, 256, 0),
                                             (420, 360, 1), (30, 18, 1)])
def test_propagate_random_slices_on_mixed_radix_grids(torch, B, oracle, nx, ny, bandlimit):
    """Random unit-modulus transmissions and random waves on grids with factors 3, 5, 7 (radix lists 8.6, 7.6.5, 8.6.5,
    7.6.5.2, 8.5.3.3 ...), rectangular ones and one mixed with a power of two; both output spaces, several frames and
    segments, probe indirection, a ragged number of waves."""
    if min(nx, ny) < 16:
        tc = None
        with pytest.raises(B.TacawError):
            tc = B.Tacaw(nx, ny, 5.0, 5.0, 0.037, 9e-4, bandlimit)       # below the supported range
        return
    nw, nframes, nsl = 5, 3, [2, 1]
    lx, ly, lam, dz = 0.09 * nx, 0.11 * ny, 0.0370144, 1.4795
    rng = np.random.default_rng(nx * 1000 + ny)
    trans = [[np.exp(1j * rng.normal(size=(s, ny, nx))) for s in nsl] for _ in range(nframes)]
    psi = rng.normal(size=(nw, ny, nx)) + 1j * rng.normal(size=(nw, ny, nx))
    psi /= np.sqrt((np.abs(psi) ** 2).sum(axis=(1, 2), keepdims=True))
    wf = np.sort(rng.integers(0, nframes, size=nw)).astype(np.int32)
    tc = B.Tacaw(nx, ny, lx, ly, lam, 9.2e-4, bandlimit)
    tr_d = [[dev(torch, t, torch.complex64) for t in fr] for fr in trans]
    probes = dev(torch, psi, torch.complex64)
    for space in (0, 1):
        ref = oracle.propagate(lx, ly, lam, bandlimit, psi, wf, trans, dz, space)
        w = torch.full((nw, ny, nx), float("nan"), dtype=torch.complex64, device="cuda")
        tc.propagate(w, wf, tr_d, dz, space, probes=probes, wave_probe=np.arange(nw, dtype=np.int32))
        got = w.cpu().numpy()
        w2 = dev(torch, psi, torch.complex64)
        tc.propagate(w2, wf, tr_d, dz, space)                    # in-place variant
        assert torch.equal(w2, w)
        for i in range(nw):
            assert rel_l2(got[i], ref[i]) <= 2e-5, (nx, ny, space, i)
    tc.close()


@pytest.mark.parametrize("n", [210])
def test_whole_path_on_a_mixed_radix_grid(torch, B, oracle, n):
    """build_slices (K1 + V -> t), probes, multislice, fused ROI gather, spectrum on an n x n grid, n = 2 3 5 7:
    against the oracle pipeline."""
    from oracle import pipeline as OP
    from paper_2607_02236_b200.pipeline import Runner
    wl = W.tiny_workload(n=32, ncell=(2, 2, 2), nframes=8, alpha_mrad=25.0)
    wl.nx = wl.ny = n
    wl.roi_mode, wl.roi_params_mrad = "disc", (60.0,)
    ref = OP.run(wl, pot_mode=0)
    for fused in (True, False):
        r = Runner(wl, frames_per_block=3, fused_gather=fused)
        out = r.run()
        assert np.array_equal(out["roi"], ref["roi"]) and np.array_equal(out["E"], ref["E"])
        buf = out["buf"].cpu().numpy()
        for f in range(wl.nframes):
            assert rel_l2(buf[0, f], ref["buf"][0, f]) <= TOL_WAVE, (fused, f)
        assert rel_l2(out["I"].cpu().numpy()[0], ref["I"][0]) <= TOL_SPEC
        r.close()


@pytest.mark.parametrize("nx,ny", [(1680, 32), (32, 1680)])
def test_whole_path_with_one_1680_edge(torch, B, oracle, nx, ny):
    """PAPER.md:162, the 1680-point transform (radices 8.7.6.5) along x (row kernel) and along y (column kernel): the whole
    path -- build_slices, probes, multislice, fused gather, spectrum -- with the paper's rectangular +-100 mrad ROI mode, on
    grids whose other edge is short so that the oracle's O(N^2) transforms of length 1680 stay cheap."""
    from oracle import pipeline as OP
    from paper_2607_02236_b200.pipeline import Runner
    wl = W.tiny_workload(n=32, ncell=(2, 2, 1), nframes=2, alpha_mrad=30.0)
    wl.nx, wl.ny = nx, ny
    wl.roi_mode, wl.roi_params_mrad = "rect", (-100.0, 100.0, -100.0, 100.0)
    ref = OP.run(wl, pot_mode=0)
    r = Runner(wl, frames_per_block=2)
    out = r.run()
    assert np.array_equal(out["roi"], ref["roi"]) and np.array_equal(out["E"], ref["E"])
    buf = out["buf"].cpu().numpy()
    for f in range(wl.nframes):
        assert rel_l2(buf[0, f], ref["buf"][0, f]) <= TOL_WAVE, f
    assert rel_l2(out["I"].cpu().numpy()[0], ref["I"][0]) <= TOL_SPEC
    r.close()


@pytest.mark.slow
def test_the_papers_1680_grid(torch, B, oracle):
    """the full 1680 x 1680 grid.  Two waves through one random slice and the free-space step, exit wave in q
    space, band limit on, against the oracle (each of its 2D transforms at this size is 9.5e9 complex multiply-adds, hence
    the single slice)."""
    n, nw = 1680, 2
    L, lam, dz = 93.0, 0.0487, 1.4795                        # the paper's 93 A cell at 60 kV
    rng = np.random.default_rng(1680)
    trans = [[np.exp(1j * rng.normal(size=(1, n, n)))]]
    psi = rng.normal(size=(nw, n, n)) + 1j * rng.normal(size=(nw, n, n))
    psi /= np.sqrt((np.abs(psi) ** 2).sum(axis=(1, 2), keepdims=True))
    wf = np.zeros(nw, np.int32)
    ref = oracle.propagate(L, L, lam, 1, psi, wf, trans, dz, 1)
    tc = B.Tacaw(n, n, L, L, lam, 9.2e-4, 1)
    w = torch.full((nw, n, n), float("nan"), dtype=torch.complex64, device="cuda")
    tc.propagate(w, wf, [[dev(torch, trans[0][0], torch.complex64)]], dz, 1, probes=dev(torch, psi, torch.complex64),
                 wave_probe=np.arange(nw, dtype=np.int32))
    got = w.cpu().numpy()
    for i in range(nw):
        assert rel_l2(got[i], ref[i]) <= 2e-5, i
    h = np.where(np.arange(n) < n // 2, np.arange(n), np.arange(n) - n)
    oob = 9 * (h[None, :] ** 2 + h[:, None] ** 2) > n * n
    assert np.all(got[:, oob] == 0)                          # out-of-band Psi_S is exactly zero
    tc.close()
