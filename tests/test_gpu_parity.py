"""GPU parity: every C-ABI call of libtacaw against the fp64 oracle on the same seeded inputs.

Tolerances (BASELINE.json north_star): complex64 exit waves rel-L2 <= 2e-4 per (probe, frame);
spectra I(q,E) rel-L2 <= 1e-3 per probe; integer ROI maps bit-exact (tests/test_library_cpu.py).
Component tests use tighter bounds derived from fp32 arithmetic.
"""
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


def random_setup(seed, nx, ny, nw, nframes, nsl):
    rng = np.random.default_rng(seed)
    trans = [[np.exp(1j * rng.normal(size=(s, ny, nx))) for s in nsl] for _ in range(nframes)]
    psi = rng.normal(size=(nw, ny, nx)) + 1j * rng.normal(size=(nw, ny, nx))
    psi /= np.sqrt((np.abs(psi) ** 2).sum(axis=(1, 2), keepdims=True))
    wf = rng.integers(0, nframes, size=nw).astype(np.int32)
    wf.sort()
    return trans, psi, wf


# ------------------------------------------------------------------------------- propagate (K4)
@pytest.mark.parametrize("n", [16, 32, 64, 128, 256, 512, 1024, 2048])
@pytest.mark.parametrize("bandlimit", [1, 0])
def test_propagate_random_slices_all_grid_sizes(torch, B, oracle, n, bandlimit):
    """Random unit-modulus transmissions and random waves: exercises every FFT plan, both output
    spaces, band-limit on/off, several frames in flight and a ragged number of waves."""
    nw, nframes, nsl = (5, 3, [2, 1]) if n <= 512 else ((3, 2, [2]) if bandlimit else (2, 1, [1]))
    L, lam, dz = 0.09 * n, 0.0370144, 1.4795
    trans, psi, wf = random_setup(n, n, n, nw, nframes, nsl)
    tc = B.Tacaw(n, n, L, L, lam, 9.2e-4, bandlimit)
    tr_d = [[dev(torch, t, torch.complex64) for t in fr] for fr in trans]
    probes = dev(torch, psi, torch.complex64)
    for space in (0, 1):
        ref = oracle.propagate(L, L, lam, bandlimit, psi, wf, trans, dz, space)
        # output buffer pre-filled with NaN: nothing of its previous content may leak into the result
        w = torch.full((nw, n, n), float("nan"), dtype=torch.complex64, device="cuda")
        tc.propagate(w, wf, tr_d, dz, space, probes=probes, wave_probe=np.arange(nw, dtype=np.int32))
        got = w.cpu().numpy()
        w2 = dev(torch, psi, torch.complex64)
        tc.propagate(w2, wf, tr_d, dz, space)                    # in-place variant (entrance waves in d_waves)
        assert torch.equal(w2, w)
        for i in range(nw):
            assert rel_l2(got[i], ref[i]) <= 2e-5, (n, space, i)
        if space == 1 and bandlimit:
            h = np.where(np.arange(n) < n // 2, np.arange(n), np.arange(n) - n)
            oob = 9 * (h[None, :] ** 2 + h[:, None] ** 2) > n * n
            assert np.all(got[:, oob] == 0)          # out-of-band Psi_S is exactly zero
    tc.close()


def test_propagate_rectangular_grid_and_probe_indirection(torch, B, oracle):
    nx, ny, lx, ly, lam, dz = 128, 64, 11.0, 7.0, 0.0370144, 1.2
    trans, psi, _ = random_setup(7, nx, ny, 2, 3, [3])
    wave_probe = np.array([1, 0, 1, 1, 0, 0, 1], dtype=np.int32)
    wave_frame = np.array([0, 0, 1, 1, 1, 2, 2], dtype=np.int32)
    tc = B.Tacaw(nx, ny, lx, ly, lam, 9.2e-4, 1)
    tr_d = [[dev(torch, t, torch.complex64) for t in fr] for fr in trans]
    probes = dev(torch, psi, torch.complex64)
    w = torch.full((7, ny, nx), float("nan"), dtype=torch.complex64, device="cuda")
    tc.propagate(w, wave_frame, tr_d, dz, 0, probes=probes, wave_probe=wave_probe)
    ref = oracle.propagate(lx, ly, lam, 1, psi[wave_probe], wave_frame, trans, dz, 0)
    got = w.cpu().numpy()
    for i in range(7):
        assert rel_l2(got[i], ref[i]) <= 2e-5
    assert torch.equal(probes, dev(torch, psi, torch.complex64))     # entrance probes untouched
    tc.close()


def test_propagate_batch_invariance_and_segments(torch, B, oracle):
    """P14: any batching of waves gives the same result; P12: segments == concatenated slices."""
    n, L, lam, dz = 64, 9.0, 0.0370144, 1.4795
    trans, psi, wf = random_setup(3, n, n, 6, 2, [2, 3])
    tc = B.Tacaw(n, n, L, L, lam, 9.2e-4, 1)
    tr_d = [[dev(torch, t, torch.complex64) for t in fr] for fr in trans]
    full = dev(torch, psi, torch.complex64)
    tc.propagate(full, wf, tr_d, dz, 1)
    for i in range(6):
        one = dev(torch, psi[i:i + 1], torch.complex64)
        tc.propagate(one, wf[i:i + 1], tr_d, dz, 1)
        assert torch.equal(one[0], full[i])
    cat_d = [[torch.cat(fr)] for fr in tr_d]
    again = dev(torch, psi, torch.complex64)
    tc.propagate(again, wf, cat_d, dz, 1)
    assert torch.equal(again, full)
    tc.close()


@pytest.mark.parametrize("n", [256, 512])
def test_propagate_wave_tuples_with_odd_frame_runs(torch, B, oracle, n):
    """The row kernel transforms tuples of waves of one frame (pairs at 256^2 / 512^2); runs of odd length leave a
    short tuple that repeats its last wave.  Result vs the oracle, and bitwise equal to one wave at a time."""
    L, lam, dz = 12.0, 0.0370144, 1.4795
    trans, psi, _ = random_setup(21, n, n, 5, 2, [2])
    wf = np.array([0, 0, 0, 1, 1], dtype=np.int32)
    tc = B.Tacaw(n, n, L, L, lam, 9.2e-4, 1)
    tr_d = [[dev(torch, t, torch.complex64) for t in fr] for fr in trans]
    full = dev(torch, psi, torch.complex64)
    tc.propagate(full, wf, tr_d, dz, 1)
    ref = oracle.propagate(L, L, lam, 1, psi, wf, trans, dz, 1)
    got = full.cpu().numpy()
    for i in range(5):
        assert rel_l2(got[i], ref[i]) <= 2e-5
        one = dev(torch, psi[i:i + 1], torch.complex64)
        tc.propagate(one, wf[i:i + 1], tr_d, dz, 1)
        assert torch.equal(one[0], full[i])
    tc.close()


def test_propagate_l2_grouping_is_transparent(torch, B, monkeypatch):
    n, L, lam, dz = 128, 9.0, 0.0370144, 1.4795
    trans, psi, wf = random_setup(11, n, n, 9, 4, [3])
    tc = B.Tacaw(n, n, L, L, lam, 9.2e-4, 1)
    tr_d = [[dev(torch, t, torch.complex64) for t in fr] for fr in trans]
    a = dev(torch, psi, torch.complex64)
    tc.propagate(a, wf, tr_d, dz, 1)
    monkeypatch.setenv("TACAW_L2_GROUP_MB", str(2.5 * n * n * 8 / 1048576))     # groups of 2 waves
    b = dev(torch, psi, torch.complex64)
    tc.propagate(b, wf, tr_d, dz, 1)
    assert torch.equal(a, b)
    tc.close()


def test_error_codes(torch, B):
    tc = B.Tacaw(64, 64, 9.0, 9.0, 0.037, 9e-4, 1)
    w = torch.zeros((1, 64, 64), dtype=torch.complex64, device="cuda")
    t = torch.ones((1, 64, 64), dtype=torch.complex64, device="cuda")
    with pytest.raises(B.TacawError):
        tc.propagate(w, [3], [[t]], 1.0, 1)                    # frame index out of range
    with pytest.raises(B.TacawError):
        tc.propagate(w, [0], [[t]], -1.0, 1)                   # bad thickness
    with pytest.raises(B.TacawError):
        tc.spectrum(torch.zeros((1, 1000, 5), dtype=torch.complex64, device="cuda"), 5.0, 1, 300.0)   # neither 2^k nor <= 512
    empty = torch.zeros((0, 64, 64), dtype=torch.complex64, device="cuda")
    tc.propagate(empty, [], [[t]], 1.0, 1)                     # empty batch is a no-op
    tc.close()


# ----------------------------------------------------------------------- build_slices (K1, K2)
@pytest.mark.parametrize("case", ["tiny16", "c1", "c2", "rect"])
def test_build_slices_vs_oracle(torch, B, oracle, case):
    if case == "tiny16":
        wl = W.tiny_workload(n=16, ncell=(1, 1, 2))
    elif case == "c1":
        wl = W.make_workload(1)
    elif case == "c2":
        wl = W.make_workload(2)
    else:
        wl = W.tiny_workload(n=32, ncell=(2, 1, 1))
        wl.ny, wl.nx = 32, 64
    seg = wl.segments[0]
    pos = seg.frames(5, 6, wl.dt_fs)[0]
    ref = oracle.build_slices(wl.nx, wl.ny, wl.lx, wl.ly, pos, seg.species, wl.a, wl.b, wl.dz, seg.nslices, 0.0,
                              wl.sigma, wl.bandlimit, 1, want_v=True)
    tc = B.Tacaw(wl.nx, wl.ny, wl.lx, wl.ly, wl.lam, wl.sigma, wl.bandlimit)
    t, ncl = tc.build_slices(dev(torch, pos), dev(torch, seg.species), wl.a, wl.b, wl.dz, seg.nslices, 0.0,
                             want_clamped=True)
    got = t.cpu().numpy()
    assert ncl == ref["n_clamped"] == 0
    # |t| = 1 and the phase sigma*v agrees: compare t itself (absolute error = phase error)
    assert np.max(np.abs(np.abs(got) - 1.0)) <= 1e-6
    phase_scale = max(1.0, wl.sigma * np.abs(ref["v"]).max())
    for n in range(seg.nslices):
        assert rel_l2(got[n], ref["trans"][n]) <= 2e-6 * phase_scale, (case, n)
    tc.close()


def test_build_slices_batched_over_frames(torch, B, oracle):
    """One call for several frames == one call per frame == oracle."""
    wl = W.make_workload(1)
    seg = wl.segments[0]
    pos = seg.frames(0, 5, wl.dt_fs)
    tc = B.Tacaw(wl.nx, wl.ny, wl.lx, wl.ly, wl.lam, wl.sigma, 1)
    out = torch.full((5, seg.nslices, wl.ny, wl.nx), float("nan"), dtype=torch.complex64, device="cuda")
    tb, ncl = tc.build_slices(dev(torch, pos), dev(torch, seg.species), wl.a, wl.b, wl.dz, seg.nslices, 0.0, out=out,
                              want_clamped=True)
    assert ncl == 0
    for f in range(5):
        t1, _ = tc.build_slices(dev(torch, pos[f]), dev(torch, seg.species), wl.a, wl.b, wl.dz, seg.nslices, 0.0)
        assert torch.equal(tb[f], t1)
        ref = oracle.build_slices(wl.nx, wl.ny, wl.lx, wl.ly, pos[f], seg.species, wl.a, wl.b, wl.dz, seg.nslices, 0.0,
                                  wl.sigma, 1, 1)
        assert rel_l2(tb[f].cpu().numpy(), ref["trans"]) <= 1e-5
    tc.close()


def test_build_slices_clamps_and_counts(torch, B, oracle):
    wl = W.tiny_workload(n=32, ncell=(1, 1, 2))
    seg = wl.segments[0]
    pos = seg.pos0.copy()
    pos[0, 2] = -0.3
    pos[1, 2] = 100.0
    pos[2, 0] += 3 * wl.lx          # x outside the cell: periodic in x/y, never in z
    ref = oracle.build_slices(wl.nx, wl.ny, wl.lx, wl.ly, pos, seg.species, wl.a, wl.b, wl.dz, seg.nslices, 0.0,
                              wl.sigma, 1, 1)
    tc = B.Tacaw(wl.nx, wl.ny, wl.lx, wl.ly, wl.lam, wl.sigma, 1)
    t, ncl = tc.build_slices(dev(torch, pos), dev(torch, seg.species), wl.a, wl.b, wl.dz, seg.nslices, 0.0,
                             want_clamped=True)
    assert ncl == ref["n_clamped"] == 2
    assert rel_l2(t.cpu().numpy(), ref["trans"]) <= 1e-5
    # no atoms at all -> t = 1
    t0, n0 = tc.build_slices(dev(torch, pos[:0]), dev(torch, seg.species[:0]), wl.a, wl.b, wl.dz, 3, 0.0, want_clamped=True)
    assert n0 == 0 and torch.all(t0 == 1)
    tc.close()


# -------------------------------------------------------------------------------- probes (K3)
@pytest.mark.parametrize("n,alpha", [(64, 0.0), (64, 30e-3), (256, 30e-3), (32, 12e-3)])
def test_make_probes_vs_oracle(torch, B, oracle, n, alpha):
    L, lam = 0.14 * n, 0.0370144
    xy = np.array([[0.0, 0.0], [1.234, 5.678], [L - 0.01, 0.37 * L]])
    ref = oracle.make_probes(n, n, L, L, lam, xy, alpha)
    tc = B.Tacaw(n, n, L, L, lam, 9.2e-4, 1)
    got = tc.make_probes(xy, alpha).cpu().numpy()
    for p in range(3):
        assert rel_l2(got[p], ref[p]) <= 5e-6
        assert abs((np.abs(got[p]) ** 2).sum() - 1.0) <= 1e-5
    tc.close()


# ---------------------------------------------------------------------- accumulate + spectrum
def test_accumulate_vs_oracle(torch, B, oracle):
    n = 32
    rng = np.random.default_rng(0)
    q = rng.normal(size=(5, n, n)) + 1j * rng.normal(size=(5, n, n))
    roi = B.make_roi(n, n, 5.0, 5.0, 0.037, "disc", [0.05])
    wp = np.array([0, 1, 1, 0, 1], np.int32)
    wf = np.array([3, 0, 2, 1, 3], np.int32)
    ref = np.zeros((2, 4, roi.size), complex)
    oracle.accumulate(q, wp, wf, roi, ref)
    tc = B.Tacaw(n, n, 5.0, 5.0, 0.037, 9e-4, 1)
    buf = torch.zeros((2, 4, roi.size), dtype=torch.complex64, device="cuda")
    tc.accumulate(dev(torch, q, torch.complex64), wp, wf, dev(torch, roi), buf)
    got = buf.cpu().numpy()
    assert np.max(np.abs(got - ref)) <= 2e-7 * np.max(np.abs(ref))
    assert np.all(got[0, 0] == 0) and np.all(got[1, 1] == 0)          # untouched slots stay untouched
    tc.close()


@pytest.mark.parametrize("T", [8, 16, 32, 64, 128, 256, 512, 1024, 2048])
def test_spectrum_vs_oracle(torch, B, oracle, T):
    rng = np.random.default_rng(T)
    P, Q = 2, 37                                   # ragged Q: not a multiple of the tile width
    buf = rng.normal(size=(P, T, Q)) + 1j * rng.normal(size=(P, T, Q))
    buf[:, :, :5] += 30.0                          # strong elastic line on some pixels
    tc = B.Tacaw(16, 16, 5.0, 5.0, 0.037, 9e-4, 1)
    for window, (emin, emax) in ((1, (-np.inf, np.inf)), (0, (-60.0, 95.0))):
        Iref, Eref = oracle.spectrum(buf, 5.0, window, 300.0, emin, emax)
        I, E = tc.spectrum(dev(torch, buf, torch.complex64), 5.0, window, 300.0, emin, emax)
        assert np.array_equal(E, Eref)
        got = I.cpu().numpy()
        assert got.shape == Iref.shape
        for p in range(P):
            assert rel_l2(got[p], Iref[p]) <= 5e-6
        assert np.max(np.abs(got - Iref) / (Iref + 1e-3 * Iref.max())) <= 1e-3   # weak bins too
    tc.close()


@pytest.mark.parametrize("T", [5, 48, 200, 500])
def test_spectrum_generic_length_vs_oracle(torch, B, oracle, T):
    """Series whose length is not a power of two (the paper's chunks of 200 snapshots): plain DFT path."""
    rng = np.random.default_rng(T)
    P, Q = 2, 45                                   # ragged Q: not a multiple of the 32-series tile
    buf = rng.normal(size=(P, T, Q)) + 1j * rng.normal(size=(P, T, Q))
    buf[:, :, :4] += 20.0
    tc = B.Tacaw(16, 16, 5.0, 5.0, 0.037, 9e-4, 1)
    for window, (emin, emax) in ((1, (-np.inf, np.inf)), (0, (-70.0, 41.0))):
        Iref, Eref = oracle.spectrum(buf, 5.0, window, 300.0, emin, emax)
        I, E = tc.spectrum(dev(torch, buf, torch.complex64), 5.0, window, 300.0, emin, emax)
        assert np.array_equal(E, Eref)
        got = I.cpu().numpy()
        assert got.shape == Iref.shape
        for p in range(P):
            assert rel_l2(got[p], Iref[p]) <= 2e-5
    tc.close()


def test_welch_with_the_papers_chunk_parameters(torch, B, oracle):
    """chunks of 200 snapshots at 15 fs, nu = 2, Hann, E-ROI +-30 THz -> 1.4 meV sampling and 181 bins;
    here on 700 snapshots after a skip of 100 (5 chunks)."""
    rng = np.random.default_rng(200)
    P, Q, L = 1, 33, 200
    buf = rng.normal(size=(P, 700, Q)) + 1j * rng.normal(size=(P, 700, Q))
    buf[:, :, 0] += 10.0
    e30 = W.H_MEV_FS * 30e12 * 1e-15
    w = B.make_window("hann", L)
    ref, Eref, nref = oracle.spectrum_welch(buf, L, 2, 15.0, oracle.window_table("hann", L), 300.0, -e30, e30, skip_init=100)
    tc = B.Tacaw(16, 16, 5.0, 5.0, 0.037, 9e-4, 1)
    I, E, n = tc.spectrum_welch(dev(torch, buf, torch.complex64), L, 2, 15.0, w, 300.0, -e30, e30, skip_init=100)
    assert n == nref == 5 and E.size == 181 and np.array_equal(E, Eref) and round(E[1] - E[0], 1) == 1.4
    assert rel_l2(I.cpu().numpy()[0], ref[0]) <= 2e-5
    tc.close()


# --------------------------------------------------------------------- whole path, configs 1-5
def _exit_wave_parity(torch, oracle, wl, frames, probes=None):
    from oracle import pipeline as OP
    from paper_2607_02236_b200.pipeline import Runner
    r = Runner(wl, frames_per_block=1, probes=probes)
    got = r.exit_waves(frames, output_space=1).cpu().numpy()
    r.close()
    del r
    ref = OP.exit_waves(wl, frames, probes=probes, output_space=1)
    worst = 0.0
    for i in range(len(frames)):
        for p in range(got.shape[1]):
            worst = max(worst, rel_l2(got[i, p], ref[i, p]))
    return worst


def test_config1_full_parity(torch, B, oracle):
    """configs[0]: every frame's exit wave and the full spectrum."""
    from oracle import pipeline as OP
    from paper_2607_02236_b200.pipeline import Runner
    wl = W.make_workload(1)
    ref = OP.run(wl, pot_mode=0)
    r = Runner(wl)
    out = r.run()
    assert np.array_equal(out["roi"], ref["roi"]) and np.array_equal(out["E"], ref["E"])
    buf = out["buf"].cpu().numpy()
    for f in range(wl.nframes):
        assert rel_l2(buf[0, f], ref["buf"][0, f]) <= TOL_WAVE
    assert rel_l2(out["I"].cpu().numpy()[0], ref["I"][0]) <= TOL_SPEC
    # inelastic-only (|bin| > 2) relative L2, reported for information (looser, R2 in SURVEY.md)
    kp = np.round(ref["E"] / (W.H_MEV_FS / (wl.nframes * wl.dt_fs))).astype(int)
    m = np.abs(kp) > 2
    print("c1 inelastic rel-L2:", rel_l2(out["I"].cpu().numpy()[0][m], ref["I"][0][m]))
    r.close()


def test_config2_sampled_exit_waves(torch, B, oracle):
    wl = W.make_workload(2)
    assert _exit_wave_parity(torch, oracle, wl, [0, 101, 255]) <= TOL_WAVE


def test_config2_full_size_bench_launch_configuration(torch, B, oracle):
    """configs[1] at full size exactly as bench.py runs it (all 256 frames in one block, 1024 waves per
    tacaw_propagate call, batched build): sampled (probe, frame) rows of the time-ordered buffer against
    exit waves the oracle computes one by one; plus properties that hold at any size."""
    from oracle import pipeline as OP
    from paper_2607_02236_b200.pipeline import Runner
    wl = W.make_workload(2)
    r = Runner(wl)
    assert r.fpb == wl.nframes
    out = r.run()
    buf = out["buf"].cpu().numpy()
    frames = [7, 128, 254]
    ref = OP.exit_waves(wl, frames, output_space=1)
    for i, f in enumerate(frames):
        for p in range(wl.nprobes):
            want = ref[i, p].ravel()[out["roi"]] / np.sqrt(wl.nx * wl.ny)
            assert rel_l2(buf[p, f], want) <= TOL_WAVE, (p, f)
    I = out["I"].cpu().numpy()
    assert I.shape == (wl.nprobes, wl.nframes, out["roi"].size) and np.all(np.isfinite(I)) and np.all(I >= 0)
    # Parseval of the spectrum normalisation (oracle pin P10) holds for the GPU result at full size
    E = out["E"]
    kbt = W.KB_EV_K * 1e3 * wl.temperature_K
    bose = np.where(E == 0, 1.0, (E / kbt) / (-np.expm1(-E / kbt + (E == 0))))
    w = 0.5 - 0.5 * np.cos(2 * np.pi * np.arange(wl.nframes) / wl.nframes)
    for p in range(wl.nprobes):
        lhs = (I[p] / bose[:, None]).sum()
        rhs = ((w ** 2)[:, None] * np.abs(buf[p]) ** 2).sum() / (w ** 2).sum()
        assert abs(lhs - rhs) <= 2e-4 * rhs
    r.close()


def test_config2_reduced_T_spectrum(torch, B, oracle):
    """configs[1] with T' = 32 frames, all four probes, full ROI: spectra parity."""
    from oracle import pipeline as OP
    from paper_2607_02236_b200.pipeline import Runner
    wl = W.make_workload(2, nframes=32)
    ref = OP.run(wl)
    r = Runner(wl, frames_per_block=8)
    out = r.run()
    I = out["I"].cpu().numpy()
    for p in range(wl.nprobes):
        assert rel_l2(I[p], ref["I"][p]) <= TOL_SPEC
    r.close()


@pytest.mark.slow
def test_config3_sampled_exit_waves(torch, B, oracle):
    """configs[2] at full depth (200 slices): two (probe, frame) pairs through all slices."""
    wl = W.make_workload(3)
    assert _exit_wave_parity(torch, oracle, wl, [517], probes=[0, 137]) <= TOL_WAVE


def test_config3_thin_sampled(torch, B, oracle):
    wl = W.make_workload(3, ncz=6)
    assert _exit_wave_parity(torch, oracle, wl, [3, 900], probes=[0, 100, 255]) <= TOL_WAVE


def test_config4_thin_segments_sampled(torch, B, oracle):
    """configs[3] shape (1024^2, four chained z-segments with their own trajectories), 4 x 3 cells thick: 6 pairs."""
    wl = W.make_workload(4, ncz=3)
    assert wl.nslices_total == 24 and len(wl.segments) == 4
    assert _exit_wave_parity(torch, oracle, wl, [0, 700, 1023], probes=[0, 63]) <= TOL_WAVE


@pytest.mark.slow
def test_config4_full_depth_chained_segments(torch, B, oracle):
    """configs[3] as specified: 4 z-segments x 170 slices = 680 slices, each segment with its own 64-mode trajectory, the exit
    wave of one segment entering the next (PAPER.md:72-84, :231 'same timestep, frequency of storing'); 2 (probe, frame)
    pairs through all 680 slices."""
    wl = W.make_workload(4)
    assert wl.nslices_total == 680 and [s.nslices for s in wl.segments] == [170] * 4 and wl.natoms == 293760
    assert _exit_wave_parity(torch, oracle, wl, [311], probes=[9, 54]) <= TOL_WAVE


def test_config5_thin_sampled(torch, B, oracle):
    """configs[4] shape (2048^2, planar fault, annular ROI), 2 cells thick: 6 pairs."""
    wl = W.make_workload(5, ncz=2)
    assert _exit_wave_parity(torch, oracle, wl, [0, 1500], probes=[5, 500, 1023]) <= TOL_WAVE


@pytest.mark.slow
def test_config5_full_depth(torch, B, oracle):
    """configs[4] as specified: 24x24x60 cells with the planar fault, 120 slices at 2048^2; 2 (probe, frame) pairs."""
    wl = W.make_workload(5)
    assert wl.nslices_total == 120 and wl.natoms == 207360
    assert _exit_wave_parity(torch, oracle, wl, [1033], probes=[17, 1000]) <= TOL_WAVE


@pytest.mark.parametrize("cfg,ncz,probes", [(3, 4, [0, 255]), (4, 1, [0, 63]), (5, 1, [0, 1023])])
def test_configs_3_to_5_reduced_T_spectra(torch, B, oracle, cfg, ncz, probes):
    """spectra parity on a reduced-T variant of configs 3-5 (T' = 64 frames, 2 probes, the config's full
    q-ROI, its window and -- c5 -- its E-ROI of +-120 meV), thinned along z so the oracle finishes: I(q,E) rel-L2 <= 1e-3
    per probe, ROI map and energy axis identical."""
    from oracle import pipeline as OP
    from paper_2607_02236_b200.pipeline import Runner
    wl = W.make_workload(cfg, nframes=64, ncz=ncz)
    ref = OP.run(wl, probes=probes)
    r = Runner(wl, frames_per_block=8, probes=probes)
    out = r.run()
    assert np.array_equal(out["roi"], ref["roi"]) and np.array_equal(out["E"], ref["E"])
    I = out["I"].cpu().numpy()
    assert I.shape == ref["I"].shape
    if cfg == 5:
        assert np.all(np.abs(out["E"]) <= 120.0 + 1e-9) and out["E"].size < 64
    buf = out["buf"].cpu().numpy()
    for p in range(len(probes)):
        assert rel_l2(I[p], ref["I"][p]) <= TOL_SPEC, (cfg, p)
        for f in (0, 63):
            assert rel_l2(buf[p, f], ref["buf"][p, f]) <= TOL_WAVE
    r.close()


@pytest.mark.parametrize("n,nw,nframes,S", [(512, 44, 4, 3), (1024, 40, 3, 3)])
def test_propagate_multi_group_multi_stream_vs_oracle(torch, B, oracle, n, nw, nframes, S):
    """The path large grids take in production: >= 40 waves over several frames and slices, so that tacaw_propagate cuts them
    into several L2 groups and forks them onto its internal streams with the default group size.  8 sampled waves against
    the oracle; every wave bitwise against a one-wave-at-a-time run (no fork, one group)."""
    L, lam, dz = 0.09 * n, 0.0370144, 1.4795
    rng = np.random.default_rng(n + nw)
    trans = [[np.exp(1j * rng.normal(size=(S, n, n))).astype(np.complex64)] for _ in range(nframes)]
    psi = (rng.normal(size=(nw, n, n)) + 1j * rng.normal(size=(nw, n, n))).astype(np.complex64)
    psi /= np.sqrt((np.abs(psi) ** 2).sum(axis=(1, 2), keepdims=True))
    wf = np.sort(rng.integers(0, nframes, size=nw)).astype(np.int32)
    tc = B.Tacaw(n, n, L, L, lam, 9.2e-4, 1)
    tr_d = [[dev(torch, t[0], torch.complex64)] for t in trans]
    full = dev(torch, psi, torch.complex64)
    l0 = tc.launches
    tc.propagate(full, wf, tr_d, dz, 1)
    ngroups = (tc.launches - l0) // (2 * S)
    assert ngroups >= 3, ngroups                     # really several groups (three streams in flight)
    got = full.cpu().numpy()
    for i in range(nw):
        one = dev(torch, psi[i:i + 1], torch.complex64)
        tc.propagate(one, wf[i:i + 1], tr_d, dz, 1)
        assert torch.equal(one[0], full[i]), i
    sample = sorted(rng.choice(nw, size=8, replace=False).tolist())
    ref = oracle.propagate(L, L, lam, 1, psi[sample].astype(np.complex128), wf[sample],
                           [[t[0].astype(np.complex128)] for t in trans], dz, 1)
    for j, i in enumerate(sample):
        assert rel_l2(got[i], ref[j]) <= 2e-5, i
    tc.close()


@pytest.mark.parametrize("cfg,kw", [(2, dict(nframes=8)), (5, dict(nframes=8, ncz=1, nprobes=3)), (1, dict())])
def test_fused_gather_equals_propagate_plus_accumulate(torch, B, oracle, cfg, kw):
    """tacaw_propagate_accumulate (the last column kernel writes the ROI pixels) against the unfused pair on the same inputs:
    equal to fp32 rounding of one scale factor, untouched buffer slots stay untouched, ROI pixels outside the band limit are
    exact zeros."""
    from paper_2607_02236_b200.pipeline import Runner
    wl = W.make_workload(cfg, **kw)
    if cfg == 1:
        wl.roi_mode, wl.roi_params_mrad = "full", ()         # full q: most ROI pixels lie outside the band limit
    outs = []
    for fused in (False, True):
        r = Runner(wl, frames_per_block=3, fused_gather=fused)
        r.alloc_buffer(wl.nframes + 1)                       # one extra time slot that no wave writes
        r.buf[:, wl.nframes] = 7.0
        for f0 in range(0, wl.nframes, r.fpb):
            nf = min(r.fpb, wl.nframes - f0)
            r.run_block(r.upload_positions(f0, f0 + nf), f0, nf)
        outs.append(r.buf.cpu().numpy())
        roi = r.roi_h
        r.close()
    a, b = outs
    assert np.all(b[:, wl.nframes] == 7.0)
    for p in range(a.shape[0]):
        for f in range(wl.nframes):
            assert rel_l2(b[p, f], a[p, f]) <= 3e-7, (p, f)
    h = np.where(roi % wl.nx < wl.nx // 2, roi % wl.nx, roi % wl.nx - wl.nx)
    k = np.where(roi // wl.nx < wl.ny // 2, roi // wl.nx, roi // wl.nx - wl.ny)
    oob = 9 * (h.astype(np.int64) ** 2 + k.astype(np.int64) ** 2) > wl.nx * wl.nx
    assert np.all(b[:, :wl.nframes][:, :, oob] == 0)


def test_segment_reassembly_per_chunk(torch, B, oracle):
    """'for each averaging chunk ... construct the stacked supercell from randomly selected segments of that
    trajectory'.  Three stack positions drawn from one 40-snapshot trajectory for two chunks of 8 frames: the time-ordered
    buffers of both chunks against the oracle's re-assembled run, and their Welch-averaged spectrum."""
    from oracle import pipeline as OP
    from paper_2607_02236_b200.pipeline import run_reassembled
    wl = W.tiny_workload(n=32, ncell=(2, 2, 1), nframes=40, alpha_mrad=25.0)
    wl.roi_mode, wl.roi_params_mrad = "disc", (40.0,)
    off = W.segment_offsets(5, 2, 3, 40, 8)
    assert off.shape == (2, 3) and off.min() >= 0 and off.max() <= 32 and len(set(off.ravel().tolist())) > 1
    ref = OP.run_reassembled(wl, off, 8)
    got = run_reassembled(wl, off, 8).cpu().numpy()
    assert got.shape == ref.shape
    for i in range(2):
        for f in range(8):
            assert rel_l2(got[i, 0, f], ref[i, 0, f]) <= TOL_WAVE
    # Eq.(2): the chunk spectra are averaged; here chunk by chunk through tacaw_spectrum on the device
    tc = B.Tacaw(wl.nx, wl.ny, wl.lx, wl.ly, wl.lam, wl.sigma, 1)
    acc, accr = 0.0, 0.0
    for i in range(2):
        I, E = tc.spectrum(dev(torch, got[i], torch.complex64), wl.dt_fs, 1, wl.temperature_K)
        Ir, Er = oracle.spectrum(ref[i], wl.dt_fs, 1, wl.temperature_K)
        acc, accr = acc + I.cpu().numpy() / 2, accr + Ir / 2
    assert rel_l2(acc[0], accr[0]) <= TOL_SPEC
    tc.close()


# ------------------------------------------------------------------------ boundary: workspace, streams
def test_workspace_is_the_callers_and_too_small_is_nomem(torch, B):
    """every device buffer is the caller's.  Without a workspace, or with one sized for smaller calls, a
    call returns TACAW_E_NOMEM (-3) and queues nothing; tacaw_workspace_bytes grows with the announced sizes."""
    import ctypes as C
    n = 64
    tc = B.Tacaw(n, n, 9.0, 9.0, 0.037, 9e-4, 1)
    small = tc.workspace_bytes(nwaves=2, nframes=1, nsegments=1)
    big = tc.workspace_bytes(nwaves=4096, nframes=8, nsegments=4, natoms=10000, nslices=40)
    assert 0 < small < big
    w = torch.zeros((4, n, n), dtype=torch.complex64, device="cuda")
    t = torch.ones((1, n, n), dtype=torch.complex64, device="cuda")
    wf = np.zeros(4, np.int32)
    nsl = np.array([1], np.int32)
    ptrs = (C.c_void_p * 1)(t.data_ptr())

    def raw_propagate(nw):
        return tc.lib.tacaw_propagate(tc._ctx, C.c_void_p(w.data_ptr()), None, C.c_int(0), None, wf.ctypes.data_as(C.c_void_p),
                                      C.c_int(nw), ptrs, C.c_int(1), nsl.ctypes.data_as(C.c_void_p), C.c_int(1),
                                      C.c_double(1.0), C.c_int(1), tc._stream())
    l0 = tc.launches
    assert raw_propagate(4) == -3 and b"workspace" in tc.lib.tacaw_last_error(tc._ctx)       # none set
    ws = torch.empty(small + 256, dtype=torch.uint8, device="cuda")
    off = (-ws.data_ptr()) % 256
    tc.set_workspace(ws[off:off + small], nwaves=2, nframes=1, nsegments=1)
    assert raw_propagate(2) == 0
    # (4 waves may still fit the 256-byte rounding of the region ...
    wbig = np.zeros(4000, np.int32)
    rc = tc.lib.tacaw_propagate(tc._ctx, C.c_void_p(w.data_ptr()), None, C.c_int(0), None, wbig.ctypes.data_as(C.c_void_p),
                                C.c_int(4000), ptrs, C.c_int(1), nsl.ctypes.data_as(C.c_void_p), C.c_int(1), C.c_double(1.0),
                                C.c_int(1), tc._stream())
    assert rc == -3                                              #  ... 4000 cannot)
    with pytest.raises(B.TacawError):
        tc.set_workspace(ws[off:off + 1024], nwaves=4096, nframes=8)   # fewer bytes than the sizes need
    with pytest.raises(B.TacawError):
        tc.set_workspace(ws[off + 8:off + 8 + small], nwaves=2, nframes=1)    # not 256-byte aligned
    torch.cuda.synchronize()
    assert tc.launches - l0 >= 2
    tc.close()


def test_bad_species_id_is_reported(torch, B):
    wl = W.tiny_workload(n=32, ncell=(1, 1, 2))
    seg = wl.segments[0]
    tc = B.Tacaw(wl.nx, wl.ny, wl.lx, wl.ly, wl.lam, wl.sigma, 1)
    sp = seg.species.copy()
    sp[3] = 7                                         # two species only
    with pytest.raises(B.TacawError):                 # synchronising variant reports at once
        tc.build_slices(dev(torch, seg.pos0), dev(torch, sp), wl.a, wl.b, wl.dz, seg.nslices, 0.0, want_clamped=True)
    tc.build_slices(dev(torch, seg.pos0), dev(torch, sp), wl.a, wl.b, wl.dz, seg.nslices, 0.0)      # asynchronous: sticky flag
    with pytest.raises(B.TacawError):
        tc.device_status()
    tc.device_status()                                # cleared by the report
    out = torch.empty((seg.nslices, wl.ny, wl.nx), dtype=torch.complex64, device="cuda")
    with pytest.raises(B.TacawError):                 # host variant validates before queueing anything
        tc.build_slices_host(seg.pos0, sp, wl.a, wl.b, wl.dz, seg.nslices, 0.0, out)
    tc.close()


def test_two_contexts_overlap_build_and_propagate_on_two_streams(torch, B, oracle):
    """tacaw.h: one stream at a time per context; overlap needs two contexts.  Context A builds the transmissions of the
    next frame on stream 1 while context B propagates the current frame on stream 2 (event-ordered hand-over); results equal
    the serial single-stream run bit for bit."""
    wl = W.make_workload(2, nframes=6)
    seg = wl.segments[0]
    pos = dev(torch, seg.frames(0, 6, wl.dt_fs))
    sp = dev(torch, seg.species)
    tA = B.Tacaw(wl.nx, wl.ny, wl.lx, wl.ly, wl.lam, wl.sigma, 1)
    tB = B.Tacaw(wl.nx, wl.ny, wl.lx, wl.ly, wl.lam, wl.sigma, 1)
    probes = tB.make_probes(wl.probes_xy, wl.alpha_mrad * 1e-3)
    P = wl.nprobes
    wp = np.arange(P, dtype=np.int32)
    # serial reference
    serial = []
    for f in range(6):
        t, _ = tA.build_slices(pos[f], sp, wl.a, wl.b, wl.dz, seg.nslices, 0.0)
        w = torch.empty((P, wl.ny, wl.nx), dtype=torch.complex64, device="cuda")
        tB.propagate(w, np.zeros(P, np.int32), [[t]], wl.dz, 1, probes=probes, wave_probe=wp)
        serial.append(w)
    torch.cuda.synchronize()
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    tbuf = [torch.empty((seg.nslices, wl.ny, wl.nx), dtype=torch.complex64, device="cuda") for _ in range(2)]
    built = [torch.cuda.Event() for _ in range(6)]
    used = [torch.cuda.Event() for _ in range(6)]
    outs = [torch.empty((P, wl.ny, wl.nx), dtype=torch.complex64, device="cuda") for _ in range(6)]
    for f in range(6):
        with torch.cuda.stream(s1):
            if f >= 2:
                s1.wait_event(used[f - 2])            # the buffer's previous frame has been propagated
            tA.build_slices(pos[f], sp, wl.a, wl.b, wl.dz, seg.nslices, 0.0, out=tbuf[f % 2])
            built[f].record(s1)
        with torch.cuda.stream(s2):
            s2.wait_event(built[f])
            tB.propagate(outs[f], np.zeros(P, np.int32), [[tbuf[f % 2]]], wl.dz, 1, probes=probes, wave_probe=wp)
            used[f].record(s2)
    torch.cuda.synchronize()
    for f in range(6):
        assert torch.equal(outs[f], serial[f]), f
    tA.close(); tB.close()


# ------------------------------------------------------------------- degenerate and empty inputs
def test_free_space_is_analytic_fresnel_on_the_gpu(torch, B, oracle):
    """No atoms: t = 1 and S slice steps must give FFT2(psi_S) = Psi_0 exp(-i pi lambda S dz q^2) inside the mask, 0 outside
    (DESIGN.md pin P1a, here for the CUDA path itself and against the oracle)."""
    n, L, lam, dz, S = 128, 18.376, 0.0370144, 1.4795, 7
    tc = B.Tacaw(n, n, L, L, lam, 9.2e-4, 1)
    a = np.array([[100.0, 50.0, 20.0, 5.0]])
    b = np.array([[0.3, 1.0, 3.0, 8.0]])
    pos = torch.zeros((0, 3), dtype=torch.float64, device="cuda")
    sp = torch.zeros((0,), dtype=torch.int32, device="cuda")
    t, ncl = tc.build_slices(pos, sp, a, b, dz, S, 0.0, want_clamped=True)
    assert ncl == 0 and torch.all(t == 1)
    xy = np.array([[3.1, 7.7], [0.0, 0.0]])
    psi0 = tc.make_probes(xy, 30e-3)
    q0 = torch.fft.fft2(psi0).cpu().numpy().astype(np.complex128)          # library FFT: test-side check only
    waves = psi0.clone()
    tc.propagate(waves, [0, 0], [[t]], dz, 1)
    got = waves.cpu().numpy().astype(np.complex128)
    h = np.fft.fftfreq(n, 1.0 / n)
    hh, kk = np.meshgrid(h, h, indexing="xy")
    q2 = (hh ** 2 + kk ** 2) / L ** 2
    mask = 9 * (hh ** 2 + kk ** 2) <= n * n
    expect = q0 * np.exp(-1j * np.pi * lam * S * dz * q2) * mask
    ref = oracle.propagate(L, L, lam, 1, psi0.cpu().numpy().astype(np.complex128), np.array([0, 0], np.int32),
                           [[np.ones((S, n, n), complex)]], dz, 1)
    for p in range(2):
        assert rel_l2(got[p], expect[p]) <= 2e-5
        assert rel_l2(got[p], ref[p]) <= 2e-5
        assert np.all(got[p][~mask] == 0)
    tc.close()


def test_empty_slice_between_occupied_ones(torch, B, oracle):
    """A slice that holds no atom has t_n = 1 exactly; its neighbours are unaffected."""
    wl = W.tiny_workload(n=32, ncell=(1, 1, 2))
    seg = wl.segments[0]
    pos = seg.pos0.copy()
    pos[:, 2] = np.where(pos[:, 2] < 2.0 * wl.dz, 0.5 * wl.dz, 2.5 * wl.dz)     # slices 0 and 2 occupied, 1 and 3 empty
    ref = oracle.build_slices(wl.nx, wl.ny, wl.lx, wl.ly, pos, seg.species, wl.a, wl.b, wl.dz, 4, 0.0, wl.sigma, 1, 1)
    tc = B.Tacaw(wl.nx, wl.ny, wl.lx, wl.ly, wl.lam, wl.sigma, 1)
    t, ncl = tc.build_slices(dev(torch, pos), dev(torch, seg.species), wl.a, wl.b, wl.dz, 4, 0.0, want_clamped=True)
    assert ncl == 0
    assert torch.all(t[1] == 1) and torch.all(t[3] == 1)
    assert rel_l2(t.cpu().numpy(), ref["trans"]) <= 1e-5
    tc.close()


def test_empty_batches_are_no_ops(torch, B):
    n = 32
    tc = B.Tacaw(n, n, 5.0, 5.0, 0.037, 9e-4, 1)
    roi = B.make_roi(n, n, 5.0, 5.0, 0.037, "disc", [0.05])
    q = torch.randn((2, n, n), dtype=torch.complex64, device="cuda")
    buf = torch.full((1, 2, roi.size), 7.0, dtype=torch.complex64, device="cuda")
    tc.accumulate(q[:0], [], [], dev(torch, roi), buf)                           # no waves
    assert torch.all(buf == 7.0)
    empty_roi = torch.zeros((0,), dtype=torch.int32, device="cuda")
    buf0 = torch.zeros((1, 2, 0), dtype=torch.complex64, device="cuda")
    tc.accumulate(q, [0, 0], [0, 1], empty_roi, buf0)                            # empty ROI
    I, E = tc.spectrum(torch.zeros((0, 16, 5), dtype=torch.complex64, device="cuda"), 5.0, 1, 300.0)   # no probes
    assert I.shape == (0, 16, 5) and E.size == 16
    I, E = tc.spectrum(torch.zeros((2, 16, 0), dtype=torch.complex64, device="cuda"), 5.0, 1, 300.0)   # no pixels
    assert I.shape == (2, 16, 0)
    assert tc.make_probes(np.zeros((0, 2)), 30e-3).shape == (0, n, n)
    torch.cuda.synchronize()
    tc.close()


def test_single_series_single_pixel_spectrum(torch, B, oracle):
    """P = Q = 1: one series alone in its tile; a pure tone on a bin gives one line scaled by the Bose factor."""
    T, dt = 64, 5.0
    f = np.arange(T)
    buf = (np.exp(2j * np.pi * 5 * f / T) + 0.25 * np.exp(-2j * np.pi * 9 * f / T)).reshape(1, T, 1)
    tc = B.Tacaw(16, 16, 5.0, 5.0, 0.037, 9e-4, 1)
    I, E = tc.spectrum(dev(torch, buf, torch.complex64), dt, 0, 300.0)
    Iref, Eref = oracle.spectrum(buf, dt, 0, 300.0)
    got = I.cpu().numpy()
    assert np.array_equal(E, Eref) and rel_l2(got, Iref) <= 5e-6
    top = np.argsort(got[0, :, 0])[-2:]
    assert sorted(top.tolist()) == sorted([T // 2 + 5, T // 2 - 9])
    tc.close()


def test_guard_bands_around_every_buffer_stay_untouched(torch, B):
    """Bounds check of our own (compute-sanitizer is closed on this pool): every device buffer the path writes -- the
    workspace, transmissions, probes, waves, the time-ordered buffer, I(q,E) -- sits between two 1 MiB guard bands filled
    with a byte pattern; after the whole path (8 frames so that the 2^k spectrum kernel runs, then 5 for the generic DFT)
    every guard byte is unchanged, and the results equal those of a run on plain allocations bit for bit."""
    G = 1 << 20
    wl = W.make_workload(1, nframes=8)
    seg = wl.segments[0]
    P, S, n = wl.nprobes, seg.nslices, wl.nx
    roi = B.make_roi(wl.nx, wl.ny, wl.lx, wl.ly, wl.lam, wl.roi_mode, [p * 1e-3 for p in wl.roi_params_mrad])
    Q = int(roi.size)
    sizes = dict(natoms=seg.pos0.shape[0], nframes=8, nslices=S, nsegments=1, nwaves=8 * P, nprobes=P, host_staging=1)
    guarded = []

    def guard(nbytes):
        nb = (nbytes + 255) // 256 * 256
        t = torch.full((nb + 2 * G,), 0xA5, dtype=torch.uint8, device="cuda")
        assert t.data_ptr() % 256 == 0
        guarded.append((t, nb))
        return t[G:G + nb]

    def cplx(shape, guarded_alloc):
        numel = int(np.prod(shape))
        if guarded_alloc:
            return guard(numel * 8)[:numel * 8].view(torch.complex64).view(shape)
        return torch.empty(shape, dtype=torch.complex64, device="cuda")

    results = []
    for use_guards in (True, False):
        tc = B.Tacaw(wl.nx, wl.ny, wl.lx, wl.ly, wl.lam, wl.sigma, wl.bandlimit)
        nws = tc.workspace_bytes(**sizes)
        ws = guard(nws)[:nws] if use_guards else torch.empty(nws, dtype=torch.uint8, device="cuda")
        tc.set_workspace(ws, **sizes)
        trans = cplx((8, S, n, n), use_guards)
        probes = cplx((P, n, n), use_guards)
        waves = cplx((8 * P, n, n), use_guards)
        buf = cplx((P, 8, Q), use_guards)
        buf.zero_()
        I = (guard(P * 8 * Q * 4)[:P * 8 * Q * 4].view(torch.float32) if use_guards
             else torch.empty(P * 8 * Q, dtype=torch.float32, device="cuda")).view(P, 8, Q)
        pos = dev(torch, seg.frames(0, 8, wl.dt_fs))
        tc.build_slices_host(seg.frames(0, 8, wl.dt_fs), seg.species, wl.a, wl.b, wl.dz, S, 0.0, trans, want_clamped=False)
        t2 = torch.empty_like(trans)
        tc.build_slices(pos, dev(torch, seg.species), wl.a, wl.b, wl.dz, S, 0.0, out=t2)
        assert torch.equal(t2, trans)
        tc.make_probes(wl.probes_xy, wl.alpha_mrad * 1e-3, out=probes)
        roi_d = dev(torch, roi)
        inv = tc.make_roi_inverse(roi_d)
        wf = np.repeat(np.arange(8, dtype=np.int32), P)
        wp = np.tile(np.arange(P, dtype=np.int32), 8)
        tr = [[trans[f]] for f in range(8)]
        tc.propagate_accumulate(waves, wp, wf, wf, tr, wl.dz, inv, Q, buf, probes=probes)
        tc.propagate(waves, wf, tr, wl.dz, 1, probes=probes, wave_probe=wp)          # unfused pair into the same buffer
        tc.accumulate(waves, wp, wf, roi_d, buf)
        Iout, E = tc.spectrum(buf, wl.dt_fs, 1, wl.temperature_K, out=I)
        I5, _ = tc.spectrum(buf[:, :5].contiguous(), wl.dt_fs, 1, wl.temperature_K)
        torch.cuda.synchronize()
        tc.device_status()
        results.append((trans.clone(), buf.clone(), Iout.clone(), I5.clone()))
        tc.close()
    for t, nb in guarded:
        assert bool((t[:G] == 0xA5).all()) and bool((t[G + nb:] == 0xA5).all())
    for a, b in zip(*results):
        assert torch.equal(a, b)
