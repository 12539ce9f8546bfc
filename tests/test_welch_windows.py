"""Welch chunk averaging (Eq.(2) :126) and the further window
functions (:170-182).  Pins of the oracle against scipy's library routines and closed forms (CPU), the host window
generator of the library against the oracle (CPU, no GPU compute), and GPU parity of tacaw_spectrum_welch."""
import os

import numpy as np
import pytest

H_MEV_FS = 4135.667696
KB_MEV = 8.617333262e-2


def rel_l2(a, b):
    return float(np.linalg.norm(np.asarray(a, dtype=np.complex128) - b) / max(np.linalg.norm(b), 1e-300))


def series(rng, P, T, Q):
    return rng.normal(size=(P, T, Q)) + 1j * rng.normal(size=(P, T, Q))


# ------------------------------------------------------------------------------------- oracle pins (CPU)
def test_w1_tukey_limits_are_hann_and_rect(oracle):
    """'Hann window can then be introduced as a special case of Tukey window ... with alpha = 1';
    no taper at all is the rectangular window."""
    for n in (8, 64, 1000):
        assert np.max(np.abs(oracle.window_table("tukey", n, 1.0) - oracle.window(1, n))) <= 1e-15
        assert np.array_equal(oracle.window_table("tukey", n, 0.0), np.ones(n))
        assert np.max(np.abs(oracle.window_table("hann", n) - oracle.window(1, n))) <= 1e-15
        assert np.array_equal(oracle.window_table("rect", n), oracle.window(0, n))


@pytest.mark.parametrize("n", [16, 256, 1024])
def test_w2_windows_match_scipy_periodic_forms(oracle, n):
    """Library routines (scipy.signal.windows, sym=False = periodic / 'fftbins') as the independent definition."""
    sw = pytest.importorskip("scipy.signal.windows")
    assert np.max(np.abs(oracle.window_table("hann", n) - sw.hann(n, sym=False))) <= 1e-14
    assert np.max(np.abs(oracle.window_table("blackman_harris", n) - sw.blackmanharris(n, sym=False))) <= 1e-14
    for a in (0.1, 0.5, 1.0):
        assert np.max(np.abs(oracle.window_table("tukey", n, a) - sw.tukey(n, a, sym=False))) <= 1e-13
    for beta in (0.0, 3 * np.pi, 5 * np.pi):
        assert np.max(np.abs(oracle.window_table("kaiser", n, beta) - sw.kaiser(n, beta, sym=False))) <= 1e-12


def test_w3_closed_form_values(oracle):
    n = 64
    bh = oracle.window_table("blackman_harris", n)
    assert abs(bh[0] - (0.35875 - 0.48829 + 0.14128 - 0.01168)) <= 1e-16      # 6e-5: -92 dB skirts
    assert abs(bh[n // 2] - 1.0) <= 1e-15                                       # the coefficients sum to one
    k = oracle.window_table("kaiser", n, 7.0)
    assert abs(k[n // 2] - 1.0) <= 1e-15 and abs(k[0] - 1.0 / np.i0(7.0)) <= 1e-15
    for kind, par in (("blackman_harris", 0.0), ("kaiser", 7.0), ("tukey", 0.3)):
        w = oracle.window_table(kind, n, par)
        assert np.max(np.abs(w[1:] - w[1:][::-1])) <= 1e-14                     # periodic form: w[f] = w[n-f]


def test_w4_chunk_starts_follow_the_paper_rule(oracle):
    """s_{n+1} = s_n + L/nu with remainder-less division, default nu = 2; complete chunks only."""
    assert oracle.chunk_starts(40, 16, 2) == [0, 8, 16, 24]
    assert oracle.chunk_starts(40, 16, 3) == [0, 5, 10, 15, 20]
    assert oracle.chunk_starts(16, 16, 2) == [0]
    assert oracle.chunk_starts(15, 16, 2) == []
    assert oracle.chunk_starts(1024 + 512, 1024, 1) == [0]


def golden():
    out = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "paper_worked_numbers.txt")) as fh:
        for line in fh:
            if line.startswith("#") or "|" not in line:
                continue
            k, v, _ = [t.strip() for t in line.split("|", 2)]
            out[k] = v
    return out


def test_w4b_the_papers_31_chunks(oracle):
    """a 51 ps trajectory stored every 15 fs (3400 snapshots), the first 3 ps (200 snapshots, Listing 1
    :443 trajectory_chunks_skip_init) discarded, chunks of 200 with nu = 2 -> 'an average over 31 chunks'."""
    g = golden()
    nsnap = round(51e3 / 15.0)
    skip = int(g["welch_skip_init_listing1"])
    assert skip == round(3e3 / 15.0)
    st = oracle.chunk_starts(nsnap, 200, 2, skip_init=skip)
    assert len(st) == int(g["welch_chunks_51ps_minus_3ps_15fs_L200_nu2"])
    assert st[0] == skip and st[1] - st[0] == 100 and st[-1] + 200 == nsnap
    # the same 48 ps without the thermalisation period in the file
    assert len(oracle.chunk_starts(nsnap - skip, 200, 2)) == 31


def test_w4c_stride_and_skip(oracle):
    """Snapshot stride (:140): chunk n holds snapshots s_n, s_n + stride, ...; complete chunks only."""
    assert oracle.chunk_starts(40, 8, 2, skip_init=3, stride=2) == [3, 11, 19]          # 3 + 7*2 = 17 <= 39, ..., 19 + 14 = 33; 27 + 14 = 41 > 39
    assert oracle.chunk_starts(40, 8, 2, stride=1) == oracle.chunk_starts(40, 8, 2)
    assert oracle.chunk_starts(16, 8, 1, stride=2) == [0]
    assert oracle.chunk_starts(15, 8, 1, stride=2) == [0]
    assert oracle.chunk_starts(14, 8, 1, stride=2) == []
    # a strided Welch average equals the plain one on the decimated series with time step stride*dt
    rng = np.random.default_rng(11)
    buf = series(rng, 2, 48, 3)
    w = oracle.window_table("hann", 8)
    I1, E1, n1 = oracle.spectrum_welch(buf, 8, 2, 5.0, w, 300.0, skip_init=4, stride=3)
    I2, E2, n2 = oracle.spectrum_welch(np.ascontiguousarray(buf[:, 4::3]), 8, 2, 15.0, w, 300.0)
    # decimated series: starts every 4 decimated snapshots = 12 stored ones, same as (L/nu)*stride
    assert n1 == n2 and np.array_equal(E1, E2) and np.max(np.abs(I1 - I2)) <= 1e-14 * np.max(I2)


def test_w8_dolph_chebyshev_100dB(oracle):
    """'the Dolph-Chebyshev window with attenuation 100 dB ... See scipy and its documentation'.
    (a) against scipy.signal.windows.chebwin in its periodic form; (b) the defining property, checked without scipy:
    every side lobe of the symmetric window's transform sits 100 dB below the main lobe (equiripple)."""
    import scipy.signal.windows as sw
    att = float(golden()["chebwin_attenuation_dB"])
    for n in (16, 17, 200, 256, 1024):
        assert np.max(np.abs(oracle.window_table("dolph_chebyshev", n, att) - sw.chebwin(n, at=att, sym=False))) <= 2e-13
    M = 65
    w = np.append(oracle.dolph_chebyshev(M - 1, att), 0.0)
    w[-1] = w[0]                                              # symmetric window of M points (periodic form + last sample)
    Wf = np.abs(np.fft.fft(w, 64 * M))
    Wf /= Wf[0]
    # main-lobe edge: first point where the response has fallen to the ripple level
    lvl = 10.0 ** (-att / 20.0)
    first = int(np.argmax(Wf < lvl * 1.0001))
    side = Wf[first: Wf.size - first]
    assert side.max() <= lvl * 1.001 and side.max() >= lvl * 0.98      # equiripple at exactly -100 dB


def test_w5_single_chunk_is_the_plain_spectrum(oracle):
    rng = np.random.default_rng(3)
    buf = series(rng, 2, 32, 5)
    I0, E0 = oracle.spectrum(buf, 5.0, 1, 300.0)
    I1, E1, n = oracle.spectrum_welch(buf, 32, 1, 5.0, oracle.window_table("hann", 32), 300.0)
    assert n == 1 and np.array_equal(E0, E1) and np.max(np.abs(I0 - I1)) <= 1e-15 * np.max(I0)


@pytest.mark.parametrize("kind,par,nu", [("hann", 0.0, 2), ("tukey", 0.25, 4), ("blackman_harris", 0.0, 2), ("rect", 0.0, 1)])
def test_w6_welch_matches_scipy_welch(oracle, kind, par, nu):
    """scipy.signal.welch (library routine) on the complex series: density scaling |X|^2/(fs sum w^2) averaged over
    segments stepping L - noverlap = L/nu; I/B must equal density * fs / L."""
    sig = pytest.importorskip("scipy.signal")
    rng = np.random.default_rng(11)
    L, Ttot, dt = 64, 64 * 3 + 17, 4.0
    buf = series(rng, 1, Ttot, 3)
    w = oracle.window_table(kind, L, par)
    I, E, n = oracle.spectrum_welch(buf, L, nu, dt, w, 300.0)
    assert n == len(range(0, Ttot - L + 1, L // nu))
    B = np.array([oracle.bose(e / (KB_MEV * 300.0)) for e in E])
    for q in range(3):
        f, pxx = sig.welch(buf[0, :, q], fs=1.0, window=w, nperseg=L, noverlap=L - L // nu, nfft=L, detrend=False,
                           return_onesided=False, scaling="density")
        order = np.argsort(np.fft.fftshift(np.fft.fftfreq(L)))          # ascending k' = -L/2 .. L/2-1
        ref = np.fft.fftshift(pxx)[order] / L
        assert np.max(np.abs(I[0, :, q] / B - ref)) <= 1e-12 * np.max(ref)
    assert np.max(np.abs(E - H_MEV_FS * np.arange(-L // 2, L // 2) / (L * dt))) <= 1e-9


def test_w7_stationary_on_bin_mode_every_chunk_alike(oracle):
    """A mode exactly on a chunk bin and a static part: every chunk has the same |Phi|^2, so the Welch average
    equals the spectrum of the first chunk, with the loss peak on its bin (P5 carried to chunks)."""
    L, nchunk, dt, m0 = 64, 5, 5.0, 7
    t = np.arange(L * nchunk)
    buf = (1.0 + 0.05 * np.exp(-2j * np.pi * m0 * t / L))[None, :, None] * np.ones((1, 1, 2))
    w = oracle.window_table("hann", L)
    I, E, n = oracle.spectrum_welch(buf, L, 2, dt, w, 300.0)
    I1, _ = oracle.spectrum_table(buf, 0, L, dt, w, 300.0)
    assert n == 2 * nchunk - 1
    assert np.max(np.abs(I - I1)) <= 1e-12 * np.max(I1)
    inel = I[0, :, 0].copy()
    inel[L // 2 - 1:L // 2 + 2] = 0                                       # elastic line and its Hann neighbours
    assert np.argmax(inel) == L // 2 - m0                                 # exp(-i w t) under the forward DFT: bin -m0


# ------------------------------------------------------------------- library host function vs oracle (CPU)
@pytest.mark.parametrize("kind,par", [("rect", 0.0), ("hann", 0.0), ("tukey", 0.0), ("tukey", 0.1), ("tukey", 1.0),
                                      ("blackman_harris", 0.0), ("kaiser", 0.0), ("kaiser", 3 * np.pi), ("kaiser", 5 * np.pi),
                                      ("dolph_chebyshev", 100.0), ("dolph_chebyshev", 60.0)])
def test_make_window_host_matches_oracle(oracle, kind, par):
    from paper_2607_02236_b200 import binding, build
    build.build_lib()
    # Dolph-Chebyshev: the oracle evaluates cos() of angles up to ~2 pi n/2 (1 ulp of the angle ~ 1e-12 at n = 2048), the
    # library reduces the angle in integers first; both agree with scipy to their own rounding
    tol = 1e-12 if kind == "dolph_chebyshev" else 2e-13
    for n in (8, 100, 2048):
        assert np.max(np.abs(binding.make_window(kind, n, par) - oracle.window_table(kind, n, par))) <= tol
    with pytest.raises(binding.TacawError):
        binding.make_window("tukey", 16, 1.5)
    with pytest.raises(binding.TacawError):
        binding.make_window("dolph_chebyshev", 16, -3.0)


# ------------------------------------------------------------------------------------------- GPU parity
@pytest.mark.gpu
@pytest.mark.parametrize("L,nu,kind,par", [(8, 1, "rect", 0.0), (64, 2, "hann", 0.0), (64, 4, "tukey", 0.1),
                                           (256, 2, "blackman_harris", 0.0), (1024, 2, "kaiser", 3 * np.pi),
                                           (2048, 3, "hann", 0.0)])
def test_spectrum_welch_vs_oracle(oracle, L, nu, kind, par):
    import torch
    from paper_2607_02236_b200 import binding, build
    build.build_lib()
    rng = np.random.default_rng(L + nu)
    P, Q = 2, 37
    Ttot = 3 * L + L // 3
    buf = series(rng, P, Ttot, Q)
    buf[:, :, 0] += 5.0                                                  # a strong static (elastic) component
    w = binding.make_window(kind, L, par)
    dt, TK = 5.0, 300.0
    span = H_MEV_FS / (2 * dt)
    for emin, emax in ((-np.inf, np.inf), (-0.31 * span, 0.5 * span)):
        ref, Eref, nref = oracle.spectrum_welch(buf, L, nu, dt, oracle.window_table(kind, L, par), TK, emin, emax)
        tc = binding.Tacaw(16, 16, 5.0, 5.0, 0.037, 9e-4, 1)
        I, E, n = tc.spectrum_welch(torch.from_numpy(buf).to("cuda", torch.complex64), L, nu, dt, w, TK, emin, emax)
        assert n == nref and np.array_equal(E, Eref)
        got = I.cpu().numpy()
        for p in range(P):
            assert rel_l2(got[p], ref[p]) <= 5e-6                        # north_star bar for spectra: 1e-3
        assert np.max(np.abs(got - ref)) <= 1e-3 * np.max(ref)
        tc.close()


@pytest.mark.gpu
@pytest.mark.parametrize("L,nu,skip,stride,kind,par", [(64, 2, 5, 1, "hann", 0.0), (32, 2, 0, 3, "dolph_chebyshev", 100.0),
                                                     (512, 2, 7, 2, "hann", 0.0), (16, 4, 200, 1, "rect", 0.0)])
def test_spectrum_welch_skip_init_and_stride_vs_oracle(oracle, L, nu, skip, stride, kind, par):
    """trajectory_chunks_skip_init (Listing 1 :443) and the snapshot stride (:140) in tacaw_spectrum_welch."""
    import torch
    from paper_2607_02236_b200 import binding, build
    build.build_lib()
    rng = np.random.default_rng(L + skip + stride)
    P, Q = 2, 21
    Ttot = skip + stride * (3 * L + 5)
    buf = series(rng, P, Ttot, Q)
    buf[:, :, 1] += 4.0
    w = binding.make_window(kind, L, par)
    ref, Eref, nref = oracle.spectrum_welch(buf, L, nu, 5.0, oracle.window_table(kind, L, par), 300.0, skip_init=skip, stride=stride)
    tc = binding.Tacaw(16, 16, 5.0, 5.0, 0.037, 9e-4, 1)
    I, E, n = tc.spectrum_welch(torch.from_numpy(buf).to("cuda", torch.complex64), L, nu, 5.0, w, 300.0, skip_init=skip, stride=stride)
    assert n == nref and n >= 3 and np.array_equal(E, Eref)
    got = I.cpu().numpy()
    for p in range(P):
        assert rel_l2(got[p], ref[p]) <= 5e-6
    tc.close()


@pytest.mark.gpu
def test_spectrum_welch_edge_cases(oracle):
    import torch
    from paper_2607_02236_b200 import binding, build
    build.build_lib()
    tc = binding.Tacaw(16, 16, 5.0, 5.0, 0.037, 9e-4, 1)
    rng = np.random.default_rng(0)
    buf = torch.from_numpy(series(rng, 1, 12, 4)).to("cuda", torch.complex64)
    w = binding.make_window("hann", 16)
    I, E, n = tc.spectrum_welch(buf, 16, 2, 5.0, w, 300.0)              # shorter than one chunk: nothing to average
    assert n == 0 and E.size == 16 and torch.all(I == 0)
    with pytest.raises(binding.TacawError):
        tc.spectrum_welch(buf, 600, 2, 5.0, np.ones(600), 300.0)        # neither a power of two nor <= 512
    with pytest.raises(binding.TacawError):
        tc.spectrum_welch(buf, 8, 0, 5.0, np.ones(8), 300.0)
    with pytest.raises(binding.TacawError):
        tc.spectrum_welch(buf, 8, 2, 5.0, np.zeros(8), 300.0)           # identically zero window
    # one chunk, Hann: identical to tacaw_spectrum
    buf2 = torch.from_numpy(series(rng, 2, 32, 9)).to("cuda", torch.complex64)
    a, Ea = tc.spectrum(buf2, 5.0, 1, 300.0)
    b, Eb, n = tc.spectrum_welch(buf2, 32, 2, 5.0, binding.make_window("hann", 32), 300.0)
    assert n == 1 and np.array_equal(Ea, Eb) and torch.equal(a, b)
    tc.close()
