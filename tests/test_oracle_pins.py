"""Pins for the fp64 oracle: what the paper and the mathematics fix, independent of the oracle's own
code path (closed forms, invariants, library routines, brute force, the paper's worked numbers).
Pin ids P1..P13 follow SURVEY.md 8(c) / DESIGN.md.  CPU only.
"""
import os

import numpy as np
import pytest

from paper_2607_02236_b200 import workloads as W

GOLD = os.path.join(os.path.dirname(__file__), "golden", "paper_worked_numbers.txt")


def golden():
    out = {}
    for line in open(GOLD):
        if line.startswith("#") or not line.strip():
            continue
        k, v, _cite = [s.strip() for s in line.split("|", 2)]
        vals = [float(x) for x in v.split()]
        out[k] = vals[0] if len(vals) == 1 else vals
    return out


def sidx(n):
    i = np.arange(n)
    return np.where(i < n // 2, i, i - n)


def random_phase_slices(rng, s, ny, nx, strength=1.0):
    return np.exp(1j * strength * rng.normal(size=(s, ny, nx)))


# --------------------------------------------------------------------------------------------- P8
@pytest.mark.parametrize("n", [1, 2, 4, 8, 16, 64, 128, 512])
def test_p8_fft_vs_naive_vs_numpy(oracle, n):
    rng = np.random.default_rng(n)
    x = rng.normal(size=n) + 1j * rng.normal(size=n)
    for sign in (-1, +1):
        ref = np.fft.fft(x) if sign < 0 else np.fft.ifft(x) * n
        scale = np.linalg.norm(ref)
        assert np.linalg.norm(oracle.fft_radix2(x, sign) - ref) <= 1e-13 * scale
        if n <= 128:
            assert np.linalg.norm(oracle.dft_naive(x, sign) - ref) <= 1e-13 * scale


@pytest.mark.parametrize("n", [200, 1680])
def test_p8_naive_dft_at_the_papers_non_power_of_two_lengths(oracle, n):
    """The paper's chunk length 200 (:164) and grid edge 1680 = 2^4 3 5 7 (:162): the oracle's dispatch falls back to
    its naive DFT for such lengths; pinned against numpy.fft (library routine, test only)."""
    rng = np.random.default_rng(n)
    x = rng.normal(size=n) + 1j * rng.normal(size=n)
    for sign, ref in ((-1, np.fft.fft(x)), (+1, np.fft.ifft(x) * n)):
        assert np.max(np.abs(oracle.dft_naive(x, sign) - ref)) <= 1e-10 * np.max(np.abs(ref))
    a = rng.normal(size=(3, n)) + 1j * rng.normal(size=(3, n))
    assert np.max(np.abs(oracle.fft2(a, -1) - np.fft.fft2(a))) <= 1e-10 * np.max(np.abs(a)) * n


@pytest.mark.parametrize("shape", [(8, 8), (16, 64), (128, 32), (256, 256)])
def test_p8_fft2_vs_numpy(oracle, shape):
    rng = np.random.default_rng(5)
    a = rng.normal(size=shape) + 1j * rng.normal(size=shape)
    assert np.allclose(oracle.fft2(a, -1), np.fft.fft2(a), rtol=0, atol=1e-12 * np.abs(a).sum() ** 0.5 * 10)
    assert np.allclose(oracle.fft2(a, +1), np.fft.ifft2(a), rtol=0, atol=1e-13)
    # both code paths (naive / radix-2) agree on the same input
    oracle.set_fft_mode(1)
    f1 = oracle.fft2(a[:32, :32], -1)
    oracle.set_fft_mode(2)
    f2 = oracle.fft2(a[:32, :32], -1)
    oracle.set_fft_mode(0)
    assert np.linalg.norm(f1 - f2) <= 1e-13 * np.linalg.norm(f1)


# --------------------------------------------------------------------------------------------- P1
def test_p1a_free_space_discrete(oracle):
    """Zero potential: FFT2(psi_S) = Psi0 * exp(-i pi lambda (S dz) q^2) for any probe."""
    n, L, lam, dz, S = 64, 13.782, 0.0370144, 1.4795, 7
    psi0 = oracle.make_probes(n, n, L, L, lam, np.array([[3.1, 7.7]]), 30e-3)
    ones = np.ones((S, n, n), dtype=np.complex128)
    out = oracle.propagate(L, L, lam, 0, psi0, None, [[ones]], dz, 1)[0]
    h = sidx(n)
    q2 = (h[None, :] / L) ** 2 + (h[:, None] / L) ** 2
    expect = np.fft.fft2(psi0[0]) * np.exp(-1j * np.pi * lam * S * dz * q2)
    assert np.linalg.norm(out - expect) <= 1e-12 * np.linalg.norm(expect)


def test_p1b_free_space_steps_compose(oracle):
    """S steps of dz == one step of S*dz (no mask)."""
    n, L, lam, dz, S = 32, 9.0, 0.0370144, 1.1, 5
    rng = np.random.default_rng(0)
    psi0 = (rng.normal(size=(1, n, n)) + 1j * rng.normal(size=(1, n, n)))
    a = oracle.propagate(L, L, lam, 0, psi0, None, [[np.ones((S, n, n), complex)]], dz, 0)
    b = oracle.propagate(L, L, lam, 0, psi0, None, [[np.ones((1, n, n), complex)]], S * dz, 0)
    assert np.linalg.norm(a - b) <= 1e-12 * np.linalg.norm(b)


def test_p1c_free_space_gaussian_closed_form(oracle):
    """Continuous Fresnel: exp(-r^2/2w^2) -> (w^2/W) exp(-r^2/2W), W = w^2 + i lambda z/(2 pi)."""
    n, L, lam = 128, 40.0, 0.0370144
    w, z = 1.5, 400.0
    x = (np.arange(n) - n // 2) * L / n
    r2 = x[None, :] ** 2 + x[:, None] ** 2
    psi0 = np.exp(-r2 / (2 * w * w))[None].astype(complex)
    S = 8
    out = oracle.propagate(L, L, lam, 0, psi0, None, [[np.ones((S, n, n), complex)]], z / S, 0)[0]
    Wc = w * w + 1j * lam * z / (2 * np.pi)
    expect = (w * w / Wc) * np.exp(-r2 / (2 * Wc))
    assert np.max(np.abs(out - expect)) <= 1e-12


# --------------------------------------------------------------------------------------------- P2
def test_p2_unitarity_without_mask(oracle):
    n, L, lam, dz, S = 32, 9.2, 0.0370144, 1.4795, 6
    rng = np.random.default_rng(1)
    t = random_phase_slices(rng, S, n, n)
    psi0 = oracle.make_probes(n, n, L, L, lam, np.array([[1.0, 2.0], [4.4, 0.3]]), 25e-3)
    _, norms = oracle.propagate(L, L, lam, 0, psi0, None, [[t]], dz, 0, want_norms=True)
    assert np.max(np.abs(norms - 1.0)) <= 1e-12


def test_p2_bandlimit_loss_identity(oracle):
    """With the 2/3 mask: norm loss per step = out-of-band power of FFT2(t psi) / (Nx Ny), exactly."""
    n, L, lam, dz = 48, 10.0, 0.0370144, 1.4795
    rng = np.random.default_rng(2)
    t = random_phase_slices(rng, 1, n, n, 2.0)
    psi0 = rng.normal(size=(1, n, n)) + 1j * rng.normal(size=(1, n, n))
    psi0 /= np.linalg.norm(psi0)
    _, norms = oracle.propagate(L, L, lam, 1, psi0, None, [[t]], dz, 0, want_norms=True)
    F = np.fft.fft2(t[0] * psi0[0])
    h = sidx(n)
    inband = 9 * (h[None, :] ** 2 + h[:, None] ** 2) <= n * n
    loss = np.sum(np.abs(F[~inband]) ** 2) / (n * n)
    assert norms[0, 1] <= norms[0, 0]
    assert abs((norms[0, 0] - norms[0, 1]) - loss) <= 1e-13
    assert loss > 1e-3          # the case actually exercises the mask


def test_p2_mask_is_two_thirds_disc(oracle):
    """The mask that propagate applies: a delta in q outside 2/3 Nyquist dies, inside survives."""
    n, L, lam = 48, 10.0, 0.0370144
    for (h, k, alive) in [(16, 0, True), (17, 0, False), (11, 11, True), (12, 12, False), (-16, 0, True), (0, -17, False)]:
        F = np.zeros((n, n), complex)
        F[k % n, h % n] = 1.0
        psi = np.fft.ifft2(F)[None]
        out = oracle.propagate(L, L, lam, 1, psi, None, [[np.ones((1, n, n), complex)]], 1.0, 1)[0]
        assert (abs(out[k % n, h % n]) > 0.5) == alive


# --------------------------------------------------------------------------------------------- P6
def test_p6_single_gaussian_atom_image_sum(oracle):
    """v(r) of one single-Gaussian atom = periodic image sum of a (pi/b) exp(-pi^2 r^2/b)."""
    n, L = 64, 13.782
    a = np.zeros((1, 4)); b = np.ones((1, 4))
    a[0, 0], b[0, 0] = 37.0, 5.0
    pos = np.array([[3.3, 5.1, 0.2]])
    r = oracle.build_slices(n, n, L, L, pos, np.zeros(1, np.int32), a, b, 1.0, 1, 0.0, 1e-3, bandlimit=0,
                            pot_mode=0, want_v=True)
    x = np.arange(n) * L / n
    v = np.zeros((n, n))
    for mx in range(-3, 4):
        for my in range(-3, 4):
            dx = x[None, :] - pos[0, 0] - mx * L
            dy = x[:, None] - pos[0, 1] - my * L
            v += a[0, 0] * (np.pi / b[0, 0]) * np.exp(-np.pi ** 2 * (dx * dx + dy * dy) / b[0, 0])
    assert np.max(np.abs(r["v"][0] - v)) <= 2e-11 * np.max(v)
    assert r["max_imag"] <= 1e-12
    assert np.allclose(r["trans"][0], np.exp(1j * 1e-3 * r["v"][0]), rtol=0, atol=1e-15)


def test_potential_modes_agree_and_slices_bin(oracle):
    """pot_mode 1 (product of per-axis phases) == pot_mode 0 (direct term); atoms land in the right slice."""
    wl = W.tiny_workload(n=16, ncell=(1, 1, 2))
    seg = wl.segments[0]
    pos = seg.frames(3, 4, wl.dt_fs)[0]
    r0 = oracle.build_slices(wl.nx, wl.ny, wl.lx, wl.ly, pos, seg.species, wl.a, wl.b, wl.dz, seg.nslices, 0.0,
                             wl.sigma, 1, 0, want_v=True, want_vq=True)
    r1 = oracle.build_slices(wl.nx, wl.ny, wl.lx, wl.ly, pos, seg.species, wl.a, wl.b, wl.dz, seg.nslices, 0.0,
                             wl.sigma, 1, 1, want_v=True, want_vq=True)
    assert np.max(np.abs(r0["vq"] - r1["vq"])) <= 1e-12 * np.max(np.abs(r0["vq"]))
    assert r0["n_clamped"] == 0
    # V_n(q=0) = sum over the atoms of slice n of f_s(0) = sum_i a_si: 3 atoms per slice (1 Ti + 2 O)
    f0 = wl.a.sum(axis=1)
    for n in range(seg.nslices):
        assert abs(r0["vq"][n, 0, 0] - (f0[0] + 2 * f0[1])) <= 1e-10
    # out-of-band V is exactly zero, Nyquist row/column carry nothing
    h = sidx(wl.nx)
    oob = 9 * (h[None, :] ** 2 + h[:, None] ** 2) > wl.nx ** 2
    assert np.all(r0["vq"][:, oob] == 0)


def test_slice_clamping_counts(oracle):
    a = np.ones((1, 4)); b = np.ones((1, 4))
    pos = np.array([[0, 0, -0.1], [0, 0, 0.5], [0, 0, 1.99], [0, 0, 2.0], [0, 0, 7.3]], dtype=float)
    r = oracle.build_slices(8, 8, 4.0, 4.0, pos, np.zeros(5, np.int32), a, b, 1.0, 2, 0.0, 1e-3, 0, 0, want_vq=True)
    assert r["n_clamped"] == 3          # z<0, z==S*dz (floor -> S), z>>top
    assert abs(r["vq"][0, 0, 0] - 2 * 4) < 1e-12 and abs(r["vq"][1, 0, 0] - 3 * 4) < 1e-12


# --------------------------------------------------------------------------------------------- P3
def test_p3_weak_phase_closed_form(oracle):
    """One thin slice, unit-norm plane wave, potential scaled by eps -> 0:
    phi[h,k] = P[h,k] (delta + i sigma V[h,k]/(Lx Ly)) + O(eps^2)."""
    n, L, lam, dz = 32, 9.188, 0.0370144, 1.4795
    sig = 9.243958e-4
    rng = np.random.default_rng(3)
    pos = np.column_stack([rng.uniform(0, L, 5), rng.uniform(0, L, 5), np.full(5, 0.5)])
    spec = np.array([0, 1, 1, 0, 1], np.int32)
    a, b = W.species_table(11)
    h = sidx(n)
    hh, kk = np.meshgrid(h, h, indexing="xy")
    q2 = (hh / L) ** 2 + (kk / L) ** 2
    inband = 9 * (hh ** 2 + kk ** 2) <= n * n
    errs = []
    for eps in (1e-2, 1e-3):
        ae = a * eps
        V = np.zeros((n, n), complex)
        for j in range(5):
            f = sum(ae[spec[j], i] * np.exp(-b[spec[j], i] * q2) for i in range(4))
            V += f * np.exp(-2j * np.pi * (hh * pos[j, 0] + kk * pos[j, 1]) / L)
        V = V * inband
        r = oracle.build_slices(n, n, L, L, pos, spec, ae, b, dz, 1, 0.0, sig, 1, 0)
        psi0 = oracle.make_probes(n, n, L, L, lam, np.zeros((1, 2)), 0.0)
        assert np.allclose(psi0, 1.0 / n, atol=1e-15)
        phi = oracle.propagate(L, L, lam, 1, psi0, None, [[r["trans"]]], dz, 1)[0] / n
        delta = np.zeros((n, n)); delta[0, 0] = 1.0
        P = np.exp(-1j * np.pi * lam * dz * q2) * inband
        expect = P * (delta + 1j * sig * V / (L * L))
        m = inband.copy(); m[0, 0] = False
        errs.append(np.linalg.norm((phi - expect)[m]) / np.linalg.norm(expect[m]))
    assert errs[0] < 5e-2 and errs[1] < 5e-3
    assert 5 < errs[0] / errs[1] < 20          # first order in eps


# --------------------------------------------------------------------------------------------- P4
def test_p4_bose_closed_forms(oracle):
    assert oracle.bose(0.0) == 1.0
    for x in (1e-9, 0.01, 0.3, 1.0, 7.5, 40.0):
        assert abs(oracle.bose(x) - oracle.bose(-x) - x) <= 1e-14 * max(1.0, x)
        assert abs(oracle.bose(x) / oracle.bose(-x) - np.exp(x)) <= 1e-13 * np.exp(x)
    kbt = 8.617333262e-5 * 300.0 * 1e3     # 25.852 meV
    assert abs(oracle.bose(20.0 / kbt) - 1.436203) < 1e-6
    assert abs(oracle.bose(-20.0 / kbt) - 0.662568) < 1e-6
    assert abs(oracle.bose(1e-12) - 1.0) < 1e-12     # no 0/0 blow-up near the elastic line


# --------------------------------------------------------------------------------- P5 / P9 / P10
def _tiny_run(oracle, **kw):
    from oracle import pipeline
    wl = W.tiny_workload(**kw)
    return wl, pipeline.run(wl, pot_mode=0)


def test_p5_harmonic_peaks_on_bins_and_detailed_balance(oracle):
    T, m0 = 64, 5
    wl, res = _tiny_run(oracle, n=16, ncell=(1, 1, 1), nframes=T, dt_fs=5.0, mode_bins=[m0], amp_A=0.01)
    I, E = res["I"][0], res["E"]
    assert I.shape == (T, 256)
    kprime = np.round(E / (W.H_MEV_FS / (T * wl.dt_fs))).astype(int)
    assert kprime[0] == -T // 2 and np.all(np.diff(kprime) == 1)
    spec = I[:, res["roi"] != 0].sum(axis=1)        # all q except the direct beam
    inel = spec.copy()
    inel[np.abs(kprime) <= 2] = 0.0                 # drop the elastic line and its Hann skirts
    assert kprime[np.argmax(np.where(kprime > 0, inel, 0.0))] == m0       # loss side
    assert kprime[np.argmax(np.where(kprime < 0, inel, 0.0))] == -m0      # gain side
    # Hann spreads an on-bin line over bins m0-1, m0, m0+1 with amplitudes 1/4, 1/2, 1/4 and nothing else
    for m in (m0, -m0):
        line = np.array([spec[kprime == m + d][0] / oracle.bose(E[kprime == m + d][0] / (W.KB_EV_K * 1e3 * wl.temperature_K))
                         for d in (-1, 0, 1)])
        assert np.allclose(line / line[1], [0.25, 1.0, 0.25], rtol=5e-2)
    loss, gain = spec[kprime == m0][0], spec[kprime == -m0][0]
    x = E[kprime == m0][0] / (W.KB_EV_K * 1e3 * wl.temperature_K)
    assert abs(loss / gain - np.exp(x)) <= 2e-3 * np.exp(x)


def test_p5_config1_like_offbin_modes_peak_within_one_bin(oracle):
    T = 32
    wl, res = _tiny_run(oracle, n=16, ncell=(1, 1, 1), nframes=T, dt_fs=5.0, amp_A=0.02)
    I, E = res["I"][0], res["E"]
    dE = E[1] - E[0]
    spec = I[:, res["roi"] != 0].sum(axis=1)
    for e_mode in (45.0, 80.0):
        k = np.argmin(np.abs(E - e_mode))
        lo, hi = max(k - 2, 0), min(k + 3, T)
        assert spec[lo:hi].max() > 3 * np.median(spec[np.abs(E) > 150.0]), (e_mode, dE)


def test_p9_static_trajectory_only_elastic_bins(oracle):
    from oracle import pipeline
    T = 16
    for window, allowed in ((1, {0, 1, -1}), (0, {0})):
        wl = W.tiny_workload(n=16, ncell=(1, 1, 1), nframes=T, amp_A=0.0)
        wl.window = window
        res = pipeline.run(wl, pot_mode=0)
        I, E = res["I"][0], res["E"]
        kprime = np.round(E / (W.H_MEV_FS / (T * wl.dt_fs))).astype(int)
        tot = I.sum()
        for e in range(T):
            if kprime[e] not in allowed:
                assert I[e].sum() <= 1e-20 * tot
        assert I[kprime == 0].sum() > 0.3 * tot


def test_p10_parseval_of_the_normalisation(oracle):
    """sum_{E,q} |Phi|^2/(T sum w^2) = sum_f w_f^2 N_f / sum_f w_f^2 with N_f = sum_q |phi(q,t_f)|^2;
    with full q and no mask N_f = 1, so the Bose-free total is 1."""
    rng = np.random.default_rng(4)
    P, T, Q = 2, 16, 37
    buf = rng.normal(size=(P, T, Q)) + 1j * rng.normal(size=(P, T, Q))
    w = 0.5 - 0.5 * np.cos(2 * np.pi * np.arange(T) / T)
    assert np.allclose(oracle.window(1, T), w, atol=1e-15) and np.all(oracle.window(0, T) == 1.0)
    I, E = oracle.spectrum(buf, 5.0, 1, 300.0)
    bose = np.array([oracle.bose(e / (W.KB_EV_K * 1e3 * 300.0)) for e in E])
    for p in range(P):
        lhs = (I[p] / bose[:, None]).sum()
        Nf = (np.abs(buf[p]) ** 2).sum(axis=1)
        rhs = (w ** 2 * Nf).sum() / (w ** 2).sum()
        assert abs(lhs - rhs) <= 1e-12 * rhs
    # against the library DFT, bin by bin
    Phi = np.fft.fft(buf * w[None, :, None], axis=1)
    order = np.argsort(np.where(np.arange(T) < T // 2, np.arange(T), np.arange(T) - T))
    ref = (np.abs(Phi[:, order, :]) ** 2) / (T * (w ** 2).sum()) * bose[None, :, None]
    assert np.max(np.abs(I - ref)) <= 1e-12 * np.max(ref)


def test_p10_full_q_unit_total(oracle):
    from oracle import pipeline
    wl = W.tiny_workload(n=16, ncell=(1, 1, 1), nframes=8)
    wl.bandlimit = 0
    res = pipeline.run(wl, pot_mode=0)
    bose = np.array([oracle.bose(e / (W.KB_EV_K * 1e3 * wl.temperature_K)) for e in res["E"]])
    assert abs((res["I"][0] / bose[:, None]).sum() - 1.0) <= 1e-12


# --------------------------------------------------------------------------------------------- P7
def test_p7_grid_aligned_translation_covariance(oracle):
    from oracle import pipeline
    wl = W.tiny_workload(n=16, ncell=(1, 1, 2), nframes=1)
    base = pipeline.exit_waves(wl, [0], output_space=1, pot_mode=0)[0, 0]
    mx, my = 3, 5
    d = np.array([mx * wl.lx / wl.nx, my * wl.ly / wl.ny, 0.0])
    wl.segments[0].pos0 = wl.segments[0].pos0 + d
    shifted = pipeline.exit_waves(wl, [0], output_space=1, pot_mode=0)[0, 0]
    h = sidx(wl.nx)
    ramp = np.exp(-2j * np.pi * (h[None, :] * mx / wl.nx + h[:, None] * my / wl.ny))
    assert np.linalg.norm(shifted - base * ramp) <= 1e-12 * np.linalg.norm(base)


# -------------------------------------------------------------------------------------------- P11
def test_p11_paper_worked_numbers(oracle):
    g = golden()
    lam60 = W.electron_wavelength_A(60.0)
    assert abs(lam60 - 0.0486606) < 2e-7 and abs(W.electron_wavelength_A(100.0) - 0.0370144) < 2e-7
    assert abs(W.interaction_sigma(100.0) - 9.243958e-4) < 1e-9
    # 0.52 mrad pixels for the 9.3 nm cell, 1.3 mrad for 8 lateral cells (a = 4.594 A)
    assert round(lam60 / 93.0 * 1e3, 2) == g["qpixel_mrad_9p3nm_60kV"]
    assert round(lam60 / (8 * 4.594) * 1e3, 1) == g["qpixel_mrad_8x8cells_60kV"]
    # +-100 mrad rectangular ROI on the 1680^2 grid -> 383 x 383
    idx = oracle.make_roi(1680, 1680, 93.0, 93.0, lam60, "rect", [-0.1, 0.1, -0.1, 0.1])
    assert idx.size == int(g["roi_px_per_axis_pm100mrad"]) ** 2
    # 200 snapshots x 15 fs: 1.4 meV sampling, 181 bins within +-30 THz
    E, bins = oracle.energy_axis(200, 15.0)
    assert round(E[1] - E[0], 1) == g["energy_sampling_meV_200x15fs"]
    e30 = W.H_MEV_FS * 30e12 * 1e-15
    Er, _ = oracle.energy_axis(200, 15.0, -e30, e30)
    assert Er.size == int(g["bins_in_pm30THz_200x15fs"])
    # Eq.(B1): eps = h/(2 tau) ~ 2000 meV fs / tau
    E1, _ = oracle.energy_axis(64, 1.0)
    assert abs(-E1[0] - W.H_MEV_FS / 2.0) < 1e-9 and round(-E1[0], -3) == g["emax_meV_per_fs"]
    # Eq.(B2)
    assert round(4 * 8 * 383 * 383 * 200 * 16 * 2 / 1e9) == g["buffer_GB_eqB2"]


def test_roi_maps_order_and_predicates(oracle):
    n, L, lam = 16, 8.0, 0.04
    full = oracle.make_roi(n, n, L, L, lam, "full", [])
    assert full.size == n * n and sorted(full.tolist()) == list(range(n * n))
    assert full[0] == (n // 2) * n + n // 2          # (k,h) = (-N/2,-N/2) first
    h = sidx(n)
    th2 = (lam / L) ** 2 * (h[None, :] ** 2 + h[:, None] ** 2)
    disc = oracle.make_roi(n, n, L, L, lam, "disc", [0.02])
    assert set(disc.tolist()) == set(np.flatnonzero((th2 <= 0.02 ** 2).ravel()).tolist())
    ann = oracle.make_roi(n, n, L, L, lam, "annulus", [0.01, 0.02])
    assert set(ann.tolist()) == set(np.flatnonzero(((th2 <= 0.02 ** 2) & (th2 >= 0.01 ** 2)).ravel()).tolist())
    # ascending (k, h) enumeration
    kk = np.where(disc // n < n // 2, disc // n, disc // n - n)
    hh = np.where(disc % n < n // 2, disc % n, disc % n - n)
    key = kk * 1000 + hh
    assert np.all(np.diff(key) > 0)


# -------------------------------------------------------------------------------------------- P12
def test_p12_segment_chaining_is_concatenation(oracle):
    n, L, lam, dz = 16, 6.0, 0.0370144, 1.4795
    rng = np.random.default_rng(6)
    t1, t2, t3 = (random_phase_slices(rng, s, n, n) for s in (2, 3, 1))
    psi0 = oracle.make_probes(n, n, L, L, lam, np.array([[1.0, 2.0]]), 30e-3)
    a = oracle.propagate(L, L, lam, 1, psi0, None, [[t1, t2, t3]], dz, 0)
    b = oracle.propagate(L, L, lam, 1, psi0, None, [[np.concatenate([t1, t2, t3])]], dz, 0)
    assert np.array_equal(a, b)
    # wave_frame picks the frame's own transmissions
    c = oracle.propagate(L, L, lam, 1, np.concatenate([psi0, psi0]), [1, 0], [[t1], [t2[:2]]], dz, 0)
    assert np.array_equal(c[0], oracle.propagate(L, L, lam, 1, psi0, None, [[t2[:2]]], dz, 0)[0])
    assert np.array_equal(c[1], oracle.propagate(L, L, lam, 1, psi0, None, [[t1]], dz, 0)[0])


# -------------------------------------------------------------------------------------------- P13
def test_p13_brute_force_tiny(oracle):
    """8x8 grid, 2 atoms, 2 slices, 4 frames: whole path with explicit O(N^4) DFT sums in numpy."""
    n, L, lam, dz, sig, T, dt, temp = 8, 5.0, 0.0370144, 1.2, 9.243958e-4, 4, 5.0, 300.0
    a, b = W.species_table(3)
    rng = np.random.default_rng(8)
    base = np.array([[1.1, 2.3, 0.4], [3.7, 0.9, 1.9]])
    spec = np.array([0, 1], np.int32)
    disp = 0.05 * rng.normal(size=(T, 2, 3)); disp[:, :, 2] = 0.0
    h = sidx(n)
    idx = np.arange(n)
    Fm = np.exp(-2j * np.pi * np.outer(idx, idx) / n)         # DFT matrix
    hh, kk = np.meshgrid(h, h, indexing="xy")
    q2 = (hh ** 2 + kk ** 2) / L ** 2
    M = (9 * (hh ** 2 + kk ** 2) <= n * n)
    P = np.exp(-1j * np.pi * lam * dz * q2) * M
    alpha = 0.012
    probe_xy = np.array([[0.7, 1.9]])
    A = (lam * lam * q2 <= alpha * alpha)
    Psi0 = A * np.exp(-2j * np.pi * (hh * probe_xy[0, 0] + kk * probe_xy[0, 1]) / L)
    psi0 = np.conj(Fm) @ Psi0 @ np.conj(Fm)
    psi0 /= np.linalg.norm(psi0)
    roi = oracle.make_roi(n, n, L, L, lam, "disc", [0.02])
    buf_ref = np.zeros((1, T, roi.size), complex)
    buf = np.zeros((1, T, roi.size), complex)
    for f in range(T):
        pos = base + disp[f]
        psi = psi0.copy()
        for s in range(2):
            V = np.zeros((n, n), complex)
            for j in range(2):
                if int(np.floor(pos[j, 2] / dz)) != s:
                    continue
                fq = sum(a[spec[j], i] * np.exp(-b[spec[j], i] * q2) for i in range(4))
                V += fq * np.exp(-2j * np.pi * (hh * pos[j, 0] + kk * pos[j, 1]) / L)
            V *= M
            v = np.real(np.conj(Fm) @ V @ np.conj(Fm)) / (L * L)
            psi = psi * np.exp(1j * sig * v)
            psi = np.conj(Fm) @ (P * (Fm @ psi @ Fm)) @ np.conj(Fm) / (n * n)
        Psi = Fm @ psi @ Fm
        buf_ref[0, f] = Psi.ravel()[roi] / n
        r = oracle.build_slices(n, n, L, L, pos, spec, a, b, dz, 2, 0.0, sig, 1, 0)
        pw = oracle.make_probes(n, n, L, L, lam, probe_xy, alpha)
        assert np.linalg.norm(pw[0] - psi0) <= 1e-13
        q = oracle.propagate(L, L, lam, 1, pw, None, [[r["trans"]]], dz, 1)
        assert np.linalg.norm(q[0] - Psi) <= 1e-13 * np.linalg.norm(Psi)
        oracle.accumulate(q, [0], [f], roi, buf)
    assert np.linalg.norm(buf - buf_ref) <= 1e-13 * np.linalg.norm(buf_ref)
    I, E = oracle.spectrum(buf, dt, 1, temp)
    w = 0.5 - 0.5 * np.cos(2 * np.pi * np.arange(T) / T)
    kp = np.arange(-T // 2, T // 2)
    Eref = W.H_MEV_FS * kp / (T * dt)
    assert np.allclose(E, Eref, rtol=0, atol=1e-9)
    Iref = np.zeros((T, roi.size))
    for e, k in enumerate(kp):
        ph = np.exp(-2j * np.pi * k * np.arange(T) / T)
        Phi = ((w * ph)[:, None] * buf_ref[0]).sum(axis=0)
        x = Eref[e] / (W.KB_EV_K * 1e3 * temp)
        B = 1.0 if x == 0 else x / (1 - np.exp(-x))
        Iref[e] = B * np.abs(Phi) ** 2 / (T * (w ** 2).sum())
    assert np.max(np.abs(I[0] - Iref)) <= 1e-12 * np.max(Iref)


def test_workload_shapes_match_configs():
    """The five configs' plain numbers (BASELINE.json configs)."""
    expect = {1: (216, 64, 1, 32, 8), 2: (7680, 256, 4, 256, 40)}
    for cfg, (na, n, p, t, s) in expect.items():
        wl = W.make_workload(cfg)
        assert (wl.natoms, wl.nx, wl.nprobes, wl.nframes, wl.nslices_total) == (na, n, p, t, s)
        assert wl.slice_steps == p * t * s
    wl = W.make_workload(1)
    z = wl.segments[0].pos0[:, 2] / wl.dz
    assert np.allclose(z - np.floor(z), 0.5)       # planes at c/4, 3c/4 = slice centres
    pts = W._raster(0.0, 0.0, 1.0, 1.0, 5, 1)[:, 0]
    assert np.allclose(pts, [0.0, 0.2, 0.4, 0.6, 0.8])     # PAPER.md:380 end point excluded
