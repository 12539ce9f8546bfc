"""DetectorSet reduction.  Oracle pins (CPU), host mask
generator vs oracle (CPU, bit-exact), GPU parity of tacaw_detect."""
import numpy as np
import pytest

LAM = 0.0370144


def grid_roi(oracle, n=64, L=13.782, mode="full", params=()):
    return oracle.make_roi(n, n, L, L, LAM, mode, list(params))


# ------------------------------------------------------------------------------------- oracle pins (CPU)
def test_d1_centred_circular_detector_is_the_disc_roi(oracle):
    """A circular detector centred on the optical axis selects exactly the pixels of the disc ROI map (O8, whose counts
    are pinned to the paper's worked numbers by P11); an annulus is the difference of two discs."""
    n, L = 64, 13.782
    full = grid_roi(oracle, n, L)
    for r in (5e-3, 20e-3, 33.3e-3):
        w = oracle.detector_weights(n, n, L, L, LAM, "circular", (0.0, 0.0), (0.0, r), full)
        disc = grid_roi(oracle, n, L, "disc", (r,))
        assert np.array_equal(np.sort(full[w > 0]), np.sort(disc))
    wa = oracle.detector_weights(n, n, L, L, LAM, "annular", (0.0, 0.0), (10e-3, 30e-3), full)
    ann = grid_roi(oracle, n, L, "annulus", (10e-3, 30e-3))
    assert np.array_equal(np.sort(full[wa > 0]), np.sort(ann))
    w0 = oracle.detector_weights(n, n, L, L, LAM, "annular", (0.0, 0.0), (0.0, 30e-3), full)
    wc = oracle.detector_weights(n, n, L, L, LAM, "circular", (0.0, 0.0), (0.0, 30e-3), full)
    assert np.array_equal(w0, wc)


def test_d2_off_axis_detector_is_the_shifted_pixel_set(oracle):
    """Moving the centre by a whole number of pixels (lambda/L per pixel) moves the selected set by that many pixels
    (the paper's off-axis detectors, Fig. 5: 'displaced 60 mrad from the center')."""
    n, L = 64, 13.782
    full = grid_roi(oracle, n, L)
    px = LAM / L
    w_c = oracle.detector_weights(n, n, L, L, LAM, "circular", (0.0, 0.0), (0.0, 12e-3), full)
    w_s = oracle.detector_weights(n, n, L, L, LAM, "circular", (5 * px, -3 * px), (0.0, 12e-3), full)
    hk = lambda idx: (np.where(idx % n < n // 2, idx % n, idx % n - n), np.where(idx // n < n // 2, idx // n, idx // n - n))
    h0, k0 = hk(full[w_c > 0])
    h1, k1 = hk(full[w_s > 0])
    assert sorted(zip(h0 + 5, k0 - 3)) == sorted(zip(h1, k1))


def test_d3_detect_is_the_brute_force_sum_and_full_detector_is_parseval(oracle):
    rng = np.random.default_rng(2)
    I = rng.random((3, 4, 11))
    w = rng.random((2, 11))
    out = oracle.detect(I, w)
    assert out.shape == (2, 4, 3)
    for d in range(2):
        for e in range(4):
            for p in range(3):
                assert abs(out[d, e, p] - sum(w[d, r] * I[p, e, r] for r in range(11))) <= 1e-14
    # an all-ones detector over full q, rect window, no mask: sum_E signal/B = 1 per probe (P10 / G10)
    T, Q = 16, 9
    phi = rng.normal(size=(1, T, Q)) + 1j * rng.normal(size=(1, T, Q))
    phi /= np.sqrt((np.abs(phi) ** 2).sum(axis=2, keepdims=True))        # unit norm at every time
    Isp, E = oracle.spectrum(phi, 5.0, 0, 300.0)
    sig = oracle.detect(Isp, np.ones((1, Q)))
    B = np.array([oracle.bose(e / (8.617333262e-2 * 300.0)) for e in E])
    assert abs((sig[0, :, 0] / B).sum() - 1.0) <= 1e-12


# ------------------------------------------------------------------- library host function vs oracle (CPU)
@pytest.mark.parametrize("kind,center,radii", [("circular", (0.0, 0.0), (0.0, 10e-3)), ("annular", (0.0, 0.0), (10e-3, 30e-3)),
                                               ("circular", (60e-3 * 0.5, -7e-3), (0.0, 30e-3 * 0.5)),
                                               ("annular", (3e-3, 4e-3), (0.0, 0.0))])
def test_make_detector_host_is_bit_exact(oracle, kind, center, radii):
    from paper_2607_02236_b200 import binding, build
    build.build_lib()
    for n, L, mode, params in ((64, 13.782, "full", ()), (256, 36.752, "disc", (60e-3,)), (128, 9.0, "rect", (-20e-3, 30e-3, -10e-3, 10e-3))):
        roi = oracle.make_roi(n, n, L, L, LAM, mode, list(params))
        ref = oracle.detector_weights(n, n, L, L, LAM, kind, center, radii, roi)
        got = binding.make_detector(n, n, L, L, LAM, kind, center, radii, roi)
        assert got.dtype == np.float32 and np.array_equal(got.astype(np.float64), ref)
    with pytest.raises(binding.TacawError):
        binding.make_detector(64, 64, 9.0, 9.0, LAM, "annular", (0, 0), (5e-3, 1e-3), np.arange(4, dtype=np.int32))


# ------------------------------------------------------------------------------------------- GPU parity
@pytest.mark.gpu
@pytest.mark.parametrize("P,nE,Q,D", [(1, 1, 1, 1), (5, 7, 1003, 3), (16, 33, 11165, 4), (3, 2, 4096, 11)])
def test_detect_vs_oracle(oracle, P, nE, Q, D):
    import torch
    from paper_2607_02236_b200 import binding, build
    build.build_lib()
    rng = np.random.default_rng(P * 1000 + D)
    I = rng.random((P, nE, Q)).astype(np.float32) * rng.choice([1e-6, 1.0, 1e3], size=(P, nE, 1)).astype(np.float32)
    w = (rng.random((D, Q)) < 0.3).astype(np.float32)
    w[-1] = rng.random(Q).astype(np.float32)                            # a "custom" weighted detector
    tc = binding.Tacaw(16, 16, 5.0, 5.0, 0.037, 9e-4, 1)
    out = tc.detect(torch.from_numpy(I).cuda(), torch.from_numpy(w).cuda())
    ref = oracle.detect(I, w)
    got = out.cpu().numpy()
    assert got.shape == (D, nE, P)
    # fp32 accumulation over Q terms of one sign: relative error <= ~sqrt(Q) eps
    assert np.all(np.abs(got - ref) <= 2e-5 * np.abs(ref) + 1e-30)
    tc.close()


@pytest.mark.gpu
def test_detectors_on_config1_spectrum(oracle):
    """End to end on configs[0]: bright-field disc + annulus of the exit-wave spectrum, GPU vs oracle."""
    import torch
    from paper_2607_02236_b200 import binding, build, workloads as W
    from paper_2607_02236_b200.pipeline import Runner
    from oracle import pipeline as OP
    build.build_lib()
    wl = W.make_workload(1)
    ref = OP.run(wl, pot_mode=0)
    r = Runner(wl, device=0)
    out = r.run()
    dets = [("circular", (0.0, 0.0), (0.0, 10e-3)), ("annular", (0.0, 0.0), (10e-3, 30e-3)), ("circular", (15e-3, 0.0), (0.0, 8e-3))]
    wg = np.stack([binding.make_detector(wl.nx, wl.ny, wl.lx, wl.ly, wl.lam, k, c, rr, out["roi"]) for k, c, rr in dets])
    wo = np.stack([oracle.detector_weights(wl.nx, wl.ny, wl.lx, wl.ly, wl.lam, k, c, rr, ref["roi"]) for k, c, rr in dets])
    assert np.array_equal(wg.astype(np.float64), wo) and wo.sum(axis=1).min() > 0
    sig = r.tc.detect(out["I"], torch.from_numpy(wg).cuda()).cpu().numpy()
    sref = oracle.detect(ref["I"], wo)
    for d in range(len(dets)):
        assert np.linalg.norm(sig[d] - sref[d]) <= 1e-3 * np.linalg.norm(sref[d])      # north_star bar for spectra
    r.tc.close()
