"""SURVEY.md 8(f) item 4 (workload variants): scan grids and scan sub-batches (Listing 1 :416-428).
Oracle pins against the paper's worked example and closed forms (CPU); host generator of the C ABI vs the oracle (CPU);
one GPU case: probes made from a parallelogram scan match the oracle's probes."""
import numpy as np
import pytest

from test_oracle_pins import golden


@pytest.fixture(scope="module")
def lib():
    from paper_2607_02236_b200 import binding, build
    build.build_lib()
    return binding.load_library()


# ------------------------------------------------------------------------------------- oracle pins (CPU)
def test_s1_paper_example_end_point_excluded(oracle):
    """:380 '5 scan points on interval [0.0, 1.0) would result in points {0.0, 0.2, 0.4, 0.6, 0.8}'."""
    g = golden()
    xy = oracle.scan_positions("box", (5, 1), (0.0, 0.0), (1.0, 1.0))
    assert np.allclose(xy[:, 0], g["scan_5pts_unit_interval"], rtol=0, atol=1e-15)
    assert np.all(xy[:, 1] == 0.0)
    xy = oracle.scan_positions("box", (1, 5), (0.0, 0.0), (1.0, 1.0))
    assert np.allclose(xy[:, 1], g["scan_5pts_unit_interval"], rtol=0, atol=1e-15)


def test_s2_listing1_box(oracle):
    """Listing 1: 16 x 16 points over [0, 4.66179)^2: spacing a/16, last point a - a/16, first axis outer."""
    g = golden()
    a = g["scan_listing1_box_end_A"]
    xy = oracle.scan_positions("box", (16, 16), (0.0, 0.0), (a, a))
    assert xy.shape == (256, 2)
    assert xy[0].tolist() == [0.0, 0.0]
    assert xy[1].tolist() == [0.0, a / 16] and xy[16].tolist() == [a / 16, 0.0]
    assert np.isclose(xy[:, 0].max(), a * 15 / 16, rtol=1e-15) and xy.max() < a
    # unique positions, all on the lattice a/16 * integers
    assert len({tuple(r) for r in np.round(xy * 16 / a).astype(int).tolist()}) == 256


def test_s3_modes_reduce_to_each_other(oracle):
    """box_relative = box in units of the cell; unitcell = box of one cell from the origin; an axis-aligned parallelogram
    = box; a sheared parallelogram keeps the area and the point count (lattice determinant)."""
    rng = np.random.default_rng(5)
    o, e = rng.uniform(0, 3, 2), rng.uniform(4, 9, 2)
    cell = (36.752, 45.94)
    box = oracle.scan_positions("box", (7, 4), o, e)
    rel = oracle.scan_positions("box_relative", (7, 4), o / cell, e / cell, cell=cell)
    assert np.allclose(box, rel, rtol=0, atol=1e-13)
    uc = oracle.scan_positions("unitcell", (7, 4), o, e - o)
    assert np.allclose(box, uc, rtol=0, atol=1e-13)
    par = oracle.scan_positions("parallelogram", (7, 4), o, (e[0] - o[0], 0.0), (0.0, e[1] - o[1]))
    assert np.allclose(box, par, rtol=0, atol=1e-13)
    a, b = np.array([3.0, 1.0]), np.array([-0.5, 2.0])
    sh = oracle.scan_positions("parallelogram", (6, 5), (1.0, 2.0), a, b)
    # solve for the fractional coordinates: they must be exactly the grid i/6, j/5
    M = np.stack([a, b], axis=1)
    frac = np.linalg.solve(M, (sh - np.array([1.0, 2.0])).T).T
    ii, jj = np.meshgrid(np.arange(6) / 6, np.arange(5) / 5, indexing="ij")
    assert np.allclose(frac[:, 0], ii.ravel(), atol=1e-13) and np.allclose(frac[:, 1], jj.ravel(), atol=1e-13)


def test_s4_batches_partition_the_scan(oracle):
    """Listing 1: a 16 x 16 scan in batches of [4, 8] = 4 x 2 tiles of 32 points; tiles partition the scan; ragged edges."""
    g = golden()
    bs = [int(v) for v in g["scan_listing1_batch_shape"]]
    tiles = oracle.scan_batches((16, 16), bs)
    assert len(tiles) == 8 and all(t.size == 32 for t in tiles)
    assert np.array_equal(np.sort(np.concatenate(tiles)), np.arange(256))
    assert tiles[0][:9].tolist() == [0, 1, 2, 3, 4, 5, 6, 7, 16]        # 4 rows x 8 columns, row-major
    assert tiles[1][0] == 8 and tiles[2][0] == 64
    rag = oracle.scan_batches((5, 7), (2, 3))
    assert [t.size for t in rag] == [6, 6, 2, 6, 6, 2, 3, 3, 1]
    assert np.array_equal(np.sort(np.concatenate(rag)), np.arange(35))


# ------------------------------------------------------------------------------------- C ABI host helpers vs oracle (CPU)
@pytest.mark.parametrize("mode", ["box", "box_relative", "unitcell", "parallelogram"])
def test_make_scan_matches_oracle(lib, oracle, mode):
    from paper_2607_02236_b200 import binding
    rng = np.random.default_rng(11)
    for shape in [(1, 1), (5, 1), (16, 16), (3, 32), (32, 32)]:
        o, a, b = rng.uniform(-2, 5, 2), rng.uniform(1, 9, 2), rng.uniform(-3, 3, 2)
        cell = (36.752, 55.128)
        if mode == "box_relative":
            o, a = o / 10, a / 10
        ours = binding.make_scan(mode, shape, o, a, b, cell)
        ref = oracle.scan_positions(mode, shape, o, a, b, cell)
        assert ours.shape == ref.shape
        assert np.max(np.abs(ours - ref)) <= 4e-15 * max(1.0, np.max(np.abs(ref)))


def test_make_scan_rejects_bad_arguments(lib):
    from paper_2607_02236_b200 import binding
    with pytest.raises(binding.TacawError):
        binding.make_scan("box", (0, 4), (0, 0), (1, 1))
    with pytest.raises(binding.TacawError):
        binding.make_scan("parallelogram", (2, 2), (0, 0), (1, 0), None)
    with pytest.raises(binding.TacawError):
        binding.make_scan("box_relative", (2, 2), (0, 0), (1, 1), None, None)


def test_scan_batch_matches_oracle(lib, oracle):
    from paper_2607_02236_b200 import binding
    for shape, bs in [((16, 16), (4, 8)), ((5, 7), (2, 3)), ((8, 8), (8, 8)), ((3, 3), (5, 5)), ((32, 32), (8, 16))]:
        ref = oracle.scan_batches(shape, bs)
        for t, r in enumerate(ref):
            idx, nb = binding.scan_batch(shape, bs, t)
            assert nb == len(ref)
            assert idx.dtype == np.int32 and np.array_equal(idx, r)
        with pytest.raises(binding.TacawError):
            binding.scan_batch(shape, bs, len(ref))


# ------------------------------------------------------------------------------------- GPU: scan -> probes
@pytest.mark.gpu
def test_probes_of_a_parallelogram_scan_match_oracle(oracle):
    """tacaw_make_scan -> tacaw_make_probes on the GPU vs oracle.scan_positions -> oracle.make_probes (O4), 60 kV
    (the paper's beam energy, Listing 1 :411), sheared 6 x 5 scan that crosses the cell boundary."""
    import torch
    from paper_2607_02236_b200 import binding
    n, L, lam, alpha = 128, 18.376, 0.0486606, 30e-3
    args = ("parallelogram", (6, 5), (16.0, 0.5), (3.0, 1.0), (-0.5, 2.0))
    xy = binding.make_scan(*args)
    ref_xy = oracle.scan_positions(*args)
    t = binding.Tacaw(n, n, L, L, lam, 1.0e-3, bandlimit=1)
    try:
        waves = torch.empty((xy.shape[0], n, n), dtype=torch.complex64, device="cuda")
        t.make_probes(xy, alpha, waves)
        torch.cuda.synchronize()
        ours = waves.cpu().numpy().astype(np.complex128)
    finally:
        t.close()
    ref = oracle.make_probes(n, n, L, L, lam, ref_xy, alpha)
    for p in range(xy.shape[0]):
        err = np.linalg.norm(ours[p] - ref[p]) / np.linalg.norm(ref[p])
        assert err <= 2e-4, (p, err)
