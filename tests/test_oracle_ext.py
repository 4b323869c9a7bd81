"""-m "not gpu": pins of the oracle's section 8(f) options: coherence-factor weighting (f1, reading A20) and
nearest-sample delays (f4, reading A21).  Nothing here comes from the CUDA path."""
import math

import numpy as np
import pytest

from paper_2203_14906_b200 import synth


@pytest.fixture(scope="module")
def c1():
    return synth.make_config("C1", n_frames=2)


def test_ex_defaults_equal_plain_beamform_bitwise(orc, c1):
    for k in (1, 3, 4):
        assert np.array_equal(orc.beamform_ex(c1.rf, c1.geom, k), orc.beamform(c1.rf, c1.geom, k))


def test_cf_hand_values(orc):
    # (1 + 2 + 3)^2 / (3 (1 + 4 + 9)) = 36 / 42 = 6/7, by hand
    assert orc.coherence_factor([1.0, 2.0, 3.0]) == pytest.approx(6.0 / 7.0, rel=1e-15)
    assert orc.coherence_factor([2.5] * 9) == pytest.approx(1.0, rel=1e-15)          # equal samples: fully coherent
    assert orc.coherence_factor([1.0, -1.0, 3.0, -3.0]) == 0.0                        # zero mean: incoherent
    assert orc.coherence_factor([0.0, 0.0, 0.0]) == 0.0                               # all zero: defined as 0
    # one non-zero channel of N: CF = 1/N (zeros count, A6)
    assert orc.coherence_factor([0.0, 0.0, 4.0, 0.0]) == pytest.approx(0.25, rel=1e-15)


def test_cf_bounds_scale_and_permutation_invariance(orc):
    rng = np.random.default_rng(3)
    for _ in range(50):
        s = rng.standard_normal(17)
        cf = orc.coherence_factor(s)
        assert 0.0 <= cf <= 1.0
        assert orc.coherence_factor(-3.7 * s) == pytest.approx(cf, rel=1e-13)
        assert orc.coherence_factor(rng.permutation(s)) == pytest.approx(cf, rel=1e-13)
        assert cf == pytest.approx(np.mean(s) ** 2 / np.mean(s ** 2), rel=1e-12)     # the same ratio, in numpy


@pytest.mark.parametrize("k", [1, 2, 3, 4, 5])
def test_cf_weighted_image(orc, c1, k):
    g = c1.geom
    plain = orc.beamform(c1.rf, g, k)
    cfw = orc.beamform_ex(c1.rf, g, k, weight="cf")
    s = orc.gather(c1.rf, g, frame=1)                                    # [nz][nx][N] delayed samples
    cf = np.mean(s, axis=-1) ** 2 / np.maximum(np.mean(s ** 2, axis=-1), 1e-300)
    assert np.allclose(cfw[1], cf * plain[1], rtol=1e-11, atol=1e-11 * np.abs(plain).max())
    assert np.all(np.abs(cfw) <= np.abs(plain) * (1 + 1e-12))            # CF <= 1 never amplifies
    # constant RF: CF = 1 on every fully in-range pixel, so the binomial closed form P4 still holds
    rf = np.full_like(c1.rf, -2.5)
    img = orc.beamform_ex(rf, g, k, weight="cf")
    full = np.all(orc.delays(g) < g.n_samp - 1.001, axis=-1) & np.all(orc.delays(g) >= 0, axis=-1)
    expect = math.comb(g.n_elem, k) * (-2.5 if k % 2 else 2.5)
    assert np.allclose(img[0][full], expect, rtol=1e-11)
    # homogeneity survives the weighting: CF is scale invariant
    a = orc.beamform_ex((2.0 * c1.rf).astype(np.float32), g, k, weight="cf")
    assert np.allclose(a, 2.0 * cfw, rtol=1e-11, atol=1e-12 * np.abs(cfw).max())


def test_nearest_index_and_gather_against_numpy(orc, c1):
    g = c1.geom
    xe = g.elem_x()
    x = g.pix_x()[None, :, None]
    z = g.pix_z()[:, None, None]
    idx = g.fs * np.sqrt((x - xe[None, None, :]) ** 2 + z ** 2) / g.c
    n = np.floor(idx + 0.5).astype(np.int64)
    ok = (n >= 0) & (n <= g.n_samp - 1)
    assert np.array_equal(orc.nearest_index(g), np.where(ok, n, -1))
    # DAS with nearest samples == numpy fancy-indexed gather, summed over elements
    rf = c1.rf[0].astype(np.float64)
    gathered = np.where(ok, rf[np.arange(g.n_elem)[None, None, :], np.clip(n, 0, g.n_samp - 1)], 0.0)
    img = orc.beamform_ex(c1.rf[:1], g, 1, interp="nearest")[0]
    assert np.allclose(img, gathered.sum(-1), rtol=1e-13, atol=1e-13)
    # order 3 on the same gathered samples through the combination pin (route B on numpy-gathered samples)
    img3 = orc.beamform_ex(c1.rf[:1], g, 3, interp="nearest")[0]
    for (m, j) in ((0, 0), (57, 9), (127, 15)):
        assert img3[m, j] == pytest.approx(orc.combine(gathered[m, j], 3), rel=1e-13)


def test_nearest_staircase_closed_form(orc):
    """RF = sample index n on every channel: nearest-sample DAS is sum_i round(idx_i) exactly; linear
    interpolation gives sum_i idx_i (P7); they differ by at most N/2."""
    g = synth.random_geometry(np.random.default_rng(8), 9, 600, 7, 33, in_range=True)
    rf = np.tile(np.arange(g.n_samp, dtype=np.float32), (1, g.n_elem, 1))
    idx = orc.delays(g)
    near = orc.beamform_ex(rf, g, 1, interp="nearest")[0]
    lin = orc.beamform_ex(rf, g, 1, interp="linear")[0]
    assert np.array_equal(near, np.floor(idx + 0.5).sum(-1))
    assert np.allclose(lin, idx.sum(-1), rtol=1e-12)
    assert np.max(np.abs(near - lin)) <= g.n_elem / 2


def test_nearest_out_of_record_is_zero(orc):
    g = synth.random_geometry(np.random.default_rng(9), 5, 200, 6, 40, in_range=False)
    rf = np.ones((1, g.n_elem, g.n_samp), dtype=np.float32)
    img = orc.beamform_ex(rf, g, 1, interp="nearest")[0]
    inside = (orc.nearest_index(g) >= 0).sum(-1)
    assert np.array_equal(img, inside.astype(np.float64)) and inside.min() < g.n_elem


# ---- row f2: orders above 5 ("this can be done for higher orders as well") ----
@pytest.mark.parametrize("k", [6, 7, 8])
def test_high_orders_recurrence_equals_definition(orc, k):
    """Route B (the reference for the GPU) against route A, the definition: all k-subsets, signed k-th root of the
    product of the un-rooted samples, the pattern of eqs. (2), (4)-(6) continued."""
    import itertools
    rng = np.random.default_rng(60 + k)
    for n in (k, k + 1, 11):
        s = rng.standard_normal(n) * 10.0 ** rng.uniform(-2, 2)
        a = orc.combine(s, k, route=orc.ROUTE_BRUTE)
        b = orc.combine(s, k, route=orc.ROUTE_RECUR)
        py = sum(math.copysign(abs(math.prod(c)) ** (1.0 / k), math.prod(c)) for c in itertools.combinations(s, k))
        assert a == pytest.approx(py, rel=1e-11, abs=1e-12 * abs(py))
        assert b == pytest.approx(a, rel=1e-10, abs=1e-11 * np.max(np.abs(s)) * math.comb(n, k))
    # fewer than k non-zero samples: exactly zero; constant samples: C(n, k) a or C(n, k) |a|
    z = np.zeros(12); z[:k - 1] = rng.standard_normal(k - 1)
    assert orc.combine(z, k) == 0.0
    c = np.full(13, -1.75)
    assert orc.combine(c, k) == pytest.approx(math.comb(13, k) * (-1.75 if k % 2 else 1.75), rel=1e-12)


@pytest.mark.parametrize("k", [6, 8])
def test_high_orders_image_homogeneity(orc, c1, k):
    img = orc.beamform(c1.rf[:1], c1.geom, k)
    twice = orc.beamform((-2.0 * c1.rf[:1]).astype(np.float32), c1.geom, k)
    assert np.allclose(twice, 2.0 * img, rtol=1e-10, atol=1e-12 * np.abs(img).max())        # even k: x |alpha|


# ---- row f3: image-quality metrics, eqs. (10)-(12) and FWHM (reading A22) ----
def test_metrics_against_numpy(orc):
    rng = np.random.default_rng(70)
    img = np.abs(rng.standard_normal((90, 70))).astype(np.float32)
    img[20:40, 10:30] += 5.0
    tgt, bkg = (20, 40, 10, 30), (50, 85, 35, 69)
    m = orc.image_metrics(img, tgt, bkg, n_bins=64, fwhm_row=30, dx=0.25e-3)
    a = img[20:40, 10:30].astype(np.float64)
    b = img[50:85, 35:69].astype(np.float64)
    assert m["mu_in"] == pytest.approx(a.mean(), rel=1e-13) and m["mu_out"] == pytest.approx(b.mean(), rel=1e-13)
    assert m["sigma_out"] == pytest.approx(b.std(), rel=1e-12)
    assert m["snr_db"] == pytest.approx(20 * np.log10(a.mean() / b.std()), rel=1e-12)          # eq. (10)
    assert m["cr_db"] == pytest.approx(20 * np.log10(a.mean() / b.mean()), rel=1e-12)          # eq. (11)
    vmax = max(a.max(), b.max())
    ha, _ = np.histogram(a / vmax, bins=64, range=(0.0, 1.0))
    hb, _ = np.histogram(b / vmax, bins=64, range=(0.0, 1.0))
    gc = 1.0 - np.minimum(ha / a.size, hb / b.size).sum()
    assert m["gcnr"] == pytest.approx(gc, abs=2.0 / min(a.size, b.size))   # bin edges: float32 here, float64 in numpy


def test_metrics_closed_forms(orc):
    img = np.full((40, 40), 2.0, dtype=np.float32)
    img[:, 20:] = 0.5
    img[::2, 20:] = 1.5                                      # background alternates 0.5 / 1.5: mean 1, std 0.5
    m = orc.image_metrics(img, (0, 40, 0, 20), (0, 40, 20, 40), n_bins=16)
    assert m["mu_in"] == 2.0 and m["mu_out"] == 1.0 and m["sigma_out"] == 0.5
    assert m["snr_db"] == pytest.approx(20 * math.log10(4.0), rel=1e-14)
    assert m["cr_db"] == pytest.approx(20 * math.log10(2.0), rel=1e-14)
    assert m["gcnr"] == 1.0                                  # disjoint amplitude sets
    same = orc.image_metrics(img, (0, 40, 20, 40), (0, 40, 20, 40), n_bins=16)
    assert same["gcnr"] == 0.0 and same["cr_db"] == 0.0      # identical regions: full overlap
    assert math.isnan(m["fwhm_m"])                           # no row asked for


def test_fwhm_of_sampled_gaussian(orc):
    x = np.arange(101, dtype=np.float64)
    for sigma in (3.0, 7.5):
        img = np.tile(np.exp(-0.5 * ((x - 48.3) / sigma) ** 2), (3, 1)).astype(np.float32)
        m = orc.image_metrics(img, (0, 3, 0, 101), (0, 3, 0, 10), fwhm_row=1, dx=0.1e-3)
        assert m["fwhm_m"] == pytest.approx(2.0 * math.sqrt(2.0 * math.log(2.0)) * sigma * 0.1e-3, rel=1e-2)   # linear interpolation of the crossings
    tri = np.zeros((1, 21), dtype=np.float32)
    tri[0, 5:16] = [0, 2, 4, 6, 8, 10, 8, 6, 4, 2, 0]       # triangle, peak 10 at column 10: half width = 5 columns
    assert orc.image_metrics(tri, (0, 1, 0, 21), (0, 1, 0, 3), fwhm_row=0, dx=1.0)["fwhm_m"] == pytest.approx(5.0, rel=1e-14)
