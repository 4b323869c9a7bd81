"""Pins for the oracle's delay / interpolation / image assembly (O1-O5).

P1: order 1 == separately written DAS loop, bitwise.
P3: on all of C1 (16 elements) route A (brute force) == route B == route C.
P4: constant RF -> C(N,k)*a on every pixel.
P7: RF linear in time -> closed-form DAS.
P8: a noiseless point absorber on a pixel centre peaks at that pixel, all orders; order-1 peak ~ N * pulse peak.
Library pin: delayed samples == numpy np.interp evaluated at numpy-computed delays.
"""
import math

import numpy as np
import pytest

from paper_2203_14906_b200 import synth


@pytest.fixture(scope="module")
def c1():
    return synth.make_config("C1")


def test_delays_and_gather_against_numpy(orc, c1):
    g = c1.geom
    xe = g.elem_x()
    X, Z = np.meshgrid(g.pix_x(), g.pix_z())                      # [nz][nx]
    idx_np = g.fs * np.sqrt((X[..., None] - xe) ** 2 + Z[..., None] ** 2) / g.c
    idx = orc.delays(g)
    assert np.max(np.abs(idx - idx_np)) < 1e-9
    # independent interpolation by the library routine np.interp, channel by channel
    s = orc.gather(c1.rf, g, frame=0)
    n = np.arange(g.n_samp)
    for i in range(g.n_elem):
        ref = np.interp(idx_np[..., i].ravel(), n, c1.rf[0, i].astype(np.float64)).reshape(g.nz, g.nx)
        inside = np.floor(idx_np[..., i]) + 1 <= g.n_samp - 1
        assert np.all(inside)   # C1 is fully in range
        assert np.max(np.abs(s[..., i] - ref)) < 1e-12


def test_element_positions_centred(orc):
    L = orc.lib()
    assert L.orc_elem_x(0, 16, 0.3e-3) == pytest.approx(-7.5 * 0.3e-3)
    assert L.orc_elem_x(15, 16, 0.3e-3) == pytest.approx(7.5 * 0.3e-3)
    assert L.orc_elem_x(2, 5, 1.0) == 0.0


def test_order1_equals_das_bitwise(orc, c1):
    a = orc.beamform(c1.rf, c1.geom, 1)
    b = orc.das(c1.rf, c1.geom)
    assert np.array_equal(a, b)


@pytest.mark.parametrize("k", [2, 3, 4, 5])
def test_c1_brute_equals_recurrence_equals_closed(orc, c1, k):
    a = orc.beamform(c1.rf, c1.geom, k, route=orc.ROUTE_BRUTE)
    b = orc.beamform(c1.rf, c1.geom, k, route=orc.ROUTE_RECUR)
    c = orc.beamform(c1.rf, c1.geom, k, route=orc.ROUTE_CLOSED)
    peak = np.max(np.abs(a))
    assert np.max(np.abs(a - b)) <= 1e-12 * peak
    assert np.max(np.abs(a - c)) <= 1e-10 * peak


@pytest.mark.parametrize("k", [1, 2, 3, 4, 5])
def test_constant_rf_closed_form(orc, k):
    g = synth.geometry("C1")
    a = -2.5
    rf = np.full((1, g.n_elem, g.n_samp), a, dtype=np.float32)
    img = orc.beamform(rf, g, k)
    exp = math.comb(g.n_elem, k) * (a if k % 2 else abs(a))
    assert np.allclose(img, exp, rtol=1e-12)


def test_linear_ramp_das_closed_form(orc):
    """P7: rf_i[n] = a_i*n + b_i is reproduced exactly by linear interpolation, so DAS = sum_i (a_i*idx_i + b_i)."""
    g = synth.geometry("C1")
    rng = np.random.default_rng(5)
    a = rng.uniform(-1, 1, g.n_elem)
    b = rng.uniform(-10, 10, g.n_elem)
    n = np.arange(g.n_samp)
    rf64 = a[:, None] * n[None, :] + b[:, None]
    rf = rf64.astype(np.float32)[None]
    idx = orc.delays(g)
    # closed form with the float32-rounded ramp: per-channel slope/intercept are not exactly linear after rounding,
    # so build the expectation from the exact piecewise-linear interpolant's bound instead: error <= max rounding step
    exp = np.sum(a * idx + b, axis=-1)
    img = orc.beamform(rf, g, 1)[0]
    assert np.max(np.abs(img - exp)) < g.n_elem * 1024 * 2.0 ** -24 * 2


def test_out_of_record_contributes_zero(orc):
    """A6: deep rows whose delays exceed the record give 0 for those channels."""
    g0 = synth.geometry("C1")
    g = synth.Geometry(g0.n_elem, 256, g0.fs, g0.c, g0.pitch, g0.nx, g0.nz, g0.x0, g0.dx, g0.z0, g0.dz)
    rf = np.ones((1, g.n_elem, g.n_samp), dtype=np.float32)
    idx = orc.delays(g)
    valid = (np.floor(idx) + 1 <= g.n_samp - 1)
    img = orc.beamform(rf, g, 1)[0]
    assert np.array_equal(img, valid.sum(-1).astype(np.float64))
    assert img.min() == 0 and img.max() == g.n_elem
    img3 = orc.beamform(rf, g, 3)[0]
    nv = valid.sum(-1)
    exp3 = np.array([[math.comb(int(v), 3) for v in row] for row in nv], dtype=np.float64)
    assert np.allclose(img3, exp3, rtol=1e-12)


@pytest.mark.parametrize("k", [1, 2, 3, 4, 5])
def test_point_absorber_peaks_at_its_pixel(orc, k):
    """P8: fixes the sign and origin conventions of O1-O3 (A5): one-way delay, t = 0 at sample 0, array centred."""
    g = synth.geometry("C1")
    ix, iz = 9, 70
    rf = synth.point_target_frame(g, ix, iz, f0=2e6, shape="gauss")     # unipolar, sigma_t = 3.2 samples
    img = orc.beamform(rf, g, k)[0]
    m, j = np.unravel_index(np.argmax(img), img.shape)
    assert (m, j) == (iz, ix)
    # every channel is delayed onto the pulse maximum: all N samples ~ 1, so every k-subset term ~ 1
    assert img[iz, ix] == pytest.approx(math.comb(g.n_elem, k), rel=0.02)
    assert img[iz, ix] <= math.comb(g.n_elem, k)


def test_n_pulse_zero_crossing_at_absorber(orc):
    """The workloads' bipolar pulse is odd about its arrival time: DAS changes sign across the absorber row."""
    g0 = synth.geometry("C1")
    # fine depth grid (one row per sample) around the absorber so the two lobes are resolved
    dz = g0.c / g0.fs
    g = synth.Geometry(g0.n_elem, g0.n_samp, g0.fs, g0.c, g0.pitch, 3, 41, -g0.dx, g0.dx, 15e-3 - 20 * dz, dz).f32()
    rf = synth.point_target_frame(g, 1, 20)
    col = orc.beamform(rf, g, 1)[0][:, 1]
    assert abs(col[20]) < 0.05 * np.max(np.abs(col))
    assert col[19] * col[21] < 0
    # g(tau) = -(tau/sigma) exp(..): positive lobe arrives first (shallower rows), peak one sigma = 1.27 samples away
    assert col[19] > 0 > col[21]
    assert 0.8 * g.n_elem < np.max(np.abs(col)) <= g.n_elem   # linear interpolation of a 8-samples-per-period pulse


def test_channel_reversal_symmetry(orc, c1):
    """P6: reversing the channel order and mirroring the grid about x = 0 leaves the image mirrored."""
    g = c1.geom
    gm = synth.Geometry(g.n_elem, g.n_samp, g.fs, g.c, g.pitch, g.nx, g.nz,
                        -(g.x0 + (g.nx - 1) * g.dx), g.dx, g.z0, g.dz)
    for k in (1, 3, 4):
        a = orc.beamform(c1.rf, g, k)[0]
        b = orc.beamform(np.ascontiguousarray(c1.rf[:, ::-1, :]), gm, k)[0]
        assert np.allclose(a, b[:, ::-1], rtol=1e-9, atol=1e-9 * np.max(np.abs(a)))


def test_int16_input_exact(orc):
    """A15: int16 counts convert exactly; same image as the float32 copy of the same counts."""
    g = synth.geometry("C1")
    rng = np.random.default_rng(11)
    rf16 = rng.integers(-2000, 2000, size=(2, g.n_elem, g.n_samp)).astype(np.int16)
    a = orc.beamform(rf16, g, 3)
    b = orc.beamform(rf16.astype(np.float32), g, 3)
    assert np.array_equal(a, b)


def test_beamform_pixels_matches_full(orc, c1):
    pix = np.array([[0, 0], [5, 3], [127, 15], [64, 8]], dtype=np.int32)
    full = orc.beamform(c1.rf, c1.geom, 3)
    sub = orc.beamform_pixels(c1.rf, c1.geom, 3, pix)
    assert np.array_equal(sub[0], full[0, pix[:, 0], pix[:, 1]])


def test_subaperture_brute_on_large_config(orc):
    """Route A on a 12-element sub-aperture of sampled C2 pixels pins route B where full brute force is unaffordable."""
    w = synth.make_config("C2")
    g = w.geom
    # gather only a few pixels: build a tiny grid that addresses them
    rng = np.random.default_rng(21)
    for _ in range(6):
        m, j = int(rng.integers(g.nz)), int(rng.integers(g.nx))
        gp = synth.Geometry(g.n_elem, g.n_samp, g.fs, g.c, g.pitch, 1, 1, g.x0 + j * g.dx, g.dx, g.z0 + m * g.dz, g.dz)
        s = orc.gather(w.rf, gp)[0, 0]
        sub = s[rng.choice(g.n_elem, 12, replace=False)]
        for k in (3, 4, 5):
            a = orc.combine(sub, k, orc.ROUTE_BRUTE)
            b = orc.combine(sub, k, orc.ROUTE_RECUR)
            assert abs(a - b) <= 1e-11 * max(1.0, abs(a))
