"""The seeded generator: shapes, determinism and the recipe of DESIGN.md / SURVEY.md §8(d)."""
import math

import numpy as np
import pytest

from paper_2203_14906_b200 import synth


def test_pulse_shapes():
    f0 = 5e6
    sigma = 1 / (2 * math.pi * f0)
    tau = np.linspace(-6 * sigma, 6 * sigma, 20001)
    g = synth.pulse_point(tau, f0)
    assert np.max(np.abs(g)) == pytest.approx(1.0, abs=1e-6)
    assert tau[np.argmax(g)] == pytest.approx(-sigma, rel=1e-3)      # positive lobe first
    assert np.allclose(g, -g[::-1])                                   # odd
    d = synth.pulse_disc(tau, f0, 0.3e-3, 1540.0)
    assert np.max(np.abs(d)) == pytest.approx(1.0, abs=1e-3)
    assert np.allclose(d, -d[::-1], atol=1e-9)


@pytest.mark.parametrize("cfg,shape,dtype", [("C1", (1, 16, 1024), np.float32), ("C3", (2, 128, 2048), np.float32),
                                              ("C5", (2, 192, 3072), np.int16)])
def test_shapes_and_determinism(cfg, shape, dtype):
    a = synth.make_config(cfg, n_frames=shape[0])
    b = synth.make_config(cfg, n_frames=shape[0])
    assert a.rf.shape == shape and a.rf.dtype == dtype
    assert np.array_equal(a.rf, b.rf)
    c = synth.make_config(cfg, seed=5, n_frames=shape[0])
    assert not np.array_equal(a.rf, c.rf)


def test_noise_level_c1():
    w = synth.make_config("C1")
    # peak-based SNR (A16): noise sigma = peak * 10^(-20/20) = 0.1 * peak of the clean frame (peak ~ 1..3 with overlap)
    quiet = w.rf[0][:, :150]                                           # before any arrival (z >= 8 mm -> n >= 207)
    assert 0.08 < quiet.std() < 0.35


def test_int16_counts_range():
    w = synth.make_config("C5", n_frames=1)
    assert np.abs(w.rf).max() <= 32767
    assert 200 <= np.abs(w.rf).max() <= 6000
    assert 6.0 < w.rf[0][:, :200].astype(np.float64).std() < 10.0       # sigma = 8 counts


def test_geometry_in_range_for_all_configs():
    """Every named config keeps every (pixel, element) delay inside the record (DESIGN.md input recipe)."""
    for cfg in ("C1", "C2", "C3", "C4", "C5"):
        g = synth.geometry(cfg)
        xe = g.elem_x()
        xmax = max(abs(g.pix_x()[0] - xe[-1]), abs(g.pix_x()[-1] - xe[0]))
        zmax = g.pix_z()[-1]
        assert g.fs * math.hypot(xmax, zmax) / g.c + 1 < g.n_samp - 1, cfg
