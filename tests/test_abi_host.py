"""-m "not gpu": the C-ABI library loads, exports every symbol include/pab.h declares, and its host-only
logic (plan, tap design, argument checks, frame sharding) behaves.  No compute call is made here."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_2203_14906_b200 import synth

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def binding():
    from paper_2203_14906_b200 import binding as b
    b.load(build_if_missing=True)
    return b


def test_library_exports_every_declared_symbol(binding):
    header = open(os.path.join(ROOT, "include", "pab.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = sorted(set(re.findall(r"\b(pab_[a-z_0-9]+)\s*\(", header)))
    assert declared == sorted(binding.SYMBOLS)
    L = binding.load()
    for name in declared:
        assert getattr(L, name) is not None
    assert binding.load().pab_version().decode().startswith("pab ")


def test_error_strings_and_null_handling(binding):
    L = binding.load()
    assert L.pab_strerror(0) == b"ok"
    for code in (-1, -2, -3, -4):
        assert L.pab_strerror(code) not in (b"ok", b"unknown error code")
    L.pab_destroy(None)                                             # documented no-op
    assert L.pab_beamform(None, None, 1, 3, None, None) == binding.ERR_INVALID
    assert L.pab_beamform_host(None, None, 1, 3, None) == binding.ERR_INVALID
    assert L.pab_set_input(None, 0, 1.0) == binding.ERR_INVALID
    assert L.pab_launch_count(None) == 0


def test_create_rejects_bad_arguments_and_needs_a_device(binding):
    import torch
    L = binding.load()
    h = C.c_void_p()
    g = synth.geometry("C1")
    gr = binding.Grid(g.nx, g.nz, g.x0, g.dx, g.z0, g.dz)
    assert L.pab_create(C.byref(h), 0, g.n_samp, g.fs, g.c, g.pitch, C.byref(gr)) == binding.ERR_INVALID
    assert L.pab_create(C.byref(h), g.n_elem, 1, g.fs, g.c, g.pitch, C.byref(gr)) == binding.ERR_INVALID
    assert L.pab_create(C.byref(h), g.n_elem, g.n_samp, -1.0, g.c, g.pitch, C.byref(gr)) == binding.ERR_INVALID
    assert L.pab_create(C.byref(h), g.n_elem, g.n_samp, g.fs, g.c, g.pitch, None) == binding.ERR_INVALID
    bad = binding.Grid(g.nx, 0, g.x0, g.dx, g.z0, g.dz)
    assert L.pab_create(C.byref(h), g.n_elem, g.n_samp, g.fs, g.c, g.pitch, C.byref(bad)) == binding.ERR_INVALID
    assert not h
    if not torch.cuda.is_available():
        # no CPU fallback: without a device the product path fails loudly
        assert L.pab_create(C.byref(h), g.n_elem, g.n_samp, g.fs, g.c, g.pitch, C.byref(gr)) == binding.ERR_DEVICE
        with pytest.raises(binding.PabError):
            binding.Beamformer(g)


@pytest.mark.parametrize("cfg", ["C1", "C2", "C3", "C4", "C5"])
def test_plan_bounds_every_tile_window(binding, cfg):
    """The staged kernel's per-channel window bound must cover the true index span of every tile."""
    g = synth.geometry(cfg)
    p = binding.plan(g)
    assert p["tile_z"] == 64 and p["tile_x"] == 8
    assert p["batch_frames"] % 16 == 0 and 16 <= p["batch_frames"] <= 256
    assert p["batch_frames"] * g.n_elem * g.n_samp * 4 <= 512 * 2 ** 20 or p["batch_frames"] == 16
    assert p["frames_per_thread"] == 16 and p["in_range"] == (0 if cfg == "C1" else 1)   # C1 starts at z = 0
    assert 0 < p["smem_bytes"] <= 232448
    assert 1 <= p["chunk_channels"] <= min(32, g.n_elem) and p["stages"] in (2, 3)
    assert p["window_samples"] % 4 == 0
    # brute-force the worst tile: idx span over the tile corners for every element
    xe = g.elem_x()
    k = g.fs / g.c
    worst = 0.0
    for r0 in range(0, g.nz, 64):
        z = (g.z0 + np.array([r0, min(r0 + 63, g.nz - 1)]) * g.dz) * k
        for c0 in range(0, g.nx, 8):
            xs = (g.x0 + np.arange(c0, min(c0 + 8, g.nx)) * g.dx)[:, None] * k - xe[None, :] * k     # [cols][N]
            lo = np.sqrt(np.min(np.abs(xs), axis=0) ** 2 + z[0] ** 2)
            lo = np.where((xs.min(axis=0) <= 0) & (xs.max(axis=0) >= 0), z[0], lo)
            hi = np.sqrt(np.max(np.abs(xs), axis=0) ** 2 + z[1] ** 2)
            worst = max(worst, float(np.max(hi - lo)))
    assert worst + 12 <= p["window_samples"] + 4 or p["window_samples"] >= g.n_samp
    assert p["window_samples"] >= worst + 8 or p["window_samples"] >= g.n_samp


def test_plan_shrinks_with_smaller_shared_memory(binding):
    g = synth.geometry("C2")
    big, small = binding.plan(g), binding.plan(g, smem_limit=64 * 1024)
    assert small["smem_bytes"] <= 64 * 1024 and small["chunk_channels"] < big["chunk_channels"]
    tiny = binding.plan(g, smem_limit=1024)
    assert tiny["smem_bytes"] == 0 and tiny["chunk_channels"] == 0       # staged kernel does not fit


def test_library_taps_match_oracle_taps(binding, orc):
    """P10: taps designed independently by the library (fp64 -> fp32) and by the oracle agree to 1e-7."""
    for T, lo, hi in ((64, 0.1875, 0.3125), (31, 0.05, 0.45), (8, 0.0, 0.25)):
        h = binding.design_bandpass(T, lo, hi)
        ref = orc.bandpass_taps(T, lo, hi)
        assert np.max(np.abs(h - ref)) <= 1e-7
        assert np.allclose(h, h[::-1], atol=1e-7)
    for L_ in (31, 10, 1):
        g = binding.design_hilbert(L_)
        ref = orc.hilbert_taps(L_)
        assert np.max(np.abs(g - ref)) <= 1e-7
        assert np.all(g[L_ % 2::2] == 0) if L_ % 2 == 0 else True
        assert np.allclose(g, -g[::-1], atol=0)
    L = binding.load()
    buf = (C.c_float * 4)()
    assert L.pab_design_bandpass(1, 0.1, 0.2, buf) == binding.ERR_INVALID
    assert L.pab_design_bandpass(4, 0.3, 0.2, buf) == binding.ERR_INVALID
    assert L.pab_design_hilbert(0, buf) == binding.ERR_INVALID


def test_shard_frames_partitions_exactly(binding):
    for n in (1, 7, 64, 1024, 3):
        for world in (1, 2, 3, 8):
            spans = [binding.shard_frames(n, r, world) for r in range(world)]
            covered = [f for lo, hi in spans for f in range(lo, hi)]
            assert covered == list(range(n))
            sizes = [hi - lo for lo, hi in spans]
            assert max(sizes) - min(sizes) <= 1
