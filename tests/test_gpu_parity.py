"""-m gpu: the CUDA path (through the C ABI, via the ctypes binding) against the fp64 oracle, element by element.

Tolerances are north_star's (BASELINE.json): pre-band-pass image relative L2 <= 1e-4; per pixel
|err| <= 1e-3 x image peak for orders <= 3 and <= 5e-3 x peak for orders 4, 5.  Post chain (DESIGN.md
"Tolerances"): band-pass / envelope relative L2 <= 2e-4; log image |delta| <= 0.05 dB where the oracle is
above -40 dB.  Pixels whose delay index lies within 1e-2 of the record end for some element are masked
(reading A17: the zero-outside-the-record rule is discontinuous there).
"""
import numpy as np
import pytest

from paper_2203_14906_b200 import synth

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

VARIANTS = ["direct", "staged"]


@pytest.fixture(scope="module")
def pab():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2203_14906_b200 import binding
    binding.load(build_if_missing=True)     # compiles libpab.so with nvcc if it is not there; raises if it cannot: no fallback
    return binding


def run_gpu(pab, g, rf, order, variant="auto", dtype="float32", scale=1.0, post=None, weight="none", interp="linear",
            delay_cache="off"):
    bf = pab.Beamformer(g, dtype=dtype, scale=scale, post=post, variant=variant, weight=weight, interp=interp,
                        delay_cache=delay_cache)
    try:
        out = bf.beamform(torch.from_numpy(rf).cuda(), order)
        torch.cuda.synchronize()
        return out.cpu().numpy().astype(np.float64), bf.launch_count()
    finally:
        bf.close()


def check_raw(gpu, ref, order, mask=None):
    peak = np.max(np.abs(ref))
    err = np.abs(gpu - ref)
    if mask is not None:
        err = np.where(mask, 0.0, err)
        ref = np.where(mask, 0.0, ref)
    rel_l2 = np.sqrt(np.sum(err ** 2) / np.sum(ref ** 2))
    tol_pix = (1e-3 if order <= 3 else 5e-3) * peak
    assert np.all(np.isfinite(gpu))
    assert rel_l2 <= 1e-4, f"order {order}: relative L2 {rel_l2:.3e}"
    assert np.max(err) <= tol_pix, f"order {order}: max |err| {np.max(err):.3e} > {tol_pix:.3e}"
    return rel_l2


def test_margin_on_fresh_seeds(pab, orc):
    """The tolerance must not hinge on the seeds of the named configs: other seeds of the headline workload, with
    a bound 4x tighter than north_star's.  (With the index carried to fp32 ulps of the index instead of ~1e-6
    samples, 3 % of such frames exceeded 1e-4: the signed root is not Lipschitz at 0.)"""
    for seed in (9001, 9005):
        w = synth.make_config("C2b", seed=seed, n_frames=16)
        for order in (1, 3):
            gpu, _ = run_gpu(pab, w.geom, w.rf, order)
            ref = orc.beamform(w.rf, w.geom, order)
            for f in range(16):
                assert check_raw(gpu[f], ref[f], order) <= 2.5e-5


def edge_mask(orc, g):
    idx = orc.delays(g)                                   # [nz][nx][N]
    return np.any(np.abs(idx - (g.n_samp - 1)) < 1e-2, axis=-1)


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("order", [1, 2, 3, 4, 5])
def test_c1_single_frame_all_orders(pab, orc, variant, order):
    w = synth.make_config("C1")
    gpu, launches = run_gpu(pab, w.geom, w.rf, order, variant)
    assert launches >= 1
    check_raw(gpu, orc.beamform(w.rf, w.geom, order), order)


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("n_frames", [2, 4, 5, 8, 9, 19])
def test_c1_multi_frame_batching(pab, orc, variant, n_frames):
    """Frame quads / octets + ragged remainders: every frame must equal its single-frame oracle image."""
    w = synth.make_config("C1", n_frames=n_frames)
    for order in (1, 3, 4):
        gpu, _ = run_gpu(pab, w.geom, w.rf, order, variant)
        ref = orc.beamform(w.rf, w.geom, order)
        for f in range(n_frames):
            check_raw(gpu[f], ref[f], order)


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("seed,n_elem,n_samp,nx,nz,frames", [(1, 7, 333, 13, 45, 1), (2, 33, 1001, 9, 70, 6),
                                                              (3, 24, 514, 37, 129, 12), (4, 1, 64, 3, 5, 1)])
def test_ragged_geometries_with_out_of_record_pixels(pab, orc, variant, seed, n_elem, n_samp, nx, nz, frames):
    """Odd sizes (ragged tiles, S not a multiple of 4) and grids that run past the end of the record (A6)."""
    rng = np.random.default_rng(seed)
    g = synth.random_geometry(rng, n_elem, n_samp, nx, nz, in_range=False)
    rf = rng.standard_normal((frames, n_elem, n_samp)).astype(np.float32)
    mask = edge_mask(orc, g)
    for order in (1, 2, 3, 4, 5):
        if order > n_elem:
            continue
        gpu, _ = run_gpu(pab, g, rf, order, variant)
        ref = orc.beamform(rf, g, order)
        for f in range(frames):
            check_raw(gpu[f], ref[f], order, mask)


@pytest.mark.parametrize("variant", VARIANTS)
def test_int16_input_and_scale(pab, orc, variant):
    w = synth.make_config("C5", n_frames=5)
    g = w.geom
    small = synth.Geometry(g.n_elem, g.n_samp, g.fs, g.c, g.pitch, 24, 96, g.x0, g.dx * 8, g.z0, g.dz * 8).f32()
    for order, scale in ((3, 1.0), (2, 0.125)):
        gpu, _ = run_gpu(pab, small, w.rf, order, variant, dtype="int16", scale=scale)
        ref = orc.beamform(w.rf, small, order, scale=scale)
        for f in range(5):
            check_raw(gpu[f], ref[f], order)


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("order", [1, 2, 3])
def test_c2_full_size_single_frame(pab, orc, variant, order):
    w = synth.make_config("C2")
    gpu, _ = run_gpu(pab, w.geom, w.rf, order, variant)
    check_raw(gpu[0], orc.beamform(w.rf, w.geom, order)[0], order)


@pytest.mark.parametrize("order", [1, 2, 3])
def test_c2_full_size_single_frame_default_path(pab, orc, order):
    """Config C2 through the default settings (automatic variant, no delay table): the table-free diagonal kernel
    (taps computed in the kernel on the FP64 pipe, one per diagonal), fp32 and int16 input."""
    w = synth.make_config("C2")
    bf = pab.Beamformer(w.geom)
    try:
        out = bf.beamform(torch.from_numpy(w.rf).cuda(), order)
        torch.cuda.synchronize()
        assert bf.plan()["diagonal"] == 2                      # the table-free diagonal kernel is what ran
        ref = orc.beamform(w.rf, w.geom, order)[0]
        assert check_raw(out.cpu().numpy().astype(np.float64)[0], ref, order) <= 2.5e-5
    finally:
        bf.close()
    rf16 = np.rint(w.rf * (8000.0 / np.max(np.abs(w.rf)))).astype(np.int16)
    gpu, _ = run_gpu(pab, w.geom, rf16, order, dtype="int16", scale=0.5)
    check_raw(gpu[0], orc.beamform(rf16, w.geom, order, scale=0.5)[0], order)


@pytest.mark.parametrize("delay_cache", ["all", "off"])
def test_c2b_headline_batch_sampled_pixels(pab, orc, delay_cache):
    """The launch configuration bench.py times (64 frames, order 3, auto variant, cached taps) on sampled pixels,
    and the same with in-kernel delays."""
    w = synth.make_config("C2b", n_frames=64)
    g = w.geom
    gpu, launches = run_gpu(pab, g, w.rf, 3, delay_cache=delay_cache)
    assert launches >= 2
    rng = np.random.default_rng(7)
    pix = np.stack([rng.integers(0, g.nz, 1500), rng.integers(0, g.nx, 1500)], axis=1)
    pix[:4] = [[0, 0], [g.nz - 1, g.nx - 1], [0, g.nx - 1], [g.nz - 1, 0]]
    ref = orc.beamform_pixels(w.rf, g, 3, pix)                      # [F][n_pix]
    got = gpu[:, pix[:, 0], pix[:, 1]]
    # Full images of ALL 64 frames: relative L2 <= 1e-4 and the per-pixel bound on every one (the oracle does a C2b
    # frame in ~0.1 s on the GPU box's cores).  Sampled pixels of all 64 frames through the oracle's per-pixel entry
    # point as well: the per-pixel bound against the image peak.  (No L2 on the sample: the error is heavy-tailed,
    # largest on the few bright absorber pixels, so the rms of a 1500-pixel sample is not an estimate of the image's.)
    full_peak, worst = 0.0, 0.0
    for f in range(64):
        full = orc.beamform(w.rf[f:f + 1], g, 3)[0]
        worst = max(worst, check_raw(gpu[f], full, 3))
        full_peak = max(full_peak, float(np.max(np.abs(full))))
    assert worst <= 2.5e-5, worst                         # the margin test_margin_on_fresh_seeds asks of other seeds
    assert np.max(np.abs(got - ref)) <= 1e-3 * full_peak


@pytest.mark.parametrize("variant", VARIANTS + ["auto"])
@pytest.mark.parametrize("order", [4, 5])
def test_c4_large_aperture(pab, orc, variant, order):
    """staged: the diagonal kernel with its tap table; direct: the direct kernel; auto (the default settings): the
    table-free diagonal kernel."""
    w = synth.make_config("C4")
    g = w.geom
    gpu, _ = run_gpu(pab, g, w.rf, order, variant, delay_cache="single" if variant == "staged" else "off")
    rng = np.random.default_rng(11)
    rows = np.unique(np.concatenate([[0, g.nz - 1], rng.integers(0, g.nz, 62)]))
    sub = synth.Geometry(g.n_elem, g.n_samp, g.fs, g.c, g.pitch, g.nx, 1, g.x0, g.dx, g.z0, g.dz)
    ref = np.empty((len(rows), g.nx))
    for r, m in enumerate(rows):                       # whole rows of the full-size image, one row at a time
        sub.z0 = float(np.float64(g.z0) + m * np.float64(g.dz))
        ref[r] = orc.beamform(w.rf, sub, order)[0, 0]
    got = gpu[0][rows]
    peak = np.max(np.abs(ref))
    err = np.abs(got - ref)
    assert np.sqrt(np.sum(err ** 2) / np.sum(ref ** 2)) <= 1e-4
    assert np.max(err) <= 5e-3 * peak


@pytest.mark.parametrize("cfg,frames", [("C3", 6), ("C5", 5)])
def test_post_chain_streaming_configs(pab, orc, cfg, frames):
    w = synth.make_config(cfg, n_frames=frames)
    g = w.geom
    dtype = "int16" if w.rf.dtype == np.int16 else "float32"
    raw = orc.beamform(w.rf, g, 3)
    post = {k: v for k, v in w.post.items() if k != "mode"}
    for mode in ("bandpass", "envelope", "log"):
        gpu, _ = run_gpu(pab, g, w.rf, 3, dtype=dtype, post=dict(post, mode=mode))
        ref = orc.post(raw, g, post["f_center"], post["f_halfwidth"], post["n_taps_bp"], post["n_taps_hilbert"],
                       post["dyn_range_db"], mode=mode)
        if mode == "log":
            sel = ref > -40.0
            assert np.max(np.abs(gpu - ref)[sel]) <= 0.05
            assert np.all(gpu <= 1e-4) and np.all(gpu >= -post["dyn_range_db"] - 1e-4)
            assert np.all(np.max(gpu.reshape(frames, -1), axis=1) > -1e-3)      # 0 dB at the frame max
        else:
            rel = np.sqrt(np.sum((gpu - ref) ** 2) / np.sum(ref ** 2))
            assert rel <= 2e-4, f"{cfg} {mode}: relative L2 {rel:.3e}"


def _check_log(gpu, ref, dr):
    sel = ref > -40.0
    assert np.max(np.abs(gpu - ref)[sel]) <= 0.05
    assert np.all(gpu <= 1e-4) and np.all(gpu >= -dr - 1e-4)
    assert np.max(gpu) > -1e-3                                            # 0 dB at the frame max


@pytest.mark.parametrize("delay_cache", ["all", "off"])
def test_c5_defining_shape_64_frame_int16_batch(pab, orc, delay_cache):
    """Config C5 as BASELINE.json states it: ONE 64-frame int16 batch at 768 x 192 pixels x 192 elements, order 3 with
    band-pass + envelope + log (16-frame groups on the int16 ingest path: the launch configuration bench.py --sweep
    times).  Frames 0 and 63 (first and last of the batch) in full against the oracle, before
    the band-pass (north_star's bound) and after the whole post chain; cached taps and in-kernel delays."""
    w = synth.make_config("C5", n_frames=64)
    g = w.geom
    assert w.rf.dtype == np.int16 and w.rf.shape == (64, 192, 3072)
    post = dict(w.post)
    raw, launches = run_gpu(pab, g, w.rf, 3, dtype="int16", delay_cache=delay_cache)
    assert launches >= 2
    out, _ = run_gpu(pab, g, w.rf, 3, dtype="int16", post=post, delay_cache=delay_cache)
    for f in (0, 63):
        ref = orc.beamform(w.rf[f:f + 1], g, 3)
        check_raw(raw[f], ref[0], 3)
        ref_log = orc.post(ref, g, post["f_center"], post["f_halfwidth"], post["n_taps_bp"], post["n_taps_hilbert"],
                           post["dyn_range_db"], mode="log")[0]
        _check_log(out[f], ref_log, post["dyn_range_db"])


def test_c3_defining_shape_256_frame_call(pab, orc):
    """Config C3 as stated: ONE call of 256 frames (512 x 128 pixels, order 3, post = log); frames 0, 63, 64, 255
    (first / last of the 64-frame batches) in full, raw and after the post chain."""
    w = synth.make_config("C3", n_frames=256)
    g = w.geom
    post = dict(w.post)
    raw, _ = run_gpu(pab, g, w.rf, 3, delay_cache="all")
    out, _ = run_gpu(pab, g, w.rf, 3, post=post, delay_cache="all")
    for f in (0, 63, 64, 255):
        ref = orc.beamform(w.rf[f:f + 1], g, 3)
        check_raw(raw[f], ref[0], 3)
        ref_log = orc.post(ref, g, post["f_center"], post["f_halfwidth"], post["n_taps_bp"], post["n_taps_hilbert"],
                           post["dyn_range_db"], mode="log")[0]
        _check_log(out[f], ref_log, post["dyn_range_db"])


@pytest.mark.parametrize("delay_cache", ["all", "off"])
@pytest.mark.parametrize("order", [4, 5])
def test_c4_16_frame_batch(pab, orc, order, delay_cache):
    """Config C4 in one 16-frame call (8 frames per thread at orders 4, 5: the sweep's batched rows): sampled whole
    rows of frames 0, 7, 8 and 15 of the full-size image."""
    w = synth.make_config("C4", n_frames=16)
    g = w.geom
    gpu, _ = run_gpu(pab, g, w.rf, order, delay_cache=delay_cache)
    rng = np.random.default_rng(13)
    rows = np.unique(np.concatenate([[0, g.nz - 1], rng.integers(0, g.nz, 22)]))
    sub = synth.Geometry(g.n_elem, g.n_samp, g.fs, g.c, g.pitch, g.nx, 1, g.x0, g.dx, g.z0, g.dz)
    frames = (0, 7, 8, 15)
    ref = np.empty((len(frames), len(rows), g.nx))
    for r, m in enumerate(rows):
        sub.z0 = float(np.float64(g.z0) + m * np.float64(g.dz))
        ref[:, r] = orc.beamform(w.rf[list(frames)], sub, order)[:, 0]
    for k, f in enumerate(frames):
        got = gpu[f][rows]
        err = np.abs(got - ref[k])
        assert np.sqrt(np.sum(err ** 2) / np.sum(ref[k] ** 2)) <= 1e-4, (order, f)
        assert np.max(err) <= 5e-3 * np.max(np.abs(ref[k])), (order, f)


@pytest.mark.parametrize("n_bp,n_h", [(31, 21), (64, 63), (50, 41), (96, 95)])
def test_post_chain_ragged_grid(pab, orc, n_bp, n_h):
    """Ragged grid and filter lengths on both post kernels: <= 32 and > 64 taps take the generic kernel,
    33..64 taps the constant-bank fast path (with and without the structural zeros of the Hilbert FIR)."""
    rng = np.random.default_rng(5)
    g = synth.random_geometry(rng, 12, 700, 41, 203, in_range=True)
    rf = rng.standard_normal((3, 12, 700)).astype(np.float32)
    raw = orc.beamform(rf, g, 2)
    fs_z = g.c / g.dz
    kw = dict(f_center=0.2 * fs_z, f_halfwidth=0.08 * fs_z, n_taps_bp=n_bp, n_taps_hilbert=n_h, dyn_range_db=50.0)
    for mode in ("bandpass", "envelope"):
        gpu, _ = run_gpu(pab, g, rf, 2, post=dict(kw, mode=mode))
        ref = orc.post(raw, g, kw["f_center"], kw["f_halfwidth"], n_bp, n_h, 50.0, mode=mode)
        assert np.sqrt(np.sum((gpu - ref) ** 2) / np.sum(ref ** 2)) <= 2e-4, mode


def test_host_entry_point_matches_device_entry_point(pab):
    w = synth.make_config("C1", n_frames=21)
    bf = pab.Beamformer(w.geom)
    try:
        dev = bf.beamform(torch.from_numpy(w.rf).cuda(), 3)
        torch.cuda.synchronize()
        host = bf.beamform_host(w.rf, 3)
        # the two entry points group the 21 frames differently (16 + 4 + 1 against 8 + 8 + 4 + 1), and in a 16-frame
        # group one frame pair takes its cube root on the FMA pipe instead of the XU pipe: the
        # same images to rounding, not to the bit
        peak = float(np.max(np.abs(host)))
        assert np.max(np.abs(dev.cpu().numpy() - host)) <= 2e-6 * peak
        pinned = torch.from_numpy(w.rf).pin_memory()
        assert np.array_equal(bf.beamform_host(pinned, 3).numpy(), host)          # same grouping: same bits
    finally:
        bf.close()


def test_host_async_stream_of_calls_matches_blocking_calls(pab):
    """pab_beamform_host_async: five calls in flight over the three device buffer sets (different frames, different frame
    counts, so a buffer handed over too early would show), one pab_host_sync; against the device entry point."""
    sizes = (16, 5, 16, 1, 12)
    w = synth.make_config("C1", n_frames=sum(sizes))
    g = w.geom
    bf = pab.Beamformer(g)
    try:
        ref = bf.beamform(torch.from_numpy(w.rf).cuda(), 3).cpu().numpy()
        torch.cuda.synchronize()
        ins, outs, f0 = [], [], 0
        for n in sizes:
            ins.append(torch.from_numpy(w.rf[f0:f0 + n].copy()).pin_memory())
            outs.append(torch.full((n, g.nz, g.nx), float("nan")).pin_memory())
            f0 += n
        for a, b in zip(ins, outs):
            bf.beamform_host_async(a, 3, b)
        bf.host_sync()
        got = np.concatenate([o.numpy() for o in outs])
        assert np.all(np.isfinite(got))
        # the calls group the frames differently (see test_host_entry_point_matches_device_entry_point): rounding only
        assert np.max(np.abs(got - ref)) <= 2e-6 * float(np.max(np.abs(ref)))
        bf.host_sync()                                      # nothing in flight: returns at once
        again = bf.beamform_host(ins[0], 3).numpy()                                   # the blocking call still works after
        assert np.max(np.abs(again - outs[0].numpy())) <= 2e-6 * float(np.max(np.abs(ref)))
    finally:
        bf.close()


def test_argument_errors_launch_nothing(pab):
    w = synth.make_config("C1")
    bf = pab.Beamformer(w.geom)
    try:
        rf = torch.from_numpy(w.rf).cuda()
        out = torch.full((1, w.geom.nz, w.geom.nx), 7.0, device="cuda")
        L = pab.load()
        n0 = bf.launch_count()
        assert L.pab_beamform(bf._h, rf.data_ptr(), 1, 0, out.data_ptr(), None) == pab.ERR_INVALID
        assert L.pab_beamform(bf._h, rf.data_ptr(), 1, 9, out.data_ptr(), None) == pab.ERR_INVALID
        assert L.pab_beamform(bf._h, rf.data_ptr(), 0, 3, out.data_ptr(), None) == pab.ERR_INVALID
        assert L.pab_beamform(bf._h, None, 1, 3, out.data_ptr(), None) == pab.ERR_INVALID
        assert L.pab_beamform(bf._h, rf.data_ptr(), 1, 3, None, None) == pab.ERR_INVALID
        assert L.pab_beamform(bf._h, rf.data_ptr() + 2, 1, 3, out.data_ptr(), None) == pab.ERR_INVALID
        torch.cuda.synchronize()
        assert bf.launch_count() == n0 and torch.all(out == 7.0)
        assert L.pab_set_post(bf._h, pab.LOG, 10e6, 2.5e6, 64, 62, 60.0) == pab.ERR_INVALID     # even Hilbert length
        assert L.pab_set_input(bf._h, 5, 1.0) == pab.ERR_INVALID
    finally:
        bf.close()


def test_homogeneity_and_zero_channels_on_gpu(pab):
    """P6 / P5 on the CUDA path: rf x alpha -> image x alpha (odd k) or x |alpha| (even k); fewer than k
    non-zero channels -> ~0 (the Newton form cancels to rounding)."""
    w = synth.make_config("C1", n_frames=4)
    for order in (2, 3):
        a, _ = run_gpu(pab, w.geom, w.rf, order)
        b, _ = run_gpu(pab, w.geom, (-2.0 * w.rf).astype(np.float32), order)
        fac = 2.0 if order % 2 == 0 else -2.0
        assert np.max(np.abs(b - fac * a)) <= 2e-5 * np.max(np.abs(a)) * 2
    rf = np.zeros_like(w.rf)
    rf[:, :2] = w.rf[:, :2]
    z, _ = run_gpu(pab, w.geom, rf, 3)
    scale = np.max(np.abs(rf)) * 1.0
    assert np.max(np.abs(z)) <= 1e-5 * scale


# ---- coherence-factor weighting (reading A20), fused into the beamforming kernel ----
@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("order", [1, 2, 3, 4, 5])
def test_cf_weighting_c1(pab, orc, variant, order):
    w = synth.make_config("C1", n_frames=9)
    ref = orc.beamform_ex(w.rf, w.geom, order, weight="cf")
    for frames in (1, 4, 9):
        gpu, _ = run_gpu(pab, w.geom, w.rf[:frames], order, variant, weight="cf")
        for f in range(frames):
            check_raw(gpu[f], ref[f], order)


@pytest.mark.parametrize("variant", VARIANTS)
def test_cf_weighting_ragged_out_of_record(pab, orc, variant):
    rng = np.random.default_rng(21)
    g = synth.random_geometry(rng, 24, 514, 37, 129, in_range=False)
    rf = rng.standard_normal((6, 24, 514)).astype(np.float32)
    mask = edge_mask(orc, g)
    for order in (2, 3):
        gpu, _ = run_gpu(pab, g, rf, order, variant, weight="cf")
        ref = orc.beamform_ex(rf, g, order, weight="cf")
        for f in range(6):
            check_raw(gpu[f], ref[f], order, mask)


def test_cf_weighting_c2b_batch(pab, orc):
    """Full-size grid, 24 frames (8 frames per thread with CF), order 3; two full frames against the oracle."""
    w = synth.make_config("C2b", n_frames=24)
    gpu, _ = run_gpu(pab, w.geom, w.rf, 3, weight="cf")
    for f in (0, 23):
        check_raw(gpu[f], orc.beamform_ex(w.rf[f:f + 1], w.geom, 3, weight="cf")[0], 3)
    # all-zero frame: CF is defined as 0, the image must be exactly 0 (no NaN from 0/0)
    z, _ = run_gpu(pab, w.geom, np.zeros_like(w.rf[:4]), 3, weight="cf")
    assert np.all(z == 0.0)


# ---- nearest-sample delays, the literal eq. (1) (reading A21) ----
@pytest.mark.parametrize("variant", VARIANTS)
def test_nearest_integer_decisions_are_the_oracles_bit_exact(pab, orc, variant):
    """RF = sample index on every channel, order 1: the image is sum_i round(idx_i), integers below 2^24, so fp32
    sums are exact and the GPU image must equal the oracle's bit for bit: every integer delay decision
    (including the out-of-record ones) is the oracle's."""
    for cfg in ("C1", "C2"):
        g = synth.geometry(cfg)
        rf = np.tile(np.arange(g.n_samp, dtype=np.float32), (1, g.n_elem, 1))
        gpu, _ = run_gpu(pab, g, rf, 1, variant, interp="nearest")
        assert np.array_equal(gpu, orc.beamform_ex(rf, g, 1, interp="nearest"))
    rng = np.random.default_rng(31)
    g = synth.random_geometry(rng, 24, 514, 37, 129, in_range=False)          # runs past the end of the record
    rf = np.tile(np.arange(g.n_samp, dtype=np.float32), (2, g.n_elem, 1))
    gpu, _ = run_gpu(pab, g, rf, 1, variant, interp="nearest")
    assert np.array_equal(gpu, orc.beamform_ex(rf, g, 1, interp="nearest"))


@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("order", [1, 2, 3, 4, 5])
def test_nearest_c1_all_orders_and_frame_counts(pab, orc, variant, order):
    w = synth.make_config("C1", n_frames=19)
    ref = orc.beamform_ex(w.rf, w.geom, order, interp="nearest")
    for frames in (1, 4, 9, 19):
        gpu, _ = run_gpu(pab, w.geom, w.rf[:frames], order, variant, interp="nearest")
        for f in range(frames):
            rel = check_raw(gpu[f], ref[f], order)
            assert rel <= 2e-5          # no fp32 delay in this path: only fp32 roots and sums remain


@pytest.mark.parametrize("variant", VARIANTS)
def test_nearest_ragged_int16_and_scale(pab, orc, variant):
    rng = np.random.default_rng(33)
    g = synth.random_geometry(rng, 33, 1001, 9, 70, in_range=False)
    rf = rng.integers(-2000, 2000, (6, 33, 1001)).astype(np.int16)
    for order, scale in ((3, 1.0), (2, 0.125), (5, 1.0)):
        gpu, _ = run_gpu(pab, g, rf, order, variant, dtype="int16", scale=scale, interp="nearest")
        ref = orc.beamform_ex(rf, g, order, interp="nearest", scale=scale)
        for f in range(6):
            check_raw(gpu[f], ref[f], order)


@pytest.mark.parametrize("dtype", ["float32", "int16"])
def test_nearest_single_frames_take_the_diagonal_kernel(pab, orc, dtype):
    """Row f4 in calls of 1..3 frames on translation-invariant in-range geometries: the single-frame diagonal kernel on a table
    of floor(idx + 1/2) with fraction 0 (one integer delay per diagonal of pairs; its interpolation then returns rf[n]
    exactly).  Integer decisions bit for bit on a sample-index ramp (ragged grid, 28-row tiles, q = 2; and config C2),
    orders 1..5 on noisy frames, fp32 and int16 with a scale."""
    rng = np.random.default_rng(44)
    fs, c, q, n_elem, nx, nz, S = 40e6, 1540.0, 2, 24, 45, 61, 900
    dx = 2.0 ** -13
    g = synth.Geometry(n_elem, S, fs, c, float(np.float32(q * np.float64(dx))), nx, nz, -(nx - 1) / 2 * dx + 0.3 * dx, dx, 2.1e-3,
                       1.1 * c / fs).f32()
    ramp = np.tile(np.arange(S, dtype=np.float32), (2, n_elem, 1))
    scale = 1.0
    base = [(rng.uniform(-1e-3, 1e-3), rng.uniform(2.5e-3, 4.5e-3), 1.0, 0.0) for _ in range(3)]
    rf, _ = synth._frames(rng, g, base, 5e6, 3, 20.0, True)
    if dtype == "int16":
        ramp, rf, scale = ramp.astype(np.int16), np.rint(rf * 4000.0).astype(np.int16), 0.25
    bf = pab.Beamformer(g, dtype=dtype, scale=scale, interp="nearest")
    try:
        assert bf.plan()["in_range"] == 1
        n0 = bf.launch_count()
        out = bf.beamform(torch.from_numpy(ramp).cuda(), 1)
        torch.cuda.synchronize()
        assert bf.launch_count() - n0 == 1                         # one kernel, no ingest pass: the diagonal kernel
        assert np.array_equal(out.cpu().numpy().astype(np.float64), orc.beamform_ex(ramp, g, 1, interp="nearest", scale=scale))
        for frames in (1, 3):
            for order in (1, 2, 3, 4, 5):
                out = bf.beamform(torch.from_numpy(rf[:frames]).cuda(), order)
                torch.cuda.synchronize()
                gpu = out.cpu().numpy().astype(np.float64)
                ref = orc.beamform_ex(rf[:frames], g, order, interp="nearest", scale=scale)
                for f in range(frames):
                    assert check_raw(gpu[f], ref[f], order) <= 2e-5
        if dtype == "float32":                 # no gather outside the staged windows (built from the rounded indices)
            assert bf.plan()["diagonal"] == 1
            for order in (3, 5):
                assert bf.self_check(torch.from_numpy(rf[:1]).cuda(), order) == 0
    finally:
        bf.close()
    if dtype == "float32":
        w = synth.make_config("C2")
        for order in (1, 2, 3):
            gpu, launches = run_gpu(pab, w.geom, w.rf, order, interp="nearest")
            assert check_raw(gpu[0], orc.beamform_ex(w.rf, w.geom, order, interp="nearest")[0], order) <= 2e-5


def test_nearest_c2b_batch_and_post_chain(pab, orc):
    w = synth.make_config("C2b", n_frames=20)
    g = w.geom
    gpu, _ = run_gpu(pab, g, w.rf, 3, interp="nearest")
    for f in (0, 19):
        check_raw(gpu[f], orc.beamform_ex(w.rf[f:f + 1], g, 3, interp="nearest")[0], 3)
    post = dict(mode="envelope", f_center=10e6, f_halfwidth=2.5e6, n_taps_bp=64, n_taps_hilbert=63, dyn_range_db=60.0)
    gpu, _ = run_gpu(pab, g, w.rf[:2], 3, interp="nearest", post=post)
    ref = orc.post(orc.beamform_ex(w.rf[:2], g, 3, interp="nearest"), g, 10e6, 2.5e6, 64, 63, 60.0, mode="envelope")
    assert np.sqrt(np.sum((gpu - ref) ** 2) / np.sum(ref ** 2)) <= 2e-4


def test_nearest_rejects_unsupported_combinations(pab):
    w = synth.make_config("C1")
    bf = pab.Beamformer(w.geom, weight="cf")
    try:
        with pytest.raises(pab.PabError):
            bf.set_interp("nearest")
        bf.set_weight("none")
        bf.set_interp("nearest")
        with pytest.raises(pab.PabError):
            bf.set_weight("cf")
    finally:
        bf.close()


# ---- orders above 5, the power-sum scheme continued ----
@pytest.mark.parametrize("variant", VARIANTS)
@pytest.mark.parametrize("order", [6, 7, 8])
def test_high_orders_c1(pab, orc, variant, order):
    """Tolerance of orders 4, 5 carried over (relative L2 <= 1e-4, per pixel <= 5e-3 x peak): an fp32 study of the
    Newton recursion at N = 128 gave 1e-6 .. 2e-6 relative L2 for k = 6..8 (DESIGN.md row f2)."""
    w = synth.make_config("C1", n_frames=9)
    ref = orc.beamform(w.rf, w.geom, order)
    for frames in (1, 4, 9):
        gpu, _ = run_gpu(pab, w.geom, w.rf[:frames], order, variant)
        for f in range(frames):
            check_raw(gpu[f], ref[f], order)


@pytest.mark.parametrize("order", [6, 8])
def test_high_orders_c2_full_size(pab, orc, order):
    w = synth.make_config("C2b", n_frames=5)
    gpu, _ = run_gpu(pab, w.geom, w.rf, order)
    for f in (0, 4):
        check_raw(gpu[f], orc.beamform(w.rf[f:f + 1], w.geom, order)[0], order)


@pytest.mark.parametrize("order", [6, 7, 8])
def test_high_orders_cached_taps(pab, orc, order):
    """Row f2 on the cached-tap kernel (4-frame groups under PAB_CACHE_ALL): C2b frames, 4 cached + 1 not."""
    w = synth.make_config("C2b", n_frames=5)
    gpu, _ = run_gpu(pab, w.geom, w.rf, order, delay_cache="all")
    for f in (0, 3, 4):
        check_raw(gpu[f], orc.beamform(w.rf[f:f + 1], w.geom, order)[0], order)


def test_high_orders_reject_weight_and_nearest(pab):
    w = synth.make_config("C1")
    rf = torch.from_numpy(w.rf).cuda()
    for kw in (dict(weight="cf"), dict(interp="nearest")):
        bf = pab.Beamformer(w.geom, **kw)
        try:
            with pytest.raises(pab.PabError):
                bf.beamform(rf, 6)
            bf.beamform(rf, 5)
        finally:
            bf.close()


# ---- image-quality metrics on the device (eqs. 10-12, FWHM; reading A22) ----
def _sim1_rois(g, depth_mm=23.0):
    r = int(round((depth_mm * 1e-3 - g.z0) / g.dz))
    c = int(round((-1.5e-3 - g.x0) / g.dx))                       # the left target of the pair
    cb = int(round((4.0e-3 - g.x0) / g.dx))                       # background: same depth, 5.5 mm to the side
    return (r - 10, r + 10, c - 8, c + 9), (r - 10, r + 10, cb - 8, cb + 9), r


def test_metrics_device_matches_oracle_on_simulation1_phantom(pab, orc):
    w = synth.simulation1_phantom()
    g = w.geom
    post = {k: v for k, v in w.post.items()}
    res = {}
    for order in (1, 3, 5):
        bf = pab.Beamformer(g, post=post)
        try:
            img = bf.beamform(torch.from_numpy(w.rf).cuda(), order)[0].contiguous()
            torch.cuda.synchronize()
            # the peak row of the target inside its box: where FWHM is measured
            tgt, bkg, r = _sim1_rois(g)
            box = img[tgt[0]:tgt[1], tgt[2]:tgt[3]]
            row = tgt[0] + int(torch.argmax(box.max(dim=1).values))
            for n_bins in (64, 256):
                got = bf.image_metrics(img, tgt, bkg, n_bins=n_bins, fwhm_row=row)
                ref = orc.image_metrics(img.cpu().numpy(), tgt, bkg, n_bins=n_bins, fwhm_row=row, dx=g.dx)
                for k in ("mu_in", "mu_out", "sigma_out", "snr_db", "cr_db", "fwhm_m"):
                    assert got[k] == pytest.approx(ref[k], rel=1e-9), (order, k)
                assert got["gcnr"] == pytest.approx(ref["gcnr"], abs=1e-12), order      # same integer bin decisions
            res[order] = got
        finally:
            bf.close()
    # the paper's qualitative claim on the synthetic phantom: contrast and SNR grow with the order,
    # the main lobe narrows
    assert res[5]["cr_db"] > res[3]["cr_db"] > res[1]["cr_db"]
    assert res[5]["snr_db"] > res[1]["snr_db"]
    assert res[5]["fwhm_m"] < res[1]["fwhm_m"]


def test_metrics_argument_errors(pab):
    w = synth.make_config("C1")
    bf = pab.Beamformer(w.geom)
    try:
        img = torch.ones((w.geom.nz, w.geom.nx), device="cuda")
        with pytest.raises(pab.PabError):
            bf.image_metrics(img, (0, 0, 0, 4), (0, 4, 0, 4))                      # empty target
        with pytest.raises(pab.PabError):
            bf.image_metrics(img, (0, 4, 0, 4), (0, 4, 0, w.geom.nx + 1))          # outside the grid
        with pytest.raises(pab.PabError):
            bf.image_metrics(img, (0, 4, 0, 4), (0, 4, 0, 4), n_bins=1)
        m = bf.image_metrics(img, (0, 4, 0, 4), (4, 8, 0, 4), n_bins=8)
        assert m["mu_in"] == 1.0 and m["cr_db"] == 0.0 and m["gcnr"] == 0.0 and np.isnan(m["fwhm_m"])
    finally:
        bf.close()


def test_beamform_is_cuda_graph_capturable(pab, orc):
    """pab_beamform only enqueues work on the caller's stream (kernels + one memset), so a whole step can be captured
    into a CUDA graph and replayed: the launch-bound tiny config C1 is where that pays."""
    w = synth.make_config("C1", n_frames=8)
    post = dict(mode="log", f_center=2.0e6, f_halfwidth=0.8e6, n_taps_bp=64, n_taps_hilbert=63, dyn_range_db=60.0)
    bf = pab.Beamformer(w.geom, post=post)
    try:
        rf = torch.from_numpy(w.rf).cuda()
        out = torch.empty((8, w.geom.nz, w.geom.nx), device="cuda")
        eager = bf.beamform(rf, 3).clone()
        s = torch.cuda.Stream()
        s.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(s):
            bf.beamform(rf, 3, out=out, stream=s)            # warm-up on the side stream
        torch.cuda.current_stream().wait_stream(s)
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=s):
            bf.beamform(rf, 3, out=out, stream=s)
        out.zero_()
        graph.replay()
        torch.cuda.synchronize()
        assert torch.equal(out, eager)
        rf.mul_(-1.0)                                        # new input in the same buffer, replay again
        graph.replay()
        torch.cuda.synchronize()
        ref = bf.beamform(rf, 3)
        torch.cuda.synchronize()
        assert torch.equal(out, ref)
    finally:
        bf.close()


@pytest.mark.parametrize("tables", ["off", "single"])
def test_cf_weighting_single_frames_take_the_diagonal_kernel(pab, orc, tables):
    """Row f1 in calls of 1..3 frames on translation-invariant in-range geometries: the diagonal kernel with the two (three
    for even orders) extra sums of the coherence factor per pixel, 8 pixels per thread at every order; both forms of the
    kernel, orders 1..5, fp32 and int16, a ragged 61-row grid (28-row tiles), an all-zero frame (exact 0), and config C2."""
    rng = np.random.default_rng(66)
    fs, c, q, n_elem, nx, nz, S = 40e6, 1540.0, 2, 24, 45, 61, 900
    dx = 2.0 ** -13
    g = synth.Geometry(n_elem, S, fs, c, float(np.float32(q * np.float64(dx))), nx, nz, -(nx - 1) / 2 * dx + 0.3 * dx, dx, 2.1e-3,
                       1.1 * c / fs).f32()
    base = [(rng.uniform(-1e-3, 1e-3), rng.uniform(2.5e-3, 4.5e-3), 1.0, 0.0) for _ in range(3)]
    rf, _ = synth._frames(rng, g, base, 5e6, 3, 20.0, True)
    rf[1] = 0.0
    for dtype, data, scale in (("float32", rf, 1.0), ("int16", np.rint(rf * 4000.0).astype(np.int16), 0.25)):
        bf = pab.Beamformer(g, dtype=dtype, scale=scale, weight="cf", delay_cache=tables)
        try:
            for frames in (1, 3):
                for order in (1, 2, 3, 4, 5):
                    n0 = bf.launch_count()
                    out = bf.beamform(torch.from_numpy(data[:frames]).cuda(), order)
                    torch.cuda.synchronize()
                    if not (tables == "off" and frames == 1 and order == 1):
                        assert bf.launch_count() - n0 == 1            # one kernel, no ingest pass: the diagonal kernel
                    gpu = out.cpu().numpy().astype(np.float64)
                    ref = orc.beamform_ex(data[:frames], g, order, weight="cf", scale=scale)
                    for f in range(frames):
                        if f == 1:
                            assert np.all(gpu[f] == 0.0) and np.all(ref[f] == 0.0)
                        else:
                            check_raw(gpu[f], ref[f], order)
            assert bf.plan()["diagonal"] == (2 if tables == "off" else 1)
        finally:
            bf.close()
    w = synth.make_config("C2")
    gpu, _ = run_gpu(pab, w.geom, w.rf, 3, weight="cf", delay_cache=tables)
    check_raw(gpu[0], orc.beamform_ex(w.rf, w.geom, 3, weight="cf")[0], 3)


def test_single_frame_default_path_under_graph_capture(pab, orc):
    """The table-free diagonal kernel builds its windows on the first 1..3-frame call (a device synchronisation), which must not
    happen inside a stream capture: a context whose FIRST such call is captured keeps the one-frame-per-thread kernel for
    it (and stays correct), builds the windows on its next eager call, and a capture made after that replays the diagonal
    kernel."""
    rng = np.random.default_rng(91)
    dx = 2.0 ** -13
    g = synth.Geometry(16, 900, 40e6, 1540.0, 2 * dx, 37, 70, -18 * dx, dx, 2.1e-3, 0.09e-3).f32()
    base = [(rng.uniform(-1e-3, 1e-3), rng.uniform(3e-3, 8e-3), 1.0, 0.0) for _ in range(3)]
    rf_np, _ = synth._frames(rng, g, base, 5e6, 1, 20.0, True)
    ref = orc.beamform(rf_np, g, 3)[0]
    bf = pab.Beamformer(g)
    try:
        rf = torch.from_numpy(rf_np).cuda()
        out = torch.empty((1, g.nz, g.nx), device="cuda")
        s = torch.cuda.Stream()
        s.wait_stream(torch.cuda.current_stream())
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=s):
            bf.beamform(rf, 3, out=out, stream=s)            # first call of the context: captured, no set-up allowed
        assert bf.plan()["diagonal"] == 0
        out.zero_()
        graph.replay()
        torch.cuda.synchronize()
        check_raw(out.cpu().numpy().astype(np.float64)[0], ref, 3)
        eager = bf.beamform(rf, 3)                           # eager call: builds the windows, runs the diagonal kernel
        torch.cuda.synchronize()
        assert bf.plan()["diagonal"] == 2
        check_raw(eager.cpu().numpy().astype(np.float64)[0], ref, 3)
        graph2 = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph2, stream=s):
            bf.beamform(rf, 3, out=out, stream=s)
        out.zero_()
        graph2.replay()
        torch.cuda.synchronize()
        assert torch.equal(out, eager)
    finally:
        bf.close()


# ---- cached interpolation taps (pab_set_delay_cache): the paper's delay table where it wins ----
@pytest.mark.parametrize("order", [1, 2, 3, 4, 5])
def test_delay_cache_single_frames_c2(pab, orc, order):
    w = synth.make_config("C2b", n_frames=3)
    ref = orc.beamform(w.rf, w.geom, order)
    for frames in (1, 3):
        gpu, _ = run_gpu(pab, w.geom, w.rf[:frames], order, delay_cache="single")
        for f in range(frames):
            assert check_raw(gpu[f], ref[f], order) <= 2.5e-5


@pytest.mark.parametrize("order", [1, 2, 3, 4, 5])
def test_delay_cache_cf_weighting_ragged(pab, orc, order):
    # row f1 on the cached-tap kernel: 8-frame (orders 1..3) and 4-frame groups, ragged grid, every order
    rng = np.random.default_rng(43)
    g = synth.random_geometry(rng, 24, 514, 37, 129, in_range=True)
    g = synth.Geometry(g.n_elem, g.n_samp, g.fs, g.c, g.pitch, g.nx, g.nz, g.x0, g.dx, max(g.z0, 2e-4), g.dz).f32()
    rf = rng.standard_normal((13, 24, 514)).astype(np.float32)
    gpu, _ = run_gpu(pab, g, rf, order, delay_cache="all", weight="cf")
    ref = orc.beamform_ex(rf, g, order, weight="cf")
    off, _ = run_gpu(pab, g, rf, order, weight="cf")
    for f in range(13):
        check_raw(gpu[f], ref[f], order)
        check_raw(off[f], ref[f], order)


def test_delay_cache_ragged_int16_and_batches(pab, orc):
    rng = np.random.default_rng(41)
    g = synth.random_geometry(rng, 24, 514, 37, 129, in_range=True)
    g = synth.Geometry(g.n_elem, g.n_samp, g.fs, g.c, g.pitch, g.nx, g.nz, g.x0, g.dx, max(g.z0, 2e-4), g.dz).f32()
    rf = rng.integers(-2000, 2000, (21, 24, 514)).astype(np.int16)
    for mode, frames in (("single", 2), ("all", 21), ("all", 16)):
        for order in (2, 3):
            gpu, _ = run_gpu(pab, g, rf[:frames], order, dtype="int16", scale=0.5, delay_cache=mode)
            ref = orc.beamform(rf[:frames], g, order, scale=0.5)
            for f in range(frames):
                check_raw(gpu[f], ref[f], order)


@pytest.mark.parametrize("tables", ["single", "off"])
@pytest.mark.parametrize("q,n_elem,nx,nz,frames,dtype", [(1, 16, 37, 70, 1, "float32"), (2, 24, 45, 33, 3, "float32"),
                                                         (3, 8, 50, 129, 2, "int16"), (2, 4, 7, 5, 1, "float32"),
                                                         (1, 64, 130, 95, 2, "int16"), (4, 12, 64, 64, 1, "float32"),
                                                         (16, 16, 300, 70, 1, "float32"), (12, 8, 100, 40, 2, "int16"),
                                                         (8, 16, 300, 70, 1, "float32")])
def test_diagonal_kernel_ragged_translation_invariant(pab, orc, q, n_elem, nx, nz, frames, dtype, tables):
    """The single-frame diagonal kernel (pitch = q dx exactly: one tap per diagonal, channel-quad staging from the caller's
    frame) on ragged grids: nx, nz off the tile sizes, arrays of 1..16 channel quads, q = 1..4, 1..3 frames, int16 input
    with a scale, every order 1..5 (16 pixels per thread for orders 1..3, 8 for orders 4, 5); q = 12 and 16: one diagonal
    part of 12 / 16 warps.  The wide ragged grids (q = 8, 16 with nx = 300) are the regression cases of an out-of-window read:
    the pixel columns past nx of their last tile lie so far out that their delays run past the record, and before table
    columns were clamped to those of real pairs (diag_ddx) the kernel gathered 1502 / 58514 samples outside the staged windows
    for them (never stored, so parity could not see it; pab_self_check did)."""
    rng = np.random.default_rng(100 + 7 * q + n_elem)
    fs, c, S = 40e6, 1540.0, 900
    dx = 2.0 ** -13                                              # 0.122 mm: q dx is a float32 for every small q
    pitch = float(np.float32(q * np.float64(dx)))
    assert pitch == q * dx                                       # exactly representable: the library's own test
    x0 = -(nx - 1) / 2 * dx + 0.3 * dx
    g = synth.Geometry(n_elem, S, fs, c, pitch, nx, nz, x0, dx, 2.1e-3, 0.09e-3).f32()
    assert float(g.pitch) == q * float(g.dx)
    base = [(rng.uniform(-1e-3, 1e-3), rng.uniform(3e-3, 9e-3), 1.0, 0.0) for _ in range(3)]
    rf, _ = synth._frames(rng, g, base, 5e6, frames, 20.0, True)
    scale = 1.0
    if dtype == "int16":
        rf, scale = np.rint(rf * 4000.0).astype(np.int16), 0.25
    bf = pab.Beamformer(g, dtype=dtype, scale=scale, delay_cache=tables)
    try:
        assert bf.plan()["in_range"] == 1
        if tables == "single":
            assert bf.plan()["diagonal"] == 1                                     # the diagonal kernel is what runs
        for order in (1, 2, 3, 4, 5):
            if order > n_elem:
                continue
            out = bf.beamform(torch.from_numpy(rf).cuda(), order)
            torch.cuda.synchronize()
            gpu = out.cpu().numpy().astype(np.float64)
            ref = orc.beamform(rf, g, order, scale=scale)
            for f in range(frames):
                assert check_raw(gpu[f], ref[f], order) <= 2.5e-5
            if tables == "off":                # delay cache off: the table-free form of the kernel (taps on the FP64 pipe)
                assert bf.plan()["diagonal"] == 2
        if dtype == "float32":               # every shared-memory gather inside the staged window of its quad (both forms)
            for order in (3, 5):
                if order <= n_elem:
                    assert bf.self_check(torch.from_numpy(rf[:1]).cuda(), order) == 0
    finally:
        bf.close()


@pytest.mark.parametrize("tables", ["off", "single", "all"])
def test_exact_integer_delays(pab, orc, tables):
    """The degenerate case of the delay index: a geometry on which many delays are EXACT integers of samples (c / fs = 2^-15 m,
    rows and z0 on multiples of it, columns on multiples of 4 samples, so every pixel under an element and every Pythagorean
    (lateral, depth) pair has an integer idx).  floor() then sits on its discontinuity: whichever way the kernels' index rounds
    (in-kernel fp64 with its rounding-constant floor and its tie rule, in-kernel fp32, or the fp64 tap table), the interpolated
    sample must be the oracle's.  Single frames (diagonal kernel), 16-frame groups and a 5-frame call, orders 1, 3, 5."""
    fs, c = float(2 ** 25), 1024.0
    dx = 2.0 ** -13
    g = synth.Geometry(16, 700, fs, c, 2 * dx, 33, 40, -16 * dx, dx, 2.0 ** -7, 2.0 ** -15).f32()
    zs = (np.float64(g.z0) + np.arange(g.nz) * np.float64(g.dz)) * fs / c
    assert np.all(zs == np.rint(zs))                                   # every row an integer number of samples deep
    idx = np.sqrt(((g.pix_x()[None, :, None] - g.elem_x()[None, None, :]) * fs / c) ** 2 + zs[:, None, None] ** 2)
    assert np.mean(idx == np.rint(idx)) > 0.02                         # thousands of exactly integer delays
    rng = np.random.default_rng(5)
    rf = rng.standard_normal((16, g.n_elem, g.n_samp)).astype(np.float32)      # white noise: adjacent samples unrelated
    bf = pab.Beamformer(g, delay_cache=tables)
    try:
        assert bf.plan()["in_range"] == 1
        for frames in (1, 5, 16):
            for order in (1, 3, 5):
                out = bf.beamform(torch.from_numpy(rf[:frames]).cuda(), order)
                torch.cuda.synchronize()
                gpu = out.cpu().numpy().astype(np.float64)
                ref = orc.beamform(rf[:frames], g, order)
                for f in range(frames):
                    peak = np.max(np.abs(ref[f]))
                    # DAS is linear in the samples: a wrong neighbour anywhere would show at 1e-2 of the peak
                    assert np.max(np.abs(gpu[f] - ref[f])) <= (2e-6 if order == 1 else 5e-3) * peak, (frames, order, f)
    finally:
        bf.close()


@pytest.mark.parametrize("tables", ["off", "all"])
@pytest.mark.parametrize("dtype", ["float32", "int16"])
def test_remainder_frames_take_the_diagonal_kernel(pab, orc, dtype, tables):
    """Frame counts that are not a multiple of 4 on a translation-invariant in-range geometry: the whole quads go through
    the frame-group kernels, the 1..3 frames left over through the single-frame diagonal kernel (straight from the caller's
    buffer), and the post chain sees all of them.  5, 7, 9 and 22 frames, orders 1..5, raw and log output."""
    rng = np.random.default_rng(77)
    q, n_elem, nx, nz, S = 2, 32, 45, 150, 900
    dx = 2.0 ** -13
    g = synth.Geometry(n_elem, S, 40e6, 1540.0, float(np.float32(q * np.float64(dx))), nx, nz, -(nx - 1) / 2 * dx, dx, 2.1e-3,
                       0.06e-3).f32()
    base = [(rng.uniform(-1e-3, 1e-3), rng.uniform(3e-3, 10e-3), 1.0, 0.0) for _ in range(4)]
    rf, _ = synth._frames(rng, g, base, 5e6, 22, 20.0, True)
    scale = 1.0
    if dtype == "int16":
        rf, scale = np.rint(rf * 4000.0).astype(np.int16), 0.25
    bf = pab.Beamformer(g, dtype=dtype, scale=scale, delay_cache=tables)
    try:
        assert bf.plan()["in_range"] == 1
        for frames in (5, 7, 9, 22):
            x = torch.from_numpy(rf[:frames]).cuda()
            for order in (1, 2, 3, 4, 5):
                out = bf.beamform(x, order)
                torch.cuda.synchronize()
                assert bf.plan()["diagonal"] in (1, 2)
                gpu = out.cpu().numpy().astype(np.float64)
                ref = orc.beamform(rf[:frames], g, order, scale=scale)
                for f in range(frames):
                    check_raw(gpu[f], ref[f], order)
    finally:
        bf.close()
    for frames, order in ((5, 3), (9, 2), (22, 5)):                 # the same with coherence-factor weighting
        gpu, _ = run_gpu(pab, g, rf[:frames], order, dtype=dtype, scale=scale, weight="cf", delay_cache=tables)
        ref = orc.beamform_ex(rf[:frames], g, order, weight="cf", scale=scale)
        for f in range(frames):
            check_raw(gpu[f], ref[f], order)
    post = dict(mode="log", f_center=10e6, f_halfwidth=2.5e6, n_taps_bp=64, n_taps_hilbert=63, dyn_range_db=60.0)
    gpu, _ = run_gpu(pab, g, rf[:7], 3, dtype=dtype, scale=scale, post=post, delay_cache=tables)
    ref = orc.post(orc.beamform(rf[:7], g, 3, scale=scale), g, post["f_center"], post["f_halfwidth"], post["n_taps_bp"],
                   post["n_taps_hilbert"], post["dyn_range_db"], mode="log")
    sel = ref > -40.0
    assert np.max(np.abs(gpu - ref)[sel]) <= 0.05


@pytest.mark.parametrize("tables", ["single", "off"])
def test_diagonal_kernel_28_row_tiles(pab, orc, tables):
    """Row pitches in (1, 8/7] samples (config C2's 1.14): the diagonal kernel takes tiles of 28 rows, seven per quarter-warp
    with the eighth lane idle, so that the gathers of a quarter-warp never meet in a bank group.  A ragged grid (61 rows:
    two whole tiles and 5 rows), 1 and 3 frames, orders 1..5, both forms of the kernel, and its bounds check."""
    rng = np.random.default_rng(28)
    fs, c, q, n_elem, nx, nz, S = 40e6, 1540.0, 2, 24, 45, 61, 900
    dx = 2.0 ** -13
    g = synth.Geometry(n_elem, S, fs, c, float(np.float32(q * np.float64(dx))), nx, nz, -(nx - 1) / 2 * dx + 0.3 * dx, dx, 2.1e-3,
                       1.1 * c / fs).f32()
    assert 1.0 < float(g.dz) * fs / c <= 8.0 / 7.0
    base = [(rng.uniform(-1e-3, 1e-3), rng.uniform(2.5e-3, 4.5e-3), 1.0, 0.0) for _ in range(3)]
    rf, _ = synth._frames(rng, g, base, 5e6, 3, 20.0, True)
    bf = pab.Beamformer(g, delay_cache=tables)
    try:
        assert bf.plan()["in_range"] == 1
        for frames in (1, 3):
            for order in (1, 2, 3, 4, 5):
                out = bf.beamform(torch.from_numpy(rf[:frames]).cuda(), order)
                torch.cuda.synchronize()
                gpu = out.cpu().numpy().astype(np.float64)
                ref = orc.beamform(rf[:frames], g, order)
                for f in range(frames):
                    assert check_raw(gpu[f], ref[f], order) <= 2.5e-5
        assert bf.plan()["diagonal"] == (1 if tables == "single" else 2)
        for order in (3, 5):
            assert bf.self_check(torch.from_numpy(rf[:1]).cuda(), order) == 0
    finally:
        bf.close()


@pytest.mark.parametrize("tables", ["single", "off"])
@pytest.mark.parametrize("cfg,order", [("C2", 3), ("C4", 5), ("C3", 1), ("C5", 4)])
def test_diagonal_kernel_self_check_named_geometries(pab, cfg, order, tables):
    """pab_self_check on the geometries of the named configs (C5's with fp32 frames): no gather of the diagonal kernel, in
    the form with its tap table or in the table-free form, leaves the staged window of its channel quad (the check
    compute-sanitizer would make; it is closed on this pool)."""
    g = synth.geometry(cfg)
    rng = np.random.default_rng(3)
    rf = rng.standard_normal((1, g.n_elem, g.n_samp)).astype(np.float32)
    bf = pab.Beamformer(g, delay_cache=tables)
    try:
        if tables == "single":
            assert bf.plan()["diagonal"] == 1
        assert bf.self_check(torch.from_numpy(rf).cuda(), order) == 0
        assert bf.plan()["diagonal"] == (1 if tables == "single" else 2)
    finally:
        bf.close()


@pytest.mark.parametrize("delay_cache", ["all", "off"])
@pytest.mark.parametrize("order", [1, 2])
def test_56_row_tiles(pab, orc, order, delay_cache):
    """Orders 1 and 2 (cached taps; order 1 also with in-kernel delays) in groups of 8 / 16 frames at a row pitch in
    (1, 8/7] samples take 56-row tiles (seven rows per quarter-warp, the eighth lane idle: pab_pipe.cuh tile_row), with
    their own tap tables under PAB_CACHE_ALL: the C2b geometry (nz = 1024 = 18 x 56 + 16: a ragged last tile) and a small
    ragged grid, 20 and 24 frames (16 + 4, 16 + 8)."""
    w = synth.make_config("C2b", n_frames=20)
    assert 1.0 < pab.plan(w.geom)["zs_per_row"] <= 8.0 / 7.0
    gpu, _ = run_gpu(pab, w.geom, w.rf, order, delay_cache=delay_cache)
    for f in (0, 15, 16, 19):
        assert check_raw(gpu[f], orc.beamform(w.rf[f:f + 1], w.geom, order)[0], order) <= 2.5e-5
    g = w.geom
    small = synth.Geometry(24, 700, g.fs, g.c, g.pitch, 37, 131, -18 * g.dx, g.dx, 4e-3, g.dz).f32()
    rng = np.random.default_rng(56)
    base = [(rng.uniform(-2e-3, 2e-3), rng.uniform(5e-3, 9e-3), 1.0, 0.0) for _ in range(3)]
    rf, _ = synth._frames(rng, small, base, 5e6, 24, 20.0, True)
    gpu, _ = run_gpu(pab, small, rf, order, delay_cache=delay_cache)
    ref = orc.beamform(rf, small, order)
    for f in range(24):
        check_raw(gpu[f], ref[f], order)


def test_delay_cache_c2b_groups_and_fallbacks(pab, orc):
    w = synth.make_config("C2b", n_frames=20)
    gpu, _ = run_gpu(pab, w.geom, w.rf, 3, delay_cache="all")                 # one 16-frame group cached + 4 frames not
    for f in (0, 15, 19):
        assert check_raw(gpu[f], orc.beamform(w.rf[f:f + 1], w.geom, 3)[0], 3) <= 2.5e-5
    gpu, _ = run_gpu(pab, w.geom, w.rf[:1], 3, delay_cache="single", weight="cf")     # weighting: in-kernel delay
    check_raw(gpu[0], orc.beamform_ex(w.rf[:1], w.geom, 3, weight="cf")[0], 3)
    gpu, _ = run_gpu(pab, w.geom, w.rf[:13], 3, delay_cache="all", weight="cf")       # CF: 8 cached + 4 cached + 1 not
    for f in (0, 7, 11, 12):
        check_raw(gpu[f], orc.beamform_ex(w.rf[f:f + 1], w.geom, 3, weight="cf")[0], 3)
    c1 = synth.make_config("C1")                                                      # z starts at 0: not in range
    bf = pab.Beamformer(c1.geom)
    try:
        with pytest.raises(pab.PabError):
            bf.set_delay_cache("single")
    finally:
        bf.close()


def test_more_frames_than_one_internal_batch(pab, orc):
    """300 frames of C1: the device entry point loops over internal batches of 256, the host entry point pipelines
    64-frame pieces (>= 256 frames) -- both must equal the per-frame oracle and each other; repeated create /
    destroy must give the memory back."""
    w = synth.make_config("C1", n_frames=300)
    assert pab.plan(w.geom)["batch_frames"] == 256
    free0 = torch.cuda.mem_get_info()[0]
    bf = pab.Beamformer(w.geom)
    try:
        dev = bf.beamform(torch.from_numpy(w.rf).cuda(), 3)
        torch.cuda.synchronize()
        host = bf.beamform_host(w.rf, 3)
        assert np.max(np.abs(dev.cpu().numpy() - host)) <= 2e-6 * float(np.max(np.abs(host)))     # 16- against 64-frame pieces
        for f in (0, 255, 256, 299):
            check_raw(host[f].astype(np.float64), orc.beamform(w.rf[f:f + 1], w.geom, 3)[0], 3)
    finally:
        bf.close()
    del dev
    torch.cuda.empty_cache()
    for _ in range(20):
        b = pab.Beamformer(synth.geometry("C3"), post=dict(mode="log"), interp="linear", delay_cache="single")
        b.close()
        b = pab.Beamformer(synth.geometry("C3"), interp="nearest")
        b.close()
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free0 - 64 * 2 ** 20          # nothing leaked beyond allocator slack


def test_constant_rf_closed_form_on_gpu(pab):
    """Pin P4 on the CUDA path, no oracle involved: constant RF a on every channel gives C(N, k) a (odd k) or
    C(N, k) |a| (even k) on every in-range pixel (eqs. 1, 2, 4-6: every k-subset product is a^k)."""
    import math
    for cfg, orders in (("C1", (1, 2, 3, 4, 5, 6, 7, 8)), ("C2", (1, 2, 3, 4, 5))):
        g = synth.geometry(cfg)
        sub = synth.Geometry(g.n_elem, g.n_samp, g.fs, g.c, g.pitch, 16, 64, g.x0, g.dx * (g.nx // 16),
                             max(g.z0, 2e-3), g.dz * (g.nz // 64) * 0.8).f32()
        rf = np.full((5, g.n_elem, g.n_samp), -2.5, dtype=np.float32)
        for order in orders:
            for frames in (1, 5):
                gpu, _ = run_gpu(pab, sub, rf[:frames], order)
                expect = math.comb(g.n_elem, order) * (-2.5 if order % 2 else 2.5)
                assert np.allclose(gpu, expect, rtol=2e-4), (cfg, order, frames, gpu.flat[0], expect)


def test_channel_reversal_symmetry_on_gpu(pab):
    """Pin P6 on the CUDA path: mirroring the channels and the pixel columns about x = 0 mirrors the image."""
    w = synth.make_config("C1", n_frames=4)
    g = w.geom
    sym = synth.Geometry(g.n_elem, g.n_samp, g.fs, g.c, g.pitch, g.nx, g.nz, -(g.nx - 1) * g.dx / 2, g.dx, 1e-3, g.dz).f32()
    for order in (2, 3):
        a, _ = run_gpu(pab, sym, w.rf, order)
        b, _ = run_gpu(pab, sym, np.ascontiguousarray(w.rf[:, ::-1, :]), order)
        assert np.max(np.abs(a - b[:, :, ::-1])) <= 2e-5 * np.max(np.abs(a))


@pytest.mark.parametrize("mode", ["cache-all", "cache-single", "nearest", "plain"])
def test_coarse_rows_large_window_fallbacks(pab, orc, mode):
    """Rows 1.07 mm apart: a tile needs a 1792-sample window per channel, one channel per stage fills shared memory.
    The cached-tap and nearest kernels need room for their table block on top and must fall back (found by a
    randomised sweep: the launch used to fail with 'invalid argument')."""
    g = synth.Geometry(25, 1978, 40e6, 1540.0, 0.0002074896910926327, 79, 46, -0.00404604896903038,
                       0.00010374484554631636, 0.01058073341846466, 0.0010749740758910775).f32()
    assert pab.plan(g)["window_samples"] >= 1500 and pab.plan(g)["chunk_channels"] == 1
    rng = np.random.default_rng(77)
    base = [(rng.uniform(-3e-3, 3e-3), rng.uniform(0.02, 0.05), 1.0, 0.0) for _ in range(3)]
    rf, _ = synth._frames(rng, g, base, 5e6, 17, 20.0, True)
    kw, okw = {}, {}
    if mode == "nearest":
        kw["interp"] = okw["interp"] = "nearest"
    elif mode.startswith("cache"):
        kw["delay_cache"] = mode[6:]
    for frames in (1, 17):
        gpu, _ = run_gpu(pab, g, rf[:frames], 3, **kw)
        ref = orc.beamform_ex(rf[:frames], g, 3, **okw)
        for f in range(frames):
            check_raw(gpu[f], ref[f], 3)


def test_randomised_api_sweep(pab, orc):
    """80 seeded random small cases over every option of the API (a short version of the sweeps DESIGN.md section 11
    describes): nothing may raise, every output is finite, and every image is grossly right (3 % relative L2 against
    the oracle; white-noise RF, so the tight tolerances do not apply: see 'Conditioning')."""
    rng = np.random.default_rng(2024)
    for case in range(80):
        n_elem = int(rng.choice([1, 2, 5, 16, 33, 64, 129])); n_samp = int(rng.choice([3, 17, 64, 333, 1024, 2047]))
        nx = int(rng.choice([1, 2, 7, 8, 9, 31, 64])); nz = int(rng.choice([1, 2, 31, 32, 33, 64, 65, 130]))
        g = synth.random_geometry(rng, n_elem, max(n_samp, 8), nx, nz, in_range=bool(rng.integers(0, 2)))
        g = synth.Geometry(g.n_elem, n_samp, g.fs, g.c, g.pitch, g.nx, g.nz, g.x0, g.dx,
                           g.z0 if rng.integers(0, 4) else 0.0, g.dz).f32()
        F = int(rng.choice([1, 2, 3, 4, 7, 8, 16, 17, 33]))
        order = int(rng.integers(1, 9))
        dtype = str(rng.choice(["float32", "int16"]))
        rf = ((rng.standard_normal((F, n_elem, n_samp)) * 300).astype(np.int16) if dtype == "int16"
              else rng.standard_normal((F, n_elem, n_samp)).astype(np.float32))
        mode = "plain" if order > 5 else str(rng.choice(["plain", "cf", "nearest", "cache-single", "cache-all"]))
        kw, okw = dict(dtype=dtype), {}
        if mode == "cf":
            kw["weight"] = okw["weight"] = "cf"
        if mode == "nearest":
            kw["interp"] = okw["interp"] = "nearest"
        bf = pab.Beamformer(g, **kw)
        try:
            try:
                bf.set_variant(str(rng.choice(["auto", "direct", "staged"])))
            except pab.PabError:
                pass                                      # staged not available for this geometry
            if mode.startswith("cache"):
                try:
                    bf.set_delay_cache(mode[6:])
                except pab.PabError:
                    pass                                  # not an in-range geometry
            if rng.integers(0, 4) == 0:
                out = np.asarray(bf.beamform_host(rf, order)).astype(np.float64)
            else:
                out = bf.beamform(torch.from_numpy(rf).cuda(), order).cpu().numpy().astype(np.float64)
        finally:
            bf.close()
        assert np.all(np.isfinite(out)), (case, mode, order)
        ref = orc.beamform_ex(rf, g, order, **okw)
        den = np.sqrt(np.sum(ref ** 2))
        if den > 0:
            assert np.sqrt(np.sum((out - ref) ** 2)) / den <= 3e-2, (case, mode, order, F, g)
