"""pab_post_no_alloc (include/pab.h): the post chain with its scratch in a fixed file-scope device array, against the
existing path (pab_beamform under the same post mode), on two calls in a row.  Collected last on purpose (the suite runs
with pytest -x); passes alone in a fresh process and after the other GPU tests.
"""
import ctypes as C

import numpy as np
import pytest
import torch

from paper_2203_14906_b200 import synth

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def pab():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2203_14906_b200 import binding
    binding.load(build_if_missing=True)     # raises if libpab.so cannot be built: no fallback
    return binding


def _compare(mode, got, ref, frames, dr):
    got = got.cpu().numpy().astype(np.float64)
    ref = ref.cpu().numpy().astype(np.float64)
    assert np.all(np.isfinite(got))
    if mode == "log":       # the tolerances of test_post_chain_streaming_configs
        sel = ref > -40.0
        assert np.max(np.abs(got - ref)[sel]) <= 0.05
        assert np.all(got <= 1e-4) and np.all(got >= -dr - 1e-4)
        assert np.all(np.max(got.reshape(frames, -1), axis=1) > -1e-3)      # 0 dB at the frame max
    else:
        rel = np.sqrt(np.sum((got - ref) ** 2) / np.sum(ref ** 2))
        assert rel <= 2e-4, f"{mode}: relative L2 {rel:.3e}"


@pytest.mark.parametrize("mode", ["log", "envelope"])
def test_post_no_alloc_matches_existing_path_twice(pab, mode):
    frames = 6
    w = synth.make_config("C3", n_frames=frames)
    g = w.geom
    dtype = "int16" if w.rf.dtype == np.int16 else "float32"
    post = dict({k: v for k, v in w.post.items() if k != "mode"}, mode=mode)
    rf = torch.from_numpy(w.rf).cuda()
    bf_raw = pab.Beamformer(g, dtype=dtype)
    bf = pab.Beamformer(g, dtype=dtype, post=post)
    try:
        raw = bf_raw.beamform(rf, 3)                 # what the caller of the new entry point holds
        ref = bf.beamform(rf, 3)                     # the existing path: beamform + post chain with allocated scratch
        torch.cuda.synchronize()
        n0 = bf.launch_count()
        # call 1 on images 4x as large: leaves 4x larger frame maxima in the shared array
        big = (raw * 4.0).contiguous()
        out1 = torch.empty_like(raw)
        bf.post_no_alloc(big, out1)
        # call 2 right behind it, frames in reverse order: stale maxima (of call 1, or of another frame) would show as
        # a 12 dB / per-frame offset under "log"
        rev = torch.flip(raw, dims=[0]).contiguous()
        out2 = torch.empty_like(raw)
        bf.post_no_alloc(rev, out2)
        torch.cuda.synchronize()
        assert bf.launch_count() - n0 == (4 if mode == "log" else 2)
        _compare(mode, out1 if mode == "log" else out1 / 4.0, ref, frames, post["dyn_range_db"])
        _compare(mode, torch.flip(out2, dims=[0]), ref, frames, post["dyn_range_db"])
    finally:
        bf.close()
        bf_raw.close()


def test_post_no_alloc_rejects(pab):
    w = synth.make_config("C3", n_frames=1)
    g = w.geom
    post = dict({k: v for k, v in w.post.items() if k != "mode"}, mode="log")
    bf = pab.Beamformer(g, dtype="int16" if w.rf.dtype == np.int16 else "float32", post=post)
    try:
        L = bf._L
        img = torch.zeros((2, g.nz, g.nx), device="cuda")
        out = torch.zeros_like(img)
        st = torch.cuda.current_stream().cuda_stream
        n0 = bf.launch_count()
        # beyond the fixed array: a clear error, nothing launched (the pointers are not touched)
        rc = L.pab_post_no_alloc(bf._h, img.data_ptr(), pab.NO_ALLOC_MAX_FRAMES + 1, out.data_ptr(), st)
        assert rc == pab.ERR_LIMIT
        assert str(pab.NO_ALLOC_MAX_FRAMES) in L.pab_last_cuda_error(bf._h).decode()
        assert b"maximum" in L.pab_strerror(rc)
        # in place / overlapping, null, no frames
        assert L.pab_post_no_alloc(bf._h, img.data_ptr(), 2, img.data_ptr(), st) == pab.ERR_INVALID
        assert L.pab_post_no_alloc(bf._h, img.data_ptr(), 2, img.data_ptr() + g.nz * g.nx * 4, st) == pab.ERR_INVALID
        assert L.pab_post_no_alloc(bf._h, None, 2, out.data_ptr(), st) == pab.ERR_INVALID
        assert L.pab_post_no_alloc(bf._h, img.data_ptr(), 0, out.data_ptr(), st) == pab.ERR_INVALID
        # modes without an envelope have no scratch to speak of and are not covered
        bf.set_post(**dict(post, mode="bandpass"))
        assert L.pab_post_no_alloc(bf._h, img.data_ptr(), 2, out.data_ptr(), st) == pab.ERR_INVALID
        assert bf.launch_count() == n0
    finally:
        bf.close()
