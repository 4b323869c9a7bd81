"""Thin ctypes binding of libpab.so (include/pab.h): argument marshalling only.

Every step of the hot path runs in the library's CUDA kernels.  PyTorch is used for device memory and
streams (torch tensors in, torch tensors out).  There is no CPU fallback: `load()` raises if libpab.so is
missing, and `Beamformer` raises if the library reports an error.
"""
from __future__ import annotations

import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpab.so")

OK, ERR_INVALID, ERR_DEVICE, ERR_ALLOC, ERR_CUDA, ERR_LIMIT = 0, -1, -2, -3, -4, -5
NO_ALLOC_MAX_FRAMES = 1024      # PAB_NO_ALLOC_MAX_FRAMES
F32, I16 = 0, 1
RAW, BANDPASS, ENVELOPE, LOG = 0, 1, 2, 3
VARIANT_AUTO, VARIANT_DIRECT, VARIANT_STAGED = 0, 1, 2
WEIGHT_NONE, WEIGHT_CF = 0, 1
INTERP_LINEAR, INTERP_NEAREST = 0, 1
STAGES = ["ingest", "beamform", "post_fir", "post_log"]
_MODES = {"raw": RAW, "bandpass": BANDPASS, "envelope": ENVELOPE, "log": LOG}
_VARIANTS = {"auto": VARIANT_AUTO, "direct": VARIANT_DIRECT, "staged": VARIANT_STAGED}

# every symbol include/pab.h declares
SYMBOLS = ["pab_create", "pab_set_input", "pab_set_post", "pab_set_variant", "pab_set_weight", "pab_set_interp", "pab_set_delay_cache", "pab_set_tuning", "pab_beamform", "pab_beamform_host", "pab_beamform_host_async", "pab_host_sync",
           "pab_destroy", "pab_plan", "pab_get_plan", "pab_design_bandpass", "pab_design_hilbert",
           "pab_launch_count", "pab_measure_peaks", "pab_self_check", "pab_post_no_alloc", "pab_image_metrics", "pab_set_profile", "pab_get_profile", "pab_strerror", "pab_last_cuda_error", "pab_version"]


class Grid(C.Structure):
    _fields_ = [("nx", C.c_int), ("nz", C.c_int), ("x0", C.c_float), ("dx", C.c_float),
                ("z0", C.c_float), ("dz", C.c_float)]


class PlanInfo(C.Structure):
    _fields_ = [("tile_z", C.c_int), ("tile_x", C.c_int), ("window_samples", C.c_int), ("chunk_channels", C.c_int),
                ("stages", C.c_int), ("smem_bytes", C.c_int), ("frames_per_thread", C.c_int),
                ("batch_frames", C.c_int), ("in_range", C.c_int), ("diagonal", C.c_int), ("zs_per_row", C.c_double), ("xs_per_col", C.c_double)]

    def asdict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


class Roi(C.Structure):
    _fields_ = [("r0", C.c_int), ("r1", C.c_int), ("c0", C.c_int), ("c1", C.c_int)]


class Metrics(C.Structure):
    _fields_ = [(k, C.c_double) for k in ("mu_in", "mu_out", "sigma_out", "snr_db", "cr_db", "gcnr", "fwhm_m")]


class PabError(RuntimeError):
    pass


_lib = None


def load(build_if_missing: bool = False):
    """dlopen libpab.so and declare the prototypes.  Fails loudly when the library is absent."""
    global _lib
    if _lib is not None:
        return _lib
    if build_if_missing and not os.path.exists(LIB_PATH):
        # absent only: a copied tree (gpurun, a checkout) does not keep modification times, so "older than a source
        # file" cannot be told from them; `python -m paper_2203_14906_b200.build` rebuilds a stale library
        from . import build as _b
        _b.build_lib()
    if not os.path.exists(LIB_PATH):
        raise PabError(f"{LIB_PATH} is missing: build it with `python -m paper_2203_14906_b200.build` "
                       "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    vp, ip, fp = C.c_void_p, C.c_int, C.c_float
    L.pab_create.argtypes = [C.POINTER(vp), ip, ip, fp, fp, fp, C.POINTER(Grid)]
    L.pab_set_input.argtypes = [vp, ip, fp]
    L.pab_set_post.argtypes = [vp, ip, fp, fp, ip, ip, fp]
    L.pab_set_variant.argtypes = [vp, ip]
    L.pab_set_weight.argtypes = [vp, ip]
    L.pab_set_interp.argtypes = [vp, ip]
    L.pab_set_delay_cache.argtypes = [vp, ip]
    L.pab_set_tuning.argtypes = [vp, ip, ip, ip, ip]
    L.pab_beamform.argtypes = [vp, vp, ip, ip, vp, vp]
    L.pab_beamform_host.argtypes = [vp, vp, ip, ip, vp]
    L.pab_beamform_host_async.argtypes = [vp, vp, ip, ip, vp]
    L.pab_host_sync.argtypes = [vp]
    L.pab_destroy.argtypes = [vp]
    L.pab_destroy.restype = None
    L.pab_plan.argtypes = [ip, ip, fp, fp, fp, C.POINTER(Grid), ip, C.POINTER(PlanInfo)]
    L.pab_get_plan.argtypes = [vp, C.POINTER(PlanInfo)]
    L.pab_design_bandpass.argtypes = [ip, C.c_double, C.c_double, C.POINTER(C.c_float)]
    L.pab_design_hilbert.argtypes = [ip, C.POINTER(C.c_float)]
    L.pab_launch_count.argtypes = [vp]
    L.pab_launch_count.restype = C.c_longlong
    L.pab_image_metrics.argtypes = [vp, vp, C.POINTER(Roi), C.POINTER(Roi), ip, ip, C.POINTER(Metrics), vp]
    L.pab_measure_peaks.argtypes = [C.POINTER(C.c_double), ip]
    L.pab_self_check.argtypes = [vp, vp, ip, C.POINTER(C.c_longlong)]
    L.pab_post_no_alloc.argtypes = [vp, vp, ip, vp, vp]
    L.pab_set_profile.argtypes = [vp, ip]
    L.pab_get_profile.argtypes = [vp, ip, C.POINTER(C.c_double), C.POINTER(C.c_longlong), ip]
    L.pab_strerror.argtypes = [ip]
    L.pab_strerror.restype = C.c_char_p
    L.pab_last_cuda_error.argtypes = [vp]
    L.pab_last_cuda_error.restype = C.c_char_p
    L.pab_version.restype = C.c_char_p
    _lib = L
    return L


def _grid(g) -> Grid:
    return Grid(int(g.nx), int(g.nz), float(g.x0), float(g.dx), float(g.z0), float(g.dz))


def plan(g, smem_limit: int = 0) -> dict:
    """pab_plan: the tiling / staging plan for a geometry (host-only, no GPU needed)."""
    info = PlanInfo()
    gr = _grid(g)
    rc = load().pab_plan(g.n_elem, g.n_samp, g.fs, g.c, g.pitch, C.byref(gr), smem_limit, C.byref(info))
    if rc != OK:
        raise PabError(f"pab_plan: {load().pab_strerror(rc).decode()}")
    return info.asdict()


def design_bandpass(n_taps: int, f_lo: float, f_hi: float):
    import numpy as np
    h = np.zeros(n_taps, dtype=np.float32)
    rc = load().pab_design_bandpass(n_taps, f_lo, f_hi, h.ctypes.data_as(C.POINTER(C.c_float)))
    if rc != OK:
        raise PabError(f"pab_design_bandpass: {load().pab_strerror(rc).decode()}")
    return h


def design_hilbert(half_len: int):
    import numpy as np
    g = np.zeros(2 * half_len + 1, dtype=np.float32)
    rc = load().pab_design_hilbert(half_len, g.ctypes.data_as(C.POINTER(C.c_float)))
    if rc != OK:
        raise PabError(f"pab_design_hilbert: {load().pab_strerror(rc).decode()}")
    return g


def measure_peaks() -> dict:
    """pab_measure_peaks on the current device: the measured unit rates behind the roofline denominators."""
    out = (C.c_double * 8)()
    rc = load().pab_measure_peaks(out, 8)
    if rc != OK:
        raise PabError(f"pab_measure_peaks: {load().pab_strerror(rc).decode()}")
    keys = ("mufu_lanes_per_clk_sm", "ffma_lanes_per_clk_sm", "ffma2_results_per_clk_sm", "lds128_bytes_per_clk_sm",
            "h2d_pinned_gbs", "d2h_pinned_gbs", "sm_clock_mhz", "sm_count")
    return dict(zip(keys, [float(v) for v in out]))


def shard_frames(n_frames: int, rank: int, world: int):
    """Replicas-only multi-GPU: contiguous frame range [lo, hi) of `rank`; frames are
    independent, so there is no exchange step and no collective on the data path."""
    base, rem = divmod(n_frames, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


class Beamformer:
    """pab_create / pab_set_* / pab_beamform / pab_destroy for one geometry on the current CUDA device."""

    def __init__(self, g, dtype: str = "float32", scale: float = 1.0, post: dict | None = None,
                 variant: str = "auto", weight: str = "none", interp: str = "linear", delay_cache: str = "off"):
        self._L = load()
        self._h = C.c_void_p()
        self.geom = g
        gr = _grid(g)
        self._check(self._L.pab_create(C.byref(self._h), g.n_elem, g.n_samp, g.fs, g.c, g.pitch, C.byref(gr)),
                    "pab_create")
        self.dtype = dtype
        self._check(self._L.pab_set_input(self._h, I16 if dtype == "int16" else F32, scale), "pab_set_input")
        if post:
            self.set_post(**post)
        if variant != "auto":
            self.set_variant(variant)
        if weight != "none":
            self.set_weight(weight)
        if interp != "linear":
            self.set_interp(interp)
        if delay_cache != "off":
            self.set_delay_cache(delay_cache)

    def _check(self, rc, what):
        if rc != OK:
            detail = self._L.pab_last_cuda_error(self._h).decode() if self._h else ""
            raise PabError(f"{what}: {self._L.pab_strerror(rc).decode()} {detail}".strip())

    def set_post(self, mode="log", f_center=10e6, f_halfwidth=2.5e6, n_taps_bp=64, n_taps_hilbert=63,
                 dyn_range_db=60.0):
        self._check(self._L.pab_set_post(self._h, _MODES[mode], f_center, f_halfwidth, n_taps_bp, n_taps_hilbert,
                                         dyn_range_db), "pab_set_post")

    def set_weight(self, weight: str):
        self._check(self._L.pab_set_weight(self._h, {"none": WEIGHT_NONE, "cf": WEIGHT_CF}[weight]), "pab_set_weight")

    def set_interp(self, interp: str):
        self._check(self._L.pab_set_interp(self._h, {"linear": INTERP_LINEAR, "nearest": INTERP_NEAREST}[interp]),
                    "pab_set_interp")

    def set_delay_cache(self, mode: str):
        self._check(self._L.pab_set_delay_cache(self._h, {"off": 0, "single": 1, "all": 2}[mode]), "pab_set_delay_cache")

    def set_variant(self, variant: str):
        self._check(self._L.pab_set_variant(self._h, _VARIANTS[variant]), "pab_set_variant")

    def set_tuning(self, frames_per_thread: int = 0, stages: int = 0, chunk_channels: int = 0,
                   host_batch_frames: int = 0):
        self._check(self._L.pab_set_tuning(self._h, frames_per_thread, stages, chunk_channels, host_batch_frames),
                    "pab_set_tuning")

    def plan(self) -> dict:
        info = PlanInfo()
        self._check(self._L.pab_get_plan(self._h, C.byref(info)), "pab_get_plan")
        return info.asdict()

    def launch_count(self) -> int:
        return int(self._L.pab_launch_count(self._h))

    def set_profile(self, max_launches: int):
        self._check(self._L.pab_set_profile(self._h, max_launches), "pab_set_profile")

    def get_profile(self, reset: bool = True) -> dict:
        """{stage: (total_ms, n_launches)} of the timed launches since the last reset."""
        out = {}
        for i, name in enumerate(STAGES):
            ms, n = C.c_double(), C.c_longlong()
            last = i == len(STAGES) - 1
            self._check(self._L.pab_get_profile(self._h, i, C.byref(ms), C.byref(n), 1 if (reset and last) else 0),
                        "pab_get_profile")
            out[name] = (ms.value, n.value)
        return out

    def beamform(self, rf, order: int, out=None, stream=None):
        """rf: CUDA tensor [F][N][S] float32 or int16 -> out: CUDA tensor [F][nz][nx] float32 (enqueue only)."""
        import torch
        g = self.geom
        assert rf.is_cuda and rf.is_contiguous() and rf.dim() == 3, "rf must be a contiguous CUDA tensor [F][N][S]"
        assert tuple(rf.shape[1:]) == (g.n_elem, g.n_samp), rf.shape
        assert rf.dtype == (torch.int16 if self.dtype == "int16" else torch.float32), rf.dtype
        F = rf.shape[0]
        if out is None:
            out = torch.empty((F, g.nz, g.nx), dtype=torch.float32, device=rf.device)
        assert out.is_cuda and out.is_contiguous() and out.dtype == torch.float32 and tuple(out.shape) == (F, g.nz, g.nx)
        st = torch.cuda.current_stream(rf.device) if stream is None else stream
        self._check(self._L.pab_beamform(self._h, rf.data_ptr(), F, order, out.data_ptr(), st.cuda_stream), "pab_beamform")
        return out

    def self_check(self, rf, order: int) -> int:
        """pab_self_check: out-of-window shared-memory gathers of the diagonal kernel on one fp32 CUDA frame [1][N][S]."""
        n = C.c_longlong(-1)
        self._check(self._L.pab_self_check(self._h, rf.data_ptr(), order, C.byref(n)), "pab_self_check")
        return int(n.value)

    def post_no_alloc(self, img, out, stream=None):
        """pab_post_no_alloc: the context's post chain (ENVELOPE / LOG) on CUDA images [F][nz][nx] float32 -> out (same
        shape, caller-allocated, not overlapping img); allocates nothing (fixed scratch array, F <= NO_ALLOC_MAX_FRAMES)."""
        import torch
        g = self.geom
        F = img.shape[0]
        for t in (img, out):
            assert t.is_cuda and t.is_contiguous() and t.dtype == torch.float32 and tuple(t.shape) == (F, g.nz, g.nx)
        st = torch.cuda.current_stream(img.device) if stream is None else stream
        self._check(self._L.pab_post_no_alloc(self._h, img.data_ptr(), F, out.data_ptr(), st.cuda_stream), "pab_post_no_alloc")
        return out

    def image_metrics(self, img, target, background, n_bins: int = 256, fwhm_row: int = -1, stream=None) -> dict:
        """pab_image_metrics on one CUDA image [nz][nx] float32; target / background = (r0, r1, c0, c1)."""
        import torch
        g = self.geom
        assert img.is_cuda and img.is_contiguous() and img.dtype == torch.float32 and tuple(img.shape) == (g.nz, g.nx)
        t, b, m = Roi(*map(int, target)), Roi(*map(int, background)), Metrics()
        st = torch.cuda.current_stream(img.device) if stream is None else stream
        self._check(self._L.pab_image_metrics(self._h, img.data_ptr(), C.byref(t), C.byref(b), n_bins, fwhm_row,
                                              C.byref(m), st.cuda_stream), "pab_image_metrics")
        return {k: getattr(m, k) for k, _ in Metrics._fields_}

    def beamform_host(self, rf, order: int, out=None):
        """rf: host array/tensor [F][N][S] (numpy or CPU torch, pinned or not) -> out: same kind, [F][nz][nx]."""
        import numpy as np
        import torch
        g = self.geom
        is_torch = isinstance(rf, torch.Tensor)
        F = rf.shape[0]
        assert tuple(rf.shape) == (F, g.n_elem, g.n_samp), rf.shape
        if is_torch:
            assert not rf.is_cuda and rf.is_contiguous()
            assert rf.dtype == (torch.int16 if self.dtype == "int16" else torch.float32), rf.dtype
            if out is None:
                out = torch.empty((F, g.nz, g.nx), dtype=torch.float32, pin_memory=rf.is_pinned())
            assert not out.is_cuda and out.is_contiguous() and out.dtype == torch.float32
            assert tuple(out.shape) == (F, g.nz, g.nx), out.shape
            src, dst = rf.data_ptr(), out.data_ptr()
        else:
            rf = np.ascontiguousarray(rf)
            assert rf.dtype == (np.int16 if self.dtype == "int16" else np.float32), rf.dtype
            if out is None:
                out = np.empty((F, g.nz, g.nx), dtype=np.float32)
            assert out.dtype == np.float32 and out.flags["C_CONTIGUOUS"] and out.shape == (F, g.nz, g.nx), out.shape
            src, dst = rf.ctypes.data, out.ctypes.data
        self._check(self._L.pab_beamform_host(self._h, src, F, order, dst), "pab_beamform_host")
        return out

    def beamform_host_async(self, rf, order: int, out):
        """pab_beamform_host_async: rf, out pinned CPU torch tensors ([F][N][S] -> [F][nz][nx]); enqueue only.  The caller
        keeps both alive and untouched until host_sync() returns."""
        import torch
        g = self.geom
        F = rf.shape[0]
        assert isinstance(rf, torch.Tensor) and not rf.is_cuda and rf.is_contiguous() and rf.is_pinned()
        assert tuple(rf.shape) == (F, g.n_elem, g.n_samp), rf.shape
        assert rf.dtype == (torch.int16 if self.dtype == "int16" else torch.float32), rf.dtype
        assert not out.is_cuda and out.is_contiguous() and out.is_pinned() and out.dtype == torch.float32
        assert tuple(out.shape) == (F, g.nz, g.nx), out.shape
        self._check(self._L.pab_beamform_host_async(self._h, rf.data_ptr(), F, order, out.data_ptr()), "pab_beamform_host_async")
        return out

    def host_sync(self):
        self._check(self._L.pab_host_sync(self._h), "pab_host_sync")

    def close(self):
        if self._h:
            self._L.pab_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
