"""ctypes loader for the fp64 CPU oracle (oracle/pab_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this package.  It
imports nothing from paper_2203_14906_b200 and shares no code with the CUDA path.

Every function is a thin marshalling wrapper: numpy arrays in, numpy float64 out.
Geometry floats are taken as Python floats (already float32-rounded by the caller,
so both sides see the same numbers) and promoted to double unchanged.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pab_oracle.c")
_LIB = os.path.join(_HERE, "libpab_oracle.so")

F32, I16 = 0, 1
ROUTE_BRUTE, ROUTE_RECUR, ROUTE_CLOSED = 0, 1, 2


class _Grid(C.Structure):
    _fields_ = [("nx", C.c_int), ("nz", C.c_int), ("x0", C.c_double), ("dx", C.c_double),
                ("z0", C.c_double), ("dz", C.c_double)]


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2 -fopenmp, no fast-math, no intrinsics)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-std=c99", "-fopenmp", "-fPIC", "-shared", "-D_GNU_SOURCE",
                               "-o", _LIB, _SRC, "-lm"])
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        dp = C.POINTER(C.c_double)
        L.orc_elem_x.restype = C.c_double
        L.orc_elem_x.argtypes = [C.c_int, C.c_int, C.c_double]
        L.orc_delay_idx.restype = C.c_double
        L.orc_delay_idx.argtypes = [C.c_double] * 5
        L.orc_combine_brute.restype = C.c_double
        L.orc_combine_brute.argtypes = [dp, C.c_int, C.c_int]
        L.orc_combine_recur.restype = C.c_double
        L.orc_combine_recur.argtypes = [dp, C.c_int, C.c_int]
        L.orc_combine_closed.restype = C.c_double
        L.orc_combine_closed.argtypes = [dp, C.c_int, C.c_int, C.c_int]
        L.orc_beamform.restype = C.c_int
        _lib = L
    return _lib


def _grid(g) -> _Grid:
    return _Grid(int(g.nx), int(g.nz), float(g.x0), float(g.dx), float(g.z0), float(g.dz))


def _rf(rf):
    rf = np.ascontiguousarray(rf)
    if rf.dtype == np.float32:
        return rf, F32
    if rf.dtype == np.int16:
        return rf, I16
    raise TypeError(f"rf must be float32 or int16, got {rf.dtype}")


def _dptr(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def delays(g) -> np.ndarray:
    """idx[nz][nx][N]: fs*sqrt((x-xe)^2+z^2)/c (O1-O3)."""
    out = np.empty((g.nz, g.nx, g.n_elem))
    gr = _grid(g)
    lib().orc_delays(C.c_int(g.n_elem), C.c_double(g.fs), C.c_double(g.c), C.c_double(g.pitch), C.byref(gr), _dptr(out))
    return out


def gather(rf, g, frame=0, scale=1.0) -> np.ndarray:
    """s[nz][nx][N]: delayed, linearly interpolated samples of one frame (O4)."""
    rf, dt = _rf(rf)
    out = np.empty((g.nz, g.nx, g.n_elem))
    gr = _grid(g)
    lib().orc_gather(C.c_void_p(rf.ctypes.data), C.c_int(dt), C.c_double(scale), C.c_int(frame), C.c_int(g.n_elem),
                     C.c_int(g.n_samp), C.c_double(g.fs), C.c_double(g.c), C.c_double(g.pitch), C.byref(gr), _dptr(out))
    return out


def combine(s, k: int, route: int = ROUTE_RECUR, repaired: bool = True) -> float:
    s = np.ascontiguousarray(s, dtype=np.float64)
    L = lib()
    if route == ROUTE_BRUTE:
        return L.orc_combine_brute(_dptr(s), C.c_int(s.size), C.c_int(k))
    if route == ROUTE_CLOSED:
        return L.orc_combine_closed(_dptr(s), C.c_int(s.size), C.c_int(k), C.c_int(1 if repaired else 0))
    return L.orc_combine_recur(_dptr(s), C.c_int(s.size), C.c_int(k))


def das(rf, g, scale=1.0) -> np.ndarray:
    rf, dt = _rf(rf)
    F = rf.shape[0]
    out = np.empty((F, g.nz, g.nx))
    gr = _grid(g)
    lib().orc_das(C.c_void_p(rf.ctypes.data), C.c_int(dt), C.c_double(scale), C.c_int(F), C.c_int(g.n_elem),
                  C.c_int(g.n_samp), C.c_double(g.fs), C.c_double(g.c), C.c_double(g.pitch), C.byref(gr), _dptr(out))
    return out


def beamform(rf, g, order: int, route: int = ROUTE_RECUR, scale=1.0, nthreads: int = 0, return_threads=False):
    """Reference image out[F][nz][nx] (fp64) of the pre-band-pass DMAS-k beamformer."""
    rf, dt = _rf(rf)
    assert rf.ndim == 3 and rf.shape[1] == g.n_elem and rf.shape[2] == g.n_samp, rf.shape
    F = rf.shape[0]
    out = np.empty((F, g.nz, g.nx))
    gr = _grid(g)
    used = lib().orc_beamform(C.c_void_p(rf.ctypes.data), C.c_int(dt), C.c_double(scale), C.c_int(F),
                              C.c_int(g.n_elem), C.c_int(g.n_samp), C.c_double(g.fs), C.c_double(g.c),
                              C.c_double(g.pitch), C.byref(gr), C.c_int(order), C.c_int(route), _dptr(out),
                              C.c_int(nthreads))
    return (out, used) if return_threads else out


def coherence_factor(s) -> float:
    s = np.ascontiguousarray(s, dtype=np.float64)
    L = lib()
    L.orc_coherence_factor.restype = C.c_double
    return L.orc_coherence_factor(_dptr(s), C.c_int(s.size))


def beamform_ex(rf, g, order: int, interp: str = "linear", weight: str = "none", route: int = ROUTE_RECUR, scale=1.0,
                nthreads: int = 0):
    """Reference image with the section 8(f) options: interp "linear" | "nearest" (A21), weight "none" | "cf" (A20)."""
    rf, dt = _rf(rf)
    F = rf.shape[0]
    out = np.empty((F, g.nz, g.nx))
    gr = _grid(g)
    lib().orc_beamform_ex(C.c_void_p(rf.ctypes.data), C.c_int(dt), C.c_double(scale), C.c_int(F), C.c_int(g.n_elem),
                          C.c_int(g.n_samp), C.c_double(g.fs), C.c_double(g.c), C.c_double(g.pitch), C.byref(gr),
                          C.c_int(order), C.c_int(route), C.c_int({"linear": 0, "nearest": 1}[interp]),
                          C.c_int({"none": 0, "cf": 1}[weight]), _dptr(out), C.c_int(nthreads))
    return out


def nearest_index(g) -> np.ndarray:
    """n[nz][nx][N]: the nearest-sample index the oracle picks, -1 outside the record (A21)."""
    out = np.empty((g.nz, g.nx, g.n_elem), dtype=np.int32)
    gr = _grid(g)
    lib().orc_nearest_index(C.c_int(g.n_elem), C.c_int(g.n_samp), C.c_double(g.fs), C.c_double(g.c),
                            C.c_double(g.pitch), C.byref(gr), out.ctypes.data_as(C.POINTER(C.c_int)))
    return out


METRIC_NAMES = ("mu_in", "mu_out", "sigma_out", "snr_db", "cr_db", "gcnr", "fwhm_m")


def image_metrics(img, target, background, n_bins: int = 256, fwhm_row: int = -1, dx: float = 1.0) -> dict:
    """Eqs. (10)-(12) + FWHM on one float32 image [nz][nx]; target / background = (r0, r1, c0, c1) (A22)."""
    img = np.ascontiguousarray(img, dtype=np.float32)
    nz, nx = img.shape
    t = np.asarray(target, dtype=np.int32)
    b = np.asarray(background, dtype=np.int32)
    out = np.empty(7)
    ip = C.POINTER(C.c_int)
    lib().orc_image_metrics(img.ctypes.data_as(C.POINTER(C.c_float)), C.c_int(nz), C.c_int(nx), t.ctypes.data_as(ip),
                            b.ctypes.data_as(ip), C.c_int(n_bins), C.c_int(fwhm_row), C.c_double(dx), _dptr(out))
    return dict(zip(METRIC_NAMES, out.tolist()))


def beamform_pixels(rf, g, order: int, pix, route: int = ROUTE_RECUR, scale=1.0) -> np.ndarray:
    """out[F][n_pix] at sampled pixels pix[n_pix][2] = (row m, column j)."""
    rf, dt = _rf(rf)
    F = rf.shape[0]
    pix = np.ascontiguousarray(pix, dtype=np.int32)
    out = np.empty((F, pix.shape[0]))
    gr = _grid(g)
    lib().orc_beamform_pixels(C.c_void_p(rf.ctypes.data), C.c_int(dt), C.c_double(scale), C.c_int(F),
                              C.c_int(g.n_elem), C.c_int(g.n_samp), C.c_double(g.fs), C.c_double(g.c),
                              C.c_double(g.pitch), C.byref(gr), C.c_int(order), C.c_int(route),
                              pix.ctypes.data_as(C.POINTER(C.c_int)), C.c_int(pix.shape[0]), _dptr(out))
    return out


def bandpass_taps(T: int, f_lo: float, f_hi: float) -> np.ndarray:
    h = np.empty(T)
    lib().orc_bandpass_taps(C.c_int(T), C.c_double(f_lo), C.c_double(f_hi), _dptr(h))
    return h


def hilbert_taps(L: int) -> np.ndarray:
    g = np.empty(2 * L + 1)
    lib().orc_hilbert_taps(C.c_int(L), _dptr(g))
    return g


def fir_axial(x, h) -> np.ndarray:
    x = np.ascontiguousarray(x, dtype=np.float64)
    h = np.ascontiguousarray(h, dtype=np.float64)
    F, nz, nx = x.shape
    y = np.empty_like(x)
    lib().orc_fir_axial(_dptr(x), C.c_int(F), C.c_int(nz), C.c_int(nx), _dptr(h), C.c_int(h.size), _dptr(y))
    return y


def envelope(y, g_taps) -> np.ndarray:
    y = np.ascontiguousarray(y, dtype=np.float64)
    g_taps = np.ascontiguousarray(g_taps, dtype=np.float64)
    F, nz, nx = y.shape
    env = np.empty_like(y)
    lib().orc_envelope(_dptr(y), C.c_int(F), C.c_int(nz), C.c_int(nx), _dptr(g_taps), C.c_int((g_taps.size - 1) // 2), _dptr(env))
    return env


def logcompress(env, dyn_range_db=60.0) -> np.ndarray:
    env = np.ascontiguousarray(env, dtype=np.float64)
    F, nz, nx = env.shape
    out = np.empty_like(env)
    lib().orc_logcompress(_dptr(env), C.c_int(F), C.c_int(nz), C.c_int(nx), C.c_double(dyn_range_db), _dptr(out))
    return out


def post(img, g, f_center, f_halfwidth, n_taps_bp=64, n_taps_hilbert=63, dyn_range_db=60.0, mode="log"):
    """O6-O8 on a beamformed image [F][nz][nx]; axial sampling rate fs_z = c/dz (one-way)."""
    fs_z = g.c / g.dz
    h = bandpass_taps(n_taps_bp, (f_center - f_halfwidth) / fs_z, (f_center + f_halfwidth) / fs_z)
    y = fir_axial(img, h)
    if mode == "bandpass":
        return y
    env = envelope(y, hilbert_taps((n_taps_hilbert - 1) // 2))
    if mode == "envelope":
        return env
    return logcompress(env, dyn_range_db)
