"""CPU oracle for the TNLM 4DCT hot path -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Thin ctypes marshalling over oracle/tnlm_oracle.c (plain C, fp64, written from the paper;
see that file's header for the passages followed).  Only tests/, __graft_entry__.smoke()
and bench.py's cpu_baseline / --impl reference legs may import this package; the CUDA
path under paper_1009_1351_b200/ never does, and nothing here imports it.
"""
import ctypes as C
from dataclasses import dataclass

import numpy as np

from . import build as _build

_lib = None
_D = C.c_double
_I = C.c_int
_P = C.c_void_p


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        geo = [_I, _I, _I, _I, _I, _D, _D, _D, _D, _D, _P]
        _lib.oracle_num_threads.restype = _I
        _lib.oracle_project.argtypes = geo + [_P, _P, _I]
        _lib.oracle_backproject.argtypes = geo + [_P, _P, _I]
        _lib.oracle_project_rays.argtypes = geo + [_P, _I, _P, _P]
        _lib.oracle_backproject_pixels.argtypes = geo + [_P, _I, _P, _P]
        _lib.oracle_cgls_step.argtypes = geo + [_P, _P, _P, _I, _P, _I]
        _lib.oracle_tnlm_raw_weight.argtypes = [_P, _P, _I, _I, _I, _D, _I, _I, _I, _I]
        _lib.oracle_tnlm_raw_weight.restype = _D
        _lib.oracle_tnlm_weights_pixel.argtypes = [_P, _P, _I, _I, _I, _I, _D, _I, _I, _P]
        _lib.oracle_tnlm_weights_pixel.restype = None
        _lib.oracle_regularize_step.argtypes = [_I, _I, _I, _I, _I, _D, _D, _P, _I, _P, _I]
        _lib.oracle_gj_sweep_pixels.argtypes = [_I, _I, _I, _I, _I, _D, _D, _P, _P, _I, _P, _P]
        _lib.oracle_reconstruct.argtypes = geo + [_I, _I, _D, _D, _P, _P, _P, _I, _I, _I, _P, _I]
        _lib.oracle_cost.argtypes = geo + [_I, _I, _D, _P, _P, _P, _P, _P]
    return _lib


def num_threads() -> int:
    return int(lib().oracle_num_threads())


@dataclass
class Geometry:
    """Fan-beam, equiangular arc detector. angles: [n_phase][n_views] radians."""
    n_views: int
    n_bins: int
    sid_mm: float
    sdd_mm: float
    bin_pitch_mm: float
    angles_rad: np.ndarray
    bin_offset: float = 0.0
    pixel_mm: float = 1.0


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _ptr(a):
    return None if a is None else a.ctypes.data_as(_P)


def _geo_args(geom: Geometry, nx, ny, n_phase):
    ang = _f64(geom.angles_rad)
    assert ang.shape == (n_phase, geom.n_views), (ang.shape, n_phase, geom.n_views)
    return ang, [nx, ny, n_phase, geom.n_views, geom.n_bins, geom.sid_mm, geom.sdd_mm,
                 geom.bin_pitch_mm, geom.bin_offset, geom.pixel_mm, _ptr(ang)]


def _split(img):
    """[N][ny][nx] or [S][N][ny][nx] -> (4-d array, had_slices)."""
    a = _f64(img)
    if a.ndim == 3:
        return a[None], False
    assert a.ndim == 4
    return a, True


def project(geom: Geometry, img):
    a, sl = _split(img)
    S, N, ny, nx = a.shape
    ang, g = _geo_args(geom, nx, ny, N)
    out = np.zeros((S, N, geom.n_views, geom.n_bins))
    lib().oracle_project(*g, _ptr(a), _ptr(out), S)
    return out if sl else out[0]


def backproject(geom: Geometry, sino, nx, ny):
    a, sl = _split(sino)
    S, N, V, B = a.shape
    ang, g = _geo_args(geom, nx, ny, N)
    out = np.zeros((S, N, ny, nx))
    lib().oracle_backproject(*g, _ptr(a), _ptr(out), S)
    return out if sl else out[0]


def project_rays(geom: Geometry, img, rays):
    a = _f64(img)
    N, ny, nx = a.shape
    ang, g = _geo_args(geom, nx, ny, N)
    idx = np.ascontiguousarray(rays, dtype=np.int64)
    out = np.zeros(idx.size)
    lib().oracle_project_rays(*g, _ptr(a), idx.size, _ptr(idx), _ptr(out))
    return out


def backproject_pixels(geom: Geometry, sino, nx, ny, pixels):
    a = _f64(sino)
    N = a.shape[0]
    ang, g = _geo_args(geom, nx, ny, N)
    idx = np.ascontiguousarray(pixels, dtype=np.int64)
    out = np.zeros(idx.size)
    lib().oracle_backproject_pixels(*g, _ptr(a), idx.size, _ptr(idx), _ptr(out))
    return out


def cgls_step(geom: Geometry, f_in, y, w, m1):
    a, sl = _split(f_in)
    S, N, ny, nx = a.shape
    ang, g = _geo_args(geom, nx, ny, N)
    yy = _f64(y).reshape(S, N, geom.n_views, geom.n_bins)
    ww = None if w is None else _f64(w).reshape(yy.shape)
    out = np.zeros_like(a)
    lib().oracle_cgls_step(*g, _ptr(a), _ptr(yy), _ptr(ww), m1, _ptr(out), S)
    return out if sl else out[0]


def raw_weight(gi, gj, patch, h, x, y):
    """exp(-||R_gi(x)-R_gj(y)||^2/h^2), the weight before normalisation."""
    gi, gj = _f64(gi), _f64(gj)
    ny, nx = gi.shape
    return float(lib().oracle_tnlm_raw_weight(_ptr(gi), _ptr(gj), ny, nx, patch, h,
                                              x[0], x[1], y[0], y[1]))


def weights_pixel(gi, gj, window, patch, h, x):
    """Normalised omega_{i,j}(x, x+delta), [W][W] over delta (0 outside the image)."""
    gi, gj = _f64(gi), _f64(gj)
    ny, nx = gi.shape
    out = np.zeros((window, window))
    lib().oracle_tnlm_weights_pixel(_ptr(gi), _ptr(gj), ny, nx, window, patch, h, x[0], x[1], _ptr(out))
    return out


def regularize_step(g, window, patch, h, mu, m2):
    a, sl = _split(g)
    S, N, ny, nx = a.shape
    out = np.zeros_like(a)
    lib().oracle_regularize_step(nx, ny, N, window, patch, h, mu, _ptr(a), m2, _ptr(out), S)
    return out if sl else out[0]


def gj_sweep_pixels(g, u, window, patch, h, mu, pixels):
    g, u = _f64(g), _f64(u)
    N, ny, nx = g.shape
    idx = np.ascontiguousarray(pixels, dtype=np.int64)
    out = np.zeros(idx.size)
    lib().oracle_gj_sweep_pixels(nx, ny, N, window, patch, h, mu, _ptr(g), _ptr(u), idx.size, _ptr(idx), _ptr(out))
    return out


def reconstruct(geom: Geometry, y, w, f0, nx, ny, window, patch, h, mu, k_outer, m1, m2):
    yy = _f64(y)
    sl = yy.ndim == 4
    if not sl:
        yy = yy[None]
    S, N, V, B = yy.shape
    ang, g = _geo_args(geom, nx, ny, N)
    ww = None if w is None else _f64(w).reshape(yy.shape)
    ff = None if f0 is None else _f64(f0).reshape(S, N, ny, nx)
    out = np.zeros((S, N, ny, nx))
    lib().oracle_reconstruct(*g, window, patch, h, mu, _ptr(yy), _ptr(ww), _ptr(ff),
                             k_outer, m1, m2, _ptr(out), S)
    return out if sl else out[0]


def cost(geom, f, gref, y, w, window, patch, h):
    """(data term, sum_i J(f_i,f_{i-1})+J(f_i,f_{i+1})) of Eq.(1); geom None skips the data term."""
    f, gref = _f64(f), _f64(gref)
    N, ny, nx = f.shape
    out = np.zeros(2)
    if geom is None:
        g = [nx, ny, N, 0, 0, 1.0, 2.0, 1.0, 0.0, 1.0, None]
        lib().oracle_cost(*g, window, patch, h, _ptr(f), _ptr(gref), None, None, _ptr(out))
    else:
        ang, g = _geo_args(geom, nx, ny, N)
        yy = _f64(y)
        ww = None if w is None else _f64(w)
        lib().oracle_cost(*g, window, patch, h, _ptr(f), _ptr(gref), _ptr(yy), _ptr(ww), _ptr(out))
    return float(out[0]), float(out[1])
