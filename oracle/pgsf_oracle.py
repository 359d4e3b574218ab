"""ctypes front end of the fp64 CPU oracle (oracle/pgsf_oracle.c).

TEST INFRASTRUCTURE, NOT PRODUCT CODE.  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this module; the product path
(paper_1507_04941_b200) never does and shares no code with it.

Everything numerical lives in the C file; this module only marshals numpy arrays, and composes
the per-scale calls into the multi-scale result the way the paper's pipeline does
(P:33 / P:49: "a series of three-dimensional Gaussian filters", then local mean / standard
deviation thresholds; "statistics and voxel selection").

Arrays are numpy, C-contiguous, shape [nz, ny, nx] (x fastest; reading C-0 in DESIGN.md).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pgsf_oracle.c")
_LIB = os.path.join(_HERE, "libpgsf_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc -O2 (+OpenMP for the timed multi-core baseline)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-fopenmp", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_LIB)
        c_int_p = ctypes.POINTER(ctypes.c_int)
        c_dbl_p = ctypes.POINTER(ctypes.c_double)
        c_flt_p = ctypes.POINTER(ctypes.c_float)
        c_u8_p = ctypes.POINTER(ctypes.c_uint8)
        lib.pgsf_oracle_set_threads.argtypes = [ctypes.c_int]
        lib.pgsf_oracle_set_threads.restype = ctypes.c_int
        lib.pgsf_oracle_radius.argtypes = [ctypes.c_double, ctypes.c_double]
        lib.pgsf_oracle_radius.restype = ctypes.c_int
        lib.pgsf_oracle_taps.argtypes = [ctypes.c_double, ctypes.c_int, c_dbl_p]
        lib.pgsf_oracle_taps.restype = None
        lib.pgsf_oracle_filter_direct.argtypes = [
            c_flt_p, ctypes.c_int, ctypes.c_int, ctypes.c_int,
            c_dbl_p, ctypes.c_int, c_dbl_p, ctypes.c_int, c_dbl_p, ctypes.c_int, c_dbl_p]
        lib.pgsf_oracle_filter_direct.restype = None
        lib.pgsf_oracle_threshold_brute.argtypes = [
            c_dbl_p, ctypes.c_int, ctypes.c_int, ctypes.c_int,
            ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_double,
            c_dbl_p, c_dbl_p, c_dbl_p, c_u8_p]
        lib.pgsf_oracle_threshold_brute.restype = None
        lib.pgsf_oracle_wfilter_direct.argtypes = [
            c_flt_p, c_flt_p, ctypes.c_int, ctypes.c_int, ctypes.c_int, c_dbl_p, ctypes.c_int, c_dbl_p,
            ctypes.c_int, c_dbl_p, ctypes.c_int, ctypes.c_int, c_dbl_p]
        lib.pgsf_oracle_wfilter_direct.restype = None
        lib.pgsf_oracle_wfilter.argtypes = lib.pgsf_oracle_wfilter_direct.argtypes
        lib.pgsf_oracle_wfilter.restype = ctypes.c_int
        lib.pgsf_oracle_filter_general.argtypes = [
            c_flt_p, ctypes.c_int, ctypes.c_int, ctypes.c_int, c_dbl_p, ctypes.c_int, ctypes.c_int, ctypes.c_int,
            c_dbl_p]
        lib.pgsf_oracle_filter_general.restype = None
        lib.pgsf_oracle_filter_region.argtypes = [
            c_flt_p, c_int_p, c_int_p, c_int_p,
            c_dbl_p, ctypes.c_int, c_dbl_p, ctypes.c_int, c_dbl_p, ctypes.c_int,
            c_int_p, c_int_p, c_dbl_p]
        lib.pgsf_oracle_filter_region.restype = ctypes.c_int
        lib.pgsf_oracle_threshold_region.argtypes = [
            c_dbl_p, c_int_p, c_int_p, c_int_p, c_int_p, ctypes.c_double,
            c_int_p, c_int_p, c_dbl_p, c_dbl_p, c_dbl_p, c_u8_p]
        lib.pgsf_oracle_threshold_region.restype = ctypes.c_int
        lib.pgsf_oracle_label26.argtypes = [c_u8_p, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.POINTER(ctypes.c_uint32)]
        lib.pgsf_oracle_label26.restype = ctypes.c_int64
        _lib = lib
    return _lib


def _p(a, ct):
    return a.ctypes.data_as(ctypes.POINTER(ct)) if a is not None else None


def _i3(v):
    return (ctypes.c_int * 3)(int(v[0]), int(v[1]), int(v[2]))


def set_threads(n: int) -> int:
    """Set the OpenMP thread count of the oracle; returns the count in effect."""
    return int(_load().pgsf_oracle_set_threads(int(n)))


def radius(sigma: float, truncate: float = 3.0) -> int:
    return int(_load().pgsf_oracle_radius(float(sigma), float(truncate)))


def taps(sigma: float, truncate: float = 3.0) -> np.ndarray:
    """fp64 taps g[-r..r] for one axis (C-1..C-3)."""
    r = radius(sigma, truncate)
    g = np.zeros(2 * r + 1, dtype=np.float64)
    _load().pgsf_oracle_taps(float(sigma), r, _p(g, ctypes.c_double))
    return g


# --------------------------------------------------------------------------- L0: definitions

def filter_direct(d: np.ndarray, sigma3: Sequence[float], truncate: float = 3.0) -> np.ndarray:
    """Eq. 2 as a direct six-deep loop (tiny cubes).  d: float32 [nz,ny,nx]; returns float64."""
    d = np.ascontiguousarray(d, dtype=np.float32)
    nz, ny, nx = d.shape
    gx, gy, gz = (taps(s, truncate) for s in sigma3)
    out = np.empty(d.shape, dtype=np.float64)
    _load().pgsf_oracle_filter_direct(
        _p(d, ctypes.c_float), nx, ny, nz,
        _p(gx, ctypes.c_double), (len(gx) - 1) // 2, _p(gy, ctypes.c_double), (len(gy) - 1) // 2,
        _p(gz, ctypes.c_double), (len(gz) - 1) // 2, _p(out, ctypes.c_double))
    return out


@dataclass
class Stats:
    mean: np.ndarray
    std: np.ndarray
    thr: np.ndarray
    mask: np.ndarray


def threshold_brute(c: np.ndarray, box_half: Sequence[int], k: float) -> Stats:
    """Local mean/std/threshold/mask by scanning every voxel's clipped window (tiny cubes)."""
    c = np.ascontiguousarray(c, dtype=np.float64)
    nz, ny, nx = c.shape
    mean = np.empty(c.shape, np.float64)
    sd = np.empty(c.shape, np.float64)
    thr = np.empty(c.shape, np.float64)
    mask = np.empty(c.shape, np.uint8)
    _load().pgsf_oracle_threshold_brute(
        _p(c, ctypes.c_double), nx, ny, nz, int(box_half[0]), int(box_half[1]), int(box_half[2]),
        float(k), _p(mean, ctypes.c_double), _p(sd, ctypes.c_double), _p(thr, ctypes.c_double),
        _p(mask, ctypes.c_uint8))
    return Stats(mean, sd, thr, mask)


# --------------------------------------------------------------------------- L1: separable, regions

def filter_general(d: np.ndarray, f: np.ndarray) -> np.ndarray:
    """Eq. 2 for an arbitrary filter array f[oz, oy, ox] with odd extents (NEXT-2): direct loops,
    correlation orientation as printed, zero outside the cube, fp64.  d: [nz, ny, nx]."""
    d = np.ascontiguousarray(d, dtype=np.float32)
    f = np.ascontiguousarray(f, dtype=np.float64)
    assert d.ndim == 3 and f.ndim == 3 and all(n % 2 == 1 for n in f.shape)
    nz, ny, nx = d.shape
    rz, ry, rx = [(n - 1) // 2 for n in f.shape]
    out = np.empty(d.shape, dtype=np.float64)
    _load().pgsf_oracle_filter_general(_p(d, ctypes.c_float), nx, ny, nz, _p(f, ctypes.c_double), rx, ry, rz,
                                       _p(out, ctypes.c_double))
    return out


def label26(mask: np.ndarray):
    """NEXT-4 (reading C-19): connected components of a mask [nz, ny, nx] under 26-connectivity by flood fill.
    Returns (labels uint32 [nz, ny, nx], count); label = 1 + smallest linear index of the component, 0 = background."""
    m = np.ascontiguousarray(mask, dtype=np.uint8)
    assert m.ndim == 3
    nz, ny, nx = m.shape
    labels = np.empty(m.shape, dtype=np.uint32)
    n = _load().pgsf_oracle_label26(_p(m, ctypes.c_uint8), nx, ny, nz, _p(labels, ctypes.c_uint32))
    return labels, int(n)


def _wfilter(fn, d, w, sigma3, mode, truncate):
    d = np.ascontiguousarray(d, dtype=np.float32)
    w = np.ascontiguousarray(w, dtype=np.float32)
    assert d.shape == w.shape and d.ndim == 3
    nz, ny, nx = d.shape
    g = [taps(s, truncate) for s in sigma3]
    r = [radius(s, truncate) for s in sigma3]
    out = np.empty(d.shape, dtype=np.float64)
    rc = fn(_p(d, ctypes.c_float), _p(w, ctypes.c_float), nx, ny, nz, _p(g[0], ctypes.c_double), r[0],
            _p(g[1], ctypes.c_double), r[1], _p(g[2], ctypes.c_double), r[2], int(mode), _p(out, ctypes.c_double))
    if rc not in (None, 0):
        raise MemoryError(f"pgsf_oracle_wfilter failed ({rc})")
    return out


def wfilter_direct(d: np.ndarray, w: np.ndarray, sigma3, mode: int = 0, truncate: float = 3.0) -> np.ndarray:
    """L0 of Eq. 1: direct loops.  d, w: [nz, ny, nx]; mode 0 = denominator as printed (sum w),
    mode 1 = sum f w."""
    return _wfilter(_load().pgsf_oracle_wfilter_direct, d, w, sigma3, mode, truncate)


def wfilter_full(d: np.ndarray, w: np.ndarray, sigma3, mode: int = 0, truncate: float = 3.0) -> np.ndarray:
    """L1 of Eq. 1: separable numerator (Eq. 2 of d*w) over box sum of w (mode 0) or Eq. 2 of w (mode 1)."""
    return _wfilter(_load().pgsf_oracle_wfilter, d, w, sigma3, mode, truncate)


def filter_region(sub: np.ndarray, sub_lo, cube, sigma3, lo, hi, truncate: float = 3.0) -> np.ndarray:
    """Separable fp64 filter on the region [lo,hi) (x,y,z order) of a cube with extents `cube`.

    `sub` (float32 [sz,sy,sx]) holds cube coordinates [sub_lo, sub_lo+shape); it must contain the
    region +- radius clipped to the cube.  Returns float64 [hi_z-lo_z, hi_y-lo_y, hi_x-lo_x]."""
    sub = np.ascontiguousarray(sub, dtype=np.float32)
    sz, sy, sx = sub.shape
    shi = (sub_lo[0] + sx, sub_lo[1] + sy, sub_lo[2] + sz)
    gx, gy, gz = (taps(s, truncate) for s in sigma3)
    out = np.empty((hi[2] - lo[2], hi[1] - lo[1], hi[0] - lo[0]), dtype=np.float64)
    rc = _load().pgsf_oracle_filter_region(
        _p(sub, ctypes.c_float), _i3(sub_lo), _i3(shi), _i3(cube),
        _p(gx, ctypes.c_double), (len(gx) - 1) // 2, _p(gy, ctypes.c_double), (len(gy) - 1) // 2,
        _p(gz, ctypes.c_double), (len(gz) - 1) // 2, _i3(lo), _i3(hi), _p(out, ctypes.c_double))
    if rc != 0:
        raise ValueError(f"pgsf_oracle_filter_region failed rc={rc} (sub does not cover region+-r?)")
    return out


def threshold_region(csub: np.ndarray, c_lo, cube, box_half, k, lo, hi) -> Stats:
    """Three directional sums + threshold on region [lo,hi); csub (float64) covers
    cube coordinates [c_lo, c_lo+shape) and must contain the region +- box_half clipped."""
    csub = np.ascontiguousarray(csub, dtype=np.float64)
    cz, cy, cx = csub.shape
    chi = (c_lo[0] + cx, c_lo[1] + cy, c_lo[2] + cz)
    shape = (hi[2] - lo[2], hi[1] - lo[1], hi[0] - lo[0])
    mean = np.empty(shape, np.float64)
    sd = np.empty(shape, np.float64)
    thr = np.empty(shape, np.float64)
    mask = np.empty(shape, np.uint8)
    rc = _load().pgsf_oracle_threshold_region(
        _p(csub, ctypes.c_double), _i3(c_lo), _i3(chi), _i3(cube), _i3(box_half), float(k),
        _i3(lo), _i3(hi), _p(mean, ctypes.c_double), _p(sd, ctypes.c_double),
        _p(thr, ctypes.c_double), _p(mask, ctypes.c_uint8))
    if rc != 0:
        raise ValueError(f"pgsf_oracle_threshold_region failed rc={rc}")
    return Stats(mean, sd, thr, mask)


def filter_full(d: np.ndarray, sigma3, truncate: float = 3.0) -> np.ndarray:
    """Separable fp64 filter of a whole cube."""
    nz, ny, nx = d.shape
    return filter_region(d, (0, 0, 0), (nx, ny, nz), sigma3, (0, 0, 0), (nx, ny, nz), truncate)


def threshold_full(c: np.ndarray, box_half, k) -> Stats:
    nz, ny, nx = c.shape
    return threshold_region(c, (0, 0, 0), (nx, ny, nz), box_half, k, (0, 0, 0), (nx, ny, nz))


@dataclass
class ScaleResult:
    f: np.ndarray       # filtered region, float64
    stats: Stats        # mean/std/thr/mask on the region (mask BEFORE halo exclusion)


@dataclass
class FindResult:
    scales: list        # list[ScaleResult]
    mask: np.ndarray    # OR over scales, halo voxels forced 0 (C-11), uint8
    count: int          # number of set voxels in `mask` (C-15)


def required_input_box(cube, sigmas, box_half, lo, hi, truncate: float = 3.0):
    """Cube-coordinate box [a,b) of input needed to evaluate region [lo,hi): region +- (r+h) clipped."""
    rmax = [max(radius(s[ax], truncate) for s in sigmas) for ax in range(3)]
    a = tuple(max(0, lo[ax] - rmax[ax] - box_half[ax]) for ax in range(3))
    b = tuple(min(cube[ax], hi[ax] + rmax[ax] + box_half[ax]) for ax in range(3))
    return a, b


def find_region(sub: np.ndarray, sub_lo, cube, sigmas, box_half, k, lo, hi,
                halo=(0, 0, 0), truncate: float = 3.0) -> FindResult:
    """Multi-scale filter + local threshold on region [lo,hi) of ONE cube (standalone, zero padded:
    C-5, C-7, C-11).  For each scale: filter on region +- box_half (clipped), then the statistics;
    masks are OR'd over scales (BASELINE.json north_star); voxels within `halo` of a cube
    face are forced to 0 and not counted (C-11, C-15)."""
    nx, ny, nz = cube
    flo = tuple(max(0, lo[ax] - box_half[ax]) for ax in range(3))
    fhi = tuple(min(cube[ax], hi[ax] + box_half[ax]) for ax in range(3))
    res = []
    shape = (hi[2] - lo[2], hi[1] - lo[1], hi[0] - lo[0])
    ormask = np.zeros(shape, np.uint8)
    for s in sigmas:
        fext = filter_region(sub, sub_lo, cube, s, flo, fhi, truncate)
        st = threshold_region(fext, flo, cube, box_half, k, lo, hi)
        f = fext[lo[2] - flo[2]: hi[2] - flo[2], lo[1] - flo[1]: hi[1] - flo[1],
                 lo[0] - flo[0]: hi[0] - flo[0]].copy()
        res.append(ScaleResult(f, st))
        ormask |= st.mask
    # halo exclusion
    zz = np.arange(lo[2], hi[2])[:, None, None]
    yy = np.arange(lo[1], hi[1])[None, :, None]
    xx = np.arange(lo[0], hi[0])[None, None, :]
    inside = ((xx >= halo[0]) & (xx < nx - halo[0]) & (yy >= halo[1]) & (yy < ny - halo[1]) &
              (zz >= halo[2]) & (zz < nz - halo[2]))
    ormask = (ormask & inside.astype(np.uint8)).astype(np.uint8)
    return FindResult(res, ormask, int(ormask.sum(dtype=np.int64)))


def find_full(d: np.ndarray, sigmas, box_half, k, halo=(0, 0, 0), truncate: float = 3.0) -> FindResult:
    nz, ny, nx = d.shape
    return find_region(d, (0, 0, 0), (nx, ny, nz), sigmas, box_half, k, (0, 0, 0), (nx, ny, nz),
                       halo, truncate)
