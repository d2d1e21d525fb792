"""ctypes front-end of the fp64 CPU oracle (oracle/tofmlem_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this package.  It imports nothing from
paper_1706_07075_b200/ and shares no code with it.  All arrays are numpy; events are dicts of
float32 arrays x1,y1,z1,x2,y2,z2[,dt].
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Dict, Optional, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "tofmlem_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")

C_MM_PER_PS = 0.299792458


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (no -ffast-math, no FMA contraction)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared", "-std=c11", "-D_GNU_SOURCE",
               "-Wall", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


class Grid(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
                ("vx", C.c_double), ("vy", C.c_double), ("vz", C.c_double),
                ("ox", C.c_double), ("oy", C.c_double), ("oz", C.c_double)]

    @property
    def nvox(self) -> int:
        return self.nx * self.ny * self.nz


class GridF32(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
                ("vx", C.c_float), ("vy", C.c_float), ("vz", C.c_float),
                ("ox", C.c_float), ("oy", C.c_float), ("oz", C.c_float)]


class _Events(C.Structure):
    _fields_ = [(k, C.c_void_p) for k in ("x1", "y1", "z1", "x2", "y2", "z2", "dt")]


class Stats(C.Structure):
    _fields_ = [("n_valid", C.c_uint64), ("n_skipped", C.c_uint64), ("visits", C.c_uint64),
                ("sum_image_sens", C.c_double)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_sigma_mm.restype = C.c_double
        _lib.orc_sigma_mm.argtypes = [C.c_double, C.c_double]
        _lib.orc_lor_weights.restype = C.c_int
        _lib.orc_em_correction.restype = C.c_uint64
        _lib.orc_em_correction_w.restype = C.c_uint64
        _lib.orc_lor_samples.restype = C.c_int
        _lib.orc_num_bins.restype = C.c_uint32
        _lib.orc_region_margin_slices.restype = C.c_int32
        _lib.orc_region_margin_slices.argtypes = [C.c_double, C.c_double, C.c_double, C.c_double]
    return _lib


def make_grid(nx, ny, nz, v, origin=None) -> Grid:
    vx, vy, vz = (v, v, v) if np.isscalar(v) else v
    if origin is None:
        origin = (-0.5 * nx * vx, -0.5 * ny * vy, -0.5 * nz * vz)
    return Grid(nx, ny, nz, vx, vy, vz, *origin)


def grid_f32(g: Grid) -> GridF32:
    return GridF32(g.nx, g.ny, g.nz, g.vx, g.vy, g.vz, g.ox, g.oy, g.oz)


def _f32(a) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(a, dtype=np.float32))


def _events(ev: Dict[str, np.ndarray], need_dt: bool) -> Tuple[_Events, int, list]:
    keep = []
    ptrs = {}
    n = None
    for k in ("x1", "y1", "z1", "x2", "y2", "z2"):
        a = _f32(ev[k])
        keep.append(a)
        ptrs[k] = a.ctypes.data
        n = a.shape[0] if n is None else n
        assert a.shape == (n,)
    if ev.get("dt") is not None:
        a = _f32(ev["dt"])
        assert a.shape == (n,)
        keep.append(a)
        ptrs["dt"] = a.ctypes.data
    else:
        assert not need_dt, "TOF mode needs dt"
        ptrs["dt"] = None
    return _Events(**ptrs), n, keep


def sigma_mm(fwhm_ps: float, c_mm_per_ps: float = C_MM_PER_PS) -> float:
    return float(lib().orc_sigma_mm(fwhm_ps, c_mm_per_ps))


def lor_weights(g: Grid, sigma: float, p1, p2, dt_ps: float = 0.0, trunc: float = 3.0):
    """(voxel indices int64, weights float64) of one LOR, in traversal order."""
    cap = int(lib().orc_lor_capacity(C.byref(g)))
    idx = np.empty(cap, np.int64)
    w = np.empty(cap, np.float64)
    scratch = np.empty(cap, np.float64)
    a = (C.c_double * 3)(*map(float, p1))
    b = (C.c_double * 3)(*map(float, p2))
    cnt = lib().orc_lor_weights(C.byref(g), C.c_double(sigma), C.c_double(trunc), a, b, C.c_double(dt_ps),
                                idx.ctypes.data_as(C.c_void_p), w.ctypes.data_as(C.c_void_p),
                                scratch.ctypes.data_as(C.c_void_p), C.c_int(cap))
    assert cnt >= 0
    return idx[:cnt].copy(), w[:cnt].copy()


def forward(g: Grid, sigma: float, ev, image, trunc: float = 3.0, K: int = 0) -> np.ndarray:
    """fwd_e = sum_j a_ej x_j; K = 0: Siddon x Gaussian rows, K >= 1: the paper's K-sample kernel."""
    e, n, keep = _events(ev, sigma > 0)
    img = np.ascontiguousarray(np.asarray(image, dtype=np.float64).reshape(-1))
    assert img.size == g.nvox
    out = np.empty(n, np.float64)
    lib().orc_forward_k(C.byref(g), C.c_double(sigma), C.c_double(trunc), C.c_int(K), C.byref(e), C.c_uint64(n),
                        img.ctypes.data_as(C.c_void_p), out.ctypes.data_as(C.c_void_p))
    return out


def backproject(g: Grid, sigma: float, ev, values: Optional[np.ndarray] = None, trunc: float = 3.0,
                K: int = 0) -> np.ndarray:
    e, n, keep = _events(ev, sigma > 0)
    out = np.zeros(g.nvox, np.float64)
    vals = None
    vp = None
    if values is not None:
        vals = np.ascontiguousarray(np.asarray(values, dtype=np.float64))
        assert vals.shape == (n,)
        vp = vals.ctypes.data_as(C.c_void_p)
    lib().orc_backproject_k(C.byref(g), C.c_double(sigma), C.c_double(trunc), C.c_int(K), C.byref(e), C.c_uint64(n),
                            vp, out.ctypes.data_as(C.c_void_p))
    return out


def sensitivity(g: Grid, lors) -> np.ndarray:
    e, m, keep = _events({**lors, "dt": None}, False)
    out = np.empty(g.nvox, np.float64)
    lib().orc_sensitivity(C.byref(g), C.byref(e), C.c_uint64(m), out.ctypes.data_as(C.c_void_p))
    return out


def mask_f32(sens_f32: np.ndarray, floor_rel: float = 1e-2) -> np.ndarray:
    s = _f32(sens_f32).reshape(-1)
    m = np.empty(s.size, np.uint8)
    lib().orc_mask_f32(s.ctypes.data_as(C.c_void_p), C.c_int64(s.size), C.c_float(floor_rel),
                       m.ctypes.data_as(C.c_void_p))
    return m


def _f64_or_none(a, n):
    if a is None:
        return None, None
    v = np.ascontiguousarray(np.asarray(a, dtype=np.float64))
    assert v.shape == (n,)
    return v, v.ctypes.data_as(C.c_void_p)


def em_correction(g: Grid, sigma: float, ev, image, trunc: float = 3.0, K: int = 0, weights=None):
    """(corr float64[nvox], n_valid, visits) of one pass; `weights`: optional per-event weights (NEXT-3)."""
    e, n, keep = _events(ev, sigma > 0)
    img = np.ascontiguousarray(np.asarray(image, dtype=np.float64).reshape(-1))
    corr = np.empty(g.nvox, np.float64)
    vis = C.c_uint64(0)
    wk, wp = _f64_or_none(weights, n)
    nv = lib().orc_em_correction_w(C.byref(g), C.c_double(sigma), C.c_double(trunc), C.c_int(K), C.byref(e),
                                   C.c_uint64(n), wp, img.ctypes.data_as(C.c_void_p),
                                   corr.ctypes.data_as(C.c_void_p), C.byref(vis), None)
    return corr, int(nv), int(vis.value)


def update(image, corr, sens_f32, mask) -> np.ndarray:
    img = np.ascontiguousarray(np.asarray(image, dtype=np.float64).reshape(-1)).copy()
    c = np.ascontiguousarray(np.asarray(corr, dtype=np.float64).reshape(-1))
    s = _f32(sens_f32).reshape(-1)
    m = np.ascontiguousarray(np.asarray(mask, dtype=np.uint8).reshape(-1))
    lib().orc_update(C.c_int64(img.size), img.ctypes.data_as(C.c_void_p), c.ctypes.data_as(C.c_void_p),
                     s.ctypes.data_as(C.c_void_p), m.ctypes.data_as(C.c_void_p))
    return img


def mlem(g: Grid, sigma: float, ev, image0, sens_f32, iters: int, floor_rel: float = 1e-2, trunc: float = 3.0,
         K: int = 0, weights=None, median: bool = False):
    """(image float64[nvox] after `iters` iterations, Stats).  K: row model (0 = Siddon x Gaussian);
    weights: optional per-event weights (NEXT-3); median: 3x3x3 median filter after every iteration (NEXT-2)."""
    e, n, keep = _events(ev, sigma > 0)
    img = np.ascontiguousarray(np.asarray(image0, dtype=np.float64).reshape(-1)).copy()
    s = _f32(sens_f32).reshape(-1)
    assert img.size == g.nvox and s.size == g.nvox
    st = Stats()
    wk, wp = _f64_or_none(weights, n)
    lib().orc_mlem_x(C.byref(g), C.c_double(sigma), C.c_double(trunc), C.c_int(K), C.byref(e), C.c_uint64(n), wp,
                     img.ctypes.data_as(C.c_void_p), s.ctypes.data_as(C.c_void_p), C.c_int(iters),
                     C.c_float(floor_rel), C.c_int(1 if median else 0), C.byref(st))
    return img, st


def sample_lut(K: int, sigma: float, trunc: float = 3.0):
    """(offsets mm float64[K], weights float64[K]) of the paper's K-sample TOF kernel."""
    off = np.empty(K, np.float64)
    w = np.empty(K, np.float64)
    lib().orc_sample_lut(C.c_int(K), C.c_double(sigma), C.c_double(trunc), off.ctypes.data_as(C.c_void_p),
                         w.ctypes.data_as(C.c_void_p))
    return off, w


def lor_samples(g: Grid, sigma: float, K: int, p1, p2, dt_ps: float = 0.0, trunc: float = 3.0):
    """(voxel indices, weights) of one event under the K-sample kernel, in sample order (dropped samples omitted)."""
    off, w = sample_lut(K, sigma, trunc)
    idx = np.empty(K, np.int64)
    ww = np.empty(K, np.float64)
    a = (C.c_double * 3)(*map(float, p1))
    b = (C.c_double * 3)(*map(float, p2))
    cnt = lib().orc_lor_samples(C.byref(g), C.c_int(K), off.ctypes.data_as(C.c_void_p), w.ctypes.data_as(C.c_void_p),
                                a, b, C.c_double(dt_ps), idx.ctypes.data_as(C.c_void_p),
                                ww.ctypes.data_as(C.c_void_p))
    return idx[:cnt].copy(), ww[:cnt].copy()


def median3(g: Grid, image) -> np.ndarray:
    """3x3x3 median filter, edges replicated (NEXT-2, R23)."""
    img = np.ascontiguousarray(np.asarray(image, dtype=np.float64).reshape(-1))
    assert img.size == g.nvox
    out = np.empty(g.nvox, np.float64)
    lib().orc_median3(C.c_int32(g.nx), C.c_int32(g.ny), C.c_int32(g.nz), img.ctypes.data_as(C.c_void_p),
                      out.ctypes.data_as(C.c_void_p))
    return out


def attenuation_weights(g: Grid, ev, mu) -> np.ndarray:
    """w_e = exp(+ line integral of mu (1/mm) along the LOR inside the grid) (NEXT-3, R19)."""
    e, n, keep = _events({**ev, "dt": None}, False)
    m = np.ascontiguousarray(np.asarray(mu, dtype=np.float64).reshape(-1))
    assert m.size == g.nvox
    out = np.empty(n, np.float64)
    lib().orc_attenuation_weights(C.byref(g), C.byref(e), C.c_uint64(n), m.ctypes.data_as(C.c_void_p),
                                  out.ctypes.data_as(C.c_void_p))
    return out


CONF95_Z = 1.959964  # two-sided 95 % point of the normal distribution ("95% confidence level")


def scatter_half_width_f32(sigma: float, conf_z: float = CONF95_Z) -> np.float32:
    return np.float32(conf_z * sigma)


def ellipsoids_f32(shapes) -> np.ndarray:
    """float32[n,6] = (cx, cy, cz, 1/ax, 1/ay, 1/az) from (centre, semi-axes) pairs; the reciprocals are taken
    in float64 and rounded once (both sides receive this same array)."""
    out = np.empty((len(shapes), 6), np.float32)
    for i, (c, s) in enumerate(shapes):
        out[i, :3] = np.asarray(c, np.float64)
        out[i, 3:] = 1.0 / np.asarray(s, np.float64)
    return out


def scatter_keep(ev, ell_f32: np.ndarray, h_f32) -> Tuple[np.ndarray, int]:
    """(keep uint8[n], n_kept): TOF-based scatter rejection against a union of ellipsoids (NEXT-4, spec F2)."""
    e, n, keepalive = _events(ev, True)
    ell = np.ascontiguousarray(np.asarray(ell_f32, dtype=np.float32).reshape(-1, 6))
    keep = np.empty(n, np.uint8)
    cnt = C.c_uint64(0)
    lib().orc_scatter_keep(C.byref(e), C.c_uint64(n), ell.ctypes.data_as(C.c_void_p), C.c_int(ell.shape[0]),
                           C.c_float(float(h_f32)), keep.ctypes.data_as(C.c_void_p), C.byref(cnt))
    return keep, int(cnt.value)


def num_bins(g: Grid, tile_log2: int = 3) -> int:
    gf = grid_f32(g)
    return int(lib().orc_num_bins(C.byref(gf), C.c_int(tile_log2)))


def bin_keys(g: Grid, ev, tile_log2: int = 3) -> np.ndarray:
    e, n, keep = _events(ev, False)
    gf = grid_f32(g)
    key = np.empty(n, np.uint32)
    lib().orc_bin_keys(C.byref(gf), C.byref(e), C.c_uint64(n), C.c_int(tile_log2), key.ctypes.data_as(C.c_void_p))
    return key


def default_region_slices(nz: int, n_regions: int = 9) -> np.ndarray:
    k = np.empty(n_regions + 1, np.int32)
    lib().orc_default_region_slices(C.c_int32(nz), C.c_int(n_regions), k.ctypes.data_as(C.c_void_p))
    return k


def region_zbounds(g: Grid, n_regions: int = 9) -> np.ndarray:
    gf = grid_f32(g)
    zb = np.empty(n_regions + 1, np.float32)
    lib().orc_region_zbounds(C.byref(gf), C.c_int(n_regions), zb.ctypes.data_as(C.c_void_p))
    return zb


def region_ids(ev, zbounds: np.ndarray):
    """(region int32[n] (-1 invalid), counts uint64[R]) for ascending float32 boundaries zb[0..R]."""
    e, n, keep = _events(ev, False)
    zb = _f32(zbounds)
    R = zb.size - 1
    region = np.empty(n, np.int32)
    counts = np.empty(R, np.uint64)
    lib().orc_region_ids(C.byref(e), C.c_uint64(n), C.c_int(R), zb.ctypes.data_as(C.c_void_p),
                         region.ctypes.data_as(C.c_void_p), counts.ctypes.data_as(C.c_void_p))
    return region, counts


def region_spans(ev, zbounds: np.ndarray, half_window_mm: float):
    """Reading R27 / specification F3: (lo int32[n], hi int32[n] (-1 invalid), counts uint64[R]): the event belongs to
    regions lo..hi, those whose core the axial extent of its +-half_window TOF window meets."""
    e, n, _keep = _events(ev, False)
    zb = _f32(zbounds)
    R = zb.size - 1
    lo = np.empty(n, np.int32)
    hi = np.empty(n, np.int32)
    counts = np.zeros(R, np.uint64)
    lib().orc_region_spans(C.byref(e), C.c_uint64(n), C.c_int(R), zb.ctypes.data_as(C.c_void_p),
                           C.c_float(np.float32(half_window_mm)), lo.ctypes.data_as(C.c_void_p),
                           hi.ctypes.data_as(C.c_void_p), counts.ctypes.data_as(C.c_void_p))
    return lo, hi, counts


def region_margin_slices(sigma: float, vz: float, trunc: float = 3.0, shell_mm: float = 6.0) -> int:
    return int(lib().orc_region_margin_slices(sigma, trunc, shell_mm, vz))


def num_threads() -> int:
    return int(lib().orc_num_threads())
