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


def forward(g: Grid, sigma: float, ev, image, trunc: float = 3.0) -> np.ndarray:
    e, n, keep = _events(ev, sigma > 0)
    img = np.ascontiguousarray(np.asarray(image, dtype=np.float64).reshape(-1))
    assert img.size == g.nvox
    out = np.empty(n, np.float64)
    lib().orc_forward(C.byref(g), C.c_double(sigma), C.c_double(trunc), C.byref(e), C.c_uint64(n),
                      img.ctypes.data_as(C.c_void_p), out.ctypes.data_as(C.c_void_p))
    return out


def backproject(g: Grid, sigma: float, ev, values: Optional[np.ndarray] = None, trunc: float = 3.0) -> np.ndarray:
    e, n, keep = _events(ev, sigma > 0)
    out = np.zeros(g.nvox, np.float64)
    vals = None
    vp = None
    if values is not None:
        vals = np.ascontiguousarray(np.asarray(values, dtype=np.float64))
        assert vals.shape == (n,)
        vp = vals.ctypes.data_as(C.c_void_p)
    lib().orc_backproject(C.byref(g), C.c_double(sigma), C.c_double(trunc), C.byref(e), C.c_uint64(n), vp,
                          out.ctypes.data_as(C.c_void_p))
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


def em_correction(g: Grid, sigma: float, ev, image, trunc: float = 3.0):
    """(corr float64[nvox], n_valid, visits) of one pass."""
    e, n, keep = _events(ev, sigma > 0)
    img = np.ascontiguousarray(np.asarray(image, dtype=np.float64).reshape(-1))
    corr = np.empty(g.nvox, np.float64)
    vis = C.c_uint64(0)
    nv = lib().orc_em_correction(C.byref(g), C.c_double(sigma), C.c_double(trunc), C.byref(e), C.c_uint64(n),
                                 img.ctypes.data_as(C.c_void_p), corr.ctypes.data_as(C.c_void_p), C.byref(vis))
    return corr, int(nv), int(vis.value)


def update(image, corr, sens_f32, mask) -> np.ndarray:
    img = np.ascontiguousarray(np.asarray(image, dtype=np.float64).reshape(-1)).copy()
    c = np.ascontiguousarray(np.asarray(corr, dtype=np.float64).reshape(-1))
    s = _f32(sens_f32).reshape(-1)
    m = np.ascontiguousarray(np.asarray(mask, dtype=np.uint8).reshape(-1))
    lib().orc_update(C.c_int64(img.size), img.ctypes.data_as(C.c_void_p), c.ctypes.data_as(C.c_void_p),
                     s.ctypes.data_as(C.c_void_p), m.ctypes.data_as(C.c_void_p))
    return img


def mlem(g: Grid, sigma: float, ev, image0, sens_f32, iters: int, floor_rel: float = 1e-2, trunc: float = 3.0):
    """(image float64[nvox] after `iters` iterations, Stats)."""
    e, n, keep = _events(ev, sigma > 0)
    img = np.ascontiguousarray(np.asarray(image0, dtype=np.float64).reshape(-1)).copy()
    s = _f32(sens_f32).reshape(-1)
    assert img.size == g.nvox and s.size == g.nvox
    st = Stats()
    lib().orc_mlem(C.byref(g), C.c_double(sigma), C.c_double(trunc), C.byref(e), C.c_uint64(n),
                   img.ctypes.data_as(C.c_void_p), s.ctypes.data_as(C.c_void_p), C.c_int(iters),
                   C.c_float(floor_rel), C.byref(st))
    return img, st


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


def region_margin_slices(sigma: float, vz: float, trunc: float = 3.0, shell_mm: float = 6.0) -> int:
    return int(lib().orc_region_margin_slices(sigma, trunc, shell_mm, vz))


def num_threads() -> int:
    return int(lib().orc_num_threads())
