"""Thin ctypes binding of libtofmlem.so (include/tofmlem.h): same names, argument marshalling only.

PyTorch is used for device memory and streams: tensors give `data_ptr()`, `torch.cuda.current_stream()`
gives the `cudaStream_t`.  Every step of the path runs inside the library's CUDA kernels; there is no CPU
fallback -- importing works without a GPU (so that the ABI can be checked), every compute call needs one.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Dict, Optional, Sequence

import torch

from . import build as _build

EVENT_FIELDS = ("x1", "y1", "z1", "x2", "y2", "z2", "dt")

TOFMLEM_OK, TOFMLEM_EINVAL, TOFMLEM_ENOMEM, TOFMLEM_ECUDA, TOFMLEM_ESTATE, TOFMLEM_EUNSUPPORTED = 0, -1, -2, -3, -4, -5
OPT_TRUNC_SIGMAS, OPT_SENS_FLOOR_REL, OPT_TILE_LOG2, OPT_PROJECTOR, OPT_SAMPLES_K, OPT_SHELL_MM = 1, 2, 3, 4, 5, 6
OPT_CTA_INTERLEAVE = 7
OPT_EM_VARIANT = 8
OPT_SUBBINS = 9
OPT_MEDIAN = 10
OPT_CACHE_SHARE = 11
OPT_CORR_BRICKS = 12
OPT_DETERMINISTIC = 13
OPT_TILE_MIN_EVENTS = 14
OPT_TILE_CHECK = 15
OPT_TILE_MAX_EVENTS = 16
OPT_REGION_PLAN = 17
OPT_REGION_OVERLAP = 18
OPT_L2_PERSIST = 19
OPT_TILE_MIN_ITEMS = 20
OPT_SENS_SORT = 21
OPT_CONCURRENT = 22
OPT_WARP_WALK = 23
PROJECTOR_SIDDON, PROJECTOR_SAMPLED = 0, 1

# every symbol include/tofmlem.h declares (checked by tests/test_abi.py against the header text)
SYMBOLS = (
    "tofmlem_create", "tofmlem_destroy", "tofmlem_set_option", "tofmlem_sigma_mm", "tofmlem_sensitivity",
    "tofmlem_forward", "tofmlem_backproject", "tofmlem_em_correction", "tofmlem_reset_stats", "tofmlem_update",
    "tofmlem_iterate", "tofmlem_iterate_host", "tofmlem_bin_events", "tofmlem_num_bins", "tofmlem_gather_events",
    "tofmlem_split_regions", "tofmlem_region_zbounds", "tofmlem_region_grid", "tofmlem_reconstruct_regions",
    "tofmlem_probe", "tofmlem_get_stats", "tofmlem_last_error", "tofmlem_launch_count", "tofmlem_version",
    "tofmlem_median3", "tofmlem_attenuation_weights", "tofmlem_em_correction_weighted", "tofmlem_iterate_weighted",
    "tofmlem_gather_f32", "tofmlem_scatter_reject", "tofmlem_permute_events", "tofmlem_reserve", "tofmlem_trim",
    "tofmlem_plan_events", "tofmlem_plan_info", "tofmlem_pass_timing", "tofmlem_split_regions_overlap",
    "tofmlem_em_correction_static", "tofmlem_static_error",
)


class Scanner(C.Structure):
    _fields_ = [("radius_mm", C.c_float), ("axial_length_mm", C.c_float)]


class Grid(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
                ("vx", C.c_float), ("vy", C.c_float), ("vz", C.c_float),
                ("ox", C.c_float), ("oy", C.c_float), ("oz", C.c_float)]

    @property
    def nvox(self) -> int:
        return self.nx * self.ny * self.nz


class Events(C.Structure):
    _fields_ = [(k, C.c_void_p) for k in EVENT_FIELDS]


class Stats(C.Structure):
    _fields_ = [("n_valid", C.c_uint64), ("n_skipped", C.c_uint64), ("visits", C.c_uint64),
                ("sum_image_sens", C.c_double), ("reductions", C.c_uint64), ("tile_events", C.c_uint64),
                ("tile_oob", C.c_uint64), ("tile_visits", C.c_uint64)]


class Plan(C.Structure):
    _fields_ = [("active", C.c_int32), ("sorted", C.c_int32), ("n_tile_items", C.c_uint32),
                ("n_direct_chunks", C.c_uint32), ("n_tile_events", C.c_uint64), ("n_direct_events", C.c_uint64),
                ("n_stragglers", C.c_uint64)]


class TofMlemError(RuntimeError):
    def __init__(self, code: int, text: str):
        super().__init__(f"libtofmlem error {code}: {text}")
        self.code = code


_lib = None


def lib():
    """Load (building if necessary) libtofmlem.so.  Fails loudly when it cannot be built or loaded."""
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        L.tofmlem_sigma_mm.restype = C.c_double
        L.tofmlem_last_error.restype = C.c_char_p
        L.tofmlem_version.restype = C.c_char_p
        L.tofmlem_num_bins.restype = C.c_uint32
        L.tofmlem_launch_count.restype = C.c_uint64
        L.tofmlem_static_error.restype = C.c_char_p
        for name in SYMBOLS:
            getattr(L, name)  # AttributeError if a declared symbol is missing
        _lib = L
    return _lib


def _ptr(t: Optional[torch.Tensor], dtype, device_type: str, numel: Optional[int] = None) -> Optional[int]:
    if t is None:
        return None
    if t.dtype != dtype or not t.is_contiguous() or t.device.type != device_type:
        raise TypeError(f"expected contiguous {dtype} tensor on {device_type}, got {t.dtype} on {t.device}")
    if numel is not None and t.numel() < numel:
        raise ValueError(f"tensor too small: {t.numel()} < {numel}")
    return t.data_ptr()


def _events(ev: Dict[str, torch.Tensor], n: int, device_type: str = "cuda") -> Events:
    e = Events()
    for k in EVENT_FIELDS:
        setattr(e, k, _ptr(ev.get(k), torch.float32, device_type, n))
    return e


class Context:
    """Owner of one tofmlem_ctx; methods carry the C names without the prefix."""

    def __init__(self, radius_mm: float, axial_length_mm: float, grid: Grid, tof_fwhm_ps: float,
                 stream: Optional[torch.cuda.Stream] = None):
        if not torch.cuda.is_available():
            raise RuntimeError("libtofmlem needs a CUDA device (B200, sm_100a); there is no CPU fallback")
        self._L = lib()
        self.grid = grid
        self.stream = stream if stream is not None else torch.cuda.current_stream()
        self._h = C.c_void_p()
        sc = Scanner(radius_mm, axial_length_mm)
        rc = self._L.tofmlem_create(C.byref(sc), C.byref(grid), C.c_float(tof_fwhm_ps),
                                    C.c_void_p(self.stream.cuda_stream), C.byref(self._h))
        if rc != TOFMLEM_OK:
            raise TofMlemError(rc, "tofmlem_create failed")

    # -- helpers
    def _check(self, rc: int):
        if rc != TOFMLEM_OK:
            raise TofMlemError(rc, self._L.tofmlem_last_error(self._h).decode())

    def close(self):
        if getattr(self, "_h", None) is not None and self._h:
            self._L.tofmlem_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def nvox(self) -> int:
        return self.grid.nvox

    # -- the ABI, one method per call
    def set_option(self, key: int, value: float):
        self._check(self._L.tofmlem_set_option(self._h, C.c_int(key), C.c_double(value)))

    def sigma_mm(self) -> float:
        return float(self._L.tofmlem_sigma_mm(self._h))

    def reserve(self, n_events: int):
        self._check(self._L.tofmlem_reserve(self._h, C.c_uint64(n_events)))

    def trim(self):
        self._check(self._L.tofmlem_trim(self._h))

    def sensitivity(self, lors: Dict[str, torch.Tensor], m: int, sens: torch.Tensor):
        e = _events({**lors, "dt": None}, m)
        self._check(self._L.tofmlem_sensitivity(self._h, C.byref(e), C.c_uint64(m),
                                                C.c_void_p(_ptr(sens, torch.float32, "cuda", self.nvox))))

    def forward(self, ev, n: int, image: torch.Tensor, fwd: torch.Tensor):
        e = _events(ev, n)
        self._check(self._L.tofmlem_forward(self._h, C.byref(e), C.c_uint64(n),
                                            C.c_void_p(_ptr(image, torch.float32, "cuda", self.nvox)),
                                            C.c_void_p(_ptr(fwd, torch.float32, "cuda", n))))

    def backproject(self, ev, n: int, values: Optional[torch.Tensor], out: torch.Tensor):
        e = _events(ev, n)
        self._check(self._L.tofmlem_backproject(self._h, C.byref(e), C.c_uint64(n),
                                                C.c_void_p(_ptr(values, torch.float32, "cuda", n)),
                                                C.c_void_p(_ptr(out, torch.float32, "cuda", self.nvox))))

    def em_correction(self, ev, n: int, image: torch.Tensor, corr: torch.Tensor):
        e = _events(ev, n)
        self._check(self._L.tofmlem_em_correction(self._h, C.byref(e), C.c_uint64(n),
                                                  C.c_void_p(_ptr(image, torch.float32, "cuda", self.nvox)),
                                                  C.c_void_p(_ptr(corr, torch.float32, "cuda", self.nvox))))

    def plan_events(self, ev, n: int) -> "Plan":
        self._check(self._L.tofmlem_plan_events(self._h, C.byref(_events(ev, n)), C.c_uint64(n)))
        return self.plan_info()

    def pass_timing(self):
        """(tile, direct, stragglers) kernel milliseconds of the last planned fused pass."""
        ms = (C.c_float * 3)()
        self._check(self._L.tofmlem_pass_timing(self._h, ms))
        return float(ms[0]), float(ms[1]), float(ms[2])

    def plan_info(self) -> "Plan":
        p = Plan()
        self._check(self._L.tofmlem_plan_info(self._h, C.byref(p)))
        return p

    def reset_stats(self):
        self._check(self._L.tofmlem_reset_stats(self._h))

    def update(self, image: torch.Tensor, corr: torch.Tensor, sens: torch.Tensor):
        self._check(self._L.tofmlem_update(self._h, C.c_void_p(_ptr(image, torch.float32, "cuda", self.nvox)),
                                           C.c_void_p(_ptr(corr, torch.float32, "cuda", self.nvox)),
                                           C.c_void_p(_ptr(sens, torch.float32, "cuda", self.nvox))))

    def iterate(self, ev, n: int, image: torch.Tensor, sens: torch.Tensor, iters: int):
        e = _events(ev, n)
        self._check(self._L.tofmlem_iterate(self._h, C.byref(e), C.c_uint64(n),
                                            C.c_void_p(_ptr(image, torch.float32, "cuda", self.nvox)),
                                            C.c_void_p(_ptr(sens, torch.float32, "cuda", self.nvox)), C.c_int(iters)))

    def iterate_host(self, h_ev, n: int, h_image: torch.Tensor, h_sens: torch.Tensor, iters: int):
        e = _events(h_ev, n, "cpu")
        self._check(self._L.tofmlem_iterate_host(self._h, C.byref(e), C.c_uint64(n),
                                                 C.c_void_p(_ptr(h_image, torch.float32, "cpu", self.nvox)),
                                                 C.c_void_p(_ptr(h_sens, torch.float32, "cpu", self.nvox)),
                                                 C.c_int(iters)))

    def num_bins(self) -> int:
        return int(self._L.tofmlem_num_bins(self._h))

    def bin_events(self, ev, n: int, key: torch.Tensor, perm: Optional[torch.Tensor],
                   bin_offsets: Optional[torch.Tensor]):
        e = _events(ev, n)
        # torch has no uint32 arithmetic everywhere: int32 tensors carry the same 32 bits
        self._check(self._L.tofmlem_bin_events(self._h, C.byref(e), C.c_uint64(n),
                                               C.c_void_p(_ptr(key, torch.int32, "cuda", n)),
                                               C.c_void_p(_ptr(perm, torch.int32, "cuda", n)),
                                               C.c_void_p(_ptr(bin_offsets, torch.int32, "cuda", self.num_bins() + 1))))

    def gather_events(self, ev, perm: torch.Tensor, n: int, out):
        a, b = _events(ev, n), _events(out, n)
        self._check(self._L.tofmlem_gather_events(self._h, C.byref(a), C.c_void_p(_ptr(perm, torch.int32, "cuda", n)),
                                                  C.c_uint64(n), C.byref(b)))

    def permute_events(self, ev, perm: torch.Tensor, n: int, out):
        """gather_events for a perm that is a permutation of 0..n-1 (bin_events / split_regions): packed fast path"""
        a, b = _events(ev, n), _events(out, n)
        self._check(self._L.tofmlem_permute_events(self._h, C.byref(a), C.c_void_p(_ptr(perm, torch.int32, "cuda", n)),
                                                   C.c_uint64(n), C.byref(b)))

    def region_zbounds(self, n_regions: int = 9) -> torch.Tensor:
        zb = torch.empty(n_regions + 1, dtype=torch.float32)
        self._check(self._L.tofmlem_region_zbounds(self._h, C.c_int(n_regions), C.c_void_p(zb.data_ptr())))
        return zb

    def split_regions(self, ev, n: int, n_regions: int, zbounds: Optional[torch.Tensor], region: torch.Tensor,
                      perm: Optional[torch.Tensor]) -> torch.Tensor:
        e = _events(ev, n)
        counts = torch.zeros(n_regions, dtype=torch.int64)
        zb = _ptr(zbounds, torch.float32, "cpu", n_regions + 1)
        self._check(self._L.tofmlem_split_regions(self._h, C.byref(e), C.c_uint64(n), C.c_int(n_regions),
                                                  C.c_void_p(zb), C.c_void_p(_ptr(region, torch.int32, "cuda", n)),
                                                  C.c_void_p(_ptr(perm, torch.int32, "cuda", n)),
                                                  C.c_void_p(counts.data_ptr())))
        return counts

    def split_regions_overlap(self, ev, n: int, n_regions: int, zbounds: Optional[torch.Tensor], span: torch.Tensor,
                              perm: Optional[torch.Tensor]) -> torch.Tensor:
        e = _events(ev, n)
        counts = torch.zeros(n_regions, dtype=torch.int64)
        zb = _ptr(zbounds, torch.float32, "cpu", n_regions + 1)
        cap = perm.numel() if perm is not None else 0
        self._check(self._L.tofmlem_split_regions_overlap(
            self._h, C.byref(e), C.c_uint64(n), C.c_int(n_regions), C.c_void_p(zb),
            C.c_void_p(_ptr(span, torch.int32, "cuda", n)), C.c_void_p(_ptr(perm, torch.int32, "cuda")),
            C.c_uint64(cap), C.c_void_p(counts.data_ptr())))
        return counts

    def region_grid(self, n_regions: int, zbounds: Optional[torch.Tensor], r: int):
        sub = Grid()
        z0, z1 = C.c_int32(), C.c_int32()
        zb = _ptr(zbounds, torch.float32, "cpu", n_regions + 1)
        self._check(self._L.tofmlem_region_grid(self._h, C.c_int(n_regions), C.c_void_p(zb), C.c_int(r),
                                                C.byref(sub), C.byref(z0), C.byref(z1)))
        return sub, z0.value, z1.value

    def reconstruct_regions(self, ev, n: int, n_regions: int, zbounds: Optional[torch.Tensor], image_out: torch.Tensor,
                            sens: torch.Tensor, iters: int):
        e = _events(ev, n)
        zb = _ptr(zbounds, torch.float32, "cpu", n_regions + 1)
        self._check(self._L.tofmlem_reconstruct_regions(
            self._h, C.byref(e), C.c_uint64(n), C.c_int(n_regions), C.c_void_p(zb),
            C.c_void_p(_ptr(image_out, torch.float32, "cuda", self.nvox)),
            C.c_void_p(_ptr(sens, torch.float32, "cuda", self.nvox)), C.c_int(iters)))

    # -- widened rows
    def median3(self, src: torch.Tensor, dst: torch.Tensor):
        self._check(self._L.tofmlem_median3(self._h, C.c_void_p(_ptr(src, torch.float32, "cuda", self.nvox)),
                                            C.c_void_p(_ptr(dst, torch.float32, "cuda", self.nvox))))

    def attenuation_weights(self, lors, n: int, mu: torch.Tensor, weight: torch.Tensor):
        e = _events({**lors, "dt": None}, n)
        self._check(self._L.tofmlem_attenuation_weights(self._h, C.byref(e), C.c_uint64(n),
                                                        C.c_void_p(_ptr(mu, torch.float32, "cuda", self.nvox)),
                                                        C.c_void_p(_ptr(weight, torch.float32, "cuda", n))))

    def em_correction_weighted(self, ev, n: int, weight: Optional[torch.Tensor], image: torch.Tensor,
                               corr: torch.Tensor):
        e = _events(ev, n)
        self._check(self._L.tofmlem_em_correction_weighted(
            self._h, C.byref(e), C.c_uint64(n), C.c_void_p(_ptr(weight, torch.float32, "cuda", n)),
            C.c_void_p(_ptr(image, torch.float32, "cuda", self.nvox)),
            C.c_void_p(_ptr(corr, torch.float32, "cuda", self.nvox))))

    def iterate_weighted(self, ev, n: int, weight: Optional[torch.Tensor], image: torch.Tensor, sens: torch.Tensor,
                         iters: int):
        e = _events(ev, n)
        self._check(self._L.tofmlem_iterate_weighted(
            self._h, C.byref(e), C.c_uint64(n), C.c_void_p(_ptr(weight, torch.float32, "cuda", n)),
            C.c_void_p(_ptr(image, torch.float32, "cuda", self.nvox)),
            C.c_void_p(_ptr(sens, torch.float32, "cuda", self.nvox)), C.c_int(iters)))

    def gather_f32(self, src: torch.Tensor, perm: torch.Tensor, n: int, dst: torch.Tensor):
        self._check(self._L.tofmlem_gather_f32(self._h, C.c_void_p(_ptr(src, torch.float32, "cuda", n)),
                                               C.c_void_p(_ptr(perm, torch.int32, "cuda", n)), C.c_uint64(n),
                                               C.c_void_p(_ptr(dst, torch.float32, "cuda", n))))

    def scatter_reject(self, ev, n: int, ellipsoids: torch.Tensor, half_width_mm: float, keep: torch.Tensor,
                       perm: Optional[torch.Tensor]) -> int:
        """ellipsoids: HOST float32 [n_ell, 6] = centre, reciprocal semi-axes; returns the number of kept events."""
        e = _events(ev, n)
        ell = _ptr(ellipsoids, torch.float32, "cpu")
        kept = C.c_uint64(0)
        self._check(self._L.tofmlem_scatter_reject(
            self._h, C.byref(e), C.c_uint64(n), C.c_void_p(ell), C.c_int(ellipsoids.numel() // 6),
            C.c_float(half_width_mm), C.c_void_p(_ptr(keep, torch.uint8, "cuda", n)),
            C.c_void_p(_ptr(perm, torch.int32, "cuda", n)), C.byref(kept)))
        return int(kept.value)

    def probe(self, kind: int, buf: torch.Tensor, n_ops: int) -> float:
        """elapsed ms of n_ops float32 REDs (kind 0,1) or gathers (2,3) against buf; see include/tofmlem.h"""
        ms = C.c_float()
        self._check(self._L.tofmlem_probe(self._h, C.c_int(kind), C.c_void_p(_ptr(buf, torch.float32, "cuda")),
                                          C.c_uint64(buf.numel()), C.c_uint64(n_ops), C.byref(ms)))
        return float(ms.value)

    def get_stats(self) -> Stats:
        st = Stats()
        self._check(self._L.tofmlem_get_stats(self._h, C.byref(st)))
        return st

    def launch_count(self) -> int:
        return int(self._L.tofmlem_launch_count(self._h))


def make_grid(nx: int, ny: int, nz: int, voxel_mm, origin: Optional[Sequence[float]] = None) -> Grid:
    vx, vy, vz = (voxel_mm,) * 3 if isinstance(voxel_mm, (int, float)) else voxel_mm
    if origin is None:
        origin = (-0.5 * nx * vx, -0.5 * ny * vy, -0.5 * nz * vz)
    return Grid(nx, ny, nz, vx, vy, vz, *origin)


def em_correction_static(grid: Grid, tof_fwhm_ps: float, ev, n: int, image: torch.Tensor, corr: torch.Tensor,
                         trunc_sigmas: float = 3.0, queues_per_sm: int = 0,
                         stream: Optional[torch.cuda.Stream] = None):
    """tofmlem_em_correction_static: the fused EM pass without a context and without any allocation (scratch in a static
    __device__ array); corr in grid order, accumulated into.  Enqueued on `stream` (default: torch's current stream)."""
    if not torch.cuda.is_available():
        raise RuntimeError("libtofmlem needs a CUDA device (B200, sm_100a); there is no CPU fallback")
    L = lib()
    e = _events(ev, n)
    s = (stream if stream is not None else torch.cuda.current_stream()).cuda_stream
    rc = L.tofmlem_em_correction_static(C.byref(grid), C.c_double(tof_fwhm_ps), C.c_double(trunc_sigmas), C.byref(e),
                                        C.c_uint64(n), C.c_void_p(_ptr(image, torch.float32, "cuda", grid.nvox)),
                                        C.c_void_p(_ptr(corr, torch.float32, "cuda", grid.nvox)),
                                        C.c_int(queues_per_sm), C.c_void_p(s))
    if rc != 0:
        raise TofMlemError(rc, L.tofmlem_static_error().decode())


def version() -> str:
    return lib().tofmlem_version().decode()
