"""Seeded synthetic list-mode PET inputs (stand-ins for the paper's GEANT4/NCAT data).

This module serves BOTH the CPU oracle's tests and the CUDA path's tests/bench, and therefore
holds none of the reconstruction method's arithmetic: it only simulates *data* (emission points,
isotropic back-to-back photons hitting a cylindrical detector, a noisy time difference,
scatter-like random LORs, detector-pair LORs for the sensitivity image).  Neither `oracle/` nor
`paper_1706_07075_b200/` is imported here, and neither of them imports this module.

Workload shapes follow BASELINE.json `configs` (cfg-1 Tiny, cfg-2 Mid, cfg-3 Full body) which in
turn take their sizes from the paper: 146 M detected coincidences, ~33 % scatter fraction, 300 ps
FWHM TOF, long axial FOV with highly inclined LORs.

Randomness is a counter-based generator (a splitmix64-style hash of (seed, event index, attempt,
draw)), written with torch int64 ops so that it runs unchanged on CPU and on CUDA tensors and
any sub-range [start, start+n) of a data set can be produced on its own.  The uniform bit streams
are identical on every device; the transcendental functions applied afterwards (sin, cos, sqrt)
may differ in the last ulp between devices, so a test always feeds ONE generated array set to both
the oracle and the CUDA path.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import Dict, List, Optional, Sequence, Tuple

import torch

C_MM_PER_PS = 0.299792458  # speed of light, mm/ps
FWHM_TO_SIGMA = 1.0 / (2.0 * math.sqrt(2.0 * math.log(2.0)))

# --------------------------------------------------------------------------------------------
# counter-based RNG
# --------------------------------------------------------------------------------------------
_M64 = (1 << 64) - 1


def _s64(x: int) -> int:
    """Wrap a python int to the signed 64-bit value with the same bit pattern."""
    x &= _M64
    return x - (1 << 64) if x >= (1 << 63) else x


_GOLD = _s64(0x9E3779B97F4A7C15)
_MIX1 = _s64(0xBF58476D1CE4E5B9)
_MIX2 = _s64(0x94D049BB133111EB)
_K_ATT = _s64(0xD1B54A32D192ED03)
_K_DRAW = _s64(0x8CB92BA72F3D8DD7)


def _lsr(z: torch.Tensor, k: int) -> torch.Tensor:
    return (z >> k) & ((1 << (64 - k)) - 1)


def _mix(z: torch.Tensor) -> torch.Tensor:
    z = z + _GOLD
    z = (z ^ _lsr(z, 30)) * _MIX1
    z = (z ^ _lsr(z, 27)) * _MIX2
    return z ^ _lsr(z, 31)


def u01(seed: int, idx: torch.Tensor, attempt: int, draw: int) -> torch.Tensor:
    """Uniform [0,1) float64, a pure function of (seed, idx, attempt, draw)."""
    z = _mix(idx + _s64(seed * 0x2545F4914F6CDD1D))
    z = _mix(z + _s64(attempt * 0xD1B54A32D192ED03) + _s64(draw * 0x8CB92BA72F3D8DD7))
    return _lsr(z, 11).to(torch.float64) * (1.0 / 9007199254740992.0)


def normal(seed: int, idx: torch.Tensor, attempt: int, draw: int) -> torch.Tensor:
    """Standard normal via Box-Muller; consumes draws `draw` and `draw+1`."""
    a = u01(seed, idx, attempt, draw)
    b = u01(seed, idx, attempt, draw + 1)
    return torch.sqrt(-2.0 * torch.log(1.0 - a)) * torch.cos(2.0 * math.pi * b)


# --------------------------------------------------------------------------------------------
# phantoms: piecewise-constant activity, painter's algorithm (later shapes override earlier ones)
# --------------------------------------------------------------------------------------------
@dataclass(frozen=True)
class Shape:
    kind: str  # "ellipsoid" | "zcylinder"
    centre: Tuple[float, float, float]
    semi: Tuple[float, float, float]  # ellipsoid semi-axes; zcylinder: (r, r, half_length)
    activity: float

    def contains(self, p: torch.Tensor) -> torch.Tensor:
        x = (p[:, 0] - self.centre[0]) / self.semi[0]
        y = (p[:, 1] - self.centre[1]) / self.semi[1]
        z = (p[:, 2] - self.centre[2]) / self.semi[2]
        if self.kind == "ellipsoid":
            return x * x + y * y + z * z <= 1.0
        return (x * x + y * y <= 1.0) & (z.abs() <= 1.0)

    def volume(self) -> float:
        a, b, c = self.semi
        if self.kind == "ellipsoid":
            return 4.0 / 3.0 * math.pi * a * b * c
        return math.pi * a * b * 2.0 * c

    def sample_inside(self, seed: int, idx: torch.Tensor, attempt: int, draw: int) -> torch.Tensor:
        """Uniform point inside the shape; consumes 3 draws."""
        u = u01(seed, idx, attempt, draw)
        v = u01(seed, idx, attempt, draw + 1)
        w = u01(seed, idx, attempt, draw + 2)
        if self.kind == "ellipsoid":
            r = u ** (1.0 / 3.0)
            ct = 2.0 * v - 1.0
            st = torch.sqrt(torch.clamp(1.0 - ct * ct, min=0.0))
            ph = 2.0 * math.pi * w
            q = torch.stack([r * st * torch.cos(ph), r * st * torch.sin(ph), r * ct], dim=1)
        else:
            r = torch.sqrt(u)
            ph = 2.0 * math.pi * v
            q = torch.stack([r * torch.cos(ph), r * torch.sin(ph), 2.0 * w - 1.0], dim=1)
        semi = torch.tensor(self.semi, dtype=torch.float64, device=idx.device)
        cen = torch.tensor(self.centre, dtype=torch.float64, device=idx.device)
        return q * semi + cen


@dataclass(frozen=True)
class Phantom:
    parts: Tuple[Shape, ...]  # pairwise DISJOINT top-level body parts (proposal distribution)
    inner: Tuple[Shape, ...]  # organs/lesions painted over the parts, in order

    def activity(self, p: torch.Tensor) -> torch.Tensor:
        a = torch.zeros(p.shape[0], dtype=torch.float64, device=p.device)
        for s in self.parts + self.inner:
            a = torch.where(s.contains(p), torch.full_like(a, s.activity), a)
        return a

    def amax(self) -> float:
        return max(s.activity for s in self.parts + self.inner)


@dataclass(frozen=True)
class Config:
    name: str
    nx: int
    ny: int
    nz: int
    voxel_mm: float
    radius_mm: float
    axial_mm: float
    phantom: Phantom
    n_events: int
    scatter_fraction: float
    tof_fwhm_ps: float
    iters: int
    sens_lors: int
    seed: int

    @property
    def origin(self) -> Tuple[float, float, float]:
        v = self.voxel_mm
        return (-0.5 * self.nx * v, -0.5 * self.ny * v, -0.5 * self.nz * v)

    @property
    def nvox(self) -> int:
        return self.nx * self.ny * self.nz


def _sph(c, r, act):
    return Shape("ellipsoid", tuple(c), (r, r, r), act)


def _ell(c, s, act):
    return Shape("ellipsoid", tuple(c), tuple(s), act)


_TINY_PHANTOM = Phantom(
    parts=(Shape("zcylinder", (0.0, 0.0, 0.0), (50.0, 50.0, 64.0), 1.0),),
    inner=(_sph((25.0, 0.0, 0.0), 5.0, 4.0), _sph((-25.0, 0.0, 0.0), 5.0, 4.0)),
)

_MID_PHANTOM = Phantom(
    parts=(_ell((0.0, 0.0, 0.0), (150.0, 100.0, 120.0), 1.0),),
    inner=(
        _ell((55.0, 10.0, 20.0), (45.0, 40.0, 50.0), 2.0),
        _ell((-50.0, 20.0, 40.0), (30.0, 30.0, 35.0), 3.0),
        _ell((-40.0, -30.0, -50.0), (40.0, 30.0, 40.0), 0.5),
        _sph((0.0, 60.0, 0.0), 4.0, 4.0),
        _sph((20.0, -55.0, 70.0), 4.5, 4.0),
        _sph((100.0, 0.0, -30.0), 5.0, 4.0),
        _sph((-95.0, 10.0, -10.0), 6.0, 4.0),
    ),
)

# Full-body table of ellipsoids: written by hand for this build (no anatomical atlas is copied).
# z runs feet (-) to head (+); the parts are pairwise disjoint (checked by tests).
_FULL_PHANTOM = Phantom(
    parts=(
        _ell((0.0, 0.0, 760.0), (80.0, 95.0, 105.0), 1.0),  # head
        _ell((0.0, 0.0, 350.0), (170.0, 110.0, 290.0), 1.0),  # torso
        _ell((215.0, 0.0, 330.0), (38.0, 40.0, 300.0), 1.0),  # arms
        _ell((-215.0, 0.0, 330.0), (38.0, 40.0, 300.0), 1.0),
        _ell((85.0, 0.0, -330.0), (72.0, 75.0, 385.0), 1.0),  # legs
        _ell((-85.0, 0.0, -330.0), (72.0, 75.0, 385.0), 1.0),
        _ell((85.0, 40.0, -790.0), (45.0, 90.0, 48.0), 1.0),  # feet
        _ell((-85.0, 40.0, -790.0), (45.0, 90.0, 48.0), 1.0),
    ),
    inner=(
        _ell((0.0, 0.0, 775.0), (62.0, 78.0, 70.0), 3.0),  # brain
        _ell((75.0, 0.0, 500.0), (50.0, 60.0, 90.0), 0.5),  # lungs
        _ell((-75.0, 0.0, 500.0), (50.0, 60.0, 90.0), 0.5),
        _ell((-15.0, 25.0, 470.0), (40.0, 35.0, 45.0), 4.0),  # heart
        _ell((70.0, 5.0, 330.0), (75.0, 60.0, 60.0), 2.0),  # liver
        _ell((-80.0, -30.0, 300.0), (25.0, 20.0, 45.0), 3.0),  # kidneys
        _ell((60.0, -45.0, 250.0), (25.0, 20.0, 45.0), 3.0),
        _ell((0.0, 15.0, 110.0), (35.0, 30.0, 30.0), 4.0),  # bladder
        _sph((0.0, 0.0, 610.0), 5.0, 4.0),  # 10 mm lesions at 4:1
        _sph((130.0, 0.0, 450.0), 5.0, 4.0),
        _sph((-215.0, 0.0, 400.0), 5.0, 4.0),
        _sph((60.0, 0.0, 95.0), 5.0, 4.0),
        _sph((85.0, 0.0, -330.0), 5.0, 4.0),
        _sph((-85.0, 60.0, -790.0), 5.0, 4.0),
    ),
)

TINY = Config("tiny", 32, 32, 32, 4.0, 200.0, 128.0, _TINY_PHANTOM, 200_000, 0.0, 300.0, 2, 1_000_000, 1)
MID = Config("mid", 128, 128, 128, 2.0, 300.0, 256.0, _MID_PHANTOM, 10_000_000, 0.30, 300.0, 5, 20_000_000, 2)
FULL = Config("full", 160, 160, 640, 3.75, 400.0, 2400.0, _FULL_PHANTOM, 146_000_000, 0.33, 300.0, 5, 100_000_000, 3)
CONFIGS: Dict[str, Config] = {c.name: c for c in (TINY, MID, FULL)}


def sweep_config(n_events: int, tof_fwhm_ps: float) -> Config:
    """cfg-5: full-body geometry/phantom, 20 % scatter, 3 iterations, seed 5 (tof<=0: non-TOF)."""
    return Config(f"sweep-{n_events}-{tof_fwhm_ps:g}", 160, 160, 640, 3.75, 400.0, 2400.0, _FULL_PHANTOM,
                  n_events, 0.20, tof_fwhm_ps, 3, 100_000_000, 5)


# --------------------------------------------------------------------------------------------
# event generation
# --------------------------------------------------------------------------------------------
_D_TYPE, _D_PART, _D_POS, _D_ACC, _D_DIR, _D_NOISE, _D_SC = 0, 1, 2, 5, 6, 8, 10  # draw slots
_MAX_ATTEMPTS = 4096


def _cyl_point(seed, idx, attempt, draw, radius, axial):
    ph = 2.0 * math.pi * u01(seed, idx, attempt, draw)
    z = (u01(seed, idx, attempt, draw + 1) - 0.5) * axial
    return torch.stack([radius * torch.cos(ph), radius * torch.sin(ph), z], dim=1)


def _true_attempt(cfg: Config, idx: torch.Tensor, attempt: int):
    """One attempt at a true coincidence for every index in idx.
    Returns (ok, p1, p2, d1_minus_d2_mm)."""
    ph = cfg.phantom
    seed = cfg.seed
    # proposal: pick a top-level part with probability ~ volume, uniform point inside it
    vols = torch.tensor([s.volume() for s in ph.parts], dtype=torch.float64, device=idx.device)
    cdf = torch.cumsum(vols, 0) / vols.sum()
    upart = u01(seed, idx, attempt, _D_PART)
    part = torch.bucketize(upart, cdf[:-1].contiguous(), right=True)
    e = torch.zeros((idx.numel(), 3), dtype=torch.float64, device=idx.device)
    for k, s in enumerate(ph.parts):
        sel = part == k
        if bool(sel.any()):
            e[sel] = s.sample_inside(seed, idx[sel], attempt, _D_POS)
    ok = u01(seed, idx, attempt, _D_ACC) * ph.amax() < ph.activity(e)
    # isotropic direction
    ct = 2.0 * u01(seed, idx, attempt, _D_DIR) - 1.0
    st = torch.sqrt(torch.clamp(1.0 - ct * ct, min=0.0))
    az = 2.0 * math.pi * u01(seed, idx, attempt, _D_DIR + 1)
    d = torch.stack([st * torch.cos(az), st * torch.sin(az), ct], dim=1)
    # intersect with the detector cylinder x^2+y^2=R^2
    a = d[:, 0] ** 2 + d[:, 1] ** 2
    b = e[:, 0] * d[:, 0] + e[:, 1] * d[:, 1]
    c = e[:, 0] ** 2 + e[:, 1] ** 2 - cfg.radius_mm ** 2
    disc = b * b - a * c
    ok &= (a > 1e-12) & (disc > 0.0)
    sq = torch.sqrt(torch.clamp(disc, min=0.0))
    a_safe = torch.where(a > 1e-12, a, torch.ones_like(a))
    t_plus = (-b + sq) / a_safe  # > 0 for a point inside the cylinder
    t_minus = (-b - sq) / a_safe  # < 0
    p1 = e + t_minus[:, None] * d
    p2 = e + t_plus[:, None] * d
    half = 0.5 * cfg.axial_mm
    ok &= (p1[:, 2].abs() <= half) & (p2[:, 2].abs() <= half)
    return ok, p1, p2, (-t_minus) - t_plus  # d1 - d2


def make_events(cfg: Config, n: Optional[int] = None, start: int = 0, device="cpu") -> Dict[str, torch.Tensor]:
    """Events [start, start+n) of the config's seeded list-mode set as SoA float32 tensors
    x1,y1,z1,x2,y2,z2 (mm) and dt (ps).  dt = (d1-d2)/c + N(0, FWHM/2.35482): positive when the
    annihilation is nearer endpoint 2."""
    n = cfg.n_events if n is None else n
    dev = torch.device(device)
    idx = torch.arange(start, start + n, dtype=torch.int64, device=dev)
    seed = cfg.seed
    p1 = torch.zeros((n, 3), dtype=torch.float64, device=dev)
    p2 = torch.zeros((n, 3), dtype=torch.float64, device=dev)
    dd = torch.zeros(n, dtype=torch.float64, device=dev)
    is_sc = u01(seed, idx, 0, _D_TYPE) < cfg.scatter_fraction
    # scatter-like: endpoints independent uniform on the detector wall, emission uniform on the LOR
    if bool(is_sc.any()):
        si = idx[is_sc]
        a = _cyl_point(seed, si, 0, _D_SC, cfg.radius_mm, cfg.axial_mm)
        b = _cyl_point(seed, si, 0, _D_SC + 2, cfg.radius_mm, cfg.axial_mm)
        ll = torch.linalg.vector_norm(b - a, dim=1)
        s = u01(seed, si, 0, _D_SC + 4) * ll
        p1[is_sc], p2[is_sc], dd[is_sc] = a, b, 2.0 * s - ll
    # trues: rejection against activity and axial acceptance, redrawing the whole event
    pending = torch.nonzero(~is_sc).flatten()
    attempt = 1
    while pending.numel() > 0:
        if attempt > _MAX_ATTEMPTS:
            raise RuntimeError("synthetic generator: acceptance too low")
        ok, a, b, d12 = _true_attempt(cfg, idx[pending], attempt)
        acc = pending[ok]
        p1[acc], p2[acc], dd[acc] = a[ok], b[ok], d12[ok]
        pending = pending[~ok]
        attempt += 1
    sigma_t = cfg.tof_fwhm_ps * FWHM_TO_SIGMA if cfg.tof_fwhm_ps > 0 else 300.0 * FWHM_TO_SIGMA
    dt = dd / C_MM_PER_PS + sigma_t * normal(seed, idx, 0, _D_NOISE)
    f32 = torch.float32
    return {
        "x1": p1[:, 0].to(f32).contiguous(), "y1": p1[:, 1].to(f32).contiguous(), "z1": p1[:, 2].to(f32).contiguous(),
        "x2": p2[:, 0].to(f32).contiguous(), "y2": p2[:, 1].to(f32).contiguous(), "z2": p2[:, 2].to(f32).contiguous(),
        "dt": dt.to(f32).contiguous(),
    }


def event_kinds(cfg: Config, n: Optional[int] = None, start: int = 0, device="cpu") -> torch.Tensor:
    """uint8[n]: 1 for the scatter-like events of make_events(cfg, n, start), 0 for the true coincidences
    (the simulation's ground truth; used to check the TOF scatter rejection statistically)."""
    n = cfg.n_events if n is None else n
    idx = torch.arange(start, start + n, dtype=torch.int64, device=torch.device(device))
    return (u01(cfg.seed, idx, 0, _D_TYPE) < cfg.scatter_fraction).to(torch.uint8)


def body_outline(cfg: Config) -> List[Tuple[Tuple[float, float, float], Tuple[float, float, float]]]:
    """The phantom's top-level body parts as (centre, semi-axes) ellipsoids: the stand-in for the NCAT / CT body
    outline of the paper's TOF scatter rejection.  Only ellipsoid parts qualify."""
    assert all(s.kind == "ellipsoid" for s in cfg.phantom.parts), "outline needs ellipsoid body parts"
    return [(s.centre, s.semi) for s in cfg.phantom.parts]


MU_WATER_511KEV = 0.0096  # 1/mm, soft tissue at 511 keV
MU_LUNG_511KEV = 0.0029


def rasterize_mu_map(cfg: Config, device="cpu") -> torch.Tensor:
    """Synthetic attenuation map (1/mm) at voxel centres, float32 [nz, ny, nx]: water inside the body parts, a
    lower value inside inner shapes of activity < 1 (lungs).  Stand-in for the NCAT mu-map."""
    act = rasterize_phantom(cfg, device)
    parts_only = Phantom(cfg.phantom.parts, ())
    body = rasterize_phantom(Config(cfg.name, cfg.nx, cfg.ny, cfg.nz, cfg.voxel_mm, cfg.radius_mm, cfg.axial_mm,
                                    parts_only, 0, 0.0, cfg.tof_fwhm_ps, 0, 0, cfg.seed), device) > 0
    mu = torch.where(body, torch.full_like(act, MU_WATER_511KEV), torch.zeros_like(act))
    return torch.where(body & (act < 1.0) & (act > 0.0), torch.full_like(act, MU_LUNG_511KEV), mu)


def make_events_chunked(cfg: Config, n: Optional[int] = None, start: int = 0, device="cpu",
                        chunk: int = 4_000_000, out_device=None) -> Dict[str, torch.Tensor]:
    """make_events in chunks (bounded scratch memory); identical values to the unchunked call."""
    n = cfg.n_events if n is None else n
    out_device = device if out_device is None else out_device
    out = {k: torch.empty(n, dtype=torch.float32, device=out_device) for k in EVENT_FIELDS}
    for s in range(0, n, chunk):
        m = min(chunk, n - s)
        part = make_events(cfg, m, start + s, device)
        for k in EVENT_FIELDS:
            out[k][s:s + m] = part[k]
    return out


EVENT_FIELDS = ("x1", "y1", "z1", "x2", "y2", "z2", "dt")
LOR_FIELDS = ("x1", "y1", "z1", "x2", "y2", "z2")


def make_sens_lors(cfg: Config, m: Optional[int] = None, start: int = 0, device="cpu") -> Dict[str, torch.Tensor]:
    """Detector-pair LORs for the Monte-Carlo sensitivity image: both endpoints independent and
    uniform on the detector cylinder (phi in [0,2pi), z in [-L/2, L/2])."""
    m = cfg.sens_lors if m is None else m
    dev = torch.device(device)
    idx = torch.arange(start, start + m, dtype=torch.int64, device=dev)
    seed = cfg.seed + 7919
    a = _cyl_point(seed, idx, 0, 0, cfg.radius_mm, cfg.axial_mm)
    b = _cyl_point(seed, idx, 0, 2, cfg.radius_mm, cfg.axial_mm)
    f32 = torch.float32
    return {
        "x1": a[:, 0].to(f32).contiguous(), "y1": a[:, 1].to(f32).contiguous(), "z1": a[:, 2].to(f32).contiguous(),
        "x2": b[:, 0].to(f32).contiguous(), "y2": b[:, 1].to(f32).contiguous(), "z2": b[:, 2].to(f32).contiguous(),
    }


def make_sens_lors_chunked(cfg: Config, m: Optional[int] = None, start: int = 0, device="cpu",
                           chunk: int = 8_000_000) -> Dict[str, torch.Tensor]:
    m = cfg.sens_lors if m is None else m
    out = {k: torch.empty(m, dtype=torch.float32, device=device) for k in LOR_FIELDS}
    for s in range(0, m, chunk):
        k = min(chunk, m - s)
        part = make_sens_lors(cfg, k, start + s, device)
        for f in LOR_FIELDS:
            out[f][s:s + k] = part[f]
    return out


def rasterize_phantom(cfg: Config, device="cpu") -> torch.Tensor:
    """Activity at voxel centres, float32 [nz, ny, nx] (a sanity image, not an oracle input)."""
    v = cfg.voxel_mm
    ox, oy, oz = cfg.origin
    dev = torch.device(device)
    xs = ox + (torch.arange(cfg.nx, dtype=torch.float64, device=dev) + 0.5) * v
    ys = oy + (torch.arange(cfg.ny, dtype=torch.float64, device=dev) + 0.5) * v
    out = torch.empty((cfg.nz, cfg.ny, cfg.nx), dtype=torch.float32, device=dev)
    yy, xx = torch.meshgrid(ys, xs, indexing="ij")
    for iz in range(cfg.nz):
        zz = torch.full_like(xx, oz + (iz + 0.5) * v)
        p = torch.stack([xx.flatten(), yy.flatten(), zz.flatten()], dim=1)
        out[iz] = cfg.phantom.activity(p).reshape(cfg.ny, cfg.nx).to(torch.float32)
    return out


def random_image(shape: Sequence[int], seed: int, device="cpu") -> torch.Tensor:
    """Positive random float32 image (uniform in [0.5, 1.5)) for projector parity tests."""
    n = 1
    for s in shape:
        n *= s
    idx = torch.arange(n, dtype=torch.int64, device=device)
    return (0.5 + u01(seed, idx, 0, 0)).to(torch.float32).reshape(tuple(shape))
