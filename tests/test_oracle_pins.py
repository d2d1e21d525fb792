"""Pins of the fp64 oracle against what the paper and the mathematics fix (no GPU, no CUDA path).

Each test is built so that a plausible mistake in oracle/tofmlem_oracle.c (dropped term, wrong sign
or index, transposed axis) fails at least one of them.  Nothing here re-types the oracle's own
crossing/sort algorithm: expected values come from the paper's printed numbers
(tests/golden/paper_values.txt), closed forms, construction of the inputs, or brute-force stepping.
"""
import math

import numpy as np
import pytest

import oracle

ERF3 = math.erf(3.0 / math.sqrt(2.0))  # mass of a Gaussian inside +-3 sigma = 0.9973002...


def gauss(t, s):
    return np.exp(-0.5 * (np.asarray(t) / s) ** 2) / (s * math.sqrt(2.0 * math.pi))


def dt_for_centre(L, s_c):
    """time difference (ps) that puts the kernel centre at arc length s_c from endpoint 1"""
    return 2.0 * (s_c - 0.5 * L) / oracle.C_MM_PER_PS


# ---------------------------------------------------------------- P1
def test_p1_sigma_from_fwhm(golden):
    """PAPER.md:111 prints sigma = 19.11 mm for 300 ps FWHM: pins c*FWHM/(2*2.3548), factor 1/2 included."""
    fwhm = golden["tof_fwhm_ps"][0]
    assert abs(oracle.sigma_mm(fwhm, 0.3) - golden["sigma_mm_at_300ps"][0]) < 0.005
    assert abs(oracle.sigma_mm(fwhm) - 19.0965) < 1e-4  # exact c
    # without the factor 1/2 the value would be 38.2, with FWHM taken as sigma 45.0
    assert abs(oracle.sigma_mm(100.0) * 3 - oracle.sigma_mm(300.0)) < 1e-12


# ---------------------------------------------------------------- P2
def _random_face_point(rng, g):
    lo = np.array([g.ox, g.oy, g.oz])
    hi = lo + np.array([g.nx * g.vx, g.ny * g.vy, g.nz * g.vz])
    p = lo + rng.random(3) * (hi - lo)
    a = rng.integers(3)
    side = rng.integers(2)
    p[a] = hi[a] if side else lo[a]
    return p, (a, side)


def test_p2_uniform_box_line_integral_is_chord():
    """Non-TOF: sum of chord lengths through an all-ones box equals the entry-exit distance, which
    is known BY CONSTRUCTION (the LOR is drawn through two chosen points on the box faces)."""
    rng = np.random.default_rng(11)
    g = oracle.make_grid(13, 9, 17, (2.0, 3.0, 1.5), origin=(-11.0, -20.0, 4.0))
    ones = np.ones(g.nvox)
    P1, P2, chord = [], [], []
    while len(chord) < 400:
        A, fa = _random_face_point(rng, g)
        B, fb = _random_face_point(rng, g)
        if fa == fb:
            continue
        d = B - A
        P1.append(A - rng.uniform(0.1, 3.0) * d)
        P2.append(B + rng.uniform(0.1, 3.0) * d)
        chord.append(np.linalg.norm(d))
    P1, P2 = np.array(P1), np.array(P2)
    ev = {"x1": P1[:, 0], "y1": P1[:, 1], "z1": P1[:, 2], "x2": P2[:, 0], "y2": P2[:, 1], "z2": P2[:, 2]}
    # the oracle takes float32 events: compare against the chord of the float32-rounded LOR
    fwd = oracle.forward(g, 0.0, ev, ones)
    chord = np.array(chord)
    assert np.max(np.abs(fwd - chord) / chord) < 2e-5  # float32 rounding of the endpoints only
    # exact in fp64 through the single-LOR entry (no float32 rounding): rel <= 1e-12
    for k in range(50):
        idx, w = oracle.lor_weights(g, 0.0, P1[k], P2[k])
        assert abs(w.sum() - chord[k]) / chord[k] < 1e-12
        assert len(set(idx.tolist())) == len(idx)  # every voxel at most once


# ---------------------------------------------------------------- P3
def test_p3_axis_aligned_rays_and_index_layout():
    """Rays through voxel centres along each axis: every chord equals the voxel size along that axis
    and the voxel indices are the row (iz*ny+iy)*nx+ix -- pins the layout and the axis order."""
    g = oracle.make_grid(5, 7, 9, (2.0, 3.0, 1.5))
    n = (g.nx, g.ny, g.nz)
    v = (g.vx, g.vy, g.vz)
    o = (g.ox, g.oy, g.oz)
    fixed = (3, 4, 6)
    for a in range(3):
        c = [o[k] + (fixed[k] + 0.5) * v[k] for k in range(3)]
        p1, p2 = list(c), list(c)
        p1[a], p2[a] = o[a] - 10.0, o[a] + n[a] * v[a] + 10.0
        idx, w = oracle.lor_weights(g, 0.0, p1, p2)
        ijk = [np.full(n[a], fixed[k]) for k in range(3)]
        ijk[a] = np.arange(n[a])
        want = (ijk[2] * g.ny + ijk[1]) * g.nx + ijk[0]
        assert idx.tolist() == want.tolist()
        assert np.allclose(w, v[a], rtol=0, atol=1e-12)
        # reversed direction visits the same voxels in reverse order
        idx_r, w_r = oracle.lor_weights(g, 0.0, p2, p1)
        assert idx_r.tolist() == want[::-1].tolist()


def test_p3_cube_diagonal_and_single_voxel():
    n, v = 6, 2.5
    g = oracle.make_grid(n, n, n, v)
    lo, hi = g.ox - 5.0, g.ox + n * v + 5.0
    idx, w = oracle.lor_weights(g, 0.0, (lo, lo, lo), (hi, hi, hi))
    big = w > 1e-9  # corner crossings may leave slivers of ~1e-15 in neighbours
    assert big.sum() == n
    assert np.allclose(w[big], v * math.sqrt(3.0), atol=1e-9)
    assert idx[big].tolist() == [(k * n + k) * n + k for k in range(n)]
    # one-voxel grid: the single weight is the box chord; here a face-to-face oblique line
    g1 = oracle.make_grid(1, 1, 1, (4.0, 6.0, 8.0))
    A, B = np.array([-2.0, 1.0, -3.0]), np.array([2.0, -2.5, 0.5])  # on the x=-2 and x=+2 faces
    idx, w = oracle.lor_weights(g1, 0.0, A - 2 * (B - A), B + 3 * (B - A))
    assert idx.tolist() == [0] and abs(w[0] - np.linalg.norm(B - A)) < 1e-12


# ---------------------------------------------------------------- P4
@pytest.mark.parametrize("v,fwhm", [(3.75, 300.0), (2.0, 300.0), (4.0, 300.0), (3.75, 600.0)])
def test_p4_tof_weights_sum_to_truncated_gaussian_mass(v, fwhm):
    """Window fully inside the grid: sum_j a_ej = erf(3/sqrt 2) within the midpoint-rule error."""
    rng = np.random.default_rng(5)
    sig = oracle.sigma_mm(fwhm)
    n = int(2 * (3 * sig + 40) / v) + 2
    g = oracle.make_grid(n, n, n, v)
    worst = 0.0
    for _ in range(200):
        d = rng.normal(size=3)
        d /= np.linalg.norm(d)
        c = rng.uniform(-30, 30, 3)  # kernel centre well inside
        p1, p2 = c - d * rng.uniform(300, 500), c + d * rng.uniform(300, 500)
        L = np.linalg.norm(p2 - p1)
        dt = dt_for_centre(L, np.linalg.norm(c - p1))
        _, w = oracle.lor_weights(g, sig, p1, p2, dt)
        worst = max(worst, abs(w.sum() - ERF3))
    assert worst < 0.04 * (v / sig) ** 2
    assert worst > 0  # not identically the closed form: it IS a midpoint rule


# ---------------------------------------------------------------- P5
def test_p5_tof_weights_closed_form_axis_aligned():
    """x-aligned ray through voxel centres, kernel centre at a voxel centre: a_k = v g(k v) for the
    interior voxels, the end segments are clipped at +-3 sigma and weighted at their clipped midpoint
    (R7).  Also pins the sign of dt (R22: dt>0 => nearer endpoint 2) and the c/2 factor."""
    v, sig = 2.0, 4.8
    g = oracle.make_grid(64, 4, 6, v)
    yc, zc = g.oy + 2.5 * v, g.oz + 3.5 * v
    p1, p2 = (-100.0, yc, zc), (100.0, yc, zc)
    ic = 40  # centre voxel, x centre = -64 + 40.5*2 = 17 -> s_c = 117
    s_c = (g.ox + (ic + 0.5) * v) - p1[0]
    dt = dt_for_centre(200.0, s_c)
    assert dt > 0  # centre nearer p2
    idx, w = oracle.lor_weights(g, sig, p1, p2, dt)
    hw = 3 * sig  # 14.4: full voxels out to |t| <= 13, then a clipped piece [13, 14.4]
    want_idx, want_w = [], []
    want_idx.append(ic - 7), want_w.append(1.4 * gauss(13.7, sig))
    for k in range(-6, 7):
        want_idx.append(ic + k), want_w.append(v * gauss(k * v, sig))
    want_idx.append(ic + 7), want_w.append(1.4 * gauss(13.7, sig))
    base = (3 * g.ny + 2) * g.nx
    assert idx.tolist() == [base + i for i in want_idx]
    assert np.allclose(w, np.array(want_w), rtol=1e-12, atol=0)
    # opposite sign of dt mirrors the centre to the other side of the LOR midpoint
    idx_m, _ = oracle.lor_weights(g, sig, p1, p2, -dt)
    assert idx_m[len(idx_m) // 2] == base + (63 - ic)


def test_p5_window_clipped_by_grid_and_lor_ends():
    """R8: the window is clipped to the grid box and to [0, L] without renormalisation."""
    v, sig = 2.0, 5.0
    g = oracle.make_grid(8, 3, 3, v)  # x in [-8, 8]
    yc, zc = g.oy + 1.5 * v, g.oz + 1.5 * v
    p1, p2 = (-50.0, yc, zc), (50.0, yc, zc)
    s_c = 50.0 + 7.0  # centre of last voxel (x=7): window [42,72] -> clipped by the grid at s=58
    idx, w = oracle.lor_weights(g, sig, p1, p2, dt_for_centre(100.0, s_c))
    assert idx.tolist() == [(1 * 3 + 1) * 8 + i for i in range(0, 8)]  # 15 mm back covers x>=-8: all 8 voxels
    assert np.allclose(w, [v * gauss((i - 7) * v, sig) for i in range(8)], rtol=1e-12)
    # LOR that ends inside the grid: nothing beyond s = L
    idx, w = oracle.lor_weights(g, sig, (-50.0, yc, zc), (1.0, yc, zc), dt_for_centre(51.0, 51.0))
    assert idx[-1] == (1 * 3 + 1) * 8 + 4 and abs(w[-1] - 1.0 * gauss(-0.5, sig)) < 1e-15


# ---------------------------------------------------------------- P6
def test_p6_infinite_sigma_reduces_to_non_tof():
    rng = np.random.default_rng(3)
    g = oracle.make_grid(12, 10, 14, (2.0, 2.5, 3.0))
    sig = 1e9
    for _ in range(50):
        p1 = rng.uniform(-60, 60, 3)
        p2 = rng.uniform(-60, 60, 3)
        i0, w0 = oracle.lor_weights(g, 0.0, p1, p2)
        i1, w1 = oracle.lor_weights(g, sig, p1, p2, rng.uniform(-100, 100))
        assert i0.tolist() == i1.tolist()
        assert np.allclose(w1 * sig * math.sqrt(2 * math.pi), w0, rtol=1e-12)


# ---------------------------------------------------------------- helpers for MLEM pins
def _small_problem(seed=7, n_ev=4000, n_lor=60000):
    import synth
    import torch

    cfg = synth.TINY
    g = oracle.make_grid(16, 16, 16, 8.0)  # same FOV as cfg-1 at coarser voxels
    ev = {k: t.numpy() for k, t in synth.make_events(cfg, n_ev).items()}
    lors = {k: t.numpy() for k, t in synth.make_sens_lors(cfg, n_lor).items()}
    sens = oracle.sensitivity(g, lors).astype(np.float32)
    return g, ev, sens


# ---------------------------------------------------------------- P7
def test_p7_mlem_preserves_counts_and_positivity():
    """After every iteration sum_j sens_j x_j = n_valid (exact identity of the EM update when x0 is
    zero off-mask) and x >= 0."""
    g, ev, sens = _small_problem()
    sig = oracle.sigma_mm(300.0)
    mask = oracle.mask_f32(sens)
    x = mask.astype(np.float64)
    for it in range(3):
        corr, n_valid, visits = oracle.em_correction(g, sig, ev, x)
        x = oracle.update(x, corr, sens, mask)
        assert x.min() >= 0.0
        assert n_valid > 3000 and visits > n_valid
        assert abs(np.dot(x, sens.astype(np.float64)) - n_valid) / n_valid < 1e-10
    # the packaged loop gives the same image
    x2, st = oracle.mlem(g, sig, ev, mask.astype(np.float64), sens, 3)
    assert np.allclose(x2, x, rtol=1e-12, atol=0)
    assert st.n_valid == n_valid and abs(st.sum_image_sens - n_valid) / n_valid < 1e-10


# ---------------------------------------------------------------- P8
def test_p8_one_voxel_and_sens_rescale():
    g1 = oracle.make_grid(1, 1, 1, 40.0)
    rng = np.random.default_rng(2)
    n = 500
    d = rng.normal(size=(n, 3))
    d /= np.linalg.norm(d, axis=1)[:, None]
    c = rng.uniform(-15, 15, (n, 3))
    p1, p2 = c - 200 * d, c + 200 * d
    ev = {"x1": p1[:, 0], "y1": p1[:, 1], "z1": p1[:, 2], "x2": p2[:, 0], "y2": p2[:, 1], "z2": p2[:, 2],
          "dt": rng.normal(0, 50, n)}
    sens = np.array([0.37], np.float32)
    for x0 in (1.0, 123.0):
        x, st = oracle.mlem(g1, oracle.sigma_mm(300.0), ev, np.array([x0]), sens, 1)
        assert st.n_valid == n
        assert abs(x[0] - n / float(sens[0])) / x[0] < 1e-12
    # rescaling sens by alpha rescales the image by 1/alpha
    g, ev, sens = _small_problem(n_ev=1500)
    sig = oracle.sigma_mm(300.0)
    x0 = oracle.mask_f32(sens).astype(np.float64)
    xa, _ = oracle.mlem(g, sig, ev, x0, sens, 2)
    xb, _ = oracle.mlem(g, sig, ev, x0, (sens * np.float32(4.0)), 2)  # power of two: exact in fp32
    assert np.allclose(xb * 4.0, xa, rtol=1e-12, atol=0)


# ---------------------------------------------------------------- P9
def _brute_segments(g, p1, p2, s_lo, s_hi, steps):
    """voxel runs along the LOR by fine stepping: list of (flat index, s_enter, s_exit)."""
    p1, p2 = np.asarray(p1, float), np.asarray(p2, float)
    L = np.linalg.norm(p2 - p1)
    u = (p2 - p1) / L
    ds = (s_hi - s_lo) / steps
    s = s_lo + (np.arange(steps) + 0.5) * ds
    q = (p1[None, :] + s[:, None] * u[None, :] - np.array([g.ox, g.oy, g.oz])) / np.array([g.vx, g.vy, g.vz])
    ijk = np.floor(q).astype(np.int64)
    inside = np.all((ijk >= 0) & (ijk < np.array([g.nx, g.ny, g.nz])), axis=1)
    flat = np.where(inside, (ijk[:, 2] * g.ny + ijk[:, 1]) * g.nx + ijk[:, 0], -1)
    return s, ds, flat, L


def test_p9_brute_force_8cube():
    """8^3 grid (NS invariant 4): per-voxel chords by fine stepping; TOF fwd by fine quadrature of
    int x(p(s)) g(s-s_c) ds over the clipped window (agrees within the midpoint bound), and the
    DEFINITION (chord x Gaussian at the clipped-chord midpoint) rebuilt from the brute-force runs."""
    rng = np.random.default_rng(9)
    v = 4.0
    g = oracle.make_grid(8, 8, 8, v)
    sig = 7.0
    img = rng.uniform(0.5, 1.5, g.nvox)
    steps = 200000
    for _ in range(12):
        p1 = rng.uniform(-40, 40, 3)
        p1[rng.integers(3)] = -45.0
        p2 = -p1 + rng.uniform(-8, 8, 3)
        L = np.linalg.norm(p2 - p1)
        # non-TOF per-voxel chord lengths
        s, ds, flat, _ = _brute_segments(g, p1, p2, 0.0, L, steps)
        idx, w = oracle.lor_weights(g, 0.0, p1, p2)
        brute = np.bincount(flat[flat >= 0], minlength=g.nvox) * ds
        mine = np.zeros(g.nvox)
        mine[idx] = w
        assert np.max(np.abs(brute - mine)) < 3 * ds
        # TOF
        s_c = 0.5 * L + rng.uniform(-12, 12)
        dt = dt_for_centre(L, s_c)
        idx, w = oracle.lor_weights(g, sig, p1, p2, dt)
        fwd = float(np.dot(w, img[idx]))
        lo, hi = max(0.0, s_c - 3 * sig), min(L, s_c + 3 * sig)
        s, ds, flat, _ = _brute_segments(g, p1, p2, lo, hi, steps)
        vals = np.where(flat >= 0, img[np.maximum(flat, 0)], 0.0)
        quad = float(np.sum(vals * gauss(s - s_c, sig)) * ds)
        assert abs(fwd - quad) < 0.04 * (v / sig) ** 2 * img.max()
        # the definition from brute-force runs: run boundaries where flat changes
        cut = np.nonzero(np.diff(flat))[0]
        starts = np.concatenate([[0], cut + 1])
        ends = np.concatenate([cut, [steps - 1]])
        defn = 0.0
        for a, b in zip(starts, ends):
            if flat[a] < 0:
                continue
            sa, sb = s[a] - 0.5 * ds, s[b] + 0.5 * ds
            defn += (sb - sa) * gauss(0.5 * (sa + sb) - s_c, sig) * img[flat[a]]
        assert abs(fwd - defn) / defn < 5e-4  # limited by the step size only


# ---------------------------------------------------------------- P10
def test_p10_forward_back_adjoint():
    rng = np.random.default_rng(4)
    g, ev, _ = _small_problem(n_ev=2000, n_lor=10)
    sig = oracle.sigma_mm(300.0)
    x = rng.uniform(0, 1, g.nvox)
    y = rng.uniform(0, 1, 2000)
    for s in (sig, 0.0):
        lhs = float(np.dot(oracle.forward(g, s, ev, x), y))
        rhs = float(np.dot(x, oracle.backproject(g, s, ev, y)))
        assert abs(lhs - rhs) / abs(lhs) < 1e-12
    # values=None means ones
    assert np.allclose(oracle.backproject(g, sig, ev), oracle.backproject(g, sig, ev, np.ones(2000)), rtol=1e-13)


def test_sensitivity_is_mean_chord():
    """sens = (1/m) sum of non-TOF chords: total over voxels = mean box chord of the LORs."""
    import synth

    g = oracle.make_grid(8, 8, 8, 16.0)
    lors = {k: t.numpy() for k, t in synth.make_sens_lors(synth.TINY, 5000).items()}
    sens = oracle.sensitivity(g, lors)
    chords = oracle.forward(g, 0.0, lors, np.ones(g.nvox))
    assert abs(sens.sum() - chords.mean()) / chords.mean() < 1e-12
    assert sens.min() >= 0


# ---------------------------------------------------------------- P11
def test_p11_region_partition(golden):
    """first region 200 slices, eight more of 100, tiling the 1000-slice matrix."""
    R = int(golden["n_regions"][0])
    nz = int(golden["axial_slices"][0])
    k = oracle.default_region_slices(nz, R)
    assert np.diff(k).tolist() == [int(t) for t in golden["region_core_slices"]]
    assert k[0] == 0 and k[-1] == nz
    assert np.diff(oracle.default_region_slices(640, 9)).tolist() == [128] + [64] * 8
    # the paper's extended sizes are >= core + (3 sigma + 6 mm shell) per open side (R12)
    m = oracle.region_margin_slices(golden["sigma_mm_at_300ps"][0], golden["voxel_mm"][0], 3.0, golden["shell_mm"][0])
    assert m == 32
    ext = golden["region_extended_slices"]
    assert ext[0] >= 200 + m and ext[1] >= 100 + 2 * m and ext[2] >= 100 + m
    assert oracle.region_margin_slices(oracle.sigma_mm(300.0), 3.75) == 17


def test_p11_region_ids_boundaries_and_counts():
    g = oracle.make_grid(160, 160, 640, 3.75)
    zb = oracle.region_zbounds(g, 9)
    assert zb.dtype == np.float32 and zb[0] == np.float32(-1200.0) and zb[-1] == np.float32(1200.0)
    assert np.all(np.diff(zb) > 0)
    # hand-placed events: vertical-ish LORs along x with dt=0 -> centre z = (z1+z2)/2 exactly
    zs = []
    for j in range(1, 9):
        b = zb[j]
        zs += [np.nextafter(b, np.float32(-np.inf)), b, np.nextafter(b, np.float32(np.inf))]
    zs += [np.float32(-5000.0), np.float32(5000.0)]  # out of range clamps to first / last
    zs = np.array(zs, np.float32)
    n = zs.size
    ev = {"x1": np.full(n, -400.0), "y1": np.zeros(n), "z1": zs, "x2": np.full(n, 400.0), "y2": np.zeros(n),
          "z2": zs, "dt": np.zeros(n)}
    region, counts = oracle.region_ids(ev, zb)
    want = []
    for j in range(1, 9):
        want += [j - 1, j, j]
    want += [0, 8]
    assert region.tolist() == want
    assert counts.sum() == n and counts.tolist() == np.bincount(want, minlength=9).tolist()
    # dt moves the centre along the LOR: z-aligned LOR, dt>0 moves towards endpoint 2 (+z here)
    ev = {"x1": [0.0], "y1": [0.0], "z1": [-1000.0], "x2": [0.0], "y2": [0.0], "z2": [1000.0], "dt": [2000.0]}
    region, _ = oracle.region_ids(ev, zb)  # centre z = +299.79 mm -> slice 400 -> region index 4
    assert region.tolist() == [int(np.searchsorted(zb[1:9], np.float32(299.79), side="right"))]
    ev["dt"] = [np.nan]
    assert oracle.region_ids(ev, zb)[0].tolist() == [-1]


# ---------------------------------------------------------------- P18 (reading R27 / specification F3)
def test_p18_region_spans_hand_built():
    """an event "always contributed to 1 or 2 image regions".  Hand-placed LORs whose window's axial extent
    is known by construction; expected spans typed in."""
    g = oracle.make_grid(160, 160, 640, 3.75)
    zb = oracle.region_zbounds(g, 9)  # borders at -720, -480, -240, 0, 240, 480, 720, 960 (cores 480 + 8 x 240 mm)
    assert zb.tolist() == [-1200.0, -720.0, -480.0, -240.0, 0.0, 240.0, 480.0, 720.0, 960.0, 1200.0]
    hw = 60.0

    def span(p1, p2, dt=0.0):
        ev = {"x1": [p1[0]], "y1": [p1[1]], "z1": [p1[2]], "x2": [p2[0]], "y2": [p2[1]], "z2": [p2[2]], "dt": [dt]}
        lo, hi, counts = oracle.region_spans(ev, zb, hw)
        assert counts.sum() == (hi[0] - lo[0] + 1 if lo[0] >= 0 else 0)
        return int(lo[0]), int(hi[0])

    # transverse LOR (dz = 0): the window has no axial extent -> exactly the single-assignment region, also on a border
    assert span((-400, 0, 100.0), (400, 0, 100.0)) == (4, 4)
    assert span((-400, 0, 240.0), (400, 0, 240.0)) == (5, 5)
    # axial LOR (|dz| / L = 1): extent = centre +- 60 mm
    assert span((0, 0, -1000), (0, 0, 1000)) == (3, 4)            # centre 0: [-60, 60] straddles the border at 0
    assert span((0, 0, -1000 + 120), (0, 0, 1000 + 120)) == (4, 4)  # centre 120: [60, 180] inside region 4
    assert span((0, 0, -1000 + 180), (0, 0, 1000 + 180)) == (4, 5)  # centre 180: [120, 240] touches the border at 240 (<=)
    assert span((0, 0, -1000 + 179), (0, 0, 1000 + 179)) == (4, 4)  # [119, 239]
    assert span((0, 0, 1000 + 180), (0, 0, -1000 + 180)) == (4, 5)  # reversed LOR: |dz|
    # 3-4-5 triangle: |dz| / L = 0.6 -> extent = centre +- 36 mm
    assert span((-400, 0, -300 + 30), (400, 0, 300 + 30)) == (3, 4)  # centre 30: [-6, 66]
    assert span((-400, 0, -300 + 40), (400, 0, 300 + 40)) == (4, 4)  # centre 40: [4, 76]
    # dt moves the centre towards end point 2 (R22): c/2 * 400 ps = 59.96 mm along +z
    assert span((0, 0, -1000), (0, 0, 1000), dt=400.0) == (3, 4)      # centre 59.96: [-0.04, 119.96] still reaches below 0
    assert span((0, 0, -1000), (0, 0, 1000), dt=401.0) == (4, 4)      # centre 60.11: [0.11, 120.11]
    assert span((0, 0, -1000), (0, 0, 1000), dt=-401.0) == (3, 3)     # centre -60.11: [-120.11, -0.11]
    # out of range: clamps to the first / last region; invalid -> (-1, -1)
    assert span((0, 0, -3000), (0, 0, 0)) == (0, 0)
    assert span((0, 0, float("nan")), (0, 0, 0)) == (-1, -1)
    # consistency with the single assignment: lo <= region <= hi, and spans of a dz = 0 set equal the single assignment
    rng = np.random.default_rng(11)
    n = 20_000
    ev = {k: rng.uniform(-400, 400, n).astype(np.float32) for k in ("x1", "y1", "x2", "y2")}
    ev["z1"] = rng.uniform(-1200, 1200, n).astype(np.float32)
    ev["z2"] = rng.uniform(-1200, 1200, n).astype(np.float32)
    ev["dt"] = rng.normal(0, 500, n).astype(np.float32)
    region, _ = oracle.region_ids(ev, zb)
    lo, hi, counts = oracle.region_spans(ev, zb, hw)
    assert np.all(lo <= region) and np.all(region <= hi) and np.all(hi - lo <= 1)
    assert counts.sum() == n + int((hi > lo).sum())
    lo0, hi0, _ = oracle.region_spans(ev, zb, 0.0)
    assert np.array_equal(lo0, region) and np.array_equal(hi0, region)


# ---------------------------------------------------------------- P12
def test_p12_bin_keys_hand_built():
    g = oracle.make_grid(32, 32, 32, 4.0)  # 4x4x4 tiles of 8^3 voxels, T = 64
    assert oracle.num_bins(g) == 12 * 64

    def key_of(p1, p2, dt=0.0):
        ev = {"x1": [p1[0]], "y1": [p1[1]], "z1": [p1[2]], "x2": [p2[0]], "y2": [p2[1]], "z2": [p2[2]], "dt": [dt]}
        return int(oracle.bin_keys(g, ev)[0])

    # centre (2,2,2) mm -> voxel (16,16,16) -> tile (2,2,2) -> 42
    t_mid = (2 * 4 + 2) * 4 + 2
    # dominant +x, dy>0, dz>0 -> class 0 ; dominant x given as -x is flipped: same class
    assert key_of((-98, -8, -3), (102, 12, 7)) == 0 * 64 + t_mid
    assert key_of((102, 12, 7), (-98, -8, -3)) == 0 * 64 + t_mid
    # dominant x, dy<0, dz>0 -> 2 ; dy>0, dz<0 -> 1 ; both <0 -> 3
    assert key_of((-98, 12, -3), (102, -8, 7)) == 2 * 64 + t_mid
    assert key_of((-98, -8, 7), (102, 12, -3)) == 1 * 64 + t_mid
    assert key_of((-98, 12, 7), (102, -8, -3)) == 3 * 64 + t_mid
    # dominant y: a=1, next axes are (z, x): dz<0 -> +2, dx<0 -> +1
    assert key_of((-8, -98, 7), (12, 102, -3)) == (4 + 2) * 64 + t_mid
    assert key_of((12, -98, -3), (-8, 102, 7)) == (4 + 1) * 64 + t_mid
    # dominant z: a=2, next axes are (x, y)
    assert key_of((-8, 12, -98), (12, -8, 102)) == (8 + 1) * 64 + t_mid
    # tie |dx| = |dy| -> lowest axis (x)
    assert key_of((-98, -98, 2), (102, 102, 2)) // 64 == 0
    # tile from the TOF centre: x-aligned LOR, dt = +200 ps moves the centre +29.98 mm towards p2
    k = key_of((-100, 2, 2), (100, 2, 2), 200.0)  # centre x = 29.98 -> voxel 23 -> tile x 2
    assert k == (2 * 4 + 2) * 4 + 2
    k = key_of((-100, 2, 2), (100, 2, 2), 250.0)  # centre x = 37.47 -> voxel 25 -> tile x 3
    assert k == (2 * 4 + 2) * 4 + 3
    # centres outside the grid clamp to the border tiles
    assert key_of((-100, 2, 2), (100, 2, 2), 2000.0) == (2 * 4 + 2) * 4 + 3
    assert key_of((-100, 2, 2), (100, 2, 2), -2000.0) == (2 * 4 + 2) * 4 + 0
    # invalid events
    assert key_of((1, 2, 3), (1, 2, 3)) == 0xFFFFFFFF
    assert key_of((np.nan, 2, 3), (1, 2, 3)) == 0xFFFFFFFF
    assert key_of((-100, 2, 2), (100, 2, 2), np.inf) == 0xFFFFFFFF


def test_bin_keys_in_range_on_synthetic_events():
    import synth

    g = oracle.make_grid(160, 160, 640, 3.75)
    ev = {k: t.numpy() for k, t in synth.make_events(synth.FULL, 20000).items()}
    key = oracle.bin_keys(g, ev)
    T = 20 * 20 * 80
    assert oracle.num_bins(g) == 12 * T and key.max() < 12 * T
    assert len(np.unique(key // T)) == 12  # the long scanner accepts every direction class


# ---------------------------------------------------------------- P17
def test_p17_mask_rule_float32():
    """R11: mask_j = (sens_j >= floor_rel * max_k sens_k) and sens_j > 0, decided in FLOAT32, default
    floor 1e-2.  The expected bytes below are typed by hand from IEEE binary32 arithmetic, not computed by any code:
      max = 100 -> thr = fl32(0.01f * 100f): 0.01f = 0.00999999977648..., the product 0.99999997765 lies between the
      neighbouring floats 0.99999994 and 1.0 and rounds to 1.0f exactly;
      max = 3 -> thr = fl32(0.01f * 3f) = 0.0299999993294... = 0.03f, whereas a double-precision threshold 0.01 * 3.0
      = 0.03 > 0.03f would reject the voxel that holds 0.03f."""
    one = np.float32(1.0)
    below, above = np.nextafter(one, np.float32(0.0)), np.nextafter(one, np.float32(2.0))
    sens = np.array([100.0, 1.0, below, above, 0.0, -5.0, np.nan, 0.5, 2.0, -0.0, 99.0],
                    np.float32)
    #                100   at  below  above  0   neg  NaN  0.5  2.0  -0   99
    want = np.array([1,    1,  0,     1,     0,  0,   0,   0,   1,   0,   1], np.uint8)
    assert np.array_equal(oracle.mask_f32(sens), want)  # default floor_rel = 1e-2
    assert np.array_equal(oracle.mask_f32(sens, 1e-2), want)
    # '>' instead of '>=' would drop element 1; a threshold taken relative to the mean or the sum instead of the max
    # would move it far from 1.0 and flip elements 7 and 8.
    # float32 product, not double: the voxel holding exactly 0.03f survives with max = 3
    s3 = np.array([3.0, np.float32(0.03), np.nextafter(np.float32(0.03), np.float32(0.0))], np.float32)
    assert np.array_equal(oracle.mask_f32(s3), np.array([1, 1, 0], np.uint8))
    # another floor: 0.5 * 100 = 50 exactly
    assert np.array_equal(oracle.mask_f32(sens, 0.5), np.array([1, 0, 0, 0, 0, 0, 0, 0, 0, 0, 1], np.uint8))
    # floor 0 keeps every strictly positive voxel and nothing else (sens > 0 is part of the rule)
    assert np.array_equal(oracle.mask_f32(sens, 0.0), np.array([1, 1, 1, 1, 0, 0, 0, 1, 1, 0, 1], np.uint8))
    # all-zero sensitivity: max = 0 -> thr = 0, and 0 >= 0 must NOT make a voxel exist
    assert not oracle.mask_f32(np.zeros(7, np.float32)).any()
    # the maximum is taken over the whole array, wherever it sits (last element here)
    assert np.array_equal(oracle.mask_f32(np.array([0.9, 1.0, 100.0], np.float32)), np.array([0, 1, 1], np.uint8))
