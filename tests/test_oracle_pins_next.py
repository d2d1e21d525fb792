"""Pins of the oracle's widened rows (NEXT-1 K-sample kernel, NEXT-2 median filter,
NEXT-3 per-event attenuation weights, NEXT-4 TOF scatter rejection).  No GPU, no CUDA path.

As in test_oracle_pins.py nothing here re-types the oracle's formulas: expected values are what the paper
prints (tests/golden/paper_values.txt), closed forms / constructions, a library routine
(scipy.ndimage.median_filter, math.erf), limits that reduce to an already pinned function, or statistics the
paper's wording fixes (the 95 % confidence level)."""
import math

import numpy as np
import pytest

import oracle
import synth

SIG300 = oracle.sigma_mm(300.0)


def dt_for_centre(L, s_c):
    return 2.0 * (s_c - 0.5 * L) / oracle.C_MM_PER_PS


# ---------------------------------------------------------------- P13: K-sample TOF kernel
def test_p13_lut_sums_to_one_symmetric_printed_K(golden):
    """PAPER.md:77 "the sum of the weights equaled one"; :79 15 samples (CPU), 32 (GPU); equally spaced."""
    for K in [int(k) for k in golden["tof_samples_cpu_gpu"]] + [1, 2, 101]:
        off, w = oracle.sample_lut(K, SIG300)
        assert off.shape == (K,) and w.shape == (K,)
        assert abs(w.sum() - 1.0) < 1e-14
        assert np.allclose(w, w[::-1], rtol=0, atol=1e-16) and np.allclose(off, -off[::-1], atol=1e-12)
        if K > 1:
            assert np.allclose(np.diff(off), 6.0 * SIG300 / (K - 1), rtol=1e-12)  # equally spaced over +-3 sigma
            assert abs(off[0] + 3.0 * SIG300) < 1e-12 and abs(off[-1] - 3.0 * SIG300) < 1e-12
            # "giving them the equivalent Gaussian weight": ratios of weights are ratios of the Gaussian
            r = w / w[K // 2]
            assert np.allclose(r, np.exp(-0.5 * (off / SIG300) ** 2) / math.exp(-0.5 * (off[K // 2] / SIG300) ** 2),
                               rtol=1e-12)
    off, w = oracle.sample_lut(15, SIG300)
    assert w.argmax() == 7 and off[7] == 0.0  # odd K: the central sample sits on the measured time difference


def test_p13_samples_land_where_constructed():
    """Axis-aligned LOR through voxel centres, spacing of the samples = one voxel: sample k must fall into
    voxel (ic + k - (K-1)/2) of the row, each with its LUT weight; index layout (iz*ny+iy)*nx+ix."""
    v, K = 4.0, 9
    sigma = (K - 1) * v / 6.0  # 6 sigma/(K-1) = v
    g = oracle.make_grid(20, 6, 5, v, origin=(-40.0, -12.0, -10.0))
    iy, iz, ic = 4, 2, 11
    y, z = g.oy + (iy + 0.5) * v, g.oz + (iz + 0.5) * v
    p1, p2 = (-100.0, y, z), (100.0, y, z)
    s_c = (g.ox + (ic + 0.5) * v) - p1[0]
    idx, w = oracle.lor_samples(g, sigma, K, p1, p2, dt_for_centre(200.0, s_c))
    off, lut = oracle.sample_lut(K, sigma)
    exp_ix = ic + np.arange(K) - (K - 1) // 2
    assert np.array_equal(idx, (iz * g.ny + iy) * g.nx + exp_ix)
    assert np.array_equal(w, lut)
    # reversed LOR and the opposite sign of dt: same voxels, traversed the other way
    idx2, w2 = oracle.lor_samples(g, sigma, K, p2, p1, -dt_for_centre(200.0, s_c))
    assert np.array_equal(idx2, idx[::-1])
    # along y and z (transposed-axis mistakes)
    g2 = oracle.make_grid(5, 20, 6, v, origin=(-10.0, -40.0, -12.0))
    x, z = g2.ox + 1.5 * v, g2.oz + 3.5 * v
    s_c = (g2.oy + (ic + 0.5) * v) + 100.0
    idx, _ = oracle.lor_samples(g2, sigma, K, (x, -100.0, z), (x, 100.0, z), dt_for_centre(200.0, s_c))
    assert np.array_equal(idx, (3 * g2.ny + exp_ix) * g2.nx + 1)


def test_p13_samples_outside_grid_or_lor_are_dropped():
    v, K = 4.0, 9
    sigma = (K - 1) * v / 6.0
    g = oracle.make_grid(8, 4, 4, v, origin=(-16.0, -8.0, -8.0))
    y = z = 2.0
    # centre in the first voxel: the 4 samples to its left fall outside the grid
    s_c = (g.ox + 0.5 * v) + 100.0
    idx, w = oracle.lor_samples(g, sigma, K, (-100.0, y, z), (100.0, y, z), dt_for_centre(200.0, s_c))
    _, lut = oracle.sample_lut(K, sigma)
    assert len(idx) == 5 and np.array_equal(w, lut[4:])
    # a LOR that starts inside the grid: samples before endpoint 1 are dropped (R8)
    p1 = (g.ox + 2.5 * v, y, z)
    idx, w = oracle.lor_samples(g, sigma, K, p1, (100.0, y, z), dt_for_centre(100.0 - p1[0], 1.0 * v))
    assert np.array_equal(idx % g.nx, np.arange(2, 8)) and np.array_equal(w, lut[3:])
    # uniform image, kernel wholly inside: forward value = sum of the weights = 1
    g3 = oracle.make_grid(40, 4, 4, v, origin=(-80.0, -8.0, -8.0))
    ev = {"x1": [-100.0], "y1": [y], "z1": [z], "x2": [100.0], "y2": [y], "z2": [z], "dt": [30.0]}
    assert abs(oracle.forward(g3, sigma, ev, np.ones(g3.nvox), K=K)[0] - 1.0) < 1e-14


def test_p13_many_samples_converge_to_siddon_tof():
    """K -> infinity: sum_k w_k x(p(s_k)) is a Riemann sum of the same integral the Siddon x Gaussian row
    evaluates chord by chord, divided by the truncated mass erf(3/sqrt 2) (the sample weights are normalised,
    R4: the chord weights are not).  Pins sample positions / centre / sign of dt against the pinned projector."""
    rng = np.random.default_rng(5)
    g = oracle.make_grid(24, 20, 28, (3.0, 3.5, 2.5))
    img = rng.random(g.nvox)
    n = 40
    ang = rng.random(n) * 2 * np.pi
    zz = (rng.random((n, 2)) - 0.5) * 60.0
    ev = {"x1": 200 * np.cos(ang), "y1": 200 * np.sin(ang), "z1": zz[:, 0],
          "x2": -200 * np.cos(ang + 0.2), "y2": -200 * np.sin(ang + 0.2), "z2": zz[:, 1],
          "dt": rng.normal(0, 120.0, n)}
    ev = {k: np.asarray(v, np.float32) for k, v in ev.items()}
    sigma = SIG300
    sid = oracle.forward(g, sigma, ev, img) / math.erf(3.0 / math.sqrt(2.0))
    # midpoint-rule error of the Siddon row on a rough image ~ (v/sigma)^2; sampling error ~ 1/K jumps
    smp = oracle.forward(g, sigma, ev, img, K=20001)
    ok = sid > 0
    assert ok.sum() > 30
    assert np.max(np.abs(smp[ok] - sid[ok]) / sid[ok]) < 0.02
    # and a coarse K = 32 is visibly different from K = 20001 (so the limit test is not vacuous)
    smp32 = oracle.forward(g, sigma, ev, img, K=32)
    assert np.max(np.abs(smp32[ok] - smp[ok]) / smp[ok]) > 0.02


def test_p13_forward_back_adjoint_and_em_invariant():
    rng = np.random.default_rng(3)
    g = oracle.make_grid(16, 16, 16, 4.0)
    cfg = synth.TINY
    ev = {k: v.numpy() for k, v in synth.make_events(cfg, 3000).items()}
    x, yv = rng.random(g.nvox), rng.random(3000)
    ax = oracle.forward(g, SIG300, ev, x, K=32)
    aty = oracle.backproject(g, SIG300, ev, yv, K=32)
    assert abs(ax @ yv - x @ aty) <= 1e-12 * abs(ax @ yv)
    # P7 for the sampled projector: sum_j corr_j x_j = n_valid (each valid event contributes fwd/fwd)
    corr, nv, vis = oracle.em_correction(g, SIG300, ev, x, K=32)
    assert nv > 2000 and abs(corr @ x - nv) < 1e-9 * nv and vis <= 32 * 3000


# ---------------------------------------------------------------- P14: median filter
@pytest.mark.parametrize("shape", [(7, 5, 9), (1, 1, 1), (2, 3, 1), (16, 16, 16)])
def test_p14_median3_matches_scipy(shape):
    from scipy import ndimage

    rng = np.random.default_rng(17)
    nx, ny, nz = shape
    g = oracle.make_grid(nx, ny, nz, 1.0)
    img = rng.random((nz, ny, nx))
    img[rng.random(img.shape) < 0.3] = 0.0  # ties
    got = oracle.median3(g, img).reshape(nz, ny, nx)
    ref = ndimage.median_filter(img, size=3, mode="nearest")
    assert np.array_equal(got, ref)


def test_p14_median3_special_cases():
    g = oracle.make_grid(9, 8, 7, 1.0)
    # constant image is a fixed point; a single hot voxel (impulse noise) is removed
    assert np.array_equal(oracle.median3(g, np.full(g.nvox, 2.5)), np.full(g.nvox, 2.5))
    img = np.zeros((7, 8, 9))
    img[3, 4, 5] = 100.0
    assert not oracle.median3(g, img).any()
    # a half-space edge is preserved (median filters keep edges)
    img = np.zeros((7, 8, 9))
    img[:, :, 5:] = 1.0
    assert np.array_equal(oracle.median3(g, img).reshape(7, 8, 9), img)
    # a linear ramp along x is preserved away from the x borders
    ramp = np.broadcast_to(np.arange(9.0), (7, 8, 9)).copy()
    out = oracle.median3(g, ramp).reshape(7, 8, 9)
    assert np.array_equal(out[:, :, 1:-1], ramp[:, :, 1:-1])


def test_p14_mlem_with_median_is_update_then_filter():
    """orc_mlem_x(median=1) = [EM pass, update, median3] per iteration ("after each iteration")."""
    cfg = synth.TINY
    g = oracle.make_grid(16, 16, 16, 8.0)
    ev = {k: v.numpy() for k, v in synth.make_events(cfg, 5000).items()}
    lors = {k: v.numpy() for k, v in synth.make_sens_lors(cfg, 40000).items()}
    sens = oracle.sensitivity(g, lors).astype(np.float32)
    mask = oracle.mask_f32(sens)
    x = mask.astype(np.float64)
    sig = oracle.sigma_mm(cfg.tof_fwhm_ps)
    got, _ = oracle.mlem(g, sig, ev, x, sens, 2, median=True)
    for _ in range(2):
        corr, _, _ = oracle.em_correction(g, sig, ev, x)
        x = oracle.median3(g, oracle.update(x, corr, sens, mask))
    assert np.allclose(got, x, rtol=1e-11, atol=0)  # the OpenMP reduction order is not fixed


# ---------------------------------------------------------------- P15: attenuation weights
def test_p15_attenuation_weight_uniform_box_is_exp_mu_chord():
    """Uniform mu over the whole grid: w = exp(mu * chord), chord known by construction (points on two faces)."""
    rng = np.random.default_rng(23)
    g = oracle.make_grid(10, 12, 14, (3.0, 2.0, 2.5))
    lo = np.array([g.ox, g.oy, g.oz])
    hi = lo + np.array([g.nx * g.vx, g.ny * g.vy, g.nz * g.vz])
    mu = 0.0096  # 1/mm, water at 511 keV
    n = 200
    A = lo + rng.random((n, 3)) * (hi - lo)
    B = lo + rng.random((n, 3)) * (hi - lo)
    A[:, 0], B[:, 0] = lo[0], hi[0]  # enter through x = lo, leave through x = hi
    d = B - A
    chord = np.linalg.norm(d, axis=1)
    u = d / chord[:, None]
    P1, P2 = A - 50.0 * u, B + 70.0 * u  # detectors outside the grid
    ev = {"x1": P1[:, 0], "y1": P1[:, 1], "z1": P1[:, 2], "x2": P2[:, 0], "y2": P2[:, 1], "z2": P2[:, 2]}
    ev = {k: v.astype(np.float32) for k, v in ev.items()}
    w = oracle.attenuation_weights(g, ev, np.full(g.nvox, mu))
    # float32 endpoints move the chord by ~1e-5 mm
    assert np.allclose(w, np.exp(mu * chord), rtol=1e-6)
    assert np.all(w >= 1.0)  # a weight "inversely proportional to the probability" of survival is >= 1
    # a LOR that misses the grid is not attenuated
    miss = {k: np.array([v], np.float32) for k, v in
            dict(x1=-100.0, y1=500.0, z1=0.0, x2=100.0, y2=500.0, z2=0.0).items()}
    assert oracle.attenuation_weights(g, miss, np.full(g.nvox, mu))[0] == 1.0


def test_p15_weighted_em_pass():
    """corr_j = sum_e w_e a_ej / fwd_e: linear in w; w = 1 is the unweighted pass; one-voxel closed form."""
    rng = np.random.default_rng(29)
    cfg = synth.TINY
    g = oracle.make_grid(16, 16, 16, 8.0)
    sig = oracle.sigma_mm(cfg.tof_fwhm_ps)
    ev = {k: v.numpy() for k, v in synth.make_events(cfg, 4000).items()}
    x = rng.random(g.nvox) + 0.1
    c0, nv0, _ = oracle.em_correction(g, sig, ev, x)
    c1, nv1, _ = oracle.em_correction(g, sig, ev, x, weights=np.ones(4000))
    assert np.allclose(c0, c1, rtol=1e-12, atol=0) and nv0 == nv1  # (OpenMP reduction order is not fixed)
    w = rng.random(4000) + 0.5
    cw, _, _ = oracle.em_correction(g, sig, ev, x, weights=w)
    c3, _, _ = oracle.em_correction(g, sig, ev, x, weights=3.0 * w)
    assert np.allclose(c3, 3.0 * cw, rtol=1e-13)
    # sum_j corr_j x_j = sum over valid events of w_e (each event contributes w_e * fwd_e / fwd_e)
    fwd = oracle.forward(g, sig, ev, x)
    assert abs(cw @ x - w[fwd > 0].sum()) < 1e-9 * w.sum()
    # weights select events: weight 0 on half of them = the pass over the other half
    half = np.arange(4000) % 2 == 0
    ch, _, _ = oracle.em_correction(g, sig, ev, x, weights=half.astype(float))
    cs, _, _ = oracle.em_correction(g, sig, {k: v[half] for k, v in ev.items()}, x)
    assert np.allclose(ch, cs, rtol=1e-12, atol=1e-15)
    # one voxel: x1 = sum of the weights of the valid events / sens, whatever x0 > 0
    g1 = oracle.make_grid(1, 1, 1, 60.0)
    sens = np.array([0.37], np.float32)
    img, st = oracle.mlem(g1, sig, ev, np.array([2.2]), sens, 1, weights=w)
    fwd1 = oracle.forward(g1, sig, ev, np.ones(1))
    assert abs(img[0] - w[fwd1 > 0].sum() / float(sens[0])) < 1e-9 * img[0]


# ---------------------------------------------------------------- P16: TOF scatter rejection
def _ev(p1, p2, dt):
    a = np.array([p1, p2], np.float64)
    return {"x1": [a[0, 0]], "y1": [a[0, 1]], "z1": [a[0, 2]], "x2": [a[1, 0]], "y2": [a[1, 1]], "z2": [a[1, 2]],
            "dt": [dt]}


def test_p16_hand_built_segments_against_a_sphere():
    """Sphere of radius 50 at (10, 0, 0); LOR along x at height y: kept iff the +-h segment around the TOF
    centre comes within 50 mm of the sphere centre (point-to-segment distance, by construction)."""
    ell = oracle.ellipsoids_f32([((10.0, 0.0, 0.0), (50.0, 50.0, 50.0))])
    h = oracle.scatter_half_width_f32(SIG300)  # 37.43 mm
    assert abs(float(h) - 1.959964 * SIG300) < 1e-5
    cases = [  # (y, x of the TOF centre, expected)
        (0.0, 10.0, 1),  # centre inside
        (0.0, 10.0 + 50.0 + 37.0, 1),  # segment end reaches the surface (50 + h - 0.43)
        (0.0, 10.0 + 50.0 + 38.0, 0),  # just too far
        (0.0, 10.0 - 50.0 - 38.0, 0),  # other side
        (0.0, 10.0 - 50.0 - 37.0, 1),
        (49.5, 10.0, 1),  # grazing LOR, centre above the sphere centre
        (50.5, 10.0, 0),  # LOR misses the sphere altogether
        (49.5, 200.0, 0),
        (30.0, 10.0 + 40.0 + 37.0, 1),  # chord half-length at y = 30 is 40
        (30.0, 10.0 + 40.0 + 38.0, 0),
    ]
    for y, xc, expect in cases:
        L = 800.0
        ev = _ev((-400.0, y, 0.0), (400.0, y, 0.0), dt_for_centre(L, xc + 400.0))
        keep, cnt = oracle.scatter_keep(ev, ell, h)
        assert keep[0] == expect and cnt == expect, (y, xc)
        # the reversed LOR with the opposite dt describes the same event
        ev = _ev((400.0, y, 0.0), (-400.0, y, 0.0), -dt_for_centre(L, xc + 400.0))
        assert oracle.scatter_keep(ev, ell, h)[0][0] == expect


def test_p16_ellipsoid_axes_union_and_invalid():
    """Anisotropic ellipsoid (semi-axes 20, 60, 100): a LOR along z at x = 19 is kept, at x = 21 rejected; the
    same offsets along y (59 / 61) pin which reciprocal goes with which axis.  Union: any ellipsoid suffices."""
    h = oracle.scatter_half_width_f32(SIG300)
    ell = oracle.ellipsoids_f32([((0.0, 0.0, 0.0), (20.0, 60.0, 100.0))])
    for (x, y, expect) in [(19.0, 0.0, 1), (21.0, 0.0, 0), (0.0, 59.0, 1), (0.0, 61.0, 0)]:
        ev = _ev((x, y, -500.0), (x, y, 500.0), 0.0)
        assert oracle.scatter_keep(ev, ell, h)[0][0] == expect, (x, y)
    # along z the surface is at 100: centre at z = 100 + 37 is kept, 100 + 38 is not
    for (zc, expect) in [(137.0, 1), (138.0, 0)]:
        ev = _ev((0.0, 0.0, -500.0), (0.0, 0.0, 500.0), dt_for_centre(1000.0, zc + 500.0))
        assert oracle.scatter_keep(ev, ell, h)[0][0] == expect
    two = oracle.ellipsoids_f32([((0.0, 0.0, 0.0), (20.0, 60.0, 100.0)), ((300.0, 0.0, 0.0), (10.0, 10.0, 10.0))])
    ev = _ev((300.0, 5.0, -500.0), (300.0, 5.0, 500.0), 0.0)
    assert oracle.scatter_keep(ev, ell, h)[0][0] == 0 and oracle.scatter_keep(ev, two, h)[0][0] == 1
    # invalid events (F1) are never kept
    bad = _ev((0.0, 0.0, 0.0), (0.0, 0.0, 0.0), 0.0)
    assert oracle.scatter_keep(bad, ell, h)[0][0] == 0
    bad = _ev((0.0, 0.0, -500.0), (0.0, 0.0, 500.0), float("nan"))
    assert oracle.scatter_keep(bad, ell, h)[0][0] == 0


def test_p16_true_events_survive_at_the_confidence_level():
    """PAPER.md:63 "limits of rejection ... at the 95% confidence level": a TRUE event's emission point lies in
    the body and within +-1.96 sigma of the TOF centre with probability 0.95, so at least ~95 % of the trues
    are kept; scatter-like LORs (random detector pairs) are rejected far more often."""
    cfg = synth.FULL
    n = 40000
    ev = {k: v.numpy() for k, v in synth.make_events(cfg, n).items()}
    kinds = synth.event_kinds(cfg, n).numpy()  # 1 = scatter-like
    ell = oracle.ellipsoids_f32([(s.centre, s.semi) for s in cfg.phantom.parts])
    h = oracle.scatter_half_width_f32(oracle.sigma_mm(cfg.tof_fwhm_ps))
    keep, cnt = oracle.scatter_keep(ev, ell, h)
    assert cnt == keep.sum()
    true_kept = keep[kinds == 0].mean()
    scat_kept = keep[kinds == 1].mean()
    assert true_kept >= 0.95 - 3 * math.sqrt(0.05 * 0.95 / (kinds == 0).sum())
    assert true_kept < 1.0  # some trues with a large timing error are lost: the cut is not vacuous
    assert scat_kept < 0.6 * true_kept
    # a tighter confidence level rejects more of both
    keep68, _ = oracle.scatter_keep(ev, ell, oracle.scatter_half_width_f32(oracle.sigma_mm(cfg.tof_fwhm_ps), 1.0))
    assert keep68.sum() < keep.sum() and not np.any(keep68 & ~keep)
