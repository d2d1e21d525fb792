"""GPU parity: the CUDA path (through the C ABI binding) against the fp64 oracle, element by element, on the
same seeded inputs.  Tolerances are BASELINE.json north_star's:
  per-LOR forward values  rel <= 1e-4;  image after N iterations rel-L2 <= 1e-3 and max rel <= 1e-2 on voxels
  above 1 % of the image maximum;  bin keys / region ids bit-exact.
"""
import numpy as np
import pytest
import torch

import oracle
import synth

pytestmark = pytest.mark.gpu

FWD_RTOL = 1e-4
IMG_L2 = 1e-3
IMG_MAX = 1e-2


@pytest.fixture(scope="module")
def pkg():
    import paper_1706_07075_b200 as p

    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return p


def grids(pkg, cfg):
    g = pkg.make_grid(cfg.nx, cfg.ny, cfg.nz, cfg.voxel_mm)
    og = oracle.make_grid(cfg.nx, cfg.ny, cfg.nz, cfg.voxel_mm)
    return g, og


def to_np(ev):
    return {k: v.cpu().numpy() for k, v in ev.items()}


def fwd_rel_err(gpu, ref):
    gpu = np.asarray(gpu, np.float64)
    pos = ref > 0
    den = np.maximum(ref, 1e-6 * np.median(ref[pos])) if pos.any() else np.ones_like(ref)
    return np.abs(gpu - ref) / den


def check_image(gpu, ref, l2=IMG_L2, mx=IMG_MAX, zero_tol=0.0):
    """zero_tol: largest value (relative to the image maximum) the CUDA path may hold in a voxel where the oracle holds
    exactly 0.  0 for dense data; sparse data on a large grid has voxels whose ONLY contribution is the sliver chord at
    a clipped window end, which exists in fp32 and not in fp64 or vice versa (SURVEY.md 8(c) "sliver < 1e-3 mm")."""
    gpu = np.asarray(gpu, np.float64).reshape(-1)
    ref = np.asarray(ref, np.float64).reshape(-1)
    rel_l2 = np.linalg.norm(gpu - ref) / np.linalg.norm(ref)
    big = ref > 0.01 * ref.max()
    max_rel = np.max(np.abs(gpu[big] - ref[big]) / ref[big])
    assert rel_l2 <= l2, f"rel-L2 {rel_l2:.3e}"
    assert max_rel <= mx, f"max rel {max_rel:.3e}"
    z = gpu[ref == 0]
    assert z.size == 0 or z.max() <= zero_tol * ref.max(), (z.max(), ref.max(), int((z != 0).sum()))
    return rel_l2, max_rel


@pytest.fixture(scope="module")
def tiny(pkg):
    cfg = synth.TINY
    ev = synth.make_events(cfg, cfg.n_events, device="cuda")
    g, og = grids(pkg, cfg)
    ctx = pkg.Context(cfg.radius_mm, cfg.axial_mm, g, cfg.tof_fwhm_ps)
    return cfg, ev, to_np(ev), g, og, ctx


@pytest.fixture(scope="module")
def tiny_sens(pkg, tiny):
    cfg, ev, ev_np, g, og, ctx = tiny
    lors = synth.make_sens_lors(cfg, cfg.sens_lors, device="cuda")
    sens = torch.empty(g.nvox, dtype=torch.float32, device="cuda")
    ctx.sensitivity(lors, cfg.sens_lors, sens)
    torch.cuda.synchronize()
    return lors, sens


def test_sigma_matches_oracle(pkg, tiny):
    ctx = tiny[5]
    assert abs(ctx.sigma_mm() - oracle.sigma_mm(300.0)) < 1e-12


def test_forward_parity_tiny(pkg, tiny):
    cfg, ev, ev_np, g, og, ctx = tiny
    n = cfg.n_events  # 200 000 = 781 blocks of 256 + a ragged tail of 64
    img = synth.random_image((g.nz, g.ny, g.nx), 123, device="cuda")
    fwd = torch.empty(n, dtype=torch.float32, device="cuda")
    ctx.forward(ev, n, img, fwd)
    ref = oracle.forward(og, oracle.sigma_mm(cfg.tof_fwhm_ps), ev_np, img.cpu().numpy())
    err = fwd_rel_err(fwd.cpu().numpy(), ref)
    assert err.max() <= FWD_RTOL, f"max rel err {err.max():.3e} at {err.argmax()}"
    assert (ref > 0).mean() > 0.95


def test_forward_parity_non_tof(pkg, tiny):
    cfg, ev, ev_np, g, og, _ = tiny
    n = 50_001
    ctx = pkg.Context(cfg.radius_mm, cfg.axial_mm, g, 0.0)
    sub = {k: v[:n].contiguous() for k, v in ev.items()}
    img = synth.random_image((g.nz, g.ny, g.nx), 5, device="cuda")
    fwd = torch.empty(n, dtype=torch.float32, device="cuda")
    ctx.forward({**sub, "dt": None}, n, img, fwd)
    ref = oracle.forward(og, 0.0, {k: v[:n] for k, v in ev_np.items() if k != "dt"}, img.cpu().numpy())
    assert fwd_rel_err(fwd.cpu().numpy(), ref).max() <= FWD_RTOL


def test_backproject_parity_tiny(pkg, tiny):
    cfg, ev, ev_np, g, og, ctx = tiny
    n = 100_003
    sub = {k: v[:n].contiguous() for k, v in ev.items()}
    sub_np = {k: v[:n] for k, v in ev_np.items()}
    vals = synth.random_image((n,), 77, device="cuda")
    out = torch.zeros(g.nvox, dtype=torch.float32, device="cuda")
    ctx.backproject(sub, n, vals, out)
    ref = oracle.backproject(og, oracle.sigma_mm(cfg.tof_fwhm_ps), sub_np, vals.cpu().numpy())
    check_image(out.cpu().numpy(), ref, l2=1e-5, mx=1e-4)
    # values = NULL means ones, and the call accumulates
    ctx.backproject(sub, n, None, out)
    ref2 = ref + oracle.backproject(og, oracle.sigma_mm(cfg.tof_fwhm_ps), sub_np, None)
    check_image(out.cpu().numpy(), ref2, l2=1e-5, mx=1e-4)


def test_sensitivity_sorted_lors_same_image(pkg, tiny, tiny_sens):
    """TOFMLEM_OPT_SENS_SORT: the LORs ordered by locality key and chord length inside the call give the same image (up
    to the order of the float32 sums)."""
    cfg, ev, ev_np, g, og, _ = tiny
    lors, sens = tiny_sens
    ctx = pkg.Context(cfg.radius_mm, cfg.axial_mm, g, cfg.tof_fwhm_ps)
    ctx.set_option(pkg.OPT_SENS_SORT, 1)
    s2 = torch.empty_like(sens)
    ctx.sensitivity(lors, cfg.sens_lors, s2)
    d = float((s2.double() - sens.double()).norm() / sens.double().norm())
    assert d < 1e-6, d


def test_sensitivity_parity_tiny(pkg, tiny, tiny_sens):
    cfg, ev, ev_np, g, og, ctx = tiny
    lors, sens = tiny_sens
    ref = oracle.sensitivity(og, to_np(lors))
    check_image(sens.cpu().numpy(), ref, l2=1e-5, mx=1e-4)


def test_iterate_parity_tiny(pkg, tiny, tiny_sens):
    """cfg-1: 2 MLEM iterations from x0 = mask; both sides get the bit-identical float32 sens (R11)."""
    cfg, ev, ev_np, g, og, ctx = tiny
    _, sens = tiny_sens
    sens_np = sens.cpu().numpy()
    mask = oracle.mask_f32(sens_np)
    x0 = torch.from_numpy(mask.astype(np.float32)).cuda()
    img = x0.clone()
    ctx.iterate(ev, cfg.n_events, img, sens, cfg.iters)
    st = ctx.get_stats()
    ref, ost = oracle.mlem(og, oracle.sigma_mm(cfg.tof_fwhm_ps), ev_np, mask.astype(np.float64), sens_np, cfg.iters)
    check_image(img.cpu().numpy(), ref)
    assert st.n_valid == ost.n_valid and st.n_skipped == ost.n_skipped
    assert abs(int(st.visits) - int(ost.visits)) <= 1e-4 * ost.visits
    # P7 on the GPU: sum(image * sens) = n_valid
    assert abs(st.sum_image_sens - st.n_valid) / st.n_valid < 1e-4
    assert float(img.min()) >= 0.0

    # the two-call form (em_correction + update) gives the same image as iterate
    img2 = x0.clone()
    corr = torch.zeros_like(img2)
    for _ in range(cfg.iters):
        ctx.reset_stats()
        half = cfg.n_events // 2 + 13  # a data set passed in two calls
        ctx.em_correction({k: v[:half] for k, v in ev.items()}, half, img2, corr)
        ctx.em_correction({k: v[half:] for k, v in ev.items()}, cfg.n_events - half, img2, corr)
        ctx.update(img2, corr, sens)
    assert float(corr.abs().max()) == 0.0
    check_image(img2.cpu().numpy(), ref)
    assert ctx.get_stats().n_valid == ost.n_valid


def test_iterate_host_parity_tiny(pkg, tiny, tiny_sens):
    cfg, ev, ev_np, g, og, ctx = tiny
    _, sens = tiny_sens
    sens_np = sens.cpu().numpy()
    mask = oracle.mask_f32(sens_np)
    h_ev = {k: v.cpu().pin_memory() for k, v in ev.items()}
    h_img = torch.from_numpy(mask.astype(np.float32)).pin_memory()
    h_sens = sens.cpu().pin_memory()
    ctx.iterate_host(h_ev, cfg.n_events, h_img, h_sens, cfg.iters)
    ref, ost = oracle.mlem(og, oracle.sigma_mm(cfg.tof_fwhm_ps), ev_np, mask.astype(np.float64), sens_np, cfg.iters)
    check_image(h_img.numpy(), ref)
    assert ctx.get_stats().n_valid == ost.n_valid


def test_mid_parity_subsample(pkg):
    """cfg-2 geometry (128^3 x 2 mm, 30 % scatter-like events, part of the body outside the grid)."""
    cfg = synth.MID
    n, m, iters = 300_000, 2_000_000, 3
    ev = synth.make_events(cfg, n, device="cuda")
    lors = synth.make_sens_lors(cfg, m, device="cuda")
    g, og = grids(pkg, cfg)
    ctx = pkg.Context(cfg.radius_mm, cfg.axial_mm, g, cfg.tof_fwhm_ps)
    sig = oracle.sigma_mm(cfg.tof_fwhm_ps)
    sens = torch.empty(g.nvox, dtype=torch.float32, device="cuda")
    ctx.sensitivity(lors, m, sens)
    img = synth.random_image((g.nz, g.ny, g.nx), 9, device="cuda")
    fwd = torch.empty(n, dtype=torch.float32, device="cuda")
    ctx.forward(ev, n, img, fwd)
    ev_np = to_np(ev)
    ref = oracle.forward(og, sig, ev_np, img.cpu().numpy())
    err = fwd_rel_err(fwd.cpu().numpy(), ref)
    assert err.max() <= FWD_RTOL, f"{err.max():.3e}"
    frac_hit = (ref > 0).mean()
    assert 0.5 < frac_hit < 0.95  # scatter-like LORs and out-of-grid activity miss the window
    assert np.all(fwd.cpu().numpy()[ref == 0] == 0)
    sens_np = sens.cpu().numpy()
    mask = oracle.mask_f32(sens_np)
    x = torch.from_numpy(mask.astype(np.float32)).cuda()
    ctx.iterate(ev, n, x, sens, iters)
    xr, ost = oracle.mlem(og, sig, ev_np, mask.astype(np.float64), sens_np, iters)
    check_image(x.cpu().numpy(), xr)
    st = ctx.get_stats()
    assert st.n_valid == ost.n_valid
    assert abs(st.sum_image_sens - st.n_valid) / st.n_valid < 1e-4


def test_full_geometry_forward_subsample(pkg):
    """cfg-3 grid (160x160x640 x 3.75 mm, coordinates to +-1200 mm, highly inclined LORs) at 100/300/600 ps
    and non-TOF: per-LOR forward parity on a seeded sub-sample."""
    cfg = synth.FULL
    n = 200_000
    ev = synth.make_events(cfg, n, start=1_000_000, device="cuda")
    ev_np = to_np(ev)
    g, og = grids(pkg, cfg)
    img = synth.random_image((g.nz, g.ny, g.nx), 31, device="cuda")
    img_np = img.cpu().numpy()
    for fwhm in (300.0, 100.0, 600.0, 0.0):
        ctx = pkg.Context(cfg.radius_mm, cfg.axial_mm, g, fwhm)
        fwd = torch.empty(n, dtype=torch.float32, device="cuda")
        ctx.forward(ev, n, img, fwd)
        ref = oracle.forward(og, oracle.sigma_mm(fwhm) if fwhm > 0 else 0.0, ev_np, img_np)
        err = fwd_rel_err(fwd.cpu().numpy(), ref)
        assert err.max() <= FWD_RTOL, f"fwhm {fwhm}: {err.max():.3e}"
        assert (ref > 0).mean() > 0.8


def test_edge_cases(pkg):
    g = pkg.make_grid(16, 12, 20, (4.0, 3.0, 2.0))
    og = oracle.make_grid(16, 12, 20, (4.0, 3.0, 2.0))
    ctx = pkg.Context(200.0, 128.0, g, 300.0)
    sig = oracle.sigma_mm(300.0)
    nan, inf = float("nan"), float("inf")
    rows = [
        # x1, y1, z1, x2, y2, z2, dt
        (-200, 0, 0, 200, 0, 0, 0),            # axis aligned, in a voxel boundary plane (y=0, z=0)
        (-200, 1.5, 1.0, 200, 1.5, 1.0, 100),  # axis aligned through voxel centres
        (0, -200, 1.0, 0, 200, 1.0, -50),      # along y, on the x=0 plane
        (1.0, 1.0, -64, 1.0, 1.0, 64, 10),     # along z
        (-200, -100, -60, 200, 100, 60, 0),    # through the grid centre (exact corner crossings)
        (-200, 0, 0, 200, 0, 0, 4000),         # window beyond the grid: misses
        (-200, 100, 0, 200, 100, 0, 0),        # LOR misses the grid
        (5, 5, 5, 5, 5, 5, 0),                 # L = 0
        (nan, 0, 0, 200, 0, 0, 0),             # non-finite coordinate
        (-200, 0, 0, 200, 0, 0, inf),          # non-finite dt
        (-200, 0, 0, 200, 0, 0, nan),
        (-32, -18, -20, 32, 18, 20, 0),        # endpoints ON the grid corners, diagonal
        (-10, 2, 3, 12, -7, 1, 20),            # both endpoints inside the grid
        (-200, 17.999, 19.99, 200, 17.999, 19.99, 0),  # grazing the top edges
    ]
    arr = np.array(rows, np.float32)
    n = arr.shape[0]
    ev_np = {k: np.ascontiguousarray(arr[:, i]) for i, k in enumerate(synth.EVENT_FIELDS)}
    ev = {k: torch.from_numpy(v).cuda() for k, v in ev_np.items()}
    img = synth.random_image((g.nz, g.ny, g.nx), 3, device="cuda")
    fwd = torch.full((n,), -1.0, dtype=torch.float32, device="cuda")
    ctx.forward(ev, n, img, fwd)
    ref = oracle.forward(og, sig, ev_np, img.cpu().numpy())
    got = fwd.cpu().numpy()
    assert np.all(got[ref == 0] == 0)
    pos = ref > 0
    assert pos.sum() >= 7
    assert np.max(np.abs(got[pos] - ref[pos]) / ref[pos]) <= FWD_RTOL
    out = torch.zeros(g.nvox, dtype=torch.float32, device="cuda")
    ctx.backproject(ev, n, None, out)
    refb = oracle.backproject(og, sig, ev_np, None)
    assert np.linalg.norm(out.cpu().numpy() - refb) / np.linalg.norm(refb) < 1e-5
    # empty input: no-ops
    ctx.forward(ev, 0, img, fwd)
    ctx.backproject(ev, 0, None, out)
    x = torch.ones(g.nvox, dtype=torch.float32, device="cuda")
    sens = torch.ones(g.nvox, dtype=torch.float32, device="cuda")
    ctx.iterate(ev, 0, x, sens, 1)  # no events: corr = 0 -> image becomes 0
    assert float(x.abs().max()) == 0.0
    # invalid arguments are reported, not crashed on
    with pytest.raises(pkg.TofMlemError):
        ctx.iterate(ev, n, x, x, 1)  # image aliases sens
    with pytest.raises(pkg.TofMlemError):
        ctx.set_option(99, 1.0)
    with pytest.raises(pkg.TofMlemError):
        ctx.forward({**ev, "dt": None}, n, img, fwd)  # TOF context needs dt


def test_trunc_option(pkg, tiny):
    cfg, ev, ev_np, g, og, _ = tiny
    ctx = pkg.Context(cfg.radius_mm, cfg.axial_mm, g, cfg.tof_fwhm_ps)
    ctx.set_option(pkg.OPT_TRUNC_SIGMAS, 2.0)
    n = 20_000
    img = synth.random_image((g.nz, g.ny, g.nx), 8, device="cuda")
    fwd = torch.empty(n, dtype=torch.float32, device="cuda")
    ctx.forward(ev, n, img, fwd)
    ref = oracle.forward(og, oracle.sigma_mm(300.0), {k: v[:n] for k, v in ev_np.items()}, img.cpu().numpy(), trunc=2.0)
    assert fwd_rel_err(fwd.cpu().numpy(), ref).max() <= FWD_RTOL


# ------------------------------------------------------------------ integer work: bit-exact
def _with_invalid(ev_np, rng):
    ev_np = {k: v.copy() for k, v in ev_np.items()}
    n = ev_np["x1"].size
    bad = rng.choice(n, 37, replace=False)
    ev_np["x1"][bad[:10]] = np.nan
    ev_np["dt"][bad[10:20]] = np.inf
    for k in ("x2", "y2", "z2"):
        ev_np[k][bad[20:]] = ev_np[k.replace("2", "1")][bad[20:]]  # L = 0
    return ev_np, bad


@pytest.mark.parametrize("cfg_name,n", [("tiny", 100_003), ("full", 300_000)])
def test_bin_events_bit_exact(pkg, cfg_name, n):
    cfg = synth.CONFIGS[cfg_name]
    g, og = grids(pkg, cfg)
    ctx = pkg.Context(cfg.radius_mm, cfg.axial_mm, g, cfg.tof_fwhm_ps)
    ev_np, bad = _with_invalid(to_np(synth.make_events(cfg, n, device="cuda")), np.random.default_rng(1))
    ev = {k: torch.from_numpy(v).cuda() for k, v in ev_np.items()}
    nb = ctx.num_bins()
    assert nb == oracle.num_bins(og)
    key = torch.empty(n, dtype=torch.int32, device="cuda")
    perm = torch.empty(n, dtype=torch.int32, device="cuda")
    offs = torch.empty(nb + 1, dtype=torch.int32, device="cuda")
    ctx.bin_events(ev, n, key, perm, offs)
    torch.cuda.synchronize()
    want = oracle.bin_keys(og, ev_np)
    got = key.cpu().numpy().view(np.uint32)
    assert np.array_equal(got, want)
    assert np.all(want[bad] == 0xFFFFFFFF) and (want == 0xFFFFFFFF).sum() == bad.size
    p = perm.cpu().numpy().view(np.uint32).astype(np.int64)
    assert np.array_equal(np.sort(p), np.arange(n))  # a permutation
    sorted_keys = want[p]
    assert np.all(np.diff(sorted_keys.astype(np.int64)) >= 0)  # sorted by key, invalid (max key) last
    o = offs.cpu().numpy().view(np.uint32).astype(np.int64)
    assert np.array_equal(o, np.searchsorted(sorted_keys, np.arange(nb + 1), side="left"))
    assert o[nb] == n - bad.size
    # bin membership (R14: order inside a bin is free): a stable argsort is one valid answer
    stable = np.argsort(want, kind="stable")
    for b in np.unique(want[want != 0xFFFFFFFF])[:: max(1, nb // 200)]:
        assert np.array_equal(np.sort(p[o[b]:o[b + 1]]), stable[o[b]:o[b + 1]])
    # gather
    out = {k: torch.empty_like(v) for k, v in ev.items()}
    ctx.gather_events(ev, perm, n, out)
    for k in synth.EVENT_FIELDS:
        a, b = out[k].cpu().numpy(), ev_np[k][p]
        assert np.array_equal(a.view(np.uint32), b.view(np.uint32))
    # the packed fast path for full permutations gives the same bits
    out2 = {k: torch.zeros_like(v) for k, v in ev.items()}
    ctx.permute_events(ev, perm, n, out2)
    for k in synth.EVENT_FIELDS:
        assert torch.equal(out[k].view(torch.int32), out2[k].view(torch.int32))


def test_split_regions_bit_exact(pkg):
    cfg = synth.FULL
    n = 400_000
    g, og = grids(pkg, cfg)
    ctx = pkg.Context(cfg.radius_mm, cfg.axial_mm, g, cfg.tof_fwhm_ps)
    ev_np, bad = _with_invalid(to_np(synth.make_events(cfg, n, device="cuda")), np.random.default_rng(2))
    # events exactly on / next to the region boundaries
    zb = oracle.region_zbounds(og, 9)
    assert np.array_equal(ctx.region_zbounds(9).numpy(), zb)
    for j in range(1, 9):
        for d, i in ((-1, 3 * j), (0, 3 * j + 1), (1, 3 * j + 2)):
            z = zb[j] if d == 0 else np.nextafter(zb[j], np.float32(d * np.inf))
            ev_np["x1"][i], ev_np["y1"][i], ev_np["z1"][i] = -400.0, 0.0, z
            ev_np["x2"][i], ev_np["y2"][i], ev_np["z2"][i] = 400.0, 0.0, z
            ev_np["dt"][i] = 0.0
    ev = {k: torch.from_numpy(v).cuda() for k, v in ev_np.items()}
    region = torch.empty(n, dtype=torch.int32, device="cuda")
    perm = torch.empty(n, dtype=torch.int32, device="cuda")
    counts = ctx.split_regions(ev, n, 9, None, region, perm)
    want, wcounts = oracle.region_ids(ev_np, zb)
    assert np.array_equal(region.cpu().numpy(), want)
    assert np.array_equal(counts.numpy().astype(np.uint64), wcounts)
    assert counts.sum().item() == n - (want < 0).sum()
    p = perm.cpu().numpy().view(np.uint32).astype(np.int64)
    assert np.array_equal(np.sort(p), np.arange(n))
    grouped = want[p]
    grouped = np.where(grouped < 0, 9, grouped)
    assert np.all(np.diff(grouped) >= 0)
    # caller-supplied boundaries (3 regions)
    zb3 = torch.tensor([-1200.0, -100.0, 250.0, 1200.0])
    counts3 = ctx.split_regions(ev, n, 3, zb3, region, None)
    want3, wc3 = oracle.region_ids(ev_np, zb3.numpy())
    assert np.array_equal(region.cpu().numpy(), want3) and np.array_equal(counts3.numpy().astype(np.uint64), wc3)
    # region sub-grids (R12): margin 17 slices at 300 ps / 3.75 mm
    m = oracle.region_margin_slices(oracle.sigma_mm(300.0), 3.75)
    ks = oracle.default_region_slices(640, 9)
    for r in range(9):
        sub, z0, z1 = ctx.region_grid(9, None, r)
        assert z0 == max(0, ks[r] - (m if r > 0 else 0)) and z1 == min(640, ks[r + 1] + (m if r < 8 else 0))
        assert sub.nz == z1 - z0 and sub.oz == np.float32(-1200.0 + 3.75 * z0) and sub.nx == 160


def test_reconstruct_regions_parity(pkg):
    """cfg-4 pipeline on a small long-axis problem: split -> independent region reconstructions on sub-grids
    -> sum, against the same pipeline assembled from oracle calls."""
    R, iters = 3, 2
    nx, ny, nz, v = 16, 16, 96, 5.0
    n, m = 60_000, 600_000
    cfg = synth.Config("long", nx, ny, nz, v, 120.0, 480.0, synth.Phantom(
        parts=(synth.Shape("ellipsoid", (0.0, 0.0, 0.0), (30.0, 25.0, 220.0), 1.0),),
        inner=(synth.Shape("ellipsoid", (10.0, 0.0, 60.0), (8.0, 8.0, 8.0), 4.0),)), n, 0.2, 300.0, iters, m, 17)
    ev = synth.make_events(cfg, n, device="cuda")
    lors = synth.make_sens_lors(cfg, m, device="cuda")
    g, og = grids(pkg, cfg)
    ctx = pkg.Context(cfg.radius_mm, cfg.axial_mm, g, cfg.tof_fwhm_ps)
    sens = torch.empty(g.nvox, dtype=torch.float32, device="cuda")
    ctx.sensitivity(lors, m, sens)
    out = torch.empty(g.nvox, dtype=torch.float32, device="cuda")
    ctx.reconstruct_regions(ev, n, R, None, out, sens, iters)
    # oracle pipeline
    sig = oracle.sigma_mm(300.0)
    ev_np, sens_np = to_np(ev), sens.cpu().numpy()
    zb = oracle.region_zbounds(og, R)
    region, counts = oracle.region_ids(ev_np, zb)
    mask = oracle.mask_f32(sens_np)
    ks = oracle.default_region_slices(nz, R)
    mg = oracle.region_margin_slices(sig, v)
    total = np.zeros(g.nvox)
    sl = nx * ny
    for r in range(R):
        z0, z1 = max(0, ks[r] - (mg if r > 0 else 0)), min(nz, ks[r + 1] + (mg if r < R - 1 else 0))
        sg = oracle.make_grid(nx, ny, z1 - z0, v, origin=(og.ox, og.oy, og.oz + z0 * v))
        sel = region == r
        sub_ev = {k: a[sel] for k, a in ev_np.items()}
        x = mask[z0 * sl:z1 * sl].astype(np.float64)
        for _ in range(iters):
            corr, _, _ = oracle.em_correction(sg, sig, sub_ev, x)
            x = oracle.update(x, corr, sens_np[z0 * sl:z1 * sl], mask[z0 * sl:z1 * sl])
        total[z0 * sl:z1 * sl] += x
    check_image(out.cpu().numpy(), total)
    # the same through per-region plans (ray records + tiles, TOFMLEM_OPT_REGION_PLAN = 1; tile thresholds lowered so that
    # these small regions really run on tiles): the same image within the tolerance of the oracle comparison
    ctx.set_option(pkg.OPT_REGION_PLAN, 1)
    ctx.set_option(pkg.OPT_TILE_MIN_EVENTS, 64)
    ctx.set_option(pkg.OPT_TILE_MIN_ITEMS, 1)
    out2 = torch.empty(g.nvox, dtype=torch.float32, device="cuda")
    ctx.reconstruct_regions(ev, n, R, None, out2, sens, iters)
    check_image(out2.cpu().numpy(), total)
    assert float((out2 - out).double().norm() / out.double().norm()) <= 1e-4
    ctx.set_option(pkg.OPT_REGION_PLAN, 0)
    # unpinned (visual only): report how far the split result is from the unsplit one
    x = torch.from_numpy(mask.astype(np.float32)).cuda()
    ctx.iterate(ev, n, x, sens, iters)
    d = (out - x).double().norm() / x.double().norm()
    print(f"split-vs-unsplit rel-L2 = {d.item():.3e} (no threshold: parity unpinned)")


def test_split_regions_overlap_bit_exact(pkg):
    """Reading R27 / specification F3: region spans (lo, hi) of 400 k cfg-3 events incl. invalid ones bit-exact against
    oracle.region_spans; the lists hold every event once per region of its span."""
    cfg = synth.FULL
    n = 400_000
    g, og = grids(pkg, cfg)
    ctx = pkg.Context(cfg.radius_mm, cfg.axial_mm, g, cfg.tof_fwhm_ps)
    ev_np, bad = _with_invalid(to_np(synth.make_events(cfg, n, device="cuda")), np.random.default_rng(4))
    zb = oracle.region_zbounds(og, 9)
    ev = {k: torch.from_numpy(v).cuda() for k, v in ev_np.items()}
    span = torch.empty(n, dtype=torch.int32, device="cuda")
    perm = torch.empty(2 * n, dtype=torch.int32, device="cuda")
    counts = ctx.split_regions_overlap(ev, n, 9, None, span, perm)
    lo, hi, wcounts = oracle.region_spans(ev_np, zb, 3.0 * oracle.sigma_mm(cfg.tof_fwhm_ps))
    sp = span.cpu().numpy()
    want = np.where(lo < 0, -1, lo | (hi << 16))
    assert np.array_equal(sp, want)
    assert np.array_equal(counts.numpy().astype(np.uint64), wcounts)
    assert 0.2 * n < int((hi > lo).sum()) < 0.7 * n  # 115 mm windows on 240 mm cores: a good part spans two regions
    p = perm.cpu().numpy().view(np.uint32).astype(np.int64)
    off = 0
    for r in range(9):
        members = np.sort(p[off:off + int(wcounts[r])])
        assert np.array_equal(members, np.nonzero((lo <= r) & (r <= hi))[0])
        off += int(wcounts[r])
    # wider margins under this reading (twice the half-window + shell)
    ctx.set_option(pkg.OPT_REGION_OVERLAP, 1)
    m2 = int(np.ceil((2 * 3.0 * oracle.sigma_mm(300.0) + 6.0) / 3.75))
    ks = oracle.default_region_slices(640, 9)
    for r in (0, 4, 8):
        _, z0, z1 = ctx.region_grid(9, None, r)
        assert z0 == max(0, ks[r] - (m2 if r > 0 else 0)) and z1 == min(640, ks[r + 1] + (m2 if r < 8 else 0))


def test_reconstruct_regions_overlap_parity(pkg):
    """cfg-4 pipeline under reading R27 (an event in every region its window reaches, wide margins, cores only) against
    the same pipeline assembled from oracle calls; and how far each reading is from the unsplit reconstruction."""
    R, iters = 3, 2
    nx, ny, nz, v = 16, 16, 96, 5.0
    n, m = 60_000, 600_000
    cfg = synth.Config("long", nx, ny, nz, v, 120.0, 480.0, synth.Phantom(
        parts=(synth.Shape("ellipsoid", (0.0, 0.0, 0.0), (30.0, 25.0, 220.0), 1.0),),
        inner=(synth.Shape("ellipsoid", (10.0, 0.0, 60.0), (8.0, 8.0, 8.0), 4.0),)), n, 0.2, 300.0, iters, m, 17)
    ev = synth.make_events(cfg, n, device="cuda")
    lors = synth.make_sens_lors(cfg, m, device="cuda")
    g, og = grids(pkg, cfg)
    ctx = pkg.Context(cfg.radius_mm, cfg.axial_mm, g, cfg.tof_fwhm_ps)
    sens = torch.empty(g.nvox, dtype=torch.float32, device="cuda")
    ctx.sensitivity(lors, m, sens)
    single = torch.empty(g.nvox, dtype=torch.float32, device="cuda")
    ctx.reconstruct_regions(ev, n, R, None, single, sens, iters)
    ctx.set_option(pkg.OPT_REGION_OVERLAP, 1)
    out = torch.empty(g.nvox, dtype=torch.float32, device="cuda")
    ctx.reconstruct_regions(ev, n, R, None, out, sens, iters)
    out2 = torch.empty_like(out)
    ctx.reconstruct_regions(ev, n, R, None, out2, sens, iters)  # second call: cached sub-contexts
    assert float((out - out2).abs().max()) <= 1e-5 * float(out.max())
    # oracle pipeline
    sig = oracle.sigma_mm(300.0)
    ev_np, sens_np = to_np(ev), sens.cpu().numpy()
    zb = oracle.region_zbounds(og, R)
    lo, hi, counts = oracle.region_spans(ev_np, zb, 3.0 * sig)
    mask = oracle.mask_f32(sens_np)
    ks = oracle.default_region_slices(nz, R)
    mg = int(np.ceil((2 * 3.0 * sig + 6.0) / v))
    total = np.zeros(g.nvox)
    sl = nx * ny
    for r in range(R):
        z0, z1 = max(0, ks[r] - (mg if r > 0 else 0)), min(nz, ks[r + 1] + (mg if r < R - 1 else 0))
        sg = oracle.make_grid(nx, ny, z1 - z0, v, origin=(og.ox, og.oy, og.oz + z0 * v))
        sel = (lo <= r) & (r <= hi)
        sub_ev = {k: a[sel] for k, a in ev_np.items()}
        x = mask[z0 * sl:z1 * sl].astype(np.float64)
        for _ in range(iters):
            corr, _, _ = oracle.em_correction(sg, sig, sub_ev, x)
            x = oracle.update(x, corr, sens_np[z0 * sl:z1 * sl], mask[z0 * sl:z1 * sl])
        total[ks[r] * sl:ks[r + 1] * sl] = x[(ks[r] - z0) * sl:(ks[r + 1] - z0) * sl]  # the core only
    check_image(out.cpu().numpy(), total)
    # unpinned ("no difference to the whole-body reconstruction", visual only): report both readings
    x = torch.from_numpy(mask.astype(np.float32)).cuda()
    ctx.iterate(ev, n, x, sens, iters)
    d13 = float((single - x).double().norm() / x.double().norm())
    d27 = float((out - x).double().norm() / x.double().norm())
    print(f"split-vs-unsplit rel-L2: single assignment (R13) {d13:.3e}, overlapping membership (R27) {d27:.3e}")
    assert d27 < d13


def test_full_size_bench_configuration(pkg):
    """BASELINE.json cfg-3 at FULL size (146 M events, 160x160x640) in the launch configuration bench.py times
    (sub-binned permutation, persistent fused EM pass, update).  The oracle cannot run 146 M events, so:
      - sampled outputs it CAN compute one by one: forward values of every 146th event of the full set (1 M events), rel <= 1e-4;
      - properties that hold at any size: the binned pass and the unbinned pass give the same correction image up to
        the float32 summation order; sum(sens * x) = n_valid after the iteration (P7); n_valid = #{fwd > 0};
        the permutation is a bijection that sorts the keys."""
    cfg = synth.FULL
    n = cfg.n_events
    free, _ = torch.cuda.mem_get_info()
    if free < 40e9:
        pytest.skip("needs 40 GB of free device memory")
    g, og = grids(pkg, cfg)
    ctx = pkg.Context(cfg.radius_mm, cfg.axial_mm, g, cfg.tof_fwhm_ps)
    ev = synth.make_events_chunked(cfg, n, device="cuda")
    img = synth.random_image((g.nvox,), 41, device="cuda")
    # sampled forward values against the oracle
    fwd = torch.empty(n, dtype=torch.float32, device="cuda")
    ctx.forward(ev, n, img, fwd)
    sub = {k: v[::146].contiguous() for k, v in ev.items()}
    ref = oracle.forward(og, oracle.sigma_mm(cfg.tof_fwhm_ps), to_np(sub), img.cpu().numpy())
    assert ref.size == 1_000_000
    err = fwd_rel_err(fwd[::146].cpu().numpy(), ref)
    assert err.max() <= FWD_RTOL, err.max()
    n_pos = int((fwd > 0).sum().item())
    del fwd
    # unbinned pass (grid-order kernel on the raw order) vs binned pass (persistent kernel on the permuted set)
    corr_a = torch.zeros(g.nvox, dtype=torch.float32, device="cuda")
    ctx.set_option(pkg.OPT_EM_VARIANT, 1)
    ctx.reset_stats()
    ctx.em_correction(ev, n, img, corr_a)
    st_a = ctx.get_stats()
    key = torch.empty(n, dtype=torch.int32, device="cuda")
    perm = torch.empty(n, dtype=torch.int32, device="cuda")
    ctx.bin_events(ev, n, key, perm, None)
    sev = {k: torch.empty_like(v) for k, v in ev.items()}
    ctx.permute_events(ev, perm, n, sev)
    skey = key[perm.long()].view(torch.int32)  # sorted as unsigned: compare through int64
    sk = skey.long() & 0xFFFFFFFF
    assert bool((sk[1:] >= sk[:-1]).all())
    del ev, key, skey, sk
    seen = torch.zeros(n, dtype=torch.uint8, device="cuda")
    seen[perm.long()] = 1
    assert int(seen.sum().item()) == n  # a bijection
    del seen, perm
    ctx.set_option(pkg.OPT_EM_VARIANT, 0)
    corr_b = torch.zeros(g.nvox, dtype=torch.float32, device="cuda")
    ctx.reset_stats()
    ctx.em_correction(sev, n, img, corr_b)
    st_b = ctx.get_stats()
    assert st_a.n_valid == st_b.n_valid == n_pos and st_a.visits == st_b.visits
    d = (corr_a.double() - corr_b.double()).norm() / corr_a.double().norm()
    assert float(d) <= 1e-5, float(d)
    big = corr_a > 0.01 * corr_a.max()
    assert float(((corr_a - corr_b).abs()[big] / corr_a[big]).max()) <= 1e-3
    # tile mode (tofmlem_plan_events: what bench.py times): the same correction image again, most events through the
    # shared-memory tiles, far fewer reductions at L2
    plan = ctx.plan_events(sev, n)
    assert plan.active and plan.n_tile_events > 0.6 * n
    corr_c = torch.zeros(g.nvox, dtype=torch.float32, device="cuda")
    ctx.reset_stats()
    ctx.em_correction(sev, n, img, corr_c)
    st_c = ctx.get_stats()
    assert st_c.n_valid == n_pos and abs(int(st_c.visits) - int(st_a.visits)) <= 1e-5 * st_a.visits and st_c.tile_oob == 0
    assert st_c.tile_events > 0.6 * n_pos and st_c.reductions < 0.6 * st_b.reductions
    d = (corr_a.double() - corr_c.double()).norm() / corr_a.double().norm()
    assert float(d) <= 1e-5, float(d)
    assert float(((corr_a - corr_c).abs()[big] / corr_a[big]).max()) <= 1e-3
    del corr_c
    # P7 at full size: after the update sum(sens * x) = n_valid (sens = any positive image; mask = all voxels)
    sens = torch.full((g.nvox,), 0.25, dtype=torch.float32, device="cuda")
    ctx.update(img, corr_b, sens)
    p7 = float((img.double() * sens.double()).sum().item())
    # sum_j x_j corr_j = n_valid holds for the image the pass was run on: rel 1e-5 covers float32 products
    assert abs(p7 - st_b.n_valid) <= 1e-5 * st_b.n_valid, (p7, st_b.n_valid)
