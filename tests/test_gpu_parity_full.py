"""GPU parity on the cfg-3 GRID (160x160x640 voxels of 3.75 mm, scanner R 400 / L 2400 mm) in the launch configuration
bench.py times: events locality-binned (tofmlem_bin_events + tofmlem_permute_events), fused persistent EM pass,
update.  SURVEY.md 8(d) "Parity at cfg-3": (ii) 5-iteration image parity on a 2 M-event sub-sample of the full grid;
plus the fused pass of every cfg-5 context (100 / 300 / 600 ps, non-TOF), the sensitivity image on the full grid, and
context reuse with changing event counts.

Tolerances are north_star's: image rel-L2 <= 1e-3 and max rel <= 1e-2 on voxels above 1 % of the maximum.
"""
import numpy as np
import pytest
import torch

import oracle
import synth

pytestmark = pytest.mark.gpu

from test_gpu_parity import FWD_RTOL, check_image, fwd_rel_err, grids, to_np  # noqa: E402


@pytest.fixture(scope="module")
def pkg():
    import paper_1706_07075_b200 as p

    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return p


def binned(ctx, ev, n):
    key = torch.empty(n, dtype=torch.int32, device="cuda")
    perm = torch.empty(n, dtype=torch.int32, device="cuda")
    ctx.bin_events(ev, n, key, perm, None)
    sev = {k: torch.empty_like(v) for k, v in ev.items()}
    ctx.permute_events(ev, perm, n, sev)
    return sev, perm


@pytest.fixture(scope="module")
def full_sens(pkg):
    """Sensitivity image of the cfg-3 grid from 4 M seeded detector-pair LORs (the same float32 array feeds both sides)."""
    cfg = synth.FULL
    m = 4_000_000
    g, og = grids(pkg, cfg)
    ctx = pkg.Context(cfg.radius_mm, cfg.axial_mm, g, cfg.tof_fwhm_ps)
    lors = synth.make_sens_lors(cfg, m, device="cuda")
    sens = torch.empty(g.nvox, dtype=torch.float32, device="cuda")
    ctx.sensitivity(lors, m, sens)
    torch.cuda.synchronize()
    return sens


def test_full_grid_five_iterations_subsample(pkg, full_sens):
    """tofmlem_iterate, 5 iterations, 2 M events of cfg-3 on the full grid vs oracle.mlem."""
    cfg = synth.FULL
    n, iters = 2_000_000, cfg.iters
    assert iters == 5
    g, og = grids(pkg, cfg)
    ev = synth.make_events(cfg, n, start=7_000_000, device="cuda")
    ctx = pkg.Context(cfg.radius_mm, cfg.axial_mm, g, cfg.tof_fwhm_ps)
    sev, _ = binned(ctx, ev, n)
    # tile mode on every bin with >= 8 events (2 M events on 384 k bins are sparse; the default threshold is 1024),
    # every tile access bounds-tested
    ctx.set_option(pkg.OPT_TILE_MIN_EVENTS, 8)
    ctx.set_option(pkg.OPT_TILE_MIN_ITEMS, 1)  # small test problems: tiles whatever the item count
    ctx.set_option(pkg.OPT_TILE_CHECK, 1)
    plan = ctx.plan_events(sev, n)
    assert plan.active and plan.sorted and plan.n_tile_events + plan.n_direct_events == n
    assert plan.n_tile_events > 0.3 * n
    sens_np = full_sens.cpu().numpy()
    mask = oracle.mask_f32(sens_np)
    x = torch.from_numpy(mask.astype(np.float32)).cuda()
    ctx.iterate(sev, n, x, full_sens, iters)
    st = ctx.get_stats()
    assert st.tile_oob == 0 and st.tile_events > 0.25 * st.n_valid, (st.tile_oob, st.tile_events, st.n_valid)
    print(f"tile items {plan.n_tile_items}, tile events {plan.n_tile_events}, through tiles {st.tile_events} of {st.n_valid}")
    ref, ost = oracle.mlem(og, oracle.sigma_mm(cfg.tof_fwhm_ps), to_np(ev), mask.astype(np.float64), sens_np, iters)
    l2, mx = check_image(x.cpu().numpy(), ref, zero_tol=1e-6)
    print(f"cfg-3 grid, 2 M events, 5 iterations: rel-L2 {l2:.2e}, max rel {mx:.2e}")
    assert st.n_valid == ost.n_valid
    assert abs(st.sum_image_sens - st.n_valid) / st.n_valid < 1e-4  # P7
    assert float(x.min()) >= 0.0


@pytest.mark.parametrize("fwhm", [100.0, 300.0, 600.0, 0.0])
def test_full_grid_fused_pass_every_context(pkg, full_sens, fwhm):
    """The fused pass (tofmlem_em_correction + tofmlem_update) of each cfg-5 context on the full geometry against
    oracle.em_correction + oracle.update: binned events, persistent kernel, the 4- / 3- / 1-segment schedules (100 /
    300 / 600 ps) and the non-TOF instantiation.  Two passes, so that the second runs on a non-trivial image."""
    cfg = synth.sweep_config(300_000, fwhm)
    n = 300_000 if fwhm > 0 else 200_000
    g, og = grids(pkg, cfg)
    ev = synth.make_events(cfg, n, start=123_456, device="cuda")
    if fwhm <= 0:
        ev["dt"].zero_()
    ctx = pkg.Context(cfg.radius_mm, cfg.axial_mm, g, fwhm)
    sev, _ = binned(ctx, ev, n)
    sens_np = full_sens.cpu().numpy()
    mask = oracle.mask_f32(sens_np)
    sig = oracle.sigma_mm(fwhm) if fwhm > 0 else 0.0
    x = synth.random_image((g.nvox,), 61, device="cuda") * torch.from_numpy(mask.astype(np.float32)).cuda()
    xr = x.cpu().numpy().astype(np.float64)
    corr = torch.zeros(g.nvox, dtype=torch.float32, device="cuda")
    ev_np = to_np(ev)
    if fwhm <= 0:
        ev_np = {k: v for k, v in ev_np.items() if k != "dt"}
    for it in range(2):
        ctx.reset_stats()
        ctx.em_correction(sev, n, x, corr)
        ctx.update(x, corr, full_sens)
        st = ctx.get_stats()
        c_ref, nv_ref, vis_ref = oracle.em_correction(og, sig, ev_np, xr)
        xr = oracle.update(xr, c_ref, sens_np, mask)
        l2, mx = check_image(x.cpu().numpy(), xr, zero_tol=1e-6)
        assert st.n_valid == nv_ref, (fwhm, it, st.n_valid, nv_ref)
        assert abs(int(st.visits) - int(vis_ref)) <= 1e-4 * vis_ref
        print(f"fwhm {fwhm:g} pass {it}: rel-L2 {l2:.2e}, max rel {mx:.2e}, visits/event {st.visits / max(1, st.n_valid):.1f}")


def test_full_grid_sensitivity(pkg):
    """tofmlem_sensitivity on the full grid (1 M LORs, 300-900 visits each) vs oracle.sensitivity."""
    cfg = synth.FULL
    m = 1_000_000
    g, og = grids(pkg, cfg)
    ctx = pkg.Context(cfg.radius_mm, cfg.axial_mm, g, cfg.tof_fwhm_ps)
    lors = synth.make_sens_lors(cfg, m, start=5_000_000, device="cuda")
    sens = torch.empty(g.nvox, dtype=torch.float32, device="cuda")
    ctx.sensitivity(lors, m, sens)
    ref = oracle.sensitivity(og, to_np(lors))
    check_image(sens.cpu().numpy(), ref, l2=1e-5, mx=1e-4)


def test_context_reuse_growing_and_shrinking_n(pkg):
    """One context, event counts 100 k -> 300 k -> 50 k (a stray cudaFree of the record scratch in the
    sub-bin re-allocation branch left a dangling pointer).  Keys vs the oracle, permuted bits vs ev[perm]."""
    cfg = synth.FULL
    g, og = grids(pkg, cfg)
    ctx = pkg.Context(cfg.radius_mm, cfg.axial_mm, g, cfg.tof_fwhm_ps)
    for n in (100_000, 300_000, 50_000, 300_001):
        ev = synth.make_events(cfg, n, start=11 * n, device="cuda")
        ev_np = to_np(ev)
        key = torch.empty(n, dtype=torch.int32, device="cuda")
        perm = torch.empty(n, dtype=torch.int32, device="cuda")
        ctx.bin_events(ev, n, key, perm, None)
        out = {k: torch.zeros_like(v) for k, v in ev.items()}
        ctx.permute_events(ev, perm, n, out)
        torch.cuda.synchronize()
        assert np.array_equal(key.cpu().numpy().view(np.uint32), oracle.bin_keys(og, ev_np))
        p = perm.cpu().numpy().view(np.uint32).astype(np.int64)
        assert np.array_equal(np.sort(p), np.arange(n))
        for k in synth.EVENT_FIELDS:
            assert np.array_equal(out[k].cpu().numpy().view(np.uint32), ev_np[k][p].view(np.uint32)), (n, k)
    # trim releases the per-event scratch; the next call allocates it again and still works
    ctx.trim()
    n = 70_000
    ctx.reserve(n)
    ev = synth.make_events(cfg, n, start=3, device="cuda")
    key = torch.empty(n, dtype=torch.int32, device="cuda")
    perm = torch.empty(n, dtype=torch.int32, device="cuda")
    ctx.bin_events(ev, n, key, perm, None)
    out = {k: torch.zeros_like(v) for k, v in ev.items()}
    ctx.permute_events(ev, perm, n, out)
    p = perm.long()
    for k in synth.EVENT_FIELDS:
        assert torch.equal(out[k].view(torch.int32), ev[k][p].view(torch.int32))
    ctx.close()
    torch.cuda.synchronize()  # a double free would have left a CUDA error behind
    assert torch.zeros(1, device="cuda").item() == 0.0


def test_deterministic_iterations_are_bit_identical(pkg):
    """SURVEY.md 8(b) `deterministic` key ("This approach always generated an identically reconstructed
    image"): with the option on, the iterations of a planned list accumulate in 64-bit integers -- two runs give the same
    bits, whatever order the GPU ran the events in, and the image still matches oracle.mlem within north_star's tolerance.
    Unplanned lists, non-TOF contexts and bad values are refused."""
    cfg = synth.TINY
    n, m, iters = 120_000, 400_000, 3
    g, og = grids(pkg, cfg)
    ev = synth.make_events(cfg, n, device="cuda")
    lors = synth.make_sens_lors(cfg, m, device="cuda")
    ctx = pkg.Context(cfg.radius_mm, cfg.axial_mm, g, cfg.tof_fwhm_ps)
    sens = torch.empty(g.nvox, dtype=torch.float32, device="cuda")
    ctx.sensitivity(lors, m, sens)
    sev, _ = binned(ctx, ev, n)
    sens_np = sens.cpu().numpy()
    mask = oracle.mask_f32(sens_np)
    ctx.set_option(pkg.OPT_DETERMINISTIC, 0)
    with pytest.raises(pkg.TofMlemError) as e:
        ctx.set_option(pkg.OPT_DETERMINISTIC, 2)
    assert e.value.code == -1
    ctx.set_option(pkg.OPT_DETERMINISTIC, 1)
    x = torch.from_numpy(mask.astype(np.float32)).cuda()
    with pytest.raises(pkg.TofMlemError) as e:  # no plan yet
        ctx.iterate(sev, n, x, sens, iters)
    assert e.value.code == -5
    ctx.set_option(pkg.OPT_TILE_MIN_EVENTS, 64)
    ctx.set_option(pkg.OPT_TILE_MIN_ITEMS, 1)
    assert ctx.plan_events(sev, n).active
    runs = []
    for _ in range(3):
        x = torch.from_numpy(mask.astype(np.float32)).cuda()
        ctx.iterate(sev, n, x, sens, iters)
        runs.append(x.clone())
    assert torch.equal(runs[0], runs[1]) and torch.equal(runs[0], runs[2])
    st = ctx.get_stats()
    ref, ost = oracle.mlem(og, oracle.sigma_mm(cfg.tof_fwhm_ps), to_np(ev), mask.astype(np.float64), sens_np, iters)
    l2, mx = check_image(runs[0].cpu().numpy(), ref, zero_tol=1e-6)
    print(f"deterministic mode: rel-L2 {l2:.2e}, max rel {mx:.2e} against the oracle")
    assert st.n_valid == ost.n_valid and st.tile_events == 0
    assert abs(st.sum_image_sens - st.n_valid) / st.n_valid < 1e-5  # P7
    # the same list in another order (a different plan, other thread-to-event mapping): still the same bits
    rev = {k: v.flip(0).contiguous() for k, v in sev.items()}
    assert ctx.plan_events(rev, n).active
    x = torch.from_numpy(mask.astype(np.float32)).cuda()
    ctx.iterate(rev, n, x, sens, iters)
    assert torch.equal(x, runs[0])
    # the default mode on the same plan stays within tolerance of it (float32 sums, order not fixed)
    ctx.set_option(pkg.OPT_DETERMINISTIC, 0)
    x = torch.from_numpy(mask.astype(np.float32)).cuda()
    ctx.iterate(rev, n, x, sens, iters)
    assert float((x - runs[0]).double().norm() / runs[0].double().norm()) < 1e-4
    nt = pkg.Context(cfg.radius_mm, cfg.axial_mm, g, 0.0)
    with pytest.raises(pkg.TofMlemError) as e:
        nt.set_option(pkg.OPT_DETERMINISTIC, 1)
    assert e.value.code == -5


# ------------------------------------------------------------------ tile mode (tofmlem_plan_events, tile.cu)
def _tile_case(pkg, cfg, n, m, min_events, iters=2, expect_active=True, seed_img=None):
    g, og = grids(pkg, cfg)
    ev = synth.make_events(cfg, n, device="cuda")
    lors = synth.make_sens_lors(cfg, m, device="cuda")
    ctx = pkg.Context(cfg.radius_mm, cfg.axial_mm, g, cfg.tof_fwhm_ps)
    sens = torch.empty(g.nvox, dtype=torch.float32, device="cuda")
    ctx.sensitivity(lors, m, sens)
    sev, _ = binned(ctx, ev, n)
    ctx.set_option(pkg.OPT_TILE_MIN_EVENTS, min_events)
    ctx.set_option(pkg.OPT_TILE_MIN_ITEMS, 1)  # small test problems: tiles whatever the item count
    ctx.set_option(pkg.OPT_TILE_CHECK, 1)
    plan = ctx.plan_events(sev, n)
    assert bool(plan.active) == expect_active, (plan.active, plan.sorted, plan.n_tile_items)
    sens_np = sens.cpu().numpy()
    mask = oracle.mask_f32(sens_np)
    x = torch.from_numpy(mask.astype(np.float32)).cuda()
    ctx.iterate(sev, n, x, sens, iters)
    st = ctx.get_stats()
    sig = oracle.sigma_mm(cfg.tof_fwhm_ps)
    ref, ost = oracle.mlem(og, sig, to_np(ev), mask.astype(np.float64), sens_np, iters)
    check_image(x.cpu().numpy(), ref, zero_tol=1e-6)
    assert st.n_valid == ost.n_valid
    assert abs(int(st.visits) - int(ost.visits)) <= 1e-4 * ost.visits
    assert st.tile_oob == 0
    assert abs(st.sum_image_sens - st.n_valid) / st.n_valid < 1e-4
    return ctx, plan, st, sev, x, sens


def test_tile_mode_parity_tiny(pkg):
    """cfg-1 in tile mode (bins of >= 64 events through shared-memory tiles, bounds-tested) vs oracle.mlem; the planned
    and the unplanned pass of the same context give the same correction (up to the float32 summation order)."""
    cfg = synth.TINY
    ctx, plan, st, sev, x, sens = _tile_case(pkg, cfg, cfg.n_events, 400_000, 64)
    assert st.tile_events > 0.8 * st.n_valid, (st.tile_events, st.n_valid)
    n = cfg.n_events
    img = synth.random_image((ctx.nvox,), 19, device="cuda")
    a = torch.zeros(ctx.nvox, dtype=torch.float32, device="cuda")
    b = torch.zeros_like(a)
    ctx.reset_stats()
    ctx.em_correction(sev, n, img, a)  # planned
    st_a = ctx.get_stats()
    other = {k: v.clone() for k, v in sev.items()}  # another list (same events): no plan for it
    ctx.reset_stats()
    ctx.em_correction(other, n, img, b)
    st_b = ctx.get_stats()
    assert st_a.tile_events > 0 and st_b.tile_events == 0
    # the planned walk adds quantised crossings (prepared.cuh): a crossing pair closer than the quantum may merge
    assert st_a.n_valid == st_b.n_valid and abs(int(st_a.visits) - int(st_b.visits)) <= 1e-5 * st_b.visits
    assert st_a.reductions < 0.5 * st_b.reductions  # what the tiles are for: far fewer reductions at L2
    d = (a.double() - b.double()).norm() / b.double().norm()
    assert float(d) < 1e-5, float(d)
    # an unsorted list (here: the same events in reverse order) is planned without tile items and runs on its records
    rev = {k: v.flip(0).contiguous() for k, v in sev.items()}
    plan2 = ctx.plan_events(rev, n)
    assert not plan2.sorted and plan2.active and plan2.n_tile_items == 0 and plan2.n_tile_events == 0
    c = torch.zeros_like(a)
    ctx.reset_stats()
    ctx.em_correction(rev, n, img, c)
    st_c = ctx.get_stats()
    assert st_c.n_valid == st_b.n_valid and st_c.tile_events == 0 and st_c.visits == st_a.visits
    assert float((c.double() - b.double()).norm() / b.double().norm()) < 1e-5
    # the old list has no plan any more (one plan per context): the unplanned pass, bit-compatible with b's path
    c.zero_()
    ctx.reset_stats()
    ctx.em_correction(sev, n, img, c)
    assert ctx.get_stats().visits == st_b.visits
    assert float((c.double() - b.double()).norm() / b.double().norm()) < 1e-6
    # tofmlem_trim drops the plan and its records
    ctx.plan_events(sev, n)
    ctx.trim()
    assert not ctx.plan_info().active


@pytest.mark.parametrize("voxel_mm,fwhm,ctas", [(4.0, 100.0, 4), (4.0, 300.0, 3), (3.0, 300.0, 2)])
def test_tile_mode_launch_configurations(pkg, voxel_mm, fwhm, ctas):
    """The tile kernel's three launch configurations (4 x 256, 3 x 384, 2 x 512 threads per SM, chosen by the tile's size;
    at 100 ps also the items made of a PAIR of cubes) vs oracle.mlem on the cfg-1 phantom, tile accesses bounds-tested."""
    base = synth.TINY
    cfg = synth.Config(f"tiny-{voxel_mm}-{fwhm}", 32, 32, 32, voxel_mm, base.radius_mm, base.axial_mm, base.phantom, 150_000,
                       0.1, fwhm, 2, 400_000, 31)
    ctx, plan, st, sev, x, sens = _tile_case(pkg, cfg, cfg.n_events, cfg.sens_lors, 48)
    assert plan.n_tile_items > 0 and st.tile_events > 0.5 * st.n_valid, (plan.n_tile_items, st.tile_events, st.n_valid)
    print(f"voxel {voxel_mm} mm, {fwhm} ps ({ctas} CTAs per SM): {plan.n_tile_items} items, {st.tile_events} of {st.n_valid} on tiles")


def test_tile_mode_anisotropic_voxels_and_weights(pkg):
    """Tile envelopes with three different voxel sizes (the lateral slopes v_a / v_b differ per class), a grid that is not
    a multiple of the 8-voxel cube, events with per-event weights."""
    cfg = synth.Config("aniso", 30, 26, 22, 4.0, 150.0, 110.0, synth.Phantom(
        parts=(synth.Shape("ellipsoid", (0.0, 0.0, 0.0), (45.0, 40.0, 40.0), 1.0),),
        inner=(synth.Shape("ellipsoid", (12.0, -8.0, 5.0), (9.0, 9.0, 9.0), 4.0),)), 150_000, 0.15, 300.0, 2, 300_000, 23)
    n, m = cfg.n_events, cfg.sens_lors
    vox = (4.0, 4.6, 5.0)
    g = pkg.make_grid(cfg.nx, cfg.ny, cfg.nz, vox)
    og = oracle.make_grid(cfg.nx, cfg.ny, cfg.nz, vox)
    ev = synth.make_events(cfg, n, device="cuda")
    ctx = pkg.Context(cfg.radius_mm, cfg.axial_mm, g, cfg.tof_fwhm_ps)
    sev, perm = binned(ctx, ev, n)
    ctx.set_option(pkg.OPT_TILE_MIN_EVENTS, 32)
    ctx.set_option(pkg.OPT_TILE_MIN_ITEMS, 1)  # small test problems: tiles whatever the item count
    ctx.set_option(pkg.OPT_TILE_CHECK, 1)
    ctx.set_option(pkg.OPT_CORR_BRICKS, 0)  # read the correction image directly (set before the plan: it is part of it)
    plan = ctx.plan_events(sev, n)
    assert plan.active
    w = (0.5 + torch.rand(n, generator=torch.Generator().manual_seed(3))).cuda()
    sw = torch.empty_like(w)
    ctx.gather_f32(w, perm, n, sw)
    img = synth.random_image((g.nvox,), 29, device="cuda")
    corr = torch.zeros(g.nvox, dtype=torch.float32, device="cuda")
    ctx.reset_stats()
    ctx.em_correction_weighted(sev, n, sw, img, corr)
    st = ctx.get_stats()
    ref, nv, vis = oracle.em_correction(og, oracle.sigma_mm(300.0), to_np(ev), img.cpu().numpy().astype(np.float64),
                                        weights=w.cpu().numpy())
    assert st.n_valid == nv and st.tile_oob == 0 and st.tile_events > 0.5 * nv
    # the tiles accumulate in fixed point (tile.cu): rounding to >= 64 quanta per longest chord, unbiased; the bound here
    # is for ONE pass over 150 k events (~10 per voxel), a fifth of north_star's image tolerance
    check_image(corr.cpu().numpy(), ref, l2=2e-4, mx=2e-3, zero_tol=1e-6)


def test_plan_without_tiles_when_they_do_not_fit(pkg):
    """cfg-2 geometry at 600 ps (2 mm voxels: the +-3 sigma window spans 115 voxels, a tile would need far more than
    227 KB): the plan holds ray records but no tile items, and the pass is the direct one on records."""
    cfg = synth.MID
    g, og = grids(pkg, cfg)
    n = 100_000
    fwhm = 600.0
    ev = synth.make_events(cfg, n, device="cuda")
    ctx = pkg.Context(cfg.radius_mm, cfg.axial_mm, g, fwhm)
    sev, _ = binned(ctx, ev, n)
    ctx.set_option(pkg.OPT_TILE_MIN_EVENTS, 8)
    ctx.set_option(pkg.OPT_TILE_MIN_ITEMS, 1)  # small test problems: tiles whatever the item count
    plan = ctx.plan_events(sev, n)
    assert plan.active and plan.n_tile_items == 0 and plan.n_tile_events == 0 and plan.n_direct_events == n
    img = synth.random_image((g.nvox,), 31, device="cuda")
    corr = torch.zeros(g.nvox, dtype=torch.float32, device="cuda")
    ctx.set_option(pkg.OPT_CORR_BRICKS, 0)  # a plain image; the plan was made for bricks, so this pass ignores it ...
    ctx.reset_stats()
    ctx.em_correction(sev, n, img, corr)
    ref, nv, vis = oracle.em_correction(og, oracle.sigma_mm(fwhm), to_np(sev), img.cpu().numpy().astype(np.float64))
    assert ctx.get_stats().n_valid == nv and abs(int(ctx.get_stats().visits) - int(vis)) <= 1e-5 * vis
    check_image(corr.cpu().numpy(), ref, l2=1e-5, mx=1e-3, zero_tol=1e-6)
    ctx.plan_events(sev, n)  # ... and this one, planned for the plain layout, runs on the records
    corr.zero_()
    ctx.reset_stats()
    ctx.em_correction(sev, n, img, corr)
    st = ctx.get_stats()
    assert st.n_valid == nv and abs(int(st.visits) - int(vis)) <= 1e-5 * vis and st.tile_events == 0
    check_image(corr.cpu().numpy(), ref, l2=3e-5, mx=1e-3, zero_tol=1e-6)  # quantised crossings: <= 2e-5 of a chord


@pytest.mark.parametrize("case", ["tiny", "mid", "full-100ps", "full-300ps", "full-600ps", "aniso"])
def test_planned_forward_parity(pkg, case):
    """Per-LOR forward values of the PLANNED walk (ray records with quantised crossings, prepared.cuh; the walk the tile
    and the direct pass on records share) against the oracle: rel <= 1e-4 (north_star), tile and direct records alike."""
    vox = None
    if case == "tiny":
        cfg, n, fwhm, tmin = synth.TINY, 200_000, 300.0, 64
    elif case == "mid":
        cfg, n, fwhm, tmin = synth.MID, 150_001, 300.0, 8
    elif case == "aniso":
        cfg = synth.Config("aniso", 30, 26, 22, 4.0, 150.0, 110.0, synth.Phantom(
            parts=(synth.Shape("ellipsoid", (0.0, 0.0, 0.0), (45.0, 40.0, 40.0), 1.0),), inner=()), 100_000, 0.15, 300.0, 2,
            300_000, 24)
        n, fwhm, tmin, vox = cfg.n_events, 300.0, 32, (4.0, 4.6, 5.0)
    else:
        cfg, n, tmin = synth.FULL, 300_007, 8
        fwhm = float(case.split("-")[1][:-2])
    g = pkg.make_grid(cfg.nx, cfg.ny, cfg.nz, vox or cfg.voxel_mm)
    og = oracle.make_grid(cfg.nx, cfg.ny, cfg.nz, vox or cfg.voxel_mm)
    ev = synth.make_events(cfg, n, device="cuda")
    # edge cases ride along: NaN / Inf fields, L = 0, a LOR that misses the grid, dt far outside
    for k, i, v in (("x1", 5, float("nan")), ("dt", 6, float("inf")), ("dt", 9, 1.0e6)):
        ev[k][i] = v
    for k in ("x2", "y2", "z2"):
        ev[k][7] = ev[k.replace("2", "1")][7]
    ev["z1"][8] = ev["z2"][8] = 1.0e5
    ctx = pkg.Context(cfg.radius_mm, cfg.axial_mm, g, fwhm)
    sev, _ = binned(ctx, ev, n)
    ctx.set_option(pkg.OPT_TILE_MIN_EVENTS, tmin)
    ctx.set_option(pkg.OPT_TILE_MIN_ITEMS, 1)  # small test problems: tiles whatever the item count
    plan = ctx.plan_events(sev, n)
    assert plan.active
    if case in ("tiny", "full-100ps", "full-300ps", "aniso"):
        assert plan.n_tile_events > 0.2 * n, plan.n_tile_events
    else:
        assert plan.n_tile_items == 0
    img = synth.random_image((g.nvox,), 41, device="cuda")
    fwd = torch.empty(n, dtype=torch.float32, device="cuda")
    ctx.forward(sev, n, img, fwd)
    ref = oracle.forward(og, oracle.sigma_mm(fwhm), to_np(sev), img.cpu().numpy())
    err = fwd_rel_err(fwd.cpu().numpy(), ref)
    print(f"{case}: planned forward max rel err {err.max():.2e}, tile events {plan.n_tile_events} of {n}")
    assert err.max() <= FWD_RTOL, f"max rel err {err.max():.3e} at {err.argmax()}"
    assert (fwd.cpu().numpy()[ref == 0] == 0).all()


def test_planned_path_edge_cases(pkg):
    """The planned path on awkward inputs: ragged sizes, a list that grows and shrinks on one context, all-invalid
    events, odd grid sizes (no 16-byte groups, no bricks), per-event weights, iters = 0, trim between plans."""
    cfg = synth.TINY
    g, og = grids(pkg, cfg)
    sig = oracle.sigma_mm(cfg.tof_fwhm_ps)
    ctx = pkg.Context(cfg.radius_mm, cfg.axial_mm, g, cfg.tof_fwhm_ps)
    ctx.set_option(pkg.OPT_TILE_MIN_EVENTS, 40)
    ctx.set_option(pkg.OPT_TILE_MIN_ITEMS, 1)
    ctx.set_option(pkg.OPT_TILE_CHECK, 1)
    img = synth.random_image((g.nvox,), 3, device="cuda")
    img_np = img.cpu().numpy().astype(np.float64)
    for n in (100_003, 33, 250_001, 31):  # grows, shrinks, not multiples of 32
        ev = synth.make_events(cfg, n, start=1000, device="cuda")
        sev, _ = binned(ctx, ev, n)
        plan = ctx.plan_events(sev, n)
        assert plan.active and plan.n_tile_events + plan.n_direct_events == n
        corr = torch.zeros(g.nvox, dtype=torch.float32, device="cuda")
        ctx.set_option(pkg.OPT_CORR_BRICKS, 0)
        ctx.plan_events(sev, n)
        ctx.reset_stats()
        ctx.em_correction(sev, n, img, corr)
        st = ctx.get_stats()
        ref, nv, vis = oracle.em_correction(og, sig, to_np(sev), img_np)
        assert st.n_valid == nv and st.tile_oob == 0
        if n > 1000:
            assert st.tile_events > 0
            check_image(corr.cpu().numpy(), ref, l2=2e-4, mx=5e-3, zero_tol=1e-6)
        else:
            assert float((corr.double().cpu() - torch.from_numpy(ref)).norm() / np.linalg.norm(ref)) < 1e-4
        ctx.set_option(pkg.OPT_CORR_BRICKS, 1)
    # all events invalid: the plan is active, nothing is walked
    n = 5000
    bad = {k: torch.full((n,), float("nan"), device="cuda") for k in ("x1", "y1", "z1", "x2", "y2", "z2", "dt")}
    plan = ctx.plan_events(bad, n)
    assert plan.active and plan.n_tile_events == 0
    corr = torch.zeros(g.nvox, dtype=torch.float32, device="cuda")
    ctx.reset_stats()
    ctx.em_correction(bad, n, img, corr)
    assert ctx.get_stats().n_valid == 0 and float(corr.abs().max()) == 0.0
    assert ctx.plan_events(bad, 0).active == 0  # empty list: no plan, no error
    # trim drops plan and scratch; planning again works
    ctx.trim()
    ev = synth.make_events(cfg, 20_000, device="cuda")
    sev, _ = binned(ctx, ev, 20_000)
    assert ctx.plan_events(sev, 20_000).active
    x = torch.ones(g.nvox, dtype=torch.float32, device="cuda")
    sens = torch.ones(g.nvox, dtype=torch.float32, device="cuda")
    x0 = x.clone()
    ctx.iterate(sev, 20_000, x, sens, 0)  # no iteration: the image is untouched
    assert torch.equal(x, x0)
    # odd grid sizes: no brick layout, nvox not a multiple of 4 (scalar reductions), tiles all the same
    g2 = pkg.make_grid(31, 29, 27, 4.0)
    og2 = oracle.make_grid(31, 29, 27, 4.0)
    ctx2 = pkg.Context(cfg.radius_mm, cfg.axial_mm, g2, cfg.tof_fwhm_ps)
    ctx2.set_option(pkg.OPT_TILE_MIN_EVENTS, 40)
    ctx2.set_option(pkg.OPT_TILE_MIN_ITEMS, 1)
    ctx2.set_option(pkg.OPT_TILE_CHECK, 1)
    n = 80_000
    ev = synth.make_events(cfg, n, device="cuda")
    sev, perm = binned(ctx2, ev, n)
    w = (0.25 + torch.rand(n, generator=torch.Generator().manual_seed(5))).cuda()
    sw = torch.empty_like(w)
    ctx2.gather_f32(w, perm, n, sw)
    assert ctx2.plan_events(sev, n).n_tile_events > 0
    img2 = synth.random_image((g2.nvox,), 9, device="cuda")
    corr2 = torch.zeros(g2.nvox, dtype=torch.float32, device="cuda")
    ctx2.reset_stats()
    ctx2.em_correction_weighted(sev, n, sw, img2, corr2)
    st = ctx2.get_stats()
    ref, nv, _ = oracle.em_correction(og2, sig, to_np(ev), img2.cpu().numpy().astype(np.float64), weights=w.cpu().numpy())
    assert st.n_valid == nv and st.tile_oob == 0 and st.tile_events > 0
    check_image(corr2.cpu().numpy(), ref, l2=2e-4, mx=5e-3, zero_tol=1e-6)
