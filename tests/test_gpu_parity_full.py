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

from test_gpu_parity import check_image, grids, to_np  # noqa: E402


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
    if hasattr(ctx, "plan_events"):
        ctx.plan_events(sev, n)
    sens_np = full_sens.cpu().numpy()
    mask = oracle.mask_f32(sens_np)
    x = torch.from_numpy(mask.astype(np.float32)).cuda()
    ctx.iterate(sev, n, x, full_sens, iters)
    st = ctx.get_stats()
    ref, ost = oracle.mlem(og, oracle.sigma_mm(cfg.tof_fwhm_ps), to_np(ev), mask.astype(np.float64), sens_np, iters)
    l2, mx = check_image(x.cpu().numpy(), ref)
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
    if hasattr(ctx, "plan_events"):
        ctx.plan_events(sev, n)
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
        l2, mx = check_image(x.cpu().numpy(), xr)
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


def test_deterministic_option_is_declared_and_refused(pkg):
    """SURVEY.md 8(b) lists a `deterministic` key.  It exists; 0 is accepted, 1 is refused with
    TOFMLEM_EUNSUPPORTED (float32 reductions are unordered)."""
    cfg = synth.TINY
    g, _ = grids(pkg, cfg)
    ctx = pkg.Context(cfg.radius_mm, cfg.axial_mm, g, cfg.tof_fwhm_ps)
    ctx.set_option(pkg.OPT_DETERMINISTIC, 0)
    with pytest.raises(pkg.TofMlemError) as e:
        ctx.set_option(pkg.OPT_DETERMINISTIC, 1)
    assert e.value.code == -5
    with pytest.raises(pkg.TofMlemError) as e:
        ctx.set_option(pkg.OPT_DETERMINISTIC, 2)
    assert e.value.code == -1
