"""GPU parity of the widened rows: K-sample TOF kernel (NEXT-1), 3x3x3 median filter (NEXT-2),
per-event attenuation weights (NEXT-3), TOF scatter rejection (NEXT-4), and of the sub-bin ordering of
tofmlem_bin_events.  CUDA path through the C-ABI binding against the fp64 oracle on the same seeded inputs.

Tolerances: forward values rel <= 1e-4 and images rel-L2 <= 1e-3 / max rel <= 1e-2 (north_star);
attenuation weights rel <= 1e-4 * max(1, ln w) (the forward tolerance carried through exp); the median
filter, the keep flags and the bin membership are bit-exact.
"""
import numpy as np
import pytest
import torch

import oracle
import synth

pytestmark = pytest.mark.gpu

from test_gpu_parity import check_image, fwd_rel_err, grids, to_np  # noqa: E402


@pytest.fixture(scope="module")
def pkg():
    import paper_1706_07075_b200 as p

    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return p


@pytest.fixture(scope="module")
def tiny(pkg):
    cfg = synth.TINY
    n = 60_000
    ev = synth.make_events(cfg, n, device="cuda")
    g, og = grids(pkg, cfg)
    lors = synth.make_sens_lors(cfg, 400_000, device="cuda")
    ctx = pkg.Context(cfg.radius_mm, cfg.axial_mm, g, cfg.tof_fwhm_ps)
    sens = torch.empty(g.nvox, dtype=torch.float32, device="cuda")
    ctx.sensitivity(lors, 400_000, sens)
    torch.cuda.synchronize()
    return cfg, n, ev, to_np(ev), g, og, sens


# ------------------------------------------------------------------ NEXT-1: K-sample kernel
@pytest.mark.parametrize("K", [32, 15, 1])
def test_sampled_forward_backproject_parity(pkg, tiny, K):
    cfg, n, ev, ev_np, g, og, sens = tiny
    ctx = pkg.Context(cfg.radius_mm, cfg.axial_mm, g, cfg.tof_fwhm_ps)
    ctx.set_option(pkg.OPT_SAMPLES_K, K)
    ctx.set_option(pkg.OPT_PROJECTOR, pkg.PROJECTOR_SAMPLED)
    sig = oracle.sigma_mm(cfg.tof_fwhm_ps)
    img = synth.random_image((g.nvox,), 77, device="cuda")
    fwd = torch.empty(n, dtype=torch.float32, device="cuda")
    ctx.forward(ev, n, img, fwd)
    ref = oracle.forward(og, sig, ev_np, img.cpu().numpy(), K=K)
    err = fwd_rel_err(fwd.cpu().numpy(), ref)
    assert err.max() <= 1e-4, err.max()
    assert np.all(fwd.cpu().numpy()[ref == 0] == 0)
    vals = (0.5 + torch.rand(n, generator=torch.Generator().manual_seed(5))).cuda()
    out = torch.zeros(g.nvox, dtype=torch.float32, device="cuda")
    ctx.backproject(ev, n, vals, out)
    refb = oracle.backproject(og, sig, ev_np, vals.cpu().numpy(), K=K)
    check_image(out.cpu().numpy(), refb)


def test_sampled_iterate_parity(pkg, tiny):
    cfg, n, ev, ev_np, g, og, sens = tiny
    ctx = pkg.Context(cfg.radius_mm, cfg.axial_mm, g, cfg.tof_fwhm_ps)
    ctx.set_option(pkg.OPT_PROJECTOR, pkg.PROJECTOR_SAMPLED)  # K = 32, the paper's GPU value
    sens_np = sens.cpu().numpy()
    mask = oracle.mask_f32(sens_np)
    img = torch.from_numpy(mask.astype(np.float32)).cuda()
    ctx.iterate(ev, n, img, sens, 2)
    st = ctx.get_stats()
    ref, ost = oracle.mlem(og, oracle.sigma_mm(cfg.tof_fwhm_ps), ev_np, mask.astype(np.float64), sens_np, 2, K=32)
    check_image(img.cpu().numpy(), ref)
    assert st.n_valid == ost.n_valid and st.visits == ost.visits
    assert 0 < st.reductions <= st.visits
    # a non-TOF context has no TOF kernel to sample
    nt = pkg.Context(cfg.radius_mm, cfg.axial_mm, g, 0.0)
    with pytest.raises(pkg.TofMlemError):
        nt.set_option(pkg.OPT_PROJECTOR, pkg.PROJECTOR_SAMPLED)


def test_sampled_full_geometry_forward(pkg):
    """cfg-3 geometry (coordinates up to +-1200 mm, 3.75 mm voxels): the fp64 voxel decision must agree."""
    cfg = synth.FULL
    n = 200_000
    ev = synth.make_events(cfg, n, device="cuda")
    g, og = grids(pkg, cfg)
    ctx = pkg.Context(cfg.radius_mm, cfg.axial_mm, g, cfg.tof_fwhm_ps)
    ctx.set_option(pkg.OPT_PROJECTOR, pkg.PROJECTOR_SAMPLED)
    img = synth.random_image((g.nvox,), 9, device="cuda")
    fwd = torch.empty(n, dtype=torch.float32, device="cuda")
    ctx.forward(ev, n, img, fwd)
    ref = oracle.forward(og, oracle.sigma_mm(cfg.tof_fwhm_ps), to_np(ev), img.cpu().numpy(), K=32)
    assert fwd_rel_err(fwd.cpu().numpy(), ref).max() <= 1e-4


# ------------------------------------------------------------------ NEXT-2: median filter
@pytest.mark.parametrize("shape", [(32, 32, 32), (37, 19, 11), (1, 1, 1), (5, 1, 3), (160, 160, 24)])
def test_median3_bit_exact(pkg, shape):
    nx, ny, nz = shape
    g = pkg.make_grid(nx, ny, nz, 2.0)
    og = oracle.make_grid(nx, ny, nz, 2.0)
    ctx = pkg.Context(200.0, 100.0, g, 300.0)
    img = synth.random_image((g.nvox,), 3, device="cuda")
    img[torch.rand(g.nvox, device="cuda") < 0.3] = 0.0  # ties
    out = torch.empty_like(img)
    ctx.median3(img, out)
    ref = oracle.median3(og, img.cpu().numpy())
    assert np.array_equal(out.cpu().numpy().astype(np.float64), ref)
    with pytest.raises(pkg.TofMlemError):
        ctx.median3(img, img)


def test_iterate_with_median_parity(pkg, tiny):
    cfg, n, ev, ev_np, g, og, sens = tiny
    ctx = pkg.Context(cfg.radius_mm, cfg.axial_mm, g, cfg.tof_fwhm_ps)
    ctx.set_option(pkg.OPT_MEDIAN, 1)
    sens_np = sens.cpu().numpy()
    mask = oracle.mask_f32(sens_np)
    img = torch.from_numpy(mask.astype(np.float32)).cuda()
    ctx.iterate(ev, n, img, sens, 3)
    ref, _ = oracle.mlem(og, oracle.sigma_mm(cfg.tof_fwhm_ps), ev_np, mask.astype(np.float64), sens_np, 3, median=True)
    # a median can pick a different neighbour when two candidates differ by rounding only: same tolerance as images
    gpu = img.cpu().numpy().astype(np.float64)
    rel_l2 = np.linalg.norm(gpu - ref) / np.linalg.norm(ref)
    big = ref > 0.01 * ref.max()
    assert rel_l2 <= 1e-3 and np.max(np.abs(gpu[big] - ref[big]) / ref[big]) <= 1e-2


# ------------------------------------------------------------------ NEXT-3: attenuation weights
def test_attenuation_weights_and_weighted_iterate(pkg):
    cfg = synth.MID
    n = 150_000
    ev = synth.make_events(cfg, n, device="cuda")
    ev_np = to_np(ev)
    g, og = grids(pkg, cfg)
    ctx = pkg.Context(cfg.radius_mm, cfg.axial_mm, g, cfg.tof_fwhm_ps)
    mu = synth.rasterize_mu_map(cfg, device="cuda").reshape(-1).contiguous()
    w = torch.empty(n, dtype=torch.float32, device="cuda")
    ctx.attenuation_weights(ev, n, mu, w)
    ref_w = oracle.attenuation_weights(og, ev_np, mu.cpu().numpy())
    got = w.cpu().numpy().astype(np.float64)
    assert ref_w.max() > 5.0  # the torso attenuates: weights well above 1
    assert np.max(np.abs(got - ref_w) / (ref_w * np.maximum(1.0, np.log(ref_w)))) <= 1e-4
    # weighted EM pass and iterations, the float32 weights fed to both sides
    m = 600_000
    lors = synth.make_sens_lors(cfg, m, device="cuda")
    sens = torch.empty(g.nvox, dtype=torch.float32, device="cuda")
    ctx.sensitivity(lors, m, sens)
    sens_np = sens.cpu().numpy()
    mask = oracle.mask_f32(sens_np)
    img = torch.from_numpy(mask.astype(np.float32)).cuda()
    ctx.iterate_weighted(ev, n, w, img, sens, 2)
    st = ctx.get_stats()
    ref, ost = oracle.mlem(og, oracle.sigma_mm(cfg.tof_fwhm_ps), ev_np, mask.astype(np.float64), sens_np, 2,
                           weights=w.cpu().numpy())
    check_image(img.cpu().numpy(), ref)
    assert st.n_valid == ost.n_valid
    # weights survive the locality permutation: bin, gather events and weights, same image
    key = torch.empty(n, dtype=torch.int32, device="cuda")
    perm = torch.empty(n, dtype=torch.int32, device="cuda")
    ctx.bin_events(ev, n, key, perm, None)
    sev = {k: torch.empty_like(v) for k, v in ev.items()}
    ctx.permute_events(ev, perm, n, sev)
    sw = torch.empty_like(w)
    ctx.gather_f32(w, perm, n, sw)
    img2 = torch.from_numpy(mask.astype(np.float32)).cuda()
    ctx.iterate_weighted(sev, n, sw, img2, sens, 2)
    check_image(img2.cpu().numpy(), ref)


# ------------------------------------------------------------------ NEXT-4: scatter rejection
@pytest.mark.parametrize("cfg_name,n", [("full", 400_003), ("mid", 100_000)])
def test_scatter_reject_bit_exact(pkg, cfg_name, n):
    cfg = synth.CONFIGS[cfg_name]
    ev = synth.make_events(cfg, n, device="cuda")
    ev_np = to_np(ev)
    # invalid events must be rejected
    for k, i, v in (("x1", 5, np.nan), ("dt", 17, np.inf)):
        ev[k][i] = v
        ev_np[k][i] = v
    for k in ("x2", "y2", "z2"):
        ev[k][29] = ev[k.replace("2", "1")][29]
        ev_np[k][29] = ev_np[k.replace("2", "1")][29]
    g, og = grids(pkg, cfg)
    ctx = pkg.Context(cfg.radius_mm, cfg.axial_mm, g, cfg.tof_fwhm_ps)
    ell = oracle.ellipsoids_f32(synth.body_outline(cfg))
    h = oracle.scatter_half_width_f32(oracle.sigma_mm(cfg.tof_fwhm_ps))
    keep = torch.empty(n, dtype=torch.uint8, device="cuda")
    perm = torch.empty(n, dtype=torch.int32, device="cuda")
    kept = ctx.scatter_reject(ev, n, torch.from_numpy(ell), float(h), keep, perm)
    ref_keep, ref_cnt = oracle.scatter_keep(ev_np, ell, h)
    assert kept == ref_cnt
    assert np.array_equal(keep.cpu().numpy(), ref_keep)
    assert not ref_keep[[5, 17, 29]].any()
    got_idx = np.sort(perm[:kept].cpu().numpy().astype(np.int64))
    assert np.array_equal(got_idx, np.nonzero(ref_keep)[0])
    # compaction: gather_events takes the kept indices (a subset whose indices exceed the output length)
    out = {k: torch.empty(kept, dtype=torch.float32, device="cuda") for k in ev}
    ctx.gather_events(ev, perm, kept, out)
    order = perm[:kept].cpu().numpy().astype(np.int64)
    for k in synth.EVENT_FIELDS:
        assert np.array_equal(out[k].cpu().numpy().view(np.uint32), ev_np[k][order].view(np.uint32))
    # default half width (<= 0) = 1.959964 sigma rounded to float32: the same flags
    keep2 = torch.empty_like(keep)
    assert ctx.scatter_reject(ev, n, torch.from_numpy(ell), 0.0, keep2, None) == ref_cnt
    assert torch.equal(keep, keep2)


# ------------------------------------------------------------------ sub-bin ordering of tofmlem_bin_events
@pytest.mark.parametrize("subbins", [1, 16, 64])
def test_subbins_keep_keys_offsets_membership(pkg, subbins):
    cfg = synth.FULL
    n = 300_000
    ev = synth.make_events(cfg, n, device="cuda")
    ev["dt"][11] = float("nan")
    ev_np = to_np(ev)
    g, og = grids(pkg, cfg)
    ctx = pkg.Context(cfg.radius_mm, cfg.axial_mm, g, cfg.tof_fwhm_ps)
    ctx.set_option(pkg.OPT_SUBBINS, subbins)
    nb = ctx.num_bins()
    key = torch.empty(n, dtype=torch.int32, device="cuda")
    perm = torch.empty(n, dtype=torch.int32, device="cuda")
    offs = torch.empty(nb + 1, dtype=torch.int32, device="cuda")
    ctx.bin_events(ev, n, key, perm, offs)
    ref_key = oracle.bin_keys(og, ev_np)
    k = key.cpu().numpy().view(np.uint32)
    assert np.array_equal(k, ref_key)
    p = perm.cpu().numpy().view(np.uint32).astype(np.int64)
    assert np.array_equal(np.sort(p), np.arange(n))  # a permutation
    sorted_keys = ref_key[p]
    assert np.all(np.diff(sorted_keys.astype(np.int64)) >= 0)  # sorted by key, invalid (0xFFFFFFFF) last
    ref_offs = np.searchsorted(sorted_keys, np.arange(nb + 1, dtype=np.uint64), side="left")
    assert np.array_equal(offs.cpu().numpy().view(np.uint32).astype(np.int64), ref_offs)


# ------------------------------------------------------------------ scheduling variants of the fused EM pass
@pytest.mark.parametrize("variant", [0, 1, 2])
def test_em_variants_parity(pkg, tiny, variant):
    """TOFMLEM_OPT_EM_VARIANT changes scheduling / accumulation only: same image within the north_star tolerance."""
    cfg, n, ev, ev_np, g, og, sens = tiny
    ctx = pkg.Context(cfg.radius_mm, cfg.axial_mm, g, cfg.tof_fwhm_ps)
    ctx.set_option(pkg.OPT_EM_VARIANT, variant)
    sens_np = sens.cpu().numpy()
    mask = oracle.mask_f32(sens_np)
    img = torch.from_numpy(mask.astype(np.float32)).cuda()
    ctx.iterate(ev, n, img, sens, 2)
    st = ctx.get_stats()
    ref, ost = oracle.mlem(og, oracle.sigma_mm(cfg.tof_fwhm_ps), ev_np, mask.astype(np.float64), sens_np, 2)
    check_image(img.cpu().numpy(), ref)
    assert st.n_valid == ost.n_valid and st.visits == ost.visits
    assert abs(st.sum_image_sens - st.n_valid) <= 1e-4 * st.n_valid  # P7


# ------------------------------------------------------------------ layout of the correction image
def test_correction_layouts(pkg, tiny):
    """TOFMLEM_OPT_CORR_BRICKS: with 0 the correction image of tofmlem_em_correction is a plain image and matches the
    oracle's element by element; with 1 (default) it is in the context's internal order, the same multiset of values,
    and em_correction + update gives the same image either way (and the same as the oracle)."""
    cfg, n, ev, ev_np, g, og, sens = tiny
    sig = oracle.sigma_mm(cfg.tof_fwhm_ps)
    x = synth.random_image((g.nvox,), 13, device="cuda")
    ref_corr, nv, _ = oracle.em_correction(og, sig, ev_np, x.cpu().numpy())
    sens_np = sens.cpu().numpy()
    ref_img = oracle.update(x.cpu().numpy().astype(np.float64), ref_corr, sens_np, oracle.mask_f32(sens_np))
    images = {}
    for bricks in (0, 1):
        ctx = pkg.Context(cfg.radius_mm, cfg.axial_mm, g, cfg.tof_fwhm_ps)
        ctx.set_option(pkg.OPT_CORR_BRICKS, bricks)
        corr = torch.zeros(g.nvox, dtype=torch.float32, device="cuda")
        ctx.em_correction(ev, n, x, corr)
        c = corr.cpu().numpy().astype(np.float64)
        if bricks == 0:
            check_image(c, ref_corr)
        else:
            # 2x2x1 bricks: value of voxel (x, y, z) sits at ((z*ny/2 + y/2)*nx/2 + x/2)*4 + (y&1)*2 + (x&1)
            lin = c.reshape(g.nz, g.ny // 2, g.nx // 2, 2, 2).transpose(0, 1, 3, 2, 4).reshape(-1)
            check_image(lin, ref_corr)
        img = x.clone()
        ctx.update(img, corr, sens)
        assert not corr.any()  # zeroed for the next pass
        images[bricks] = img.cpu().numpy()
        check_image(images[bricks], ref_img)
    assert np.allclose(images[0], images[1], rtol=1e-4, atol=0)


# ------------------------------------------------------------------ the paper's whole chain (Table 2)
def test_paper_pipeline_parity(pkg):
    """Pre-processing (TOF scatter rejection, attenuation weights), starting backprojection as x0,
    then MLEM iterations with the per-event weights and the median filter after each iteration,
    on locality-binned events: the CUDA chain against the same chain of oracle calls."""
    cfg = synth.MID
    n, m, iters = 120_000, 500_000, 3
    ev = synth.make_events(cfg, n, device="cuda")
    ev_np = to_np(ev)
    g, og = grids(pkg, cfg)
    sig = oracle.sigma_mm(cfg.tof_fwhm_ps)
    ctx = pkg.Context(cfg.radius_mm, cfg.axial_mm, g, cfg.tof_fwhm_ps)
    ctx.set_option(pkg.OPT_MEDIAN, 1)
    # 1. scatter rejection against the body outline, compaction
    ell = oracle.ellipsoids_f32(synth.body_outline(cfg))
    h = oracle.scatter_half_width_f32(sig)
    keep = torch.empty(n, dtype=torch.uint8, device="cuda")
    perm = torch.empty(n, dtype=torch.int32, device="cuda")
    kept = ctx.scatter_reject(ev, n, torch.from_numpy(ell), float(h), keep, perm)
    ref_keep, ref_cnt = oracle.scatter_keep(ev_np, ell, h)
    assert kept == ref_cnt and np.array_equal(keep.cpu().numpy(), ref_keep)
    kev = {k: torch.empty(kept, dtype=torch.float32, device="cuda") for k in ev}
    ctx.gather_events(ev, perm, kept, kev)
    kev_np = to_np(kev)  # the oracle works on the same compacted order
    # 2. attenuation weights
    mu = synth.rasterize_mu_map(cfg, device="cuda").reshape(-1).contiguous()
    w = torch.empty(kept, dtype=torch.float32, device="cuda")
    ctx.attenuation_weights(kev, kept, mu, w)
    # 3. sensitivity, 4. starting backprojection
    lors = synth.make_sens_lors(cfg, m, device="cuda")
    sens = torch.empty(g.nvox, dtype=torch.float32, device="cuda")
    ctx.sensitivity(lors, m, sens)
    x0 = torch.zeros(g.nvox, dtype=torch.float32, device="cuda")
    ctx.backproject(kev, kept, None, x0)
    ref_x0 = oracle.backproject(og, sig, kev_np)
    check_image(x0.cpu().numpy(), ref_x0)
    # 5. locality binning of events and weights, 6. iterations
    key = torch.empty(kept, dtype=torch.int32, device="cuda")
    bperm = torch.empty(kept, dtype=torch.int32, device="cuda")
    ctx.bin_events(kev, kept, key, bperm, None)
    sev = {k: torch.empty_like(v) for k, v in kev.items()}
    ctx.permute_events(kev, bperm, kept, sev)
    sw = torch.empty_like(w)
    ctx.gather_f32(w, bperm, kept, sw)
    img = x0.clone()
    ctx.iterate_weighted(sev, kept, sw, img, sens, iters)
    # the oracle chain starts from the SAME float32 x0, weights and sensitivity (so that only the iterations differ)
    ref, _ = oracle.mlem(og, sig, kev_np, x0.cpu().numpy().astype(np.float64), sens.cpu().numpy(), iters,
                         weights=w.cpu().numpy(), median=True)
    gpu = img.cpu().numpy().astype(np.float64)
    rel_l2 = np.linalg.norm(gpu - ref) / np.linalg.norm(ref)
    big = ref > 0.01 * ref.max()
    assert rel_l2 <= 1e-3 and np.max(np.abs(gpu[big] - ref[big]) / ref[big]) <= 1e-2, rel_l2
