"""The warp-per-LOR walk of whole chords (csrc/warpwalk.cu, TOFMLEM_OPT_WARP_WALK; north_star bullet 2 "a thread or warp
per event chosen by chord length") against the fp64 oracle: sensitivity image, attenuation line integrals, forward /
backprojection / fused pass of a non-TOF context -- on hand-built degenerate LORs, on ragged anisotropic grids (the
transposes' tails) and on the full cfg-3 grid, and against the thread-per-LOR walk it replaces."""
import numpy as np
import pytest
import torch

import oracle
import synth

pytestmark = pytest.mark.gpu

FWD_RTOL = 1e-4


@pytest.fixture(scope="module")
def pkg():
    import paper_1706_07075_b200 as p

    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return p


def _lors(rows):
    arr = np.array(rows, np.float32)
    ev_np = {k: np.ascontiguousarray(arr[:, i]) for i, k in enumerate(synth.LOR_FIELDS)}
    ev = {k: torch.from_numpy(v).cuda() for k, v in ev_np.items()}
    ev["dt"] = None
    return ev, ev_np, arr.shape[0]


def _fwd_err(got, ref):
    got = np.asarray(got, np.float64)
    pos = ref > 0
    den = np.maximum(ref, 1e-6 * np.median(ref[pos]))
    return np.abs(got - ref) / den


def _img_err(got, ref):
    got = np.asarray(got, np.float64).reshape(-1)
    ref = np.asarray(ref, np.float64).reshape(-1)
    big = ref > 0.01 * ref.max()
    return np.linalg.norm(got - ref) / np.linalg.norm(ref), np.max(np.abs(got[big] - ref[big]) / ref[big])


def test_degenerate_lors(pkg):
    """Axis-parallel LORs, LORs inside voxel boundary planes, exact corner crossings, end points on the grid faces and
    inside the grid, clipped corners (chords of a fraction of a voxel), grazing rays, invalid LORs."""
    dims, vox = (16, 12, 20), (4.0, 3.0, 2.0)
    g = pkg.make_grid(*dims, vox)
    og = oracle.make_grid(*dims, vox)
    nan = float("nan")
    rows = [
        (-200, 0, 0, 200, 0, 0),              # along x, in the planes y = 0 and z = 0
        (-200, 1.5, 1.0, 200, 1.5, 1.0),      # along x through voxel centres
        (200, 1.5, 1.0, -200, 1.5, 1.0),      # ... towards -x
        (0, -200, 1.0, 0, 200, 1.0),          # along y, in the plane x = 0
        (1.0, 1.0, -64, 1.0, 1.0, 64),        # along z
        (1.0, 1.0, 64, 1.0, 1.0, -64),        # along -z
        (-200, -100, -60, 200, 100, 60),      # through the grid centre: exact corner crossings
        (-32, -18, -20, 32, 18, 20),          # end points ON the grid corners, main diagonal
        (32, -18, 20, -32, 18, -20),          # another diagonal, mixed signs
        (-10, 2, 3, 12, -7, 1),               # both end points inside the grid
        (-200, 17.999, 19.99, 200, 17.999, 19.99),  # grazing the top edges
        (-200, 100, 0, 200, 100, 0),          # misses the grid
        (5, 5, 5, 5, 5, 5),                   # L = 0
        (nan, 0, 0, 200, 0, 0),               # non-finite
        (-33, -17.9, 0.5, -31.5, -19, 0.7),   # clips the corner x = -32, y = -18: a chord of a fraction of a voxel
        (31.9, 0.2, -21, 32.3, 0.25, -19.5),  # clips the edge x = 32, z = -20
        (-200, -17.5, -19.0, 200, 17.5, 19.0),  # shallow in y and z, x-dominant
        (-3.0, -200, -19.0, 3.5, 200, 19.5),  # y-dominant, shallow in x
        (-31.0, 17.0, -200, 31.0, -17.0, 200),  # z-dominant
        (0.0, -18.0, -20.0, 0.0, 18.0, 20.0),   # in the plane x = 0, slope exactly along the y-z diagonal of the grid
        (-32.0, -18.0, 0.0, 32.0, 18.0, 0.0),   # |dx / vx| = |dy / vy|: a tie between two dominant axes
    ]
    ev, ev_np, n = _lors(rows)
    img = synth.random_image((g.nz, g.ny, g.nx), 3, device="cuda").reshape(-1).contiguous()
    ref = oracle.forward(og, 0.0, ev_np, img.cpu().numpy())
    refb = oracle.backproject(og, 0.0, ev_np, None)
    assert (ref > 0).sum() >= 16
    for ww in (1, 0):
        ctx = pkg.Context(200.0, 128.0, g, 0.0)
        ctx.set_option(pkg.OPT_WARP_WALK, ww)
        fwd = torch.full((n,), -1.0, dtype=torch.float32, device="cuda")
        ctx.forward(ev, n, img, fwd)
        got = fwd.cpu().numpy()
        assert np.all(got[ref == 0] == 0), (ww, got[ref == 0])
        err = _fwd_err(got, ref)
        assert err.max() <= FWD_RTOL, (ww, int(err.argmax()), err.max())
        out = torch.zeros(g.nvox, dtype=torch.float32, device="cuda")
        ctx.backproject(ev, n, None, out)
        assert np.linalg.norm(out.cpu().numpy() - refb) / np.linalg.norm(refb) < 1e-5, ww
        assert not np.any(out.cpu().numpy()[refb == 0] > 1e-4), ww  # nothing lands in voxels no chord meets
        ctx.forward(ev, 0, img, fwd)  # empty input: no-ops
        ctx.backproject(ev, 0, None, out)


@pytest.mark.parametrize("dims,vox", [((33, 47, 29), (3.0, 2.0, 4.5)), ((64, 20, 70), (2.0, 5.0, 1.5)),
                                      ((7, 5, 130), (6.0, 7.0, 1.0))])
def test_ragged_anisotropic_grids(pkg, dims, vox):
    """Odd sizes (tails of the transposes, unaligned rows, nvox % 4 != 0) and anisotropic voxels (the dominant axis is
    decided in voxel units): sensitivity, line integrals and the fused pass against the oracle."""
    g = pkg.make_grid(*dims, vox)
    og = oracle.make_grid(*dims, vox)
    cfg = synth.Config("ragged", dims[0], dims[1], dims[2], vox[0], 120.0, 260.0, synth.TINY.phantom, 0, 0.0, 0.0, 1,
                       60_001, 17)
    m = cfg.sens_lors
    lors = synth.make_sens_lors(cfg, m, device="cuda")
    lors_np = {k: v.cpu().numpy() for k, v in lors.items()}
    ctx = pkg.Context(cfg.radius_mm, cfg.axial_mm, g, 0.0)
    sens = torch.empty(g.nvox, dtype=torch.float32, device="cuda")
    ctx.sensitivity(lors, m, sens)
    ref = oracle.sensitivity(og, lors_np)
    l2, mx = _img_err(sens.cpu().numpy(), ref)
    assert l2 <= 1e-5 and mx <= 1e-4, (l2, mx)
    mu = synth.random_image((g.nz, g.ny, g.nx), 9, device="cuda").reshape(-1).contiguous() * 2e-3
    w = torch.empty(m, dtype=torch.float32, device="cuda")
    ctx.attenuation_weights(lors, m, mu, w)
    line = oracle.forward(og, 0.0, lors_np, mu.cpu().numpy())
    assert np.max(np.abs(w.cpu().numpy() - np.exp(line)) / np.exp(line)) <= FWD_RTOL
    img = synth.random_image((g.nz, g.ny, g.nx), 4, device="cuda").reshape(-1).contiguous()
    corr = torch.zeros(g.nvox, dtype=torch.float32, device="cuda")
    ctx.reset_stats()
    ctx.em_correction({**lors, "dt": None}, m, img, corr)
    oc, nv, vis = oracle.em_correction(og, 0.0, lors_np, img.cpu().numpy().astype(np.float64))
    l2, mx = _img_err(corr.cpu().numpy(), oc)
    assert l2 <= 1e-5 and mx <= 1e-3, (l2, mx)
    st = ctx.get_stats()
    assert st.n_valid == nv
    assert abs(int(st.visits) - vis) <= 1e-4 * vis
    # the update after a warp-walk pass reads the correction image in grid order
    s1 = torch.ones(g.nvox, dtype=torch.float32, device="cuda")
    x = img.clone()
    ctx.update(x, corr, s1)
    assert float((x.double() - img.double() * torch.from_numpy(oc).cuda()).abs().max()) <= 1e-3 * float(oc.max())


def test_full_grid_against_oracle_and_thread_walk(pkg):
    """cfg-3 geometry (160 x 160 x 640 x 3.75 mm, chords of up to 900 voxels): 200 k detector pairs."""
    cfg = synth.FULL
    g = pkg.make_grid(cfg.nx, cfg.ny, cfg.nz, cfg.voxel_mm)
    og = oracle.make_grid(cfg.nx, cfg.ny, cfg.nz, cfg.voxel_mm)
    m = 200_000
    lors = synth.make_sens_lors(cfg, m, device="cuda")
    lors_np = {k: v.cpu().numpy() for k, v in lors.items()}
    img = synth.random_image((g.nz, g.ny, g.nx), 5, device="cuda").reshape(-1).contiguous()
    ref = oracle.forward(og, 0.0, lors_np, img.cpu().numpy())
    refs = oracle.sensitivity(og, lors_np)
    res = {}
    for ww in (1, 0):
        ctx = pkg.Context(cfg.radius_mm, cfg.axial_mm, g, 0.0)
        ctx.set_option(pkg.OPT_WARP_WALK, ww)
        fwd = torch.empty(m, dtype=torch.float32, device="cuda")
        ctx.forward({**lors, "dt": None}, m, img, fwd)
        got = fwd.cpu().numpy()
        assert np.array_equal(got == 0, ref == 0)
        assert _fwd_err(got, ref).max() <= FWD_RTOL, ww
        sens = torch.empty(g.nvox, dtype=torch.float32, device="cuda")
        ctx.sensitivity(lors, m, sens)
        l2, mx = _img_err(sens.cpu().numpy(), refs)
        assert l2 <= 1e-5 and mx <= 1e-3, (ww, l2, mx)
        vals = synth.random_image((m,), 77, device="cuda")
        out = torch.zeros(g.nvox, dtype=torch.float32, device="cuda")
        ctx.backproject({**lors, "dt": None}, m, vals, out)
        res[ww] = out
    refb = oracle.backproject(og, 0.0, lors_np, synth.random_image((m,), 77).numpy())
    for ww in (1, 0):
        l2, mx = _img_err(res[ww].cpu().numpy(), refb)
        assert l2 <= 1e-5 and mx <= 1e-3, (ww, l2, mx)


def test_non_tof_iterations_parity(pkg):
    """Two MLEM iterations of a non-TOF context through the warp walk (tiny grid) against oracle.mlem."""
    cfg = synth.TINY
    g = pkg.make_grid(cfg.nx, cfg.ny, cfg.nz, cfg.voxel_mm)
    og = oracle.make_grid(cfg.nx, cfg.ny, cfg.nz, cfg.voxel_mm)
    n = 60_000
    ev = synth.make_events(cfg, n, device="cuda")
    lor = {k: v for k, v in ev.items() if k != "dt"}
    lor_np = {k: v.cpu().numpy() for k, v in lor.items()}
    ctx = pkg.Context(cfg.radius_mm, cfg.axial_mm, g, 0.0)
    lors = synth.make_sens_lors(cfg, 300_000, device="cuda")
    sens = torch.empty(g.nvox, dtype=torch.float32, device="cuda")
    ctx.sensitivity(lors, 300_000, sens)
    sens_np = sens.cpu().numpy()
    mask = oracle.mask_f32(sens_np)
    img = torch.from_numpy(mask.astype(np.float32)).cuda()
    ctx.iterate({**lor, "dt": None}, n, img, sens, 2)
    ref, ost = oracle.mlem(og, 0.0, lor_np, mask.astype(np.float64), sens_np, 2)
    l2, mx = _img_err(img.cpu().numpy(), ref)
    assert l2 <= 1e-3 and mx <= 1e-2, (l2, mx)
    st = ctx.get_stats()
    assert st.n_valid == ost.n_valid
