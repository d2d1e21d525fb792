"""tofmlem_em_correction_static (include/tofmlem.h): the fused EM pass for callers that cannot call cudaMalloc -- no
context, scratch in a static __device__ array.  Its correction image is compared with the existing path's (a context's
unplanned pass in grid order) and with the fp64 oracle, on two calls in a row (the second call finds the first call's
counters in the shared array).  Collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest
import torch

import oracle
import synth

pytestmark = pytest.mark.gpu

# two float32 passes with the same arithmetic and a different order of the sums (tests/test_gpu_parity.py uses the same
# bounds for the backprojection against the oracle)
L2_TOL = 1e-5
MAX_TOL = 1e-4


def _compare(a, b, l2=L2_TOL, mx=MAX_TOL, zeros=True):
    a = np.asarray(a, np.float64).reshape(-1)
    b = np.asarray(b, np.float64).reshape(-1)
    rel_l2 = np.linalg.norm(a - b) / np.linalg.norm(b)
    big = b > 0.01 * b.max()
    max_rel = np.max(np.abs(a[big] - b[big]) / b[big])
    assert rel_l2 <= l2, f"rel-L2 {rel_l2:.3e}"
    assert max_rel <= mx, f"max rel {max_rel:.3e}"
    assert not zeros or not np.any(a[b == 0] != 0)  # same voxels touched (same walk)


@pytest.fixture(scope="module")
def pkg():
    import paper_1706_07075_b200 as p

    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return p


def test_static_em_correction_matches_context_path(pkg):
    cfg = synth.TINY
    n = 120_003  # several 32-event pieces per queue and a ragged tail
    ev = synth.make_events(cfg, n, device="cuda")
    ev_np = {k: v.cpu().numpy() for k, v in ev.items()}
    g = pkg.make_grid(cfg.nx, cfg.ny, cfg.nz, cfg.voxel_mm)
    og = oracle.make_grid(cfg.nx, cfg.ny, cfg.nz, cfg.voxel_mm)
    ctx = pkg.Context(cfg.radius_mm, cfg.axial_mm, g, cfg.tof_fwhm_ps)
    ctx.set_option(pkg.OPT_CORR_BRICKS, 0)  # the existing path with its correction image in grid order
    images = [torch.ones(g.nvox, dtype=torch.float32, device="cuda"),
              synth.random_image((g.nz, g.ny, g.nx), 11, device="cuda").reshape(-1).contiguous() + 0.25]
    sigma = oracle.sigma_mm(cfg.tof_fwhm_ps)
    for call, img in enumerate(images):  # two calls in a row on the shared scratch
        ref = torch.zeros(g.nvox, dtype=torch.float32, device="cuda")
        ctx.em_correction(ev, n, img, ref)
        out = torch.zeros(g.nvox, dtype=torch.float32, device="cuda")
        pkg.em_correction_static(g, cfg.tof_fwhm_ps, ev, n, img, out, queues_per_sm=(0 if call == 0 else 2))
        torch.cuda.synchronize()
        _compare(out.cpu().numpy(), ref.cpu().numpy())
        orc, _, _ = oracle.em_correction(og, sigma, ev_np, img.cpu().numpy().astype(np.float64))
        _compare(out.cpu().numpy(), orc, l2=1e-3, mx=1e-2, zeros=False)
    # accumulation: a third call into the same array doubles it
    pkg.em_correction_static(g, cfg.tof_fwhm_ps, ev, n, images[1], out)
    torch.cuda.synchronize()
    _compare(out.cpu().numpy(), 2.0 * ref.cpu().numpy().astype(np.float64))


def test_static_em_correction_non_tof_and_unaligned(pkg):
    """Non-TOF pass (dt = NULL) and a correction image that is not 16-byte aligned (scalar reductions)."""
    cfg = synth.TINY
    n = 20_001
    ev = synth.make_events(cfg, n, device="cuda")
    lor = {k: v for k, v in ev.items() if k != "dt"}
    g = pkg.make_grid(cfg.nx, cfg.ny, cfg.nz, cfg.voxel_mm)
    ctx = pkg.Context(cfg.radius_mm, cfg.axial_mm, g, 0.0)
    ctx.set_option(pkg.OPT_CORR_BRICKS, 0)
    img = synth.random_image((g.nz, g.ny, g.nx), 3, device="cuda").reshape(-1).contiguous() + 0.5
    ref = torch.zeros(g.nvox, dtype=torch.float32, device="cuda")
    ctx.em_correction({**lor, "dt": None}, n, img, ref)
    for _ in range(2):
        buf = torch.zeros(g.nvox + 1, dtype=torch.float32, device="cuda")
        out = buf[1:]  # 4 bytes off a 16-byte boundary
        pkg.em_correction_static(g, 0.0, {**lor, "dt": None}, n, img, out)
        torch.cuda.synchronize()
        _compare(out.cpu().numpy(), ref.cpu().numpy())


def test_static_em_correction_rejects_oversize(pkg):
    cfg = synth.TINY
    n = 1000
    ev = synth.make_events(cfg, n, device="cuda")
    g = pkg.make_grid(cfg.nx, cfg.ny, cfg.nz, cfg.voxel_mm)
    img = torch.ones(g.nvox, dtype=torch.float32, device="cuda")
    out = torch.zeros(g.nvox, dtype=torch.float32, device="cuda")
    n_sm = torch.cuda.get_device_properties(0).multi_processor_count
    too_many = 1024 // n_sm + 1  # SMs x queues_per_sm > TOFMLEM_STATIC_MAX_QUEUES
    if too_many <= 8:
        with pytest.raises(pkg.TofMlemError) as ei:
            pkg.em_correction_static(g, cfg.tof_fwhm_ps, ev, n, img, out, queues_per_sm=too_many)
        assert ei.value.code == -1 and "static scratch" in str(ei.value)
    with pytest.raises(pkg.TofMlemError) as ei:
        pkg.em_correction_static(g, cfg.tof_fwhm_ps, ev, n, img, out, queues_per_sm=9)
    assert ei.value.code == -1
    with pytest.raises(pkg.TofMlemError):  # a TOF pass without dt
        pkg.em_correction_static(g, cfg.tof_fwhm_ps, {**ev, "dt": None}, n, img, out)
    assert float(out.abs().sum()) == 0.0  # a refused call launches nothing
    pkg.em_correction_static(g, cfg.tof_fwhm_ps, ev, 0, img, out)  # n = 0: nothing to do
    torch.cuda.synchronize()
