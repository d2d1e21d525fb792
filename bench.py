#!/usr/bin/env python
"""bench.py -- events/s per TOF-MLEM iteration on the full-body workload (BASELINE.json cfg-3).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl b200|reference] [--workload full|mid|tiny]

One "step" = one MLEM iteration over the whole (locality-binned) event set: fused forward+back EM pass
(`tofmlem_em_correction`), [sum of the correction image across ranks when N > 1], multiplicative update
(`tofmlem_update`).  Binning and the sensitivity image are one-off per data set and are reported separately
(`setup`), as is the whole-reconstruction time (binning + `cfg.iters` iterations).
Prints ONE JSON line (rank 0).  See DESIGN.md "Measurement" for the roofline model.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "events/s per TOF-MLEM iteration (fwd+backproj)"
UNIT = "events/s"


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi sampled every 200 ms during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "200"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            out, _ = self.proc.communicate(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
            out, _ = self.proc.communicate()
        sm, mx, reasons, power = [], [], set(), []
        for line in out.strip().splitlines():
            f = [t.strip() for t in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
                power.append(float(f[2]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------------
def run_reference(args):
    """--impl reference: the fp64 oracle, as it stands, on the host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    import numpy as np

    import oracle
    import synth

    cfg = synth.CONFIGS[args.workload]
    og = oracle.make_grid(cfg.nx, cfg.ny, cfg.nz, cfg.voxel_mm)
    sig = oracle.sigma_mm(cfg.tof_fwhm_ps)
    n = args.ref_events
    ev = {k: v.numpy() for k, v in synth.make_events_chunked(cfg, n, chunk=500_000).items()}
    x = np.ones(og.nvox)
    sens = np.ones(og.nvox, np.float32)
    mask = np.ones(og.nvox, np.uint8)
    times = []
    for step in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        corr, n_valid, visits = oracle.em_correction(og, sig, ev, x)
        x = oracle.update(x, corr, sens, mask)
        x *= og.nvox / max(x.sum(), 1e-300)  # keep the image scale stable without a real sensitivity image
        if step >= args.warmup:
            times.append(time.perf_counter() - t0)
    ms = 1e3 * sum(times) / len(times)
    value = n / (ms * 1e-3)
    cores = oracle.num_threads()
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"{cfg.name}: {cfg.nx}x{cfg.ny}x{cfg.nz} x {cfg.voxel_mm} mm, TOF {cfg.tof_fwhm_ps:g} ps",
                   "events_per_step": n},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": f"{n}-event prefix of the seeded {cfg.name} set, one EM pass + update per step, full grid"},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


# ------------------------------------------------------------------------------------------------
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--workload", default="full", choices=["full", "mid", "tiny"])
    ap.add_argument("--events", type=int, default=0, help="override the event count (debugging only)")
    ap.add_argument("--sens-lors", type=int, default=0, help="override the number of sensitivity LORs")
    ap.add_argument("--ref-events", type=int, default=1_000_000, help="events per step of the oracle legs")
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="target duration of the cpu_baseline sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-bin", action="store_true", help="skip locality binning (for comparison)")
    ap.add_argument("--subbins", type=int, default=0, help="TOFMLEM_OPT_SUBBINS override (0 = library default)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist

    import paper_1706_07075_b200 as pkg
    import synth
    from paper_1706_07075_b200 import sharding

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device; there is no CPU fallback"
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dev = torch.device("cuda", local)

    cfg = synth.CONFIGS[args.workload]
    n = args.events or cfg.n_events  # per rank: weak scaling, every rank reconstructs its own shard
    m = args.sens_lors or cfg.sens_lors
    g = pkg.make_grid(cfg.nx, cfg.ny, cfg.nz, cfg.voxel_mm)
    ctx = pkg.Context(cfg.radius_mm, cfg.axial_mm, g, cfg.tof_fwhm_ps)
    if args.subbins:
        ctx.set_option(pkg.OPT_SUBBINS, args.subbins)
    nvox = g.nvox

    def timed(fn):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        fn()
        b.record()
        b.synchronize()
        return a.elapsed_time(b)

    # ---- inputs (synthetic, seeded; resident in HBM before any timed region)
    ev_start, _ = sharding.weak_shard_range(n, rank)
    ev = synth.make_events_chunked(cfg, n, start=ev_start, device=dev)
    sens = torch.empty(nvox, dtype=torch.float32, device=dev)
    lors = synth.make_sens_lors_chunked(cfg, m, device=dev)
    sens_ms = timed(lambda: ctx.sensitivity(lors, m, sens))
    del lors
    # ---- a1: locality binning (one-off per data set)
    bin_ms = 0.0
    if not args.no_bin:
        key = torch.empty(n, dtype=torch.int32, device=dev)
        perm = torch.empty(n, dtype=torch.int32, device=dev)
        sev = {k: torch.empty_like(v) for k, v in ev.items()}

        def do_bin():
            ctx.bin_events(ev, n, key, perm, None)
            ctx.gather_events(ev, perm, n, sev)

        bin_ms = timed(do_bin)
        n_valid_keys = int((key != -1).sum().item())
        del key, perm, ev
        ev = sev
    torch.cuda.empty_cache()

    image = torch.ones(nvox, dtype=torch.float32, device=dev)
    corr = torch.zeros(nvox, dtype=torch.float32, device=dev)

    k_start = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
    k_stop = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]

    def step(i=None):
        ctx.reset_stats()
        if i is not None:
            k_start[i].record()
        ctx.em_correction(ev, n, image, corr)
        if i is not None:
            k_stop[i].record()
        sharding.allreduce_correction(corr)  # N > 1: the iteration's one exchange (NCCL sum of the partial corrections)
        ctx.update(image, corr, sens)

    for _ in range(args.warmup):
        step()
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    launches0 = ctx.launch_count()
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0.record()
    for i in range(args.steps):
        step(i)
    t1.record()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    total_ms = t0.elapsed_time(t1)
    launches = ctx.launch_count() - launches0
    clocks = sampler.stop() if rank == 0 else None
    total_ms = sharding.max_over_ranks_ms(total_ms, dev)
    ms_per_step = total_ms / args.steps
    value = world * n / (ms_per_step * 1e-3)
    st = ctx.get_stats()
    kern_ms = statistics.mean(a.elapsed_time(b) for a, b in zip(k_start, k_stop))
    p7 = float((image.double() * sens.double()).sum().item())

    # ---- roofline of the dominant kernel (em_correction): see DESIGN.md "Measurement"
    hbm_peak, peak_src = load_peaks()
    visits = int(st.visits)
    probe_buf = torch.zeros(nvox, dtype=torch.float32, device=dev)
    n_ops = 1 << 30
    red_rand = n_ops / (ctx.probe(0, probe_buf, n_ops) * 1e-3)
    red_row = n_ops / (ctx.probe(1, probe_buf, n_ops) * 1e-3)
    ld_rand = n_ops / (ctx.probe(2, probe_buf, n_ops) * 1e-3)
    ld_row = n_ops / (ctx.probe(3, probe_buf, n_ops) * 1e-3)
    del probe_buf
    hbm_bytes = 28.0 * n  # algorithmic HBM bytes per launch: 7 float32 per event
    t_hbm = hbm_bytes / (hbm_peak * 1e9)
    t_red = visits / red_rand  # one RED per visit (events with fwd = 0 do none: a few %)
    t_ld = visits / ld_rand
    t_roof = max(t_hbm, t_red, t_ld)
    achieved = visits / (kern_ms * 1e-3)
    roofline = {
        "bound": "l2_atomic", "achieved": achieved / 1e9, "peak": red_rand / 1e9, "unit": "Gvisit/s",
        "frac": achieved / red_rand, "traffic": None,
        "kernel": "em_correction_kernel<TOF>", "kernel_ms": kern_ms, "visits_per_launch": visits,
        "peak_source": "tofmlem_probe kind 0 (random-address RED.ADD.F32 into an L2-resident array of nvox floats), measured in this run",
        "probes_Gops": {"red_random": red_rand / 1e9, "red_row": red_row / 1e9, "gather_random": ld_rand / 1e9,
                        "gather_row": ld_row / 1e9},
        "t_roof_ms": {"hbm": t_hbm * 1e3, "red": t_red * 1e3, "gather": t_ld * 1e3},
        "hbm": {"algorithmic_bytes": hbm_bytes, "achieved_GBs": hbm_bytes / (kern_ms * 1e-3) / 1e9, "peak_GBs": hbm_peak,
                "peak_source": peak_src},
    }

    # ---- e2e: the same step through the C ABI with HOST buffers (pinned), copies inside the timed region
    e2e = None
    if not args.no_e2e:
        h_ev = {k: v.cpu().pin_memory() for k, v in ev.items()}
        h_img = torch.ones(nvox, dtype=torch.float32).pin_memory()
        h_sens = sens.cpu().pin_memory()
        ctx.iterate_host(h_ev, n, h_img, h_sens, 1)  # warm-up (allocates the staging buffers)
        if world > 1:
            dist.barrier()
        reps = max(1, min(3, args.steps))
        tt = time.perf_counter()
        for _ in range(reps):
            ctx.iterate_host(h_ev, n, h_img, h_sens, 1)
        e2e_s = (time.perf_counter() - tt) / reps
        e2e_s = sharding.max_over_ranks_ms(e2e_s, dev)
        e2e = {"value": world * n / e2e_s, "unit": UNIT, "h2d_bytes_per_step": 28 * n + 8 * nvox,
               "d2h_bytes_per_step": 4 * nvox, "ms_per_step": e2e_s * 1e3,
               "call": "tofmlem_iterate_host(iters=1), pinned host buffers, binned event order"}
        del h_ev, h_img, h_sens

    # ---- cpu_baseline: the oracle on this box's host cores, bounded sample (rank 0, N = 1 only)
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        import numpy as np

        import oracle

        og = oracle.make_grid(cfg.nx, cfg.ny, cfg.nz, cfg.voxel_mm)
        x = image.cpu().numpy().astype(np.float64)
        sens_np, ones = sens.cpu().numpy(), np.ones(nvox, np.uint8)
        # events are binned (spatially ordered): a strided sample keeps the workload's mix of LORs
        ns, dt = min(n, 500_000), 0.0
        for attempt in range(3):
            stride = max(1, n // ns)
            sub = {k: v[::stride][:ns].cpu().numpy() for k, v in ev.items()}
            tt = time.perf_counter()
            c_ref, nv_ref, vis_ref = oracle.em_correction(og, oracle.sigma_mm(cfg.tof_fwhm_ps), sub, x)
            oracle.update(x.copy(), c_ref, sens_np, ones)
            dt = time.perf_counter() - tt
            ns2 = min(max(n // 4, 1), int(ns * args.cpu_seconds / max(dt, 1e-3)))
            if attempt == 2 or ns2 <= 1.5 * ns:
                break
            ns = ns2
        cpu = {"value": ns / dt, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
               "sample": f"{ns} events (every {stride}th of the binned set), one EM pass + update on the full grid, {dt:.1f} s"}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {
                "workload": f"{cfg.name}: {cfg.nx}x{cfg.ny}x{cfg.nz} voxels of {cfg.voxel_mm} mm, scanner R={cfg.radius_mm:g} L={cfg.axial_mm:g} mm, "
                            f"{n} events/GPU, {cfg.scatter_fraction:.0%} scatter-like, TOF {cfg.tof_fwhm_ps:g} ps FWHM",
                "events_per_gpu": n, "l2": "inputs larger than L2 (events 28 B x n >> 126 MB); no flush",
                "binned": not args.no_bin, "sens_lors": m,
                "parallelism": "event shards + one fp32 all-reduce of the correction image per iteration" if world > 1 else "single GPU",
            },
            "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks,
            "setup": {"sensitivity_ms": sens_ms, "bin_sort_gather_ms": bin_ms,
                      "recon_wall_s": (bin_ms + cfg.iters * ms_per_step) * 1e-3,
                      "recon_wall_note": f"binning + {cfg.iters} iterations, events resident in HBM"},
            "stats": {"n_valid": int(st.n_valid), "visits": visits, "visits_per_valid_event": visits / max(1, int(st.n_valid)),
                      "sum_image_sens": p7, "p7_rel_err": abs(p7 - st.n_valid) / max(1, int(st.n_valid))},
            "paper_context": "PAPER.md:17,:299 -- 3.5 min for the slowest of nine regions (20 iterations, Tesla C2075 + 16 CPU threads); context, not the target",
        }
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
