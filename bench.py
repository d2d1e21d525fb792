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
# DRAM bytes of one launch of the dominant kernel at cfg-3 (ncu --set full; refresh with the capture)
TRAFFIC_BYTES = 6.868e9
TRAFFIC_SOURCE = ("profiles/r05_em_tile_ncu_full_metrics.txt: em_tile_kernel 6.411 GB read + 0.456 GB written per launch "
                  "(algorithmic: 56 B x 97.9 M tile events = 5.48 GB of records + scale scratch)")
UNIT = "events/s"


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi sampled every 50 ms during the timed region (B200_PROFILING.md recipe)."""
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
                 "-lms", "50"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
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
def make_config(cfg, n, m, world, binned=True):
    """The `config` object of the JSON line: the same for the b200 arm and the reference (oracle) arm."""
    return {
        "workload": f"{cfg.name}: {cfg.nx}x{cfg.ny}x{cfg.nz} voxels of {cfg.voxel_mm} mm, scanner R={cfg.radius_mm:g} L={cfg.axial_mm:g} mm, "
                    f"{n} events/GPU, {cfg.scatter_fraction:.0%} scatter-like, TOF {cfg.tof_fwhm_ps:g} ps FWHM",
        "events_per_gpu": n, "l2": "inputs larger than L2 (events 28 B x n >> 126 MB); no flush",
        "binned": binned, "sens_lors": m,
        "parallelism": "event shards + one fp32 all-reduce of the correction image per iteration" if world > 1 else "single GPU",
    }


def oracle_arm(cfg, n_sample, steps, warmup):
    """The oracle, as it stands, on the host cores: one EM pass + update per step over a bounded sample of the workload.
    The sample is the first `n_sample` events of the seeded set in generation order -- the events are independent draws,
    so a prefix is an unbiased sample of the workload's LOR mix -- on the full grid, image = 1, sensitivity = 1 (the
    oracle's cost does not depend on the image values).  Used by --impl reference and by the b200 arm's `cpu_baseline`,
    so that both report the same thing."""
    import numpy as np

    import oracle
    import synth

    og = oracle.make_grid(cfg.nx, cfg.ny, cfg.nz, cfg.voxel_mm)
    sig = oracle.sigma_mm(cfg.tof_fwhm_ps)
    n = min(n_sample, cfg.n_events)
    ev = {k: v.numpy() for k, v in synth.make_events_chunked(cfg, n, chunk=500_000).items()}
    x = np.ones(og.nvox)
    sens = np.ones(og.nvox, np.float32)
    mask = np.ones(og.nvox, np.uint8)
    times = []
    for step in range(warmup + steps):
        t0 = time.perf_counter()
        corr, n_valid, visits = oracle.em_correction(og, sig, ev, x)
        x = oracle.update(x, corr, sens, mask)
        x *= og.nvox / max(x.sum(), 1e-300)  # keep the image scale stable without a real sensitivity image
        if step >= warmup:
            times.append(time.perf_counter() - t0)
    ms = 1e3 * sum(times) / len(times)
    return {"value": n / (ms * 1e-3), "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
            "sample": f"first {n} events of the seeded {cfg.name} set in generation order (independent draws: an unbiased "
                      f"sample), one EM pass + update per step on the full grid, {steps} timed steps of {ms / 1e3:.2f} s"}, ms


def run_reference(args):
    """--impl reference: the fp64 oracle, as it stands, on the host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    import synth

    cfg = synth.CONFIGS[args.workload]
    cpu, ms = oracle_arm(cfg, args.ref_events, args.steps, args.warmup)
    value = cpu["value"]
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": make_config(cfg, args.events or cfg.n_events, args.sens_lors or cfg.sens_lors, max(1, args.gpus)),
        "cpu_baseline": cpu,
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


# ------------------------------------------------------------------------------------------------
def run_report(args):
    """Single-GPU reports beside the bench line: cfg-5 sweep, cfg-4 division, widened rows.  Device-timed with CUDA
    events after a warm-up pass; inputs (>= 280 MB of events) are larger than L2 except where noted."""
    import torch

    import paper_1706_07075_b200 as pkg
    import synth

    assert torch.cuda.is_available(), "bench.py needs a CUDA device; there is no CPU fallback"
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)

    def timed(fn, reps=1):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(reps):
            fn()
        b.record()
        b.synchronize()
        return a.elapsed_time(b) / reps

    def binned(ctx, ev, n):
        key = torch.empty(n, dtype=torch.int32, device=dev)
        perm = torch.empty(n, dtype=torch.int32, device=dev)
        sev = {k: torch.empty_like(v) for k, v in ev.items()}
        ms = timed(lambda: (ctx.bin_events(ev, n, key, perm, None), ctx.permute_events(ev, perm, n, sev)))
        return sev, perm, ms

    full = synth.FULL
    g = pkg.make_grid(full.nx, full.ny, full.nz, full.voxel_mm)
    nvox = g.nvox
    base = pkg.Context(full.radius_mm, full.axial_mm, g, full.tof_fwhm_ps)
    m = args.sens_lors or 20_000_000
    lors = synth.make_sens_lors_chunked(full, m, device=dev)
    sens = torch.empty(nvox, dtype=torch.float32, device=dev)
    base.sensitivity(lors, m, sens)
    del lors
    probe_buf = torch.zeros(nvox, dtype=torch.float32, device=dev)
    red_rand = (1 << 30) / (base.probe(0, probe_buf, 1 << 30) * 1e-3)
    del probe_buf
    out = {"report": args.report, "data": "synthetic", "dtype": "f32", "sens_lors": m,
           "red_random_Gps": red_rand / 1e9}

    if args.report == "sweep":
        # cfg-5: full-body geometry and phantom, 20 % scatter, 3 iterations, seed 5
        points = []
        for n in [int(t) for t in args.sweep_events.split(",")]:
            for fwhm in [float(t) for t in args.sweep_fwhm.split(",")]:
                cfg = synth.sweep_config(n, fwhm)
                ev = synth.make_events_chunked(cfg, n, device=dev)
                if fwhm <= 0:
                    ev["dt"].zero_()
                ctx = pkg.Context(cfg.radius_mm, cfg.axial_mm, g, fwhm)
                ctx.reserve(n)  # scratch of binning and plan: allocated outside the timed calls
                sev, _, bin_ms = binned(ctx, ev, n)
                del ev
                plan_ms = timed(lambda: ctx.plan_events(sev, n)) if args.tile else 0.0  # inactive for non-TOF
                plan = ctx.plan_info()
                image = torch.ones(nvox, dtype=torch.float32, device=dev)
                corr = torch.zeros(nvox, dtype=torch.float32, device=dev)

                def step():
                    ctx.reset_stats()
                    ctx.em_correction(sev, n, image, corr)
                    ctx.update(image, corr, sens)

                step()  # warm-up = iteration 1
                ms = timed(step, reps=cfg.iters - 1)  # iterations 2..3
                st = ctx.get_stats()
                p7 = float((image.double() * sens.double()).sum().item())
                points.append({
                    "events": n, "tof_fwhm_ps": fwhm, "ms_per_iteration": ms, "events_per_s": n / (ms * 1e-3),
                    "n_valid": int(st.n_valid), "visits": int(st.visits), "reductions": int(st.reductions),
                    "visits_per_valid_event": st.visits / max(1, st.n_valid), "Gvisits_per_s": st.visits / ms / 1e6,
                    "roofline_frac": st.reductions / (ms * 1e-3) / red_rand, "bin_sort_gather_ms": bin_ms,
                    "plan_ms": plan_ms, "planned": int(plan.active), "tile_items": int(plan.n_tile_items),
                    "tile_events": int(st.tile_events),
                    "p7_rel_err": abs(p7 - st.n_valid) / max(1, st.n_valid)})
                print(json.dumps(points[-1]), file=sys.stderr, flush=True)
                del sev, image, corr, ctx
                torch.cuda.empty_cache()
        out["config"] = {"workload": "cfg-5 sweep: 160x160x640 x 3.75 mm, 20% scatter-like, 3 iterations (first = warm-up)"}
        out["points"] = points

    elif args.report == "division":
        # cfg-4: the cfg-3 event set split into nine axial regions, each reconstructed on its sub-volume + margin on its
        # own stream, the extended images summed; compared with the unsplit reconstruction (same x0 = mask).
        cfg = full
        n = args.events or cfg.n_events
        it = args.division_iters or cfg.iters
        ev = synth.make_events_chunked(cfg, n, device=dev)
        sev, _, bin_ms = binned(base, ev, n)
        mx = sens.max()
        x0 = (sens >= 0.01 * mx).float()
        whole = x0.clone()
        plan_ms = timed(lambda: base.plan_events(sev, n)) if args.tile else 0.0
        base.iterate(sev, n, whole, sens, 1)  # warm-up
        whole = x0.clone()
        whole_ms = timed(lambda: base.iterate(sev, n, whole, sens, it))
        del sev
        base.trim()  # drop the unsplit plan's records
        split = torch.empty(nvox, dtype=torch.float32, device=dev)
        if args.region_plan >= 0:
            base.set_option(pkg.OPT_REGION_PLAN, args.region_plan)
        base.reconstruct_regions(ev, n, 9, None, split, sens, it)  # warm-up: builds the sub-contexts and scratch
        split_runs = []
        for _ in range(5):
            t0 = time.perf_counter()
            base.reconstruct_regions(ev, n, 9, None, split, sens, it)  # synchronises
            split_runs.append((time.perf_counter() - t0) * 1e3)
        split_ms = statistics.median(split_runs)
        region = torch.empty(n, dtype=torch.int32, device=dev)
        counts = base.split_regions(ev, n, 9, None, region, None)
        d = (split.double() - whole.double())
        big = whole > 0.01 * whole.max()
        # where the difference sits: slices within the region margin of an internal border vs the region interiors
        zb = base.region_zbounds(9)
        ks = [int(round((float(z) - g.oz) / g.vz)) for z in zb]
        _, z0r, z1r = base.region_grid(9, None, 1)
        margin = ks[1] - z0r
        near = torch.zeros(cfg.nz, dtype=torch.bool, device=dev)
        for k in ks[1:-1]:
            near[max(0, k - margin):min(cfg.nz, k + margin)] = True
        near_v = near.repeat_interleave(cfg.nx * cfg.ny)
        w2 = whole.double()
        interior_l2 = float(d[~near_v].norm() / w2[~near_v].norm())
        border_l2 = float(d[near_v].norm() / w2[near_v].norm())

        def overlap_report():
            # the other reading of PAPER.md:101 (R27): an event in every region its window reaches, wide margins, cores only
            base.set_option(pkg.OPT_REGION_OVERLAP, 1)
            o = torch.empty(nvox, dtype=torch.float32, device=dev)
            base.reconstruct_regions(ev, n, 9, None, o, sens, it)  # warm-up (new sub-contexts: other margins)
            runs = []
            for _ in range(3):
                t0 = time.perf_counter()
                base.reconstruct_regions(ev, n, 9, None, o, sens, it)
                runs.append((time.perf_counter() - t0) * 1e3)
            span = torch.empty(n, dtype=torch.int32, device=dev)
            oc = base.split_regions_overlap(ev, n, 9, None, span, None)
            dd = o.double() - whole.double()
            base.set_option(pkg.OPT_REGION_OVERLAP, 0)
            return {"split_runs_ms": runs, "list_entries": int(oc.sum()), "region_counts": [int(c) for c in oc],
                    "rel_l2_split_vs_unsplit": float(dd.norm() / w2.norm()),
                    "max_rel_on_voxels_above_1pct": float((dd.abs()[big] / w2[big]).max()),
                    "rel_l2_region_interiors": float(dd[~near_v].norm() / w2[~near_v].norm()),
                    "rel_l2_within_margin_of_borders": float(dd[near_v].norm() / w2[near_v].norm())}

        out["config"] = {"workload": f"cfg-4 division: {n} events of cfg-3, 9 regions, {it} iterations each"}
        out.update({
            "unsplit_ms": whole_ms, "unsplit_bin_ms": bin_ms, "unsplit_plan_ms": plan_ms, "split_total_ms": split_ms,
            "split_runs_ms": split_runs,
            "split_note": "split + permute + nine per-region reconstructions on nine streams + sum, host wall clock of the synchronising call",
            "region_counts": [int(c) for c in counts],
            "rel_l2_split_vs_unsplit": float(d.norm() / whole.double().norm()),
            "max_rel_on_voxels_above_1pct": float((d.abs()[big] / whole.double()[big]).max()),
            "margin_slices": margin, "rel_l2_region_interiors": interior_l2, "rel_l2_within_margin_of_borders": border_l2,
            "border_slice_fraction": float(near.float().mean()),
            "overlap_reading_R27": overlap_report(),
            "paper": "PAPER.md:212 'no difference to the whole-body reconstruction' (visual); parity unpinned, no threshold"})

    elif args.report == "pipeline":
        # The paper's whole chain on the cfg-3 data (Table 2): pre-processing (TOF scatter rejection,
        # attenuation weights), starting backprojection, locality binning, 20 MLEM iterations with per-event weights and
        # the median filter after each iteration.  Host wall clock around each stage (every stage ends in a
        # synchronisation), events resident in HBM at the start.
        import numpy as np
        cfg = full
        n = args.events or cfg.n_events
        iters = 20
        ev = synth.make_events_chunked(cfg, n, device=dev)
        mu = synth.rasterize_mu_map(cfg, device=dev).reshape(-1).contiguous()
        ell = np.empty((len(cfg.phantom.parts), 6), np.float32)
        for i, (c, sa) in enumerate(synth.body_outline(cfg)):
            ell[i, :3] = c
            ell[i, 3:] = 1.0 / np.asarray(sa, np.float64)
        ell_t = torch.from_numpy(ell)
        base.set_option(pkg.OPT_MEDIAN, 1)
        stages = {}

        def stage(name, fn):
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            out_ = fn()
            torch.cuda.synchronize()
            stages[name] = (time.perf_counter() - t0) * 1e3
            return out_

        def run_chain():
            keep = torch.empty(n, dtype=torch.uint8, device=dev)
            perm = torch.empty(n, dtype=torch.int32, device=dev)
            kept = stage("scatter_rejection", lambda: base.scatter_reject(ev, n, ell_t, 0.0, keep, perm))
            kev = {k: torch.empty(kept, dtype=torch.float32, device=dev) for k in ev}
            stage("compaction", lambda: base.gather_events(ev, perm, kept, kev))
            del keep, perm
            x = torch.zeros(nvox, dtype=torch.float32, device=dev)
            stage("starting_backprojection", lambda: base.backproject(kev, kept, None, x))
            key = torch.empty(kept, dtype=torch.int32, device=dev)
            bperm = torch.empty(kept, dtype=torch.int32, device=dev)
            sev = {k: torch.empty_like(v) for k, v in kev.items()}
            stage("binning_and_permutation", lambda: (base.bin_events(kev, kept, key, bperm, None),
                                                      base.permute_events(kev, bperm, kept, sev)))
            del kev, key, bperm
            # on the binned events: neighbouring LORs are nearly parallel and close, so the mu-map gathers hit L1
            sw = torch.empty(kept, dtype=torch.float32, device=dev)
            stage("attenuation_weights", lambda: base.attenuation_weights(sev, kept, mu, sw))
            if args.tile:
                stage("plan_ray_records", lambda: base.plan_events(sev, kept))
            stage("mlem_20_iterations_with_median", lambda: base.iterate_weighted(sev, kept, sw, x, sens, iters))
            return kept, x

        run_chain()  # warm-up (allocations, lazy module loading)
        kept, x = run_chain()
        st = base.get_stats()
        total = sum(stages.values())
        out["config"] = {"workload": f"the paper's chain on cfg-3: {n} detected events, 160x160x640 x 3.75 mm, {iters} iterations"}
        out.update({"stages_ms": stages, "total_ms": total, "events_kept": kept, "n_valid_last_pass": int(st.n_valid),
                    "image_sum": float(x.double().sum().item()),
                    "paper_context": "PAPER.md Table 2 (:292-297): whole body, SRF 300 ps, 20 iterations with median filter: "
                                     "21:11 min on Tesla C2075 + 16 CPU threads, of which pre-processing 1:08 and starting "
                                     "backprojection 1:40 (350x350x1000 voxels of 2 mm, ~73 M events after rejection); "
                                     "another machine, another grid: context, not a comparison"})

    else:  # widened rows, cfg-3 sizes
        cfg = full
        n = args.events or cfg.n_events
        ev = synth.make_events_chunked(cfg, n, device=dev)
        res = {}
        # NEXT-4 first (it is a pre-processing step): TOF scatter rejection against the phantom's body outline
        import numpy as np
        ell = np.empty((len(cfg.phantom.parts), 6), np.float32)
        for i, (c, sa) in enumerate(synth.body_outline(cfg)):
            ell[i, :3] = c
            ell[i, 3:] = 1.0 / np.asarray(sa, np.float64)
        ell_t = torch.from_numpy(ell)
        keep = torch.empty(n, dtype=torch.uint8, device=dev)
        perm = torch.empty(n, dtype=torch.int32, device=dev)
        base.scatter_reject(ev, n, ell_t, 0.0, keep, perm)
        t0 = time.perf_counter()
        kept = base.scatter_reject(ev, n, ell_t, 0.0, keep, perm)
        ms = (time.perf_counter() - t0) * 1e3
        kinds = synth.event_kinds(cfg, min(n, 4_000_000), device=dev).bool()
        kk = keep[:kinds.numel()].bool()
        res["scatter_reject"] = {"ms": ms, "events_per_s": n / (ms * 1e-3), "kept": kept, "kept_fraction": kept / n,
                                 "hbm_GBs": (28.0 * n + n + 4.0 * kept) / (ms * 1e-3) / 1e9,
                                 "trues_kept": float(kk[~kinds].float().mean()),
                                 "scatter_like_kept": float(kk[kinds].float().mean())}
        del keep, perm
        # NEXT-3: attenuation weights (non-TOF line integral of a synthetic mu-map) and the weighted EM pass
        mu = synth.rasterize_mu_map(cfg, device=dev).reshape(-1).contiguous()
        w = torch.empty(n, dtype=torch.float32, device=dev)
        base.attenuation_weights(ev, n, mu, w)
        ms = timed(lambda: base.attenuation_weights(ev, n, mu, w))
        res["attenuation_weights"] = {"ms": ms, "lors_per_s": n / (ms * 1e-3), "mean_weight": float(w.mean())}
        sev, perm, _ = binned(base, ev, n)
        sw = torch.empty_like(w)
        base.gather_f32(w, perm, n, sw)
        del ev, w, perm, mu
        image = torch.ones(nvox, dtype=torch.float32, device=dev)
        corr = torch.zeros(nvox, dtype=torch.float32, device=dev)

        def pass_w():
            base.em_correction_weighted(sev, n, sw, image, corr)
            base.update(image, corr, sens)

        if args.tile:
            base.reserve(n)
            res["plan_events"] = {"ms": timed(lambda: base.plan_events(sev, n))}
        pass_w()
        ms = timed(pass_w, reps=3)
        res["weighted_iteration"] = {"ms": ms, "events_per_s": n / (ms * 1e-3)}
        # NEXT-2: 3x3x3 median filter on the full volume (65.5 MB in + 65.5 MB out: L2-sized, HBM-cold between reps)
        tmp = torch.empty_like(image)
        base.median3(image, tmp)
        ms = timed(lambda: base.median3(image, tmp), reps=5)
        hbm_peak, _ = load_peaks()
        res["median3"] = {"ms": ms, "voxels_per_s": nvox / (ms * 1e-3), "algorithmic_GBs": 8.0 * nvox / (ms * 1e-3) / 1e9,
                          "hbm_frac": 8.0 * nvox / (ms * 1e-3) / 1e9 / hbm_peak}
        # NEXT-1: the paper's K-sample kernel (K = 32 GPU value, 15 CPU value), fused EM pass + update
        for K in (32, 15):
            ctx = pkg.Context(cfg.radius_mm, cfg.axial_mm, g, cfg.tof_fwhm_ps)
            ctx.set_option(pkg.OPT_SAMPLES_K, K)
            ctx.set_option(pkg.OPT_PROJECTOR, pkg.PROJECTOR_SAMPLED)
            image.fill_(1.0)
            corr.zero_()

            def pass_k():
                ctx.reset_stats()
                ctx.em_correction(sev, n, image, corr)
                ctx.update(image, corr, sens)

            pass_k()
            ms = timed(pass_k, reps=3)
            st = ctx.get_stats()
            res[f"sampled_K{K}_iteration"] = {"ms": ms, "events_per_s": n / (ms * 1e-3), "samples_kept": int(st.visits),
                                             "reductions": int(st.reductions), "n_valid": int(st.n_valid),
                                             "roofline_frac": st.reductions / (ms * 1e-3) / red_rand}
        out["config"] = {"workload": f"widened rows on cfg-3: {n} events, 160x160x640 x 3.75 mm"}
        out["results"] = res
    print(json.dumps(out))


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
    ap.add_argument("--ref-events", type=int, default=8_000_000,
                    help="events per step of --impl reference (the oracle's per-call cost of ~0.75 s -- one private fp64 "
                         "correction image per thread -- is amortised from a few million events on)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-bin", action="store_true", help="skip locality binning (for comparison)")
    ap.add_argument("--subbins", type=int, default=0, help="TOFMLEM_OPT_SUBBINS override (0 = library default)")
    ap.add_argument("--tile-log2", type=int, default=0, help="TOFMLEM_OPT_TILE_LOG2 override (0 = library default, 3)")
    ap.add_argument("--em-variant", type=int, default=-1, help="TOFMLEM_OPT_EM_VARIANT override (-1 = library default)")
    ap.add_argument("--cache-share", type=int, default=-1, help="TOFMLEM_OPT_CACHE_SHARE override")
    ap.add_argument("--tile", type=int, default=1,
                    help="1 (default): tofmlem_plan_events on the binned list (ray records + shared-memory tiles); 0: the "
                         "unplanned fused pass of round 1")
    ap.add_argument("--tile-min", type=int, default=0, help="TOFMLEM_OPT_TILE_MIN_EVENTS override")
    ap.add_argument("--tile-max", type=int, default=0, help="TOFMLEM_OPT_TILE_MAX_EVENTS override")
    ap.add_argument("--report", default="", choices=["", "sweep", "division", "next", "pipeline"],
                    help="extra single-GPU reports (one JSON line each, not the driver's bench line): cfg-5 TOF/scale "
                         "sweep, cfg-4 nine-region division vs unsplit, timings of the widened rows (NEXT-1..4)")
    ap.add_argument("--sens-sort", type=int, default=-1, help="TOFMLEM_OPT_SENS_SORT override")
    ap.add_argument("--concurrent", type=int, default=-1, help="TOFMLEM_OPT_CONCURRENT override")
    ap.add_argument("--l2-persist", type=int, default=-1, help="TOFMLEM_OPT_L2_PERSIST override")
    ap.add_argument("--region-plan", type=int, default=-1, help="TOFMLEM_OPT_REGION_PLAN override (division report)")
    ap.add_argument("--division-iters", type=int, default=0, help="iterations of the division report (0 = the config's 5)")
    ap.add_argument("--sweep-events", default="10000000,146000000,500000000")
    ap.add_argument("--sweep-fwhm", default="100,300,600,0")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.report:
        return run_report(args)

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
    if args.tile_log2:
        ctx.set_option(pkg.OPT_TILE_LOG2, args.tile_log2)
    if args.em_variant >= 0:
        ctx.set_option(pkg.OPT_EM_VARIANT, args.em_variant)
    if args.cache_share >= 0:
        ctx.set_option(pkg.OPT_CACHE_SHARE, args.cache_share)
    if args.l2_persist >= 0:
        ctx.set_option(pkg.OPT_L2_PERSIST, args.l2_persist)
    if args.concurrent >= 0:
        ctx.set_option(pkg.OPT_CONCURRENT, args.concurrent)
    if args.sens_sort >= 0:
        ctx.set_option(pkg.OPT_SENS_SORT, args.sens_sort)
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
    # ---- a1: locality binning (one-off per data set); scratch of binning and plan allocated beforehand (tofmlem_reserve)
    bin_ms = 0.0
    ctx.reserve(n)
    if not args.no_bin:
        key = torch.empty(n, dtype=torch.int32, device=dev)
        perm = torch.empty(n, dtype=torch.int32, device=dev)
        sev = {k: torch.empty_like(v) for k, v in ev.items()}

        def do_bin():
            ctx.bin_events(ev, n, key, perm, None)
            ctx.permute_events(ev, perm, n, sev)

        bin_ms = timed(do_bin)
        n_valid_keys = int((key != -1).sum().item())
        del key, perm, ev
        ev = sev
    torch.cuda.empty_cache()
    plan, plan_ms = None, 0.0
    if args.tile and not args.no_bin:
        if args.tile_min:
            ctx.set_option(pkg.OPT_TILE_MIN_EVENTS, args.tile_min)
        if args.tile_max:
            ctx.set_option(pkg.OPT_TILE_MAX_EVENTS, args.tile_max)
        plan_ms = timed(lambda: ctx.plan_events(ev, n))
        plan = ctx.plan_info()

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
    n_valid_all = sharding.sum_over_ranks(int(st.n_valid), dev)  # the image was updated with the all-reduced correction

    # ---- roofline of the dominant kernel: see DESIGN.md "Measurement"
    hbm_peak, peak_src = load_peaks()
    visits = int(st.visits)
    tile_visits = int(st.tile_visits)
    t_tile_ms, t_direct_ms, t_strag_ms = ctx.pass_timing()  # CUDA events around the kernels of the last planned pass
    probe_buf = torch.zeros(nvox, dtype=torch.float32, device=dev)
    n_ops = 1 << 30
    red_rand = n_ops / (ctx.probe(0, probe_buf, n_ops) * 1e-3)
    red_row = n_ops / (ctx.probe(1, probe_buf, n_ops) * 1e-3)
    ld_rand = n_ops / (ctx.probe(2, probe_buf, n_ops) * 1e-3)
    ld_row = n_ops / (ctx.probe(3, probe_buf, n_ops) * 1e-3)
    red_rand_v4 = n_ops / (ctx.probe(5, probe_buf, n_ops) * 1e-3)  # the direct kernel's own instruction
    smem_add = n_ops / (ctx.probe(6, probe_buf, n_ops) * 1e-3)     # ATOMS.ADD on a 72 KB tile, 3 CTAs per SM
    smem_ld = n_ops / (ctx.probe(7, probe_buf, n_ops) * 1e-3)      # LDS, same pattern
    red_peak = max(red_rand, red_rand_v4)  # the roofline uses the HIGHER of the two request rates
    del probe_buf
    planned = plan is not None and bool(plan.active)
    rec_bytes = 48.0 if planned else 28.0
    hbm_bytes = rec_bytes * n  # algorithmic HBM bytes per pass: one ray record (or 7 float32) per event
    reds = int(st.reductions)  # reduction requests to the L2 atomic units (direct pass + tile flushes)
    t_hbm = hbm_bytes / (hbm_peak * 1e9)
    # the same pass against SURVEY.md 8(d)'s visit-based formula, T_roof = max(HBM, visits / R_gather, visits / R_red)
    # with the conflict-free RANDOM L2 rates, and against the COALESCED L2 rates of the same probes (what the method
    # would need with full sectors)
    t_roof_visits = max(t_hbm, visits / ld_rand, visits / red_rand)
    t_roof_row = max(t_hbm, visits / ld_row, visits / red_row)
    full_default = args.workload == "full" and not args.events and not args.no_bin
    probes = {"red_random": red_rand / 1e9, "red_random_v4": red_rand_v4 / 1e9, "red_row": red_row / 1e9,
              "gather_random": ld_rand / 1e9, "gather_row": ld_row / 1e9, "smem_add_random": smem_add / 1e9,
              "smem_load_random": smem_ld / 1e9}
    common = {
        "frac_visits": t_roof_visits / (kern_ms * 1e-3), "frac_l2_coalesced": t_roof_row / (kern_ms * 1e-3),
        "kernel_ms": kern_ms, "visits_per_launch": visits, "reductions_per_launch": reds,
        "visits_Gps": visits / (kern_ms * 1e-3) / 1e9, "probes_Gops": probes,
        "hbm": {"algorithmic_bytes": hbm_bytes, "achieved_GBs": hbm_bytes / (kern_ms * 1e-3) / 1e9, "peak_GBs": hbm_peak,
                "frac": hbm_bytes / (kern_ms * 1e-3) / 1e9 / hbm_peak, "peak_source": peak_src},
    }
    if planned and t_tile_ms > 0.0 and t_tile_ms >= t_direct_ms:
        # Dominant kernel: em_tile_kernel.  Every tile visit is one shared-memory load (forward walk) and one
        # shared-memory integer add (scatter walk) through the SM's shared-memory pipe: algorithmic time = visits x
        # (1 / R_load + 1 / R_add) with both rates measured on the tile pass's own footprint (probe kinds 6, 7).
        peak_vis = 1.0 / (1.0 / smem_ld + 1.0 / smem_add)
        ach = tile_visits / (t_tile_ms * 1e-3)
        roofline = {
            "bound": "smem_atomic", "achieved": ach / 1e9, "peak": peak_vis / 1e9, "unit": "G tile visits/s",
            "frac": ach / peak_vis,
            "kernel": "em_tile_kernel<384, 3, BRICK>", "dominant_kernel_ms": t_tile_ms,
            "tile_visits_per_launch": tile_visits,
            "traffic": TRAFFIC_BYTES if full_default else None,
            "traffic_source": TRAFFIC_SOURCE if full_default else None,
            "peak_source": "tofmlem_probe kinds 6 / 7: random ATOMS.ADD.U32 and LDS on a 72 KB shared-memory tile, 3 CTAs "
                           "of 384 threads per SM, measured in this run; one tile visit = one load + one add",
            # the second kernel of the step: the direct pass on records, bound by L2 reduction requests as in round 1
            "direct": {"kernel": "em_planned_kernel<v4, BRICK>", "kernel_ms": t_direct_ms + t_strag_ms,
                       "bound": "l2_atomic", "peak": red_peak / 1e9, "unit": "G reductions/s",
                       "note": "reductions_per_launch counts the direct pass's 16-byte reductions and the tiles' flushes"},
            # both kernels together: algorithmic time of the step over its measured time
            "frac_step": (tile_visits / peak_vis + (visits - tile_visits) / 1.5 / red_peak) / (kern_ms * 1e-3),
            **common,
        }
    else:
        achieved = reds / (kern_ms * 1e-3)
        roofline = {
            "bound": "l2_atomic", "achieved": achieved / 1e9, "peak": red_peak / 1e9, "unit": "G reductions/s",
            "frac": achieved / red_peak,
            "traffic": None, "traffic_source": None,
            "kernel": "em_planned_kernel<v4, BRICK>" if planned else "em_persistent_kernel<TOF, v4, BRICK>",
            "visits_per_reduction": visits / max(1, reds),
            "peak_source": "tofmlem_probe: random-address reductions into an L2-resident array of nvox floats, the higher of "
                           "the 4-byte (kind 0) and the 16-byte (kind 5) request rates, measured in this run",
            "t_roof_ms": {"hbm": t_hbm * 1e3, "red": reds / red_peak * 1e3, "gather": visits / ld_rand * 1e3},
            **common,
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

    # ---- cpu_baseline: the oracle on this box's host cores, bounded sample (rank 0, N = 1 only): exactly what
    # `--impl reference` times (same events, same order, same image), so the two arms describe one configuration
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu, _ = oracle_arm(cfg, args.ref_events, 3, 1)

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": make_config(cfg, n, m, world, binned=not args.no_bin),
            "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks,
            "setup": {"sensitivity_ms": sens_ms, "bin_sort_gather_ms": bin_ms, "plan_ms": plan_ms,
                      "recon_wall_s": (bin_ms + plan_ms + cfg.iters * ms_per_step) * 1e-3,
                      "recon_wall_note": f"binning + plan (ray records) + {cfg.iters} iterations, events resident in HBM"},
            "stats": {"n_valid": int(st.n_valid), "visits": visits, "visits_per_valid_event": visits / max(1, int(st.n_valid)),
                      "sum_image_sens": p7, "p7_rel_err": abs(p7 - n_valid_all) / max(1, n_valid_all),
                      "tile_events": int(st.tile_events),
                      "plan": None if plan is None else {"active": int(plan.active), "items": int(plan.n_tile_items),
                                                         "tile_events": int(plan.n_tile_events),
                                                         "direct_events": int(plan.n_direct_events),
                                                         "stragglers": int(plan.n_stragglers)}},
            "paper_context": "PAPER.md:17,:299 -- 3.5 min for the slowest of nine regions (20 iterations, Tesla C2075 + 16 CPU threads); context, not the target",
        }
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
