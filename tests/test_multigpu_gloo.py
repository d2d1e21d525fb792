"""N > 1 path on CPU: two gloo ranks run the host-side logic of the event-sharded iteration (shard ranges, the one
all-reduce of the correction image, identical update on every rank).  The per-shard EM pass itself is stood in for by
the oracle here (there is no GPU in this test); what is checked is the sharding/exchange logic that bench.py --gpus N
uses: the sharded result equals the single-process result and is identical on both ranks."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import oracle
import synth
from paper_1706_07075_b200 import sharding


def test_shard_ranges_tile():
    for n in (0, 1, 7, 200_000, 146_000_000):
        for world in (1, 2, 3, 8):
            r = [sharding.shard_range(n, k, world) for k in range(world)]
            assert r[0][0] == 0 and sum(c for _, c in r) == n
            for (s0, c0), (s1, _) in zip(r, r[1:]):
                assert s0 + c0 == s1
            assert max(c for _, c in r) - min(c for _, c in r) <= 1
    assert sharding.weak_shard_range(1000, 3) == (3000, 1000)
    with pytest.raises(ValueError):
        sharding.shard_range(10, 2, 2)


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _problem():
    cfg = synth.TINY
    n = 6001
    g = oracle.make_grid(16, 16, 16, 8.0)
    ev = {k: v.numpy() for k, v in synth.make_events(cfg, n).items()}
    lors = {k: v.numpy() for k, v in synth.make_sens_lors(cfg, 50_000).items()}
    sens = oracle.sensitivity(g, lors).astype(np.float32)
    return cfg, n, g, ev, sens


def _rank_main(rank: int, world: int, port: int, out_dir: str):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        cfg, n, g, ev, sens = _problem()
        sig = oracle.sigma_mm(cfg.tof_fwhm_ps)
        mask = oracle.mask_f32(sens)
        x = mask.astype(np.float64)
        start, count = sharding.shard_range(n, rank, world)
        shard = {k: v[start:start + count] for k, v in ev.items()}
        n_valid = 0
        for _ in range(2):
            corr, nv, _ = oracle.em_correction(g, sig, shard, x)
            t = torch.from_numpy(corr)
            sharding.allreduce_correction(t)  # the iteration's one exchange
            x = oracle.update(x, t.numpy(), sens, mask)
            n_valid = nv
        ms = sharding.max_over_ranks_ms(10.0 + rank)
        nv_all = sharding.sum_over_ranks(n_valid)  # what bench.py compares sum(image * sens) with (P7)
        np.savez(os.path.join(out_dir, f"rank{rank}.npz"), x=x, ms=ms, n_valid=nv_all)
    finally:
        dist.destroy_process_group()


def test_two_rank_gloo_iteration_matches_single_process(tmp_path):
    world = 2
    mp.start_processes(_rank_main, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True,
                       start_method="spawn")
    cfg, n, g, ev, sens = _problem()
    sig = oracle.sigma_mm(cfg.tof_fwhm_ps)
    mask = oracle.mask_f32(sens)
    ref, st = oracle.mlem(g, sig, ev, mask.astype(np.float64), sens, 2)
    r0 = np.load(os.path.join(tmp_path, "rank0.npz"))
    r1 = np.load(os.path.join(tmp_path, "rank1.npz"))
    assert np.array_equal(r0["x"], r1["x"])  # every rank applies the same update to the same summed correction
    assert np.allclose(r0["x"], ref, rtol=1e-11, atol=0)
    assert int(r0["n_valid"]) == st.n_valid
    assert float(r0["ms"]) == 11.0 and float(r1["ms"]) == 11.0  # max over ranks
    # P7 holds for the sharded iteration as well
    assert abs(float((r0["x"] * sens.astype(np.float64)).sum()) - st.n_valid) <= 1e-9 * st.n_valid
