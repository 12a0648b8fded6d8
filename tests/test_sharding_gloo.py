"""World-size-2 (gloo, CPU) test of the multi-rank plumbing: conformer sharding, max-over-ranks timing and the
gather of per-rank profiles.  The per-rank 'profiles' here are oracle outputs -- the data path has no collective,
so what is tested is only that the shards tile the batch and are reassembled in order."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1306_2258_b200 import sharding


def test_shard_range_tiles_everything():
    for n in (0, 1, 5, 1024, 1031):
        for world in (1, 2, 3, 8):
            cover = []
            for r in range(world):
                lo, hi = sharding.shard_range(n, r, world)
                cover += list(range(lo, hi))
                assert 0 <= hi - lo <= n // world + 1
            assert cover == list(range(n))


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close(); return p


def _worker(rank, world, port, tmp):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from oracle import oracle as orc
    from paper_1306_2258_b200 import workloads as wl
    w = wl.cfg4(B=5, N=120)
    lo, hi = sharding.shard_range(w.B, rank, world)
    local = torch.from_numpy(orc.debye_batch(w.xyz[lo:hi], w.type, w.fftab, w.q))
    full = sharding.gather_profiles(local, w.B, rank, world)
    # q-grid split of ONE structure: each rank computes a slice of q, the slices are gathered
    one = wl.small_random(3, 90, 3, 23)
    fn = lambda f, q: torch.from_numpy(orc.debye_sym(one.xyz, one.type, f.numpy(), q.numpy()))
    loc, (qlo, qhi) = sharding.profile_q_slice(fn, torch.from_numpy(one.fftab), torch.from_numpy(one.q), rank, world)
    fullq = sharding.gather_q_slices(loc, one.M, rank, world)
    if rank == 0:
        np.save(os.path.join(tmp, "fullq.npy"), fullq.numpy())
    # tile split of ONE structure: each rank contributes partial sums, all-gathered in rank order
    part = torch.full((2, 3, 7), float(rank + 1), dtype=torch.float64) * torch.arange(7, dtype=torch.float64)
    allp = sharding.gather_partials(part, world)
    if rank == 1:
        np.save(os.path.join(tmp, "allp.npy"), allp.numpy())
    # the whole helper with stand-ins for the two library calls: every rank must end with the rank-ordered sum
    tot = sharding.profile_tile_split(lambda r, wd: (torch.full((1, 3, 7), float(10 ** r), dtype=torch.float64), None),
                                      lambda S, n, f: (S * torch.arange(1, S.shape[0] + 1, dtype=torch.float64)[:, None, None, None]).sum(0),
                                      None, rank, world)
    np.save(os.path.join(tmp, f"tot{rank}.npy"), tot.numpy())
    # every rank must have built the same static schedule (same pairs grid): agreeing grids pass, differing ones raise everywhere
    sharding.assert_same_schedule(2368, world)
    try:
        sharding.assert_same_schedule(2368 + rank, world)
        raised = False
    except RuntimeError:
        raised = True
    np.save(os.path.join(tmp, f"raised{rank}.npy"), np.array([raised]))
    t = sharding.max_over_ranks(1.0 + rank)
    s = sharding.sum_over_ranks(hi - lo)
    if rank == 0:
        np.save(os.path.join(tmp, "full.npy"), full.numpy())
        np.save(os.path.join(tmp, "ts.npy"), np.array([t, s]))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_gloo_shards_and_gathers(tmp_path):
    mp.spawn(_worker, args=(2, _free_port(), str(tmp_path)), nprocs=2, join=True)
    from oracle import oracle as orc
    from paper_1306_2258_b200 import workloads as wl
    w = wl.cfg4(B=5, N=120)
    full = np.load(tmp_path / "full.npy")
    assert full.shape == (5, w.M)
    assert np.array_equal(full, orc.debye_batch(w.xyz, w.type, w.fftab, w.q))
    one = wl.small_random(3, 90, 3, 23)
    assert np.array_equal(np.load(tmp_path / "fullq.npy"), orc.debye_sym(one.xyz, one.type, one.fftab, one.q))
    allp = np.load(tmp_path / "allp.npy")
    assert allp.shape == (2, 2, 3, 7)
    for r in range(2):
        assert np.array_equal(allp[r], np.broadcast_to((r + 1) * np.arange(7.0), (2, 3, 7)))
    for r in range(2):      # 1 * 10^0 + 2 * 10^1: the parts arrive in rank order on every rank
        assert np.array_equal(np.load(tmp_path / f"tot{r}.npy"), np.full((1, 3, 7), 21.0))
    t, s = np.load(tmp_path / "ts.npy")
    assert t == 2.0 and s == 5.0
    assert np.load(tmp_path / "raised0.npy")[0] and np.load(tmp_path / "raised1.npy")[0]


def test_bench_refuses_more_gpus_than_the_node_has():
    """`python bench.py --gpus N` starts N ranks itself (torch.distributed.run on 127.0.0.1) -- and says so, with a non-zero
    exit status, when the node has fewer than N CUDA devices (here: none) instead of measuring fewer GPUs than it reports."""
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK")}
    env["CUDA_VISIBLE_DEVICES"] = ""
    r = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--steps", "1", "--warmup", "1"],
                       capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode != 0 and "needs 2 CUDA devices" in (r.stderr + r.stdout)
    env["WORLD_SIZE"] = "4"            # under a launcher the two counts must agree
    r = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2"], capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode != 0 and "WORLD_SIZE=4" in (r.stderr + r.stdout)
