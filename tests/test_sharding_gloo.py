"""world_size-2 gloo test of the multi-GPU path (CPU): chains are sharded over ranks with no data-path collective, and
because the RNG is keyed by the global chain id the union of the per-rank results equals the single-process result.
The per-rank work is done by the ORACLE here (no GPU on this box); the GPU path takes the same (chain0, count)."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _worker(rank, world, port, n_chains, n_steps, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from oracle import hea_oracle as ho
    from paper_2411_18906_b200 import sharding, workloads
    w = workloads.config(1)
    o = ho.Oracle(*w.create_args())
    chain0, count = sharding.strong_chain_range(rank, world, n_chains)
    occ = o.init_random(count, w.seed, chain0=chain0)
    cnt, _, _ = o.sro_full(occ)
    st, _ = o.mc_run(occ, cnt, n_steps, w.K, w.seed, chain0=chain0, eval_all=False)
    # the only exchange is the read-out of the per-chain results (not on the data path)
    mine = torch.tensor(np.stack([st["hash"].astype(np.int64), st["n_accept"].astype(np.int64)], 1))
    sizes = [sharding.strong_chain_range(r, world, n_chains)[1] for r in range(world)]
    bufs = [torch.zeros((s, 2), dtype=torch.int64) for s in sizes]
    for r in range(world):                        # ragged split (3 + 2 chains): one broadcast per rank
        if rank == r:
            bufs[r] = mine
        dist.broadcast(bufs[r], src=r)
    if rank == 0:
        np.save(os.path.join(out_dir, "gathered.npy"), torch.cat(bufs).numpy())
    ranges = torch.tensor([chain0, count])
    all_ranges = [torch.zeros(2, dtype=torch.int64) for _ in range(world)]
    dist.all_gather(all_ranges, ranges)
    if rank == 0:
        np.save(os.path.join(out_dir, "ranges.npy"), torch.stack(all_ranges).numpy())
    dist.destroy_process_group()


def test_chain_sharding_matches_single_process(tmp_path):
    from oracle import hea_oracle as ho
    from paper_2411_18906_b200 import workloads
    n_chains, n_steps, world = 5, 120, 2            # ragged: 3 + 2 chains
    port = 29500 + (os.getpid() % 2000)
    mp.spawn(_worker, args=(world, port, n_chains, n_steps, str(tmp_path)), nprocs=world, join=True)
    got = np.load(tmp_path / "gathered.npy")
    ranges = np.load(tmp_path / "ranges.npy")
    assert ranges[:, 1].sum() == n_chains and ranges[0, 0] == 0
    assert all(ranges[r, 0] + ranges[r, 1] == ranges[r + 1, 0] for r in range(world - 1))     # a partition, in order
    w = workloads.config(1)
    o = ho.Oracle(*w.create_args())
    occ = o.init_random(n_chains, w.seed)
    cnt, _, _ = o.sro_full(occ)
    st, _ = o.mc_run(occ, cnt, n_steps, w.K, w.seed, eval_all=False)
    np.testing.assert_array_equal(got[:, 0], st["hash"].astype(np.int64))
    np.testing.assert_array_equal(got[:, 1], st["n_accept"].astype(np.int64))


def test_weak_and_strong_ranges():
    from paper_2411_18906_b200 import sharding
    assert [sharding.weak_chain_range(r, 16) for r in range(3)] == [(0, 16), (16, 16), (32, 16)]
    for world in (1, 2, 3, 8):
        for n in (0, 1, 7, 16, 1024):
            parts = [sharding.strong_chain_range(r, world, n) for r in range(world)]
            assert sum(c for _, c in parts) == n
            pos = 0
            for c0, c in parts:
                assert c0 == pos
                pos += c
            assert max(c for _, c in parts) - min(c for _, c in parts) <= 1
