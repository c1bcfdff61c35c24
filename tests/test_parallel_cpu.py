"""Host-side logic of the N > 1 path on CPU: two gloo ranks exchange ragged key
lists exactly as paper_2112_06613_b200.parallel does over NCCL, and the union / degree sum equal
the oracle's network.  (The shards' keys themselves come from the CUDA kernels: test_parity_gpu.py
checks on one GPU that the shards partition the edge set.)"""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from cdr3_synth import generate


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, keys_by_rank, n: int, out_dir: str):
    from paper_2112_06613_b200 import parallel
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    try:
        mine = torch.from_numpy(keys_by_rank[rank])
        allk = parallel.all_gather_v(mine)
        # degrees of this rank's shard, then the all-reduce of the rank-partitioned variant
        u, v = (mine >> 32).numpy(), (mine & 0xffffffff).numpy()
        deg = np.bincount(u, minlength=n) + np.bincount(v, minlength=n)
        total = parallel.sum_degrees(torch.from_numpy(deg.astype(np.int64)))
        np.save(os.path.join(out_dir, f"keys{rank}.npy"), allk.numpy())
        np.save(os.path.join(out_dir, f"deg{rank}.npy"), total.numpy())
        # ragged edge case: one rank contributes nothing
        empty = parallel.all_gather_v(mine[:0] if rank == 0 else mine[:5])
        assert empty.numel() == 5 and torch.equal(empty, torch.from_numpy(keys_by_rank[1][:5]))

        # parallel.build_distributed itself, end to end, on a stand-in for the context: build_shard hands out this
        # rank's share of the oracle's keys (what tcrnet_build_shard does with the work items), assemble collects
        class Net:
            def __init__(self):
                self.calls = []

            def build_shard(self, l_max, shard, n_shards):
                self.calls.append((l_max, shard, n_shards))
                return torch.from_numpy(keys_by_rank[shard])

            def assemble(self, keys):
                self.keys = keys
                return int(keys.numel())

        net = Net()
        n_edges = parallel.build_distributed(net, 2)
        assert net.calls == [(2, rank, world)]
        assert n_edges == sum(k.size for k in keys_by_rank)
        np.save(os.path.join(out_dir, f"built{rank}.npy"), net.keys.numpy())
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(300)
def test_two_rank_key_exchange_matches_oracle(tmp_path):
    import oracle
    d = generate("cfg1")
    pairs, _ = oracle.edges(d.residues, d.lengths, 2, tier=0)
    row_ptr, col, deg = oracle.csr(pairs, d.n)
    keys = (pairs[:, 0] << 32) | pairs[:, 1]
    # any partition of the edge set will do for the exchange logic: interleave like the work items
    keys_by_rank = [np.ascontiguousarray(keys[r::2]) for r in range(2)]
    port = _free_port()
    mp.spawn(_worker, args=(2, port, keys_by_rank, d.n, str(tmp_path)), nprocs=2, join=True)
    for r in range(2):
        got = np.load(tmp_path / f"keys{r}.npy")
        assert got.shape == keys.shape
        assert np.array_equal(got, np.concatenate(keys_by_rank))          # rank order, nothing lost
        assert np.array_equal(np.sort(got), keys)                          # the union is the edge set
        assert np.array_equal(np.load(tmp_path / f"deg{r}.npy"), deg.astype(np.int64))
        assert np.array_equal(np.sort(np.load(tmp_path / f"built{r}.npy")), keys)  # build_distributed: every rank, all edges


def test_single_process_is_identity():
    from paper_2112_06613_b200 import parallel
    t = torch.arange(7, dtype=torch.int64)
    assert parallel.sum_degrees(t).equal(t)
