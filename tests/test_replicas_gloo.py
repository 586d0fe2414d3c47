"""The N>1 plumbing (replicas only) on CPU: two gloo ranks run the same
helpers bench.py uses -- barrier, max/sum over ranks, by-sequence sharding -- and each rank runs
the ORACLE on its own shard of one batch; the union of the shards must equal the unsharded result
bit for bit (the path has no exchange step, so sharding by sequence cannot change any row)."""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, tmpdir: str):
    sys.path.insert(0, ROOT)
    os.environ.update({"RANK": str(rank), "LOCAL_RANK": str(rank), "WORLD_SIZE": str(world),
                       "MASTER_ADDR": "127.0.0.1", "MASTER_PORT": str(port)})
    import oracle
    from paper_2605_30842_b200 import replicas
    from paper_2605_30842_b200 import workloads as W

    r, lr, ws = replicas.init("gloo")
    assert (r, lr, ws) == (rank, rank, world)
    replicas.barrier()
    # timing reduction: max over ranks; work reduction: sum over ranks
    assert replicas.max_over_ranks(10.0 + rank) == 10.0 + (world - 1)
    assert replicas.sum_over_ranks(100 * (rank + 1)) == 100 * world * (world + 1) / 2

    lens = [700, 33, 0, 1500, 16, 257, 900]
    batch = W.make_batch(lens, 8, 2, 64, 16, seed=77, device="cpu")
    shards = replicas.shard_sequences(lens, world)
    mine = shards[rank]
    pairs = [(b, h) for b in mine for h in range(8)]
    out, lse = oracle.decode_attn(batch.q, batch.k_pages, batch.v_pages, batch.block_table,
                                  batch.seq_lens, batch.softmax_scale, pairs=pairs, num_threads=1)
    np.save(os.path.join(tmpdir, f"out_{rank}.npy"), out)
    np.save(os.path.join(tmpdir, f"idx_{rank}.npy"), np.array(mine, dtype=np.int64))
    replicas.barrier()
    replicas.finalize()


@pytest.mark.timeout(180)
def test_two_rank_replicas_gloo(tmp_path, oracle):
    world = 2
    port = _free_port()
    mp.spawn(_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True)

    from paper_2605_30842_b200 import workloads as W
    lens = [700, 33, 0, 1500, 16, 257, 900]
    batch = W.make_batch(lens, 8, 2, 64, 16, seed=77, device="cpu")
    full, _ = oracle.decode_attn(batch.q, batch.k_pages, batch.v_pages, batch.block_table,
                                 batch.seq_lens, batch.softmax_scale, num_threads=1)
    full = full.reshape(len(lens), 8, 64)
    seen = []
    for r in range(world):
        idx = np.load(tmp_path / f"idx_{r}.npy").tolist()
        out = np.load(tmp_path / f"out_{r}.npy").reshape(len(idx), 8, 64)
        for j, b in enumerate(idx):
            assert np.array_equal(out[j], full[b])      # bit-identical: no exchange step exists
        seen += idx
    assert sorted(seen) == list(range(len(lens)))       # every sequence on exactly one rank


def test_shard_sequences_is_balanced_and_deterministic():
    from paper_2605_30842_b200 import replicas
    from paper_2605_30842_b200 import workloads as W

    lens = W.ragged_lens(32, 8192, 65536, 1003)
    for world in (1, 2, 4, 8):
        sh = replicas.shard_sequences(lens, world)
        assert sh == replicas.shard_sequences(lens, world)
        assert sorted(i for s in sh for i in s) == list(range(32))
        loads = [sum(lens[i] for i in s) for s in sh]
        assert max(loads) - min(loads) <= max(lens)     # greedy longest-first bound
