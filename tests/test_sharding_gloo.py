"""world_size-2 gloo test (CPU) of the N>1 path: the path shards over independent batches
with no data-path collective, so the host logic to cover is the shard
arithmetic and the max-over-ranks timing reduction.  The per-rank compute stand-in is the
oracle (tests may use it); concatenating the ranks' slices must equal the unsharded result."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2606_00601_b200.sharding import max_over_ranks, shard_range, sum_over_ranks


def test_shard_range_partitions_exactly():
    for n in (0, 1, 7, 8, 9, 4096):
        for world in (1, 2, 3, 8):
            spans = [shard_range(n, r, world) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == n
            for (a, b), (c, d) in zip(spans, spans[1:]):
                assert b == c and a <= b and c <= d
            sizes = [b - a for a, b in spans]
            assert max(sizes) - min(sizes) <= 1


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import oracle
        from workloads import config, make_selective_inputs, to_f64_numpy
        c = config(2, batch=5, d_inner=6, L=64)
        inp = {k: to_f64_numpy(v) for k, v in make_selective_inputs(c).items()}
        lo, hi = shard_range(c.batch, rank, world)
        y, hl = oracle.selective_scan_fwd(inp["x"][lo:hi], inp["delta"][lo:hi], inp["A"],
                                          inp["B"][lo:hi], inp["C"][lo:hi], inp["D"], None)
        np.save(os.path.join(out_dir, f"y{rank}.npy"), y)
        np.save(os.path.join(out_dir, f"hl{rank}.npy"), hl)
        # timing reduction: max over ranks, and unit counts sum over ranks
        assert max_over_ranks(10.0 + rank) == 10.0 + world - 1
        assert sum_over_ranks(float(hi - lo)) == float(c.batch)
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_two_rank_batch_sharding_matches_unsharded(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    import oracle
    from workloads import config, make_selective_inputs, to_f64_numpy
    c = config(2, batch=5, d_inner=6, L=64)
    inp = {k: to_f64_numpy(v) for k, v in make_selective_inputs(c).items()}
    y, hl = oracle.selective_scan_fwd(inp["x"], inp["delta"], inp["A"], inp["B"], inp["C"],
                                      inp["D"], None)
    ys = np.concatenate([np.load(tmp_path / f"y{r}.npy") for r in range(world)])
    hls = np.concatenate([np.load(tmp_path / f"hl{r}.npy") for r in range(world)])
    assert np.array_equal(ys, y) and np.array_equal(hls, hl)
