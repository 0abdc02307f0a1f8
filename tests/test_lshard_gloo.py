"""world_size-2 (and 3) gloo tests, on CPU, of the L-sharded scan's plumbing
(paper_2606_00601_b200/sharding.py::selective_scan_fwd_l_sharded): slice ->
aggregate -> all-gather -> compose the carry -> final scan.  The three compute steps are injected:
here they are the float64 oracle (tests may use it), so what is tested is the exchange step, the
rank order of the composition (Eq.7: later on the left) and the slicing."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2606_00601_b200.sharding import selective_scan_fwd_l_sharded, shard_range_aligned


def test_aligned_shards_partition_exactly_on_vector_boundaries():
    for n in (0, 8, 15, 16, 2048, 2049, 65536 + 3):
        for world in (1, 2, 3, 8):
            spans = [shard_range_aligned(n, r, world, 8) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == n
            for (a, b), (c, d) in zip(spans, spans[1:]):
                assert b == c and a <= b and b % 8 == 0 or b == n


class OracleOps:
    """The three compute steps of the L-sharded scan, stated with the oracle (float64 inside,
    fp32 tensors at the interface like the CUDA entry points)."""

    calls = {"aggregate": 0, "compose": 0, "fwd": 0}

    @staticmethod
    def _np(t):
        return None if t is None else t.double().numpy()

    @classmethod
    def selective_scan_slice_aggregate(cls, x, delta, A, B, C, P, U):
        import oracle
        cls.calls["aggregate"] += 1
        f = cls._np
        # U: state after the slice entered with h = 0; P: the same call's response to h0 = 1
        # with u = 0 (x = 0): the total product of a_t -- two oracle calls, no closed form
        _, u = oracle.selective_scan_fwd(f(x), f(delta), f(A), f(B), f(C), None, None)
        ones = np.ones(tuple(P.shape))
        _, p = oracle.selective_scan_fwd(np.zeros_like(f(x)), f(delta), f(A), f(B), f(C), None, ones)
        P.copy_(torch.from_numpy(p))
        U.copy_(torch.from_numpy(u))

    @classmethod
    def compose_carry(cls, P_all, U_all, h0, h_in, rank):
        import oracle
        cls.calls["compose"] += 1
        assert P_all.shape[0] > rank
        h = np.zeros(tuple(h_in.shape)) if h0 is None else h0.double().numpy().copy()
        for j in range(rank):                     # earlier ranks first; later on the left
            Pj, Uj = P_all[j].double().numpy(), U_all[j].double().numpy()
            flat = [oracle.compose((float(p), float(u)), (0.0, float(v)))[1]
                    for p, u, v in zip(Pj.ravel(), Uj.ravel(), h.ravel())]
            h = np.asarray(flat).reshape(h.shape)
        h_in.copy_(torch.from_numpy(h))

    @classmethod
    def selective_scan_fwd(cls, x, delta, A, B, C, D, h0, y, h_last):
        import oracle
        cls.calls["fwd"] += 1
        f = cls._np
        yy, hl = oracle.selective_scan_fwd(f(x), f(delta), f(A), f(B), f(C), f(D), f(h0))
        y.copy_(torch.from_numpy(yy))
        h_last.copy_(torch.from_numpy(hl))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _problem():
    from workloads import config, make_selective_inputs
    c = config(2, batch=2, d_inner=5, N=4, L=203, dtype=torch.float64)
    return make_selective_inputs(c, with_h0=True)


def _worker(rank, world, port, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        inp = _problem()
        L = inp["x"].shape[2]
        lo, hi = shard_range_aligned(L, rank, world, 8)
        sl = {k: (v[..., lo:hi].contiguous() if k in ("x", "delta", "B", "C") else v)
              for k, v in inp.items()}
        y = torch.empty_like(sl["x"])
        h_last = torch.empty((2, 5, 4), dtype=torch.float64)
        # the interface tensors of the CUDA path are fp32; the oracle ops accept any float dtype
        selective_scan_fwd_l_sharded(sl["x"], sl["delta"], sl["A"].double(), sl["B"], sl["C"],
                                     sl["D"].double(), sl["h0"].double(), y, h_last, ops=OracleOps)
        # rank 0 needs no carry, nobody consumes the last rank's aggregate: neither is computed
        assert OracleOps.calls == {"aggregate": int(rank < world - 1), "compose": int(rank > 0),
                                   "fwd": 1}, OracleOps.calls
        np.save(os.path.join(out_dir, f"y{rank}.npy"), y.numpy())
        np.save(os.path.join(out_dir, f"hl{rank}.npy"), h_last.numpy())
        dist.barrier()
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_l_sharded_scan_equals_unsharded(tmp_path, world):
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    import oracle
    inp = _problem()
    f = lambda t: None if t is None else t.double().numpy()  # noqa: E731
    y, hl = oracle.selective_scan_fwd(f(inp["x"]), f(inp["delta"]), f(inp["A"]), f(inp["B"]),
                                      f(inp["C"]), f(inp["D"]), f(inp["h0"]))
    ys = np.concatenate([np.load(tmp_path / f"y{r}.npy") for r in range(world)], axis=2)
    # fp32 P/U messages between the ranks (as on the GPU path) bound the agreement
    np.testing.assert_allclose(ys, y, rtol=2e-6, atol=2e-6)
    for r in range(world):                                    # every rank returns the global h_last
        np.testing.assert_allclose(np.load(tmp_path / f"hl{r}.npy"), hl, rtol=2e-6, atol=2e-6)
