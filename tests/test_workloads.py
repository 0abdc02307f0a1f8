"""CPU checks of the seeded input generators (workloads/gen.py): determinism, independence
of chunking, the distributions BASELINE.json's configs state, and that the module holds no
method arithmetic of its own (it imports neither the oracle nor the CUDA package)."""
import os

import torch

import workloads
import workloads.gen as gen


def test_counter_based_and_chunk_independent():
    a = gen.uniform((3, 100_000), 0, 1, seed=1, stream=0)
    old = gen._CHUNK
    try:
        gen._CHUNK = 4096
        b = gen.uniform((3, 100_000), 0, 1, seed=1, stream=0)
        n1 = gen.normal((50_000,), seed=2, stream=3)
        gen._CHUNK = old
        n2 = gen.normal((50_000,), seed=2, stream=3)
    finally:
        gen._CHUNK = old
    assert torch.equal(a, b) and torch.equal(n1, n2)
    assert not torch.equal(a, gen.uniform((3, 100_000), 0, 1, seed=2, stream=0))
    assert not torch.equal(a, gen.uniform((3, 100_000), 0, 1, seed=1, stream=1))
    # a prefix of a longer draw is the shorter draw (values depend on the flat index only)
    assert torch.equal(gen.uniform((1000,), 0, 1, seed=1, stream=0), a.reshape(-1)[:1000])


def test_moments():
    u = gen.uniform((1 << 20,), 0.5, 0.99, seed=3, stream=0)
    assert 0.5 <= u.min() and u.max() <= 0.99
    assert abs(u.mean().item() - 0.745) < 1e-3
    n = gen.normal((1 << 20,), seed=3, stream=1)
    assert abs(n.mean().item()) < 5e-3 and abs(n.std().item() - 1) < 5e-3
    assert abs((n ** 4).mean().item() - 3) < 0.05
    # streams are uncorrelated
    m = gen.normal((1 << 20,), seed=3, stream=2)
    assert abs((n * m).mean().item()) < 5e-3


def test_configs_match_baseline_json():
    c1 = workloads.config(1)
    assert (c1.num_seq, c1.L, c1.dtype) == (16, 1024, torch.float32)
    c2 = workloads.config(2)
    assert (c2.batch, c2.d_inner, c2.N, c2.L, c2.dtype) == (2, 768, 16, 2048, torch.float32)
    c3 = workloads.config(3)
    assert (c3.batch, c3.d_inner, c3.N, c3.L, c3.dtype) == (8, 4096, 16, 2048, torch.bfloat16)
    c4 = workloads.config(4)
    assert (c4.batch, c4.d_inner, c4.N, c4.L, c4.delta_shift) == (1, 1536, 16, 65536, -4.0)
    for logL in (10, 12, 14, 16, 18, 20):
        c5 = workloads.config(5, L=1 << logL)
        assert c5.elements == 1 << 30 and c5.h0_recipe == "normal"
    assert len({workloads.config(k).seed for k in range(1, 6)}) == 5


def test_input_recipes():
    inp = workloads.make_affine_inputs(workloads.config(1))
    assert inp["h0"] is None and inp["a"].dtype == torch.float32
    assert 0.5 <= inp["a"].min() and inp["a"].max() <= 0.99
    inp = workloads.make_affine_inputs(workloads.config(5, L=1024, total=1 << 16))
    assert inp["a"].shape == (64, 1024) and inp["h0"].shape == (64,)
    assert 0.9 <= inp["a"].min() and inp["a"].max() <= 0.9999
    c = workloads.config(3, d_inner=64, L=512, batch=2)
    inp = workloads.make_selective_inputs(c)
    assert inp["x"].dtype == torch.bfloat16 and inp["A"].dtype == torch.float32
    assert inp["B"].shape == (2, 16, 512) and inp["D"].shape == (64,)
    assert (inp["delta"].float() > 0).all()
    assert (inp["A"] < 0).all() and inp["A"].min() >= -2.7183 and inp["A"].max() <= -0.3678
    # delta = softplus(N(0,1) - 2): mean ≈ 0.175
    d = workloads.make_selective_inputs(workloads.config(2, d_inner=256))["delta"]
    assert abs(d.mean().item() - 0.175) < 0.01


def test_generator_module_is_independent():
    with open(os.path.join(os.path.dirname(gen.__file__), "gen.py")) as f:
        src = f.read()
    assert "import oracle" not in src and "paper_2606_00601_b200" not in src
