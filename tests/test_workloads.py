"""The seeded input generator: deterministic, counter-based, right moments, exact bf16 widening."""
import numpy as np
import torch

from paper_2507_16697_b200 import workloads as w


def test_counter_based_and_deterministic():
    a = w.normal_f32(5000, seed=7, tensor_id=1)
    b = w.normal_f32(5000, seed=7, tensor_id=1, chunk=777)     # chunking must not matter
    assert torch.equal(a, b)
    assert not torch.equal(a, w.normal_f32(5000, seed=8, tensor_id=1))
    assert not torch.equal(a, w.normal_f32(5000, seed=7, tensor_id=2))


def test_moments():
    x = w.normal_f32(1 << 20, seed=3, tensor_id=0).double()
    assert abs(x.mean()) < 5e-3 and abs(x.std() - 1) < 5e-3
    assert abs((x ** 4).mean() - 3) < 5e-2
    assert abs((x[:-1] * x[1:]).mean()) < 5e-3


def test_config_tensors_and_exact_widening():
    cfg = w.CONFIGS["C1"]
    q, k, v = w.make_qkv(cfg)
    assert q.shape == (1, 1, 1024, 64) and q.dtype == torch.float32 and q.is_contiguous()
    assert not torch.equal(q, k)
    qb = w.make_tensor((1, 2, 128, 64), "q", seed=5, dtype="bf16", gain=3.0)
    assert qb.dtype == torch.bfloat16
    wide = w.to_f64_numpy(qb)
    assert wide.dtype == np.float64
    assert torch.equal(torch.from_numpy(wide).to(torch.bfloat16), qb)       # lossless round trip
    assert abs(wide.std() - 3.0) < 0.1


def test_flop_counts_match_baseline_md():
    assert abs(w.CONFIGS["C3"].fwd_flops - 2.81e14) / 2.81e14 < 5e-3
    assert abs(w.CONFIGS["C4"].bwd_flops - 8.80e13) / 8.80e13 < 5e-3
    assert w.voxel_token_index(1, 2, 3, 32) == 1 + 32 * (2 + 32 * 3)
