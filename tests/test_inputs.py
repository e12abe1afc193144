"""Host-side checks of the seeded input generator (no method arithmetic lives there)."""
import numpy as np
import torch

import hcms_inputs as I


def test_counter_based_and_deterministic():
    a = I.normal_f32(3, 1, 10000, threads=1)
    b = I.normal_f32(3, 1, 10000, threads=4)
    assert np.array_equal(a, b)
    # value i depends only on (seed, tensor, i): a longer stream has the same prefix
    c = I.normal_f32(3, 1, 5_000_000, threads=4)
    assert np.array_equal(c[:10000], a)
    assert not np.array_equal(I.normal_f32(4, 1, 1000), a[:1000])
    assert not np.array_equal(I.normal_f32(3, 2, 1000), a[:1000])


def test_distribution_is_standard_normal():
    x = I.normal_f32(0, 0, 2_000_000).astype(np.float64)
    assert abs(x.mean()) < 3e-3 and abs(x.std() - 1) < 3e-3
    assert abs((x ** 3).mean()) < 1e-2 and abs((x ** 4).mean() - 3) < 3e-2
    assert np.isfinite(x).all() and np.abs(x).max() < 9


def test_bf16_rounding_matches_library():
    x = I.normal_f32(1, 0, 100000)
    x = np.concatenate([x, np.float32([0.0, -0.0, 1.0, 1.00390625, 1.01171875, 3.3895314e38, np.inf, -np.inf, 1e-40])])
    bits = I.f32_to_bf16_bits(x)
    ref = torch.from_numpy(x).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)
    assert np.array_equal(bits, ref)
    assert np.array_equal(I.bf16_bits_to_f32(bits), torch.from_numpy(x).to(torch.bfloat16).float().numpy())


def test_workloads_match_baseline_json():
    w = I.WORKLOADS
    assert [(w[i].S, w[i].H, w[i].D, w[i].P, w[i].C) for i in range(1, 6)] == [
        (1024, 4, 64, 2, 2), (8192, 12, 64, 4, 2), (32760, 40, 128, 4, 4),
        (56160, 40, 128, 8, 2), (98304, 24, 128, 8, 3)]
    assert w[1].dtype == "f32" and w[1].seed == 0 and w[3].k_scale == 0.5
    q, k, v = I.make_qkv(w[1])
    assert q.dtype == np.float32 and q.shape == (1024, 4, 64)
    small = I.Workload("t", 64, 4, 8, 2, 2, 2, "bf16", 0.5)
    q, k, v = I.make_qkv(small)
    assert k.dtype == np.uint16
    k_unscaled = I.f32_to_bf16_bits(I.normal_f32(2, 1, 64 * 4 * 8).reshape(64, 4, 8))
    assert np.array_equal(I.bf16_bits_to_f32(k), I.bf16_bits_to_f32(k_unscaled) * np.float32(0.5))


def test_index_pattern_distinguishes_neighbours():
    x = I.index_pattern(16, 4, 8, np.uint32)
    assert len(np.unique(x)) == x.size
    y = I.index_pattern(16, 4, 8, np.uint16)
    assert len(np.unique(y)) > 0.95 * y.size
