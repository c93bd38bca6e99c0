"""The seeded input generator: determinism, logical-position addressing, distribution shape."""
import numpy as np
import torch

from paper_2511_20982_b200 import workloads as W


def test_mix64_tensor_matches_python_int():
    xs = [0, 1, 2, 0x9E3779B97F4A7C15, (1 << 63) + 12345, (1 << 64) - 1]
    t = torch.tensor([W._s64(x) for x in xs], dtype=torch.int64)
    got = [int(v) & W._MASK64 for v in W.mix64_t(t).tolist()]
    assert got == [W.mix64_i(x) for x in xs]
    # splitmix64 reference value: state 0 + gamma -> first output of splitmix64(seed=0)
    assert W.mix64_i(0x9E3779B97F4A7C15) == 0xE220A8397B1DCDAF


def test_normal_table_shape():
    t = W.normal_table().to(torch.float64)
    assert t.numel() == 65536 and torch.all(t[1:] >= t[:-1])
    assert abs(t.mean().item()) < 1e-3 and abs(t.std().item() - 1.0) < 5e-3
    assert torch.all(t == -t.flip(0))


def test_kv_values_are_a_function_of_logical_position():
    a = W.kv_values(7, W.KIND_K, 3, 2, 64, 0, 3, 0, 50)
    b = W.kv_values(7, W.KIND_K, 3, 2, 64, 1, 1, 10, 20)
    assert torch.equal(a[1:2, :, 10:20], b)                      # slice == regenerated slice
    assert not torch.equal(a, W.kv_values(7, W.KIND_V, 3, 2, 64, 0, 3, 0, 50))
    assert not torch.equal(a, W.kv_values(7, W.KIND_K, 4, 2, 64, 0, 3, 0, 50))
    assert not torch.equal(a, W.kv_values(8, W.KIND_K, 3, 2, 64, 0, 3, 0, 50))
    x = W.kv_values(1, W.KIND_V, 0, 8, 128, 0, 1, 0, 2048).to(torch.float64)
    assert abs(x.mean().item()) < 5e-3 and abs(x.std().item() - 1) < 5e-3
    q = W.q_values(1, 5, 2, 4, 8, 64)
    assert q.shape == (4, 8, 64) and q.dtype == torch.bfloat16
    assert torch.equal(q, W.q_values(1, 5, 2, 4, 8, 64))


def test_length_laws_follow_baseline_configs():
    c = W.CONFIGS
    assert list(c["cfg1_tiny"].draw_lengths()) == [17, 64, 130, 255]
    l2 = c["cfg2_7b_mha"].draw_lengths()
    assert l2.shape == (64,) and l2.min() >= 512 and l2.max() <= 2048
    l3 = c["cfg3_8b_gqa"].draw_lengths(20000)
    assert l3.min() >= 128 and l3.max() <= 8192 and 950 < np.median(l3) < 1100 and 1300 < l3.mean() < 1500
    l4 = c["cfg4_70b_long"].draw_lengths(20000)
    assert l4.min() >= 4096 and l4.max() <= 32768 and 18000 < l4.mean() < 18900
    l5 = c["cfg5_stress"].draw_lengths(20000)
    long = l5 >= 8192
    assert 0.18 < long.mean() < 0.22 and l5[~long].max() <= 256 and l5[~long].min() >= 64 and l5.max() <= 16384
    assert np.array_equal(c["cfg3_8b_gqa"].draw_lengths(), c["cfg3_8b_gqa"].draw_lengths())
    assert not np.array_equal(c["cfg3_8b_gqa"].draw_lengths(salt=1), c["cfg3_8b_gqa"].draw_lengths())
    for w in c.values():
        assert w.max_len >= int(w.draw_lengths(1000).max())
