"""Pins of the input recipe: frequency tables (inputs of the kvr_* calls) and the structure of the five
BASELINE.json configs.  No method arithmetic is tested here."""
import os

import numpy as np
import pytest

from workloads import config, config_small, inv_freq_llama3, inv_freq_standard, pos_map_with_gaps

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def test_llama3_inv_freq_spot_values_and_classes():
    f = inv_freq_llama3(5e5, 128, 8.0, 1.0, 4.0, 8192)
    base = inv_freq_standard(5e5, 128)
    for line in open(os.path.join(GOLDEN, "llama3_inv_freq_spots.txt")):
        if line.startswith("#") or not line.strip():
            continue
        i, v = line.split()
        assert abs(f[int(i)] / float(v) - 1) <= 1e-13
    assert np.array_equal(f[:29], base[:29])                  # high-frequency pairs unchanged
    assert np.allclose(f[35:], base[35:] / 8.0, rtol=1e-15)   # low-frequency pairs / factor
    assert np.all(f[29:35] < base[29:35]) and np.all(f[29:35] > base[29:35] / 8.0)
    assert np.all(np.diff(f) < 0)                             # monotone decreasing


def test_llama3_inv_freq_vs_transformers():
    ru = pytest.importorskip("transformers.modeling_rope_utils")
    cfg_mod = pytest.importorskip("transformers")
    cfg = cfg_mod.LlamaConfig(hidden_size=4096, num_attention_heads=32, max_position_embeddings=131072,
                              rope_parameters=dict(rope_type="llama3", rope_theta=5e5, factor=8.0,
                                                   low_freq_factor=1.0, high_freq_factor=4.0,
                                                   original_max_position_embeddings=8192))
    inv, _ = ru.ROPE_INIT_FUNCTIONS["llama3"](cfg, "cpu")
    ours = inv_freq_llama3(5e5, 128, 8.0, 1.0, 4.0, 8192)
    assert np.max(np.abs(inv.double().numpy() / ours - 1)) <= 4e-7     # the library table is fp32


def test_standard_inv_freq():
    f = inv_freq_standard(1e4, 64)
    assert f[0] == 1.0 and abs(f[16] - 1e-2) < 1e-15 and f.shape == (32,)
    assert abs(inv_freq_standard(1e6, 128)[32] - 1e-3) < 1e-15


def test_pos_map_law():
    pm = pos_map_with_gaps(65536, 100000, 0.05, 64, 1)
    d = np.diff(pm.astype(np.int64))
    assert pm[0] == 100000 and d.min() == 1 and d.max() <= 65
    assert 0.04 < np.mean(d > 1) < 0.06
    assert np.array_equal(pm, pos_map_with_gaps(65536, 100000, 0.05, 64, 1))     # seeded


def test_config_shapes():
    w0, w1, w2, w3, w4 = (config(c) for c in range(5))
    assert (w0.layers, w0.kv_heads, w0.head_dim, w0.tokens, w0.num_blocks) == (2, 2, 64, 128, 16)
    assert (w1.layers, w1.kv_heads, w1.head_dim, w1.tokens) == (36, 8, 128, 4096)
    assert w1.block_table.shape == (1, 381) and w1.num_blocks == 1024
    assert sorted(s.len for s in w2.segments) == [512, 2048, 8192, 16384] and w2.tokens == 27136
    assert max(s.dst_token_start + s.len for s in w2.segments) <= 32768 and w2.num_blocks == 4096
    assert len(w3.segments) == 192 and w3.dtype == "fp8" and w3.k_scale.shape == (256,)
    assert all(256 <= s.len <= 4096 for s in w3.segments)
    assert 0.5 <= w3.k_scale.min() and w3.k_scale.max() <= 2.0
    assert (w4.layers, w4.kv_heads, w4.rotary_dim, w4.pairing, w4.tokens) == (48, 4, 64, "gptj", 65536)
    assert np.all(w4.block_table[0, :6250] == -1) and np.all(w4.block_table[0, 6250:] >= 0)
    for w in (w0, w1, w2, w3, w4):
        # segments of one sequence never overlap; every touched block is allocated and distinct
        used = w.block_table[w.block_table >= 0]
        assert len(np.unique(used)) == len(used) and used.max() < w.num_blocks
        for q in range(w.block_table.shape[0]):
            iv = sorted((s.dst_token_start, s.dst_token_start + s.len) for s in w.segments if s.dst_seq == q)
            assert all(a[1] <= b[0] for a, b in zip(iv, iv[1:]))
            for a, b in iv:
                assert np.all(w.block_table[q, a // w.block_size:-(-b // w.block_size)] >= 0)


def test_small_configs_span_tiles_and_ragged_tails():
    for c in range(1, 5):
        w = config_small(c)
        assert w.tokens >= 512 and w.tokens * w.layers * w.kv_heads * w.head_dim <= 40e6
    assert any(s.dst_token_start % 16 for s in config_small(2).segments)
