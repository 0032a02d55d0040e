"""GPU parity for the representation adapters (Fig. 22):
M-RoPE image-KV (only the temporal pairs rotate; sectioned and interleaved layouts; Delta = 161) and the MLA
[latent | k_pe] cache (rotary window at an offset, no V tensor), plus rows that are not a power of two.
Same bar as tests/test_gpu_parity.py: slots, V and untouched bytes bit-exact, K within 2 bf16 ulps / 1 e4m3 step."""
import numpy as np
import pytest
import torch

from tests.helpers import K_TOL, k_distance, materialize_cpu, np_bits, run_oracle, torch_bits
from tests.test_gpu_parity import PATHS, _gpu, check_parity
from workloads import ADAPTERS, SENTINEL_BF16, adapter_config, adapter_small, make_workload

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("path", ["generic", "generic_vec", "ring"])
@pytest.mark.parametrize("layout", ["NHD", "HND"])
@pytest.mark.parametrize("name", ADAPTERS)
def test_adapter_small(name, layout, path):
    w = adapter_small(name, layout)
    d = check_parity(w, path)
    assert np.mean(d == 0) > 0.95


@pytest.mark.parametrize("name", ADAPTERS)
def test_adapter_auto_dispatch_takes_the_ring_kernel(name):
    w = adapter_small(name)
    srcs, _, _ = materialize_cpu(w)
    _, _, status, info = _gpu(w, srcs, dict(path=0))
    assert status[0] == 0 and info["path"] == PATHS["ring"], info


def _mla(pairing, dtype="bf16", layout="NHD", scales_differ=False, D=576, off=512, R=64, heads=1, bs=64, pad=0):
    return make_workload(name="mla", layers=3, kv_heads=heads, head_dim=D, rotary_dim=R, rotary_offset=off,
                         pairing=pairing, dtype=dtype, theta=1e4, block_size=bs, seed=43, has_v=False, layout=layout,
                         scales_differ=scales_differ, dst_head_pad=pad, slack=1.5,
                         seq_segments=[[dict(len=1, dst_token_start=3, new_start=3),
                                        dict(len=209, dst_token_start=7, new_start=1000, old_start=17),
                                        dict(len=66, dst_token_start=250, new_start=5, old_start=4000, src_row_pad=pad)],
                                       [dict(len=5, dst_token_start=0, new_start=0),
                                        dict(len=131, dst_token_start=6, new_start=161)]])


@pytest.mark.parametrize("path", ["generic", "generic_vec", "ring"])
@pytest.mark.parametrize("pairing,dtype,scales_differ,pad", [("gptj", "bf16", False, 0), ("neox", "bf16", False, 8),
                                                             ("gptj", "fp8", False, 0), ("neox", "fp8", True, 16),
                                                             ("gptj", "fp8", True, 0)])
def test_mla_edge_cases(pairing, dtype, scales_differ, pad, path):
    """1-token segment, negative Delta, Delta = 0, Delta = 161, two sequences, padded rows, fp8 with a scale change
    (the latent is then requantised)."""
    check_parity(_mla(pairing, dtype, scales_differ=scales_differ, pad=pad), path)


@pytest.mark.parametrize("tuning", [dict(max_ctas=3, stages=2, consumer_warps=1),
                                    dict(max_ctas=2, stages=7, consumer_warps=3),
                                    dict(max_ctas=1, stages=4, consumer_warps=4, layers_per_unit=1)])
def test_mla_ring_wraps(tuning):
    check_parity(adapter_small("mla-dsv2-lite"), "ring", **tuning)


@pytest.mark.parametrize("path", ["generic", "generic_vec", "ring"])
@pytest.mark.parametrize("layout", ["NHD", "HND"])
@pytest.mark.parametrize("pairing,D,R,off,dtype,has_v", [
    ("neox", 96, 64, 0, "bf16", True),      # head_dim 96 (192-byte rows): window mode with a V tensor
    ("gptj", 96, 32, 32, "bf16", True),     # rotary window in the middle of the row
    ("neox", 80, 64, 16, "bf16", True),     # 160-byte rows
    ("neox", 192, 64, 128, "fp8", True),    # fp8, window at the end
    ("gptj", 128, 64, 64, "bf16", True),    # power-of-two row, but an offset window
    ("neox", 48, 32, 16, "bf16", False)])
def test_rows_that_are_not_a_power_of_two(pairing, D, R, off, dtype, has_v, layout, path):
    pad = 8 if dtype == "bf16" else 16
    w = make_workload(name="win", layers=3, kv_heads=3, head_dim=D, rotary_dim=R, rotary_offset=off, pairing=pairing,
                      dtype=dtype, theta=1e4, block_size=8, layout=layout, seed=47, dst_head_pad=pad, slack=1.5,
                      has_v=has_v, scales_differ=(dtype == "fp8"),
                      seq_segments=[[dict(len=1, dst_token_start=3, new_start=3),
                                     dict(len=37, dst_token_start=7, new_start=1000, old_start=17),
                                     dict(len=14, dst_token_start=49, new_start=5, old_start=4000, src_row_pad=pad)],
                                    [dict(len=5, dst_token_start=0, new_start=0),
                                     dict(len=23, dst_token_start=6, new_start=161)]])
    check_parity(w, path)


@pytest.mark.parametrize("path", ["auto", "generic", "generic_vec"])
@pytest.mark.parametrize("pairing", ["neox", "gptj"])
def test_mla_inplace_refloat(pairing, path):
    """kvr_reposition_inplace on a resident [latent | k_pe] chunk: only the k_pe window changes; v_cache is NULL."""
    from oracle import kvr_oracle as orc
    from paper_2606_17107_b200 import kvr
    from paper_2606_17107_b200.harness import DeviceWorkload
    w = _mla(pairing)
    srcs, kc, _ = materialize_cpu(w)
    run_oracle(w, srcs, kc, None)                       # the chunk as spliced (oracle)
    dw = DeviceWorkload(w, "cuda:0", sources=[(torch_bits(k), None) for k, _ in srcs])
    dw.k_cache.copy_(torch_bits(kc))
    deltas = [9, 161, -1000, 0, 4097]
    with kvr.Context(dw.model) as ctx:
        ctx.set_tuning(path=0 if path == "auto" else PATHS[path])
        dw.run_inplace(ctx, dw.inplace_spans(deltas))
        assert ctx.last_device_status()[0] == 0
        assert ctx.last_launch_info()["path"] == (kvr.PATH_WINDOW if path == "auto" else PATHS[path])
    torch.cuda.synchronize()
    orc.inplace_workload(w, kc, deltas=deltas)
    got = np_bits(dw.k_cache)
    assert k_distance(w, got, kc).max() <= K_TOL[w.dtype]
    untouched = kc == SENTINEL_BF16
    assert np.array_equal(got[untouched], kc[untouched])


def test_mla_host_sources_and_write_span():
    from paper_2606_17107_b200 import kvr
    from paper_2606_17107_b200.harness import DeviceWorkload
    w = adapter_small("mla-dsv2-lite")
    srcs, kc, vc = materialize_cpu(w)
    dw = DeviceWorkload(w, "cuda:0", sources=[(torch_bits(k), None) for k, _ in srcs])
    dw.make_host_sources()
    with kvr.Context(dw.model) as ctx:
        dw.run_host(ctx)
        assert ctx.last_device_status()[0] == 0
        assert ctx.last_h2d_bytes() >= dw.bytes_moved() // 2
        torch.cuda.synchronize()
        run_oracle(w, srcs, kc, vc)
        assert k_distance(w, np_bits(dw.k_cache), kc).max() <= K_TOL[w.dtype]
        # span overwrite (Delta = 0 scatter) of the same rows: byte-exact source rows in the slots
        ctx.write_span(dw.dst, dw.write_spans())
        assert ctx.last_device_status()[0] == 0
    torch.cuda.synchronize()
    for s in w.segments:
        s.new_start = s.old_start
    run_oracle(w, srcs, kc, vc)
    assert np.array_equal(np_bits(dw.k_cache), kc)


@pytest.mark.parametrize("name", ["mla-dsv2-lite", "image-kv-qwen25vl-7b", "image-kv-qwen3vl-8b", "compose-qwen3-8b"])
def test_adapter_full_size_every_layer(name):
    """The launch configuration bench.py times (full-size workload, auto dispatch); the oracle checks every layer."""
    from paper_2606_17107_b200 import kvr
    from paper_2606_17107_b200.harness import DeviceWorkload, bits_to_numpy
    from oracle import kvr_oracle as orc
    w = adapter_config(name)
    layers = range(w.layers)
    dw = DeviceWorkload(w, "cuda:0", guard_bytes=1 << 16)
    with kvr.Context(dw.model) as ctx:
        dw.run(ctx)
        assert ctx.last_device_status()[0] == 0
        assert ctx.last_launch_info()["path"] == PATHS["ring"]
    torch.cuda.synchronize()
    s_l = w.dst_strides()[0]
    for l in layers:
        srcs = [(bits_to_numpy(k[l:l + 1]), None if v is None else bits_to_numpy(v[l:l + 1])) for k, v in dw.sources]
        import copy
        w1 = copy.copy(w)
        w1.layers = 1
        if w.k_scale is not None:
            w1.k_scale = w.k_scale[l * w.kv_heads:(l + 1) * w.kv_heads]
        from workloads import make_pool
        kc, vc = make_pool(w1, "cpu")
        kc, vc = np_bits(kc).copy(), None if vc is None else np_bits(vc).copy()
        run_oracle(w1, srcs, kc, vc, n_threads=orc.host_threads())
        gk = bits_to_numpy(dw.k_cache[l * s_l:(l + 1) * s_l])
        diff = np.flatnonzero(gk != kc)
        if diff.size:
            assert not np.any(kc[diff] == SENTINEL_BF16), (name, l, "an untouched K element changed")
            assert k_distance(w, gk[diff], kc[diff]).max() <= K_TOL[w.dtype], (name, l)
        if vc is not None:
            assert np.array_equal(bits_to_numpy(dw.v_cache[l * s_l:(l + 1) * s_l]), vc), (name, l, "V")
    dw.check_guards()


# ------------------------------------------------------------------ NEXT-4: skills + seam token + fresh suffix in ONE call
def _compose(dtype="bf16", layout="NHD", pairing="neox", with_map=False, D=128, heads=4):
    """Two sequences; each gets a precompiled skill, and then -- in the same call -- a repaired seam token (Delta = 0
    row) and/or the freshly projected suffix keys (KVR_SEG_PRE_ROPE), optionally at mapped positions with gaps."""
    pm = (3000 + np.cumsum(np.r_[0, 1 + (np.arange(76) % 7 == 0) * 5])).astype(np.int32) if with_map else None
    return make_workload(
        name="compose", layers=3, kv_heads=heads, head_dim=D, pairing=pairing, dtype=dtype, theta=1e6, block_size=16,
        layout=layout, seed=61, slack=1.5,
        seq_segments=[[dict(len=300, dst_token_start=20, new_start=20),                                # skill
                       dict(len=1, dst_token_start=320, new_start=0),                                  # seam row, Delta = 0
                       dict(len=77, dst_token_start=321, new_start=321, pre_rope=True, pos_map=pm)],   # suffix
                      [dict(len=130, dst_token_start=5, new_start=161),
                       dict(len=40, dst_token_start=135, new_start=135, pre_rope=True)]])


@pytest.mark.parametrize("path", ["generic", "generic_vec", "ring"])
@pytest.mark.parametrize("dtype,layout,pairing,with_map,heads", [("bf16", "NHD", "neox", False, 4), ("bf16", "HND", "gptj", True, 8),
                                                              ("fp8", "NHD", "neox", True, 8), ("bf16", "NHD", "neox", True, 2)])
def test_compose_skill_seam_and_fresh_suffix_in_one_call(dtype, layout, pairing, with_map, heads, path):
    check_parity(_compose(dtype, layout, pairing, with_map, heads=heads), path)
