"""GPU parity of the widened rows: kvr_reposition_inplace (NEXT-1) and
kvr_write_span (NEXT-2) through the C ABI against the oracle, element by element.
Bar: every byte the call does not address (other slots, pass-through dims, padding, all of V) bit-exact;
K within 2 bf16 ulps / 1 e4m3 step of the fp64 result rounded once."""
import copy

import ml_dtypes
import numpy as np
import pytest
import torch

from tests.helpers import K_TOL, k_distance, materialize_cpu, np_bits, run_oracle, torch_bits
from workloads import config, config_small, make_workload

pytestmark = pytest.mark.gpu

PATHS = {"generic": 1, "ring": 2, "generic_vec": 5}
WINDOW = 4                      # kvr_last_launch_info path of the window in-place kernel (auto dispatch only)


def _random_pool(w, seed):
    rng = np.random.default_rng(seed)
    n = w.pool_elems()
    if w.dtype == "bf16":
        f = lambda: rng.standard_normal(n).astype(np.float32).astype(ml_dtypes.bfloat16).view(np.uint16).copy()
    else:
        f = lambda: np.clip(rng.standard_normal(n) * 2, -400, 400).astype(np.float32).astype(
            ml_dtypes.float8_e4m3fn).view(np.uint8).copy()
    return f(), f()


def _deltas(w, seed=3):
    base = [161, -37, 0, 2000, 100000, -4000, 7]
    rng = np.random.default_rng(seed)
    return [base[i] if i < len(base) else int(rng.integers(-5000, 100000)) for i in range(len(w.segments))]


def check_inplace(w, path, with_pos_map=False, null_v=False, declined_ok=False, **tuning):
    from oracle import kvr_oracle as orc
    from paper_2606_17107_b200 import kvr
    kc, vc = _random_pool(w, 41)
    deltas = _deltas(w)
    # device pool = the same bytes
    dk, dv = torch_bits(kc.copy()).cuda(), torch_bits(vc.copy()).cuda()
    dw = _PoolOnly(w, dk, None if null_v else dv)
    with kvr.Context(dw.model) as ctx:
        ctx.set_tuning(path=0 if path == "window" else PATHS[path], **tuning)
        spans = dw.inplace_spans(deltas, with_pos_map=with_pos_map)
        moved_dims = w.rotary_dim if getattr(w, "rotary_offset", 0) else w.head_dim        # kvr.h: only the window moves
        assert kvr.kvr_inplace_bytes_moved(dw.model, spans) == 2 * w.layers * w.kv_heads * moved_dims * w.elt_bytes * w.tokens
        try:
            dw.run_inplace(ctx, spans)
        except kvr.KvrError as e:
            if e.status == kvr.KVR_ERR_UNSUPPORTED and path == "ring" and declined_ok:
                return None, None          # outside the ring kernel's domain: declined before any launch
            raise
        st = ctx.last_device_status()
        info = ctx.last_launch_info()
    torch.cuda.synchronize()
    assert st[0] == 0 and info["path"] == (WINDOW if path == "window" else PATHS[path]), (st, info)
    ref = kc.copy()
    orc.inplace_workload(w, ref, deltas=deltas)
    gk = np_bits(dk)
    assert np.array_equal(np_bits(dv), vc), "V must not be touched"
    same = ref == kc                                   # bytes the oracle left alone ...
    d = k_distance(w, gk, ref)
    assert d.max() <= K_TOL[w.dtype], (int(d.max()), int((d > K_TOL[w.dtype]).sum()))
    untouched = _untouched_mask(w, kc.shape)
    assert np.array_equal(gk[untouched], kc[untouched]), "bytes outside the addressed rotary dims changed"
    assert not np.array_equal(gk, kc)
    return d, same


def _untouched_mask(w, shape):
    """True for every pool element no (segment, token, rotary dim) addresses -- by brute force."""
    from tests.helpers import brute_force_offsets
    m = np.ones(shape, dtype=bool)
    off = getattr(w, "rotary_offset", 0)               # the rotary window starts at rotary_offset inside the row
    for o in brute_force_offsets(w).values():
        m[o + off:o + off + w.rotary_dim] = False
    return m


class _PoolOnly:
    """DeviceWorkload-like view with a caller-made pool and no sources (in-place needs none)."""

    def __init__(self, w, k_cache, v_cache):
        from paper_2606_17107_b200 import kvr
        from paper_2606_17107_b200.harness import DeviceWorkload
        self._dw = DeviceWorkload.__new__(DeviceWorkload)
        dw = self._dw
        dw.w, dw.device = w, torch.device("cuda:0")
        from paper_2606_17107_b200.harness import model_of
        dw.model, dw._inv_keep = model_of(w)
        dw.block_table = torch.from_numpy(np.ascontiguousarray(w.block_table)).cuda()
        dw.k_scale = None if w.k_scale is None else torch.from_numpy(w.k_scale).cuda()
        dw.k_scale_src = None
        dw.k_cache, dw.v_cache = k_cache, v_cache
        dw.dst = dw.dst_for(k_cache, v_cache)
        self.model = dw.model

    def __getattr__(self, name):
        return getattr(self._dw, name)


@pytest.mark.parametrize("path", ["generic", "generic_vec", "ring"])
@pytest.mark.parametrize("layout", ["NHD", "HND"])
@pytest.mark.parametrize("c", [0, 1, 2, 3, 4])
def test_inplace_small_configs(c, layout, path):
    w = config_small(c, layout)
    for s in w.segments:
        s.pos_map = None
    d, _ = check_inplace(w, path)
    if w.dtype == "bf16":
        assert np.mean(d == 0) > 0.95


@pytest.mark.parametrize("path", ["generic", "generic_vec", "ring"])
@pytest.mark.parametrize("layout", ["NHD", "HND"])
def test_inplace_with_position_map_and_without_v(layout, path):
    w = config_small(1, layout)
    check_inplace(w, path, with_pos_map=True, null_v=True)


@pytest.mark.parametrize("tuning", [dict(max_ctas=3, stages=2, consumer_warps=1),
                                    dict(max_ctas=2, stages=7, consumer_warps=3),
                                    dict(max_ctas=1, stages=4, consumer_warps=4, layers_per_unit=1)])
@pytest.mark.parametrize("c", [2, 3])
def test_inplace_ring_wraps(c, tuning):
    w = config_small(c, "NHD" if c % 2 else "HND")
    check_inplace(w, "ring", **tuning)


@pytest.mark.parametrize("path", ["generic", "generic_vec", "ring"])
@pytest.mark.parametrize("layout", ["NHD", "HND"])
@pytest.mark.parametrize("pairing,D,R,dtype", [("neox", 32, 32, "bf16"), ("gptj", 32, 16, "bf16"),
                                               ("neox", 64, 64, "fp8"), ("gptj", 64, 32, "fp8"),
                                               ("neox", 256, 256, "bf16")])
def test_inplace_edge_cases(layout, pairing, D, R, dtype, path):
    """Padded pool rows (the per-row copy mode), block size 4, ragged first/last blocks, two sequences."""
    pad = 8 if dtype == "bf16" else 16
    w = make_workload(name="edge", layers=3, kv_heads=3, head_dim=D, rotary_dim=R, pairing=pairing, dtype=dtype,
                      theta=1e4, block_size=4, layout=layout, seed=99, dst_head_pad=pad, slack=1.5,
                      seq_segments=[[dict(len=1, dst_token_start=3), dict(len=9, dst_token_start=7),
                                     dict(len=6, dst_token_start=17)],
                                    [dict(len=5, dst_token_start=0), dict(len=7, dst_token_start=6)]])
    check_inplace(w, path)


@pytest.mark.parametrize("path", ["generic", "generic_vec", "ring"])
def test_inplace_bad_block_sets_status_and_skips(path):
    from paper_2606_17107_b200 import kvr
    w = make_workload(name="bad", layers=2, kv_heads=2, head_dim=64, theta=1e4, block_size=4, seed=2,
                      seq_segments=[[dict(len=10, dst_token_start=2)]])
    good = int(w.block_table[0, 2])
    w.block_table[0, 2] = -1
    kc, vc = _random_pool(w, 5)
    dk = torch_bits(kc.copy()).cuda()
    dw = _PoolOnly(w, dk, None)
    with kvr.Context(dw.model) as ctx:
        ctx.set_tuning(path=PATHS[path])
        dw.run_inplace(ctx, dw.inplace_spans([9]))
        st = ctx.last_device_status()
    assert st[0] == kvr.KVR_ERR_OUT_OF_RANGE and st[1] == 0 and st[2] == 6
    s_l, s_b, _, _ = w.dst_strides()
    gk = np_bits(dk)
    for l in range(w.layers):
        o = l * s_l + good * s_b
        assert np.array_equal(gk[o:o + s_b], kc[o:o + s_b])          # the unreachable block kept its bytes


def test_inplace_host_validation():
    from paper_2606_17107_b200 import kvr
    w = make_workload(name="val", layers=1, kv_heads=1, head_dim=64, theta=1e4, block_size=4, seed=3,
                      seq_segments=[[dict(len=8, dst_token_start=0)]])
    kc, _ = _random_pool(w, 6)
    dk = torch_bits(kc.copy()).cuda()
    dw = _PoolOnly(w, dk, None)
    with kvr.Context(dw.model) as ctx:
        sp = dw.inplace_spans([5])
        for field, value, expect in [("len", 0, kvr.KVR_ERR_INVALID_ARG), ("seq", 1, kvr.KVR_ERR_INVALID_ARG),
                                     ("token_start", 1, kvr.KVR_ERR_OUT_OF_RANGE), ("old_start", -1, kvr.KVR_ERR_INVALID_ARG)]:
            old = getattr(sp[0], field)
            setattr(sp[0], field, value)
            assert ctx.reposition_inplace(dw.dst, sp, check=False) == expect, field
            setattr(sp[0], field, old)
        assert ctx.launch_count() == 0
        torch.cuda.synchronize()
        assert np.array_equal(np_bits(dk), kc)
        assert ctx.reposition_inplace(dw.dst, kvr.resident_span_array([]), check=False) == kvr.KVR_OK


# ------------------------------------------------------------------ splice then re-float = the agent loop
def test_splice_then_refloat_every_turn_matches_oracle():
    """the chunk is spliced once, then re-floated in place turn after turn."""
    from oracle import kvr_oracle as orc
    from paper_2606_17107_b200 import kvr
    from paper_2606_17107_b200.harness import DeviceWorkload
    w = config_small(2, "NHD")
    srcs, kc, vc = materialize_cpu(w)
    dw = DeviceWorkload(w, "cuda:0", sources=[(torch_bits(k), torch_bits(v)) for k, v in srcs])
    run_oracle(w, srcs, kc, vc)
    with kvr.Context(dw.model) as ctx:
        dw.run(ctx)
        for turn in range(3):
            deltas = [37 * (turn + 1) + i for i in range(len(w.segments))]
            # the oracle follows the GPU's own bytes turn by turn, so the tolerance does not compound
            before = np_bits(dw.k_cache)
            ref = before.copy()
            orc.inplace_workload(w, ref, deltas=deltas)
            dw.run_inplace(ctx, dw.inplace_spans(deltas))
            assert ctx.last_device_status()[0] == 0
            assert k_distance(w, np_bits(dw.k_cache), ref).max() <= K_TOL[w.dtype]
            assert np.array_equal(np_bits(dw.v_cache), vc)


# ------------------------------------------------------------------ full size, the launch configuration bench.py times
@pytest.mark.parametrize("c,layout", [(1, "NHD"), (1, "HND"), (2, "NHD"), (4, "HND")])
def test_inplace_full_size_every_layer(c, layout):
    """Splice (fills the slots with finite keys), snapshot the pool, re-float in place; the oracle re-floats the
    snapshot layer by layer: every layer, every element; V and everything outside the addressed rows unchanged."""
    from oracle import kvr_oracle as orc
    from paper_2606_17107_b200 import kvr
    from paper_2606_17107_b200.harness import DeviceWorkload
    w = config(c, layout)
    for s in w.segments:
        s.pos_map = None
    dw = DeviceWorkload(w, "cuda:0", guard_bytes=1 << 16)
    s_l = w.dst_strides()[0]
    deltas = [161 + 7 * i for i in range(len(w.segments))]
    with kvr.Context(dw.model) as ctx:
        dw.run(ctx)
        torch.cuda.synchronize()
        before_k, before_v = dw.k_cache.clone(), dw.v_cache.clone()
        dw.run_inplace(ctx, dw.inplace_spans(deltas))
        assert ctx.last_device_status()[0] == 0 and ctx.last_launch_info()["path"] == 2
    torch.cuda.synchronize()
    dw.check_guards()
    assert torch.equal(dw.v_cache, before_v), "V must not be touched"
    w1 = config(c, layout, layers=1)
    w1.block_table, w1.num_blocks, w1.segments = w.block_table, w.num_blocks, w.segments
    for l in range(w.layers):
        ref = np_bits(before_k[l * s_l:(l + 1) * s_l]).copy()
        orc.inplace_workload(w1, ref, deltas=deltas, n_threads=orc.host_threads())
        got = np_bits(dw.k_cache[l * s_l:(l + 1) * s_l])
        diff = np.flatnonzero(got != ref)
        if diff.size:
            d = k_distance(w, got[diff], ref[diff])
            assert d.max() <= K_TOL[w.dtype], (c, layout, l, int(d.max()))


# ------------------------------------------------------------------ NEXT-2: span overwrite
@pytest.mark.parametrize("path", ["generic", "generic_vec", "ring"])
@pytest.mark.parametrize("layout", ["NHD", "HND"])
@pytest.mark.parametrize("c", [0, 3, 4])
def test_write_span_is_a_byte_exact_scatter(c, layout, path):
    from paper_2606_17107_b200 import kvr
    from paper_2606_17107_b200.harness import DeviceWorkload
    w = config_small(c, layout)
    w0 = copy.deepcopy(w)
    for s in w0.segments:                                   # the oracle's Delta = 0 splice is the definition
        s.pos_map, s.old_start, s.new_start = None, 0, 0
    srcs, kc, vc = materialize_cpu(w0)
    dw = DeviceWorkload(w0, "cuda:0", sources=[(torch_bits(k), torch_bits(v)) for k, v in srcs])
    with kvr.Context(dw.model) as ctx:
        ctx.set_tuning(path=PATHS[path])
        ctx.write_span(dw.dst, dw.write_spans())
        assert ctx.last_device_status()[0] == 0
    torch.cuda.synchronize()
    run_oracle(w0, srcs, kc, vc)
    assert np.array_equal(np_bits(dw.k_cache), kc) and np.array_equal(np_bits(dw.v_cache), vc)


def test_seam_repair_overwrites_the_first_token_of_a_spliced_chunk():
    """PAPER.md:141/:528 'one boundary token repaired': splice, then overwrite token 0 of the chunk with new K/V."""
    from paper_2606_17107_b200 import kvr
    from paper_2606_17107_b200.harness import DeviceWorkload
    w = config_small(1, "NHD")
    srcs, kc, vc = materialize_cpu(w)
    dw = DeviceWorkload(w, "cuda:0", sources=[(torch_bits(k), torch_bits(v)) for k, v in srcs])
    seg = w.segments[0]
    rng = np.random.default_rng(1)
    shape = (w.layers, w.kv_heads, 2, w.head_dim)
    nk = rng.standard_normal(shape).astype(np.float32).astype(ml_dtypes.bfloat16).view(np.uint16)
    nv = rng.standard_normal(shape).astype(np.float32).astype(ml_dtypes.bfloat16).view(np.uint16)
    dk, dv = torch_bits(nk.copy()).cuda(), torch_bits(nv.copy()).cuda()
    with kvr.Context(dw.model) as ctx:
        dw.run(ctx)
        sp = kvr.span(dk, dv, (w.kv_heads * 2 * w.head_dim, 2 * w.head_dim, w.head_dim), 2, seg.dst_seq, seg.dst_token_start)
        ctx.write_span(dw.dst, [sp])
        assert ctx.last_device_status()[0] == 0
    torch.cuda.synchronize()
    run_oracle(w, srcs, kc, vc)
    gk, gv = np_bits(dw.k_cache), np_bits(dw.v_cache)
    s_l, s_b, s_t, s_h = w.dst_strides()
    repaired = np.zeros(kc.shape, dtype=bool)
    for t in range(2):
        j = seg.dst_token_start + t
        blk, off = int(w.block_table[seg.dst_seq, j // w.block_size]), j % w.block_size
        for l in range(w.layers):
            for h in range(w.kv_heads):
                o = l * s_l + blk * s_b + off * s_t + h * s_h
                repaired[o:o + w.head_dim] = True
                assert np.array_equal(gk[o:o + w.head_dim], nk[l, h, t]) and np.array_equal(gv[o:o + w.head_dim], nv[l, h, t])
    assert np.array_equal(gv[~repaired], vc[~repaired])
    assert k_distance(w, gk[~repaired], kc[~repaired]).max() <= K_TOL["bf16"]


@pytest.mark.parametrize("path", ["window", "generic", "generic_vec"])
@pytest.mark.parametrize("layout", ["NHD", "HND"])
@pytest.mark.parametrize("pairing,D,R,off,dtype", [
    ("neox", 576, 64, 512, "bf16"),      # the MLA [latent 512 | k_pe 64] row
    ("gptj", 576, 64, 512, "bf16"),
    ("neox", 96, 64, 16, "bf16"),        # head_dim 96: 192-byte rows, window in the middle
    ("gptj", 96, 32, 32, "bf16"),
    ("neox", 80, 16, 64, "bf16"),        # one lane per row (32-byte window)
    ("neox", 192, 64, 128, "fp8"),       # fp8 codes rotated as they are (one scale in place)
    ("gptj", 192, 128, 64, "fp8"),
    ("neox", 1024, 512, 512, "bf16")])   # 16 lanes per row
def test_inplace_window_kernel(pairing, D, R, off, dtype, layout, path):
    """kvr_reposition_inplace on rows that carry position-free dims besides the rotary window (kvr_window.cu): auto
    dispatch takes the window kernel, which touches the window alone; the generic kernel is the cross-check.  Several
    heads, padded pool rows, block size 8, ragged chunks, five spans over two sequences, shifts of both signs and 0."""
    pad = 8 if dtype == "bf16" else 16
    w = make_workload(name="winip", layers=3, kv_heads=2 if D < 500 else 1, head_dim=D, rotary_dim=R, rotary_offset=off,
                      pairing=pairing, dtype=dtype, theta=1e4, block_size=8, layout=layout, seed=1234, dst_head_pad=pad,
                      slack=1.5, seq_segments=[[dict(len=1, dst_token_start=3), dict(len=37, dst_token_start=7),
                                                dict(len=14, dst_token_start=49)],
                                               [dict(len=5, dst_token_start=0), dict(len=23, dst_token_start=6)]])
    check_inplace(w, path)


def test_inplace_window_kernel_bad_block_and_many_spans():
    """A bad block-table entry skips its chunk and raises the sticky status; 40 spans (staged descriptors) in one call."""
    from paper_2606_17107_b200 import kvr
    w = make_workload(name="winbad", layers=2, kv_heads=1, head_dim=576, rotary_dim=64, rotary_offset=512, theta=1e4,
                      block_size=4, seed=2, has_v=False, seq_segments=[[dict(len=10, dst_token_start=2)]])
    good = int(w.block_table[0, 2])
    w.block_table[0, 2] = -1
    kc, _ = _random_pool(w, 5)
    dk = torch_bits(kc.copy()).cuda()
    dw = _PoolOnly(w, dk, None)
    with kvr.Context(dw.model) as ctx:
        dw.run_inplace(ctx, dw.inplace_spans([9]))
        st = ctx.last_device_status()
        assert ctx.last_launch_info()["path"] == WINDOW
    assert st[0] == kvr.KVR_ERR_OUT_OF_RANGE and st[1] == 0 and st[2] == 6
    s_l, s_b, _, _ = w.dst_strides()
    gk = np_bits(dk)
    for l in range(w.layers):
        o = l * s_l + good * s_b
        assert np.array_equal(gk[o:o + s_b], kc[o:o + s_b])
    assert not np.array_equal(gk, kc)
    w2 = make_workload(name="winmany", layers=2, kv_heads=1, head_dim=576, rotary_dim=64, rotary_offset=512, theta=1e4,
                       block_size=16, seed=3, has_v=False,
                       seq_segments=[[dict(len=11, dst_token_start=13 * i) for i in range(40)]])
    check_inplace(w2, "window", null_v=True)
