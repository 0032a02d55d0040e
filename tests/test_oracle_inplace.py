"""Pins of the oracle's IN-PLACE reposition (kvr_oracle_reposition_inplace; R20)
against things other than itself: brute-force slot enumeration + an independent numpy rotation with exact
rational rounding, the pi/2 closed form, Delta = 0, Delta then -Delta, and the RoPE identity through the pool."""
import math
from fractions import Fraction

import ml_dtypes
import numpy as np
import pytest

from oracle import kvr_oracle as orc
from tests.helpers import PAIRING, brute_force_offsets, rope_direct_np
from tests.test_oracle_splice import bf16_exact, e4m3_exact_sat
from workloads import make_workload, pos_map_with_gaps


def _random_pool(w, seed):
    """A pool full of finite random values of the cache dtype (every slot, touched or not)."""
    rng = np.random.default_rng(seed)
    n = w.pool_elems()
    if w.dtype == "bf16":
        return rng.standard_normal(n).astype(np.float32).astype(ml_dtypes.bfloat16).view(np.uint16).copy()
    return np.clip(rng.standard_normal(n) * 2, -400, 400).astype(np.float32).astype(ml_dtypes.float8_e4m3fn).view(np.uint8).copy()


def _inplace(w, kc, si, old_start, new_start, pos_map=None, **kw):
    seg = w.segments[si]
    s_l, s_b, s_t, s_h = w.dst_strides()
    return orc.reposition_inplace(
        layers=w.layers, kv_heads=w.kv_heads, head_dim=w.head_dim, rotary_dim=w.rotary_dim,
        pairing=PAIRING[w.pairing], dtype=orc.BF16 if w.dtype == "bf16" else orc.FP8_E4M3, inv_freq=w.inv_freq,
        k_cache=kc, stride_layer=s_l, stride_block=s_b, stride_token=s_t, stride_head=s_h,
        num_blocks=w.num_blocks, block_size=w.block_size, block_table=w.block_table, k_scale=w.k_scale,
        seq=seg.dst_seq, token_start=seg.dst_token_start, len=seg.len, old_start=old_start, new_start=new_start,
        pos_map=pos_map, **kw)


def _edge_workload(layout, pairing, D, R, dtype="bf16"):
    return make_workload(name="ip", layers=2, kv_heads=3, head_dim=D, rotary_dim=R, pairing=pairing, dtype=dtype,
                         theta=1e4, block_size=4, layout=layout, seed=77, dst_head_pad=8 if dtype == "bf16" else 16,
                         slack=1.5,
                         seq_segments=[[dict(len=1, dst_token_start=3), dict(len=9, dst_token_start=7),
                                        dict(len=6, dst_token_start=17)],
                                       [dict(len=5, dst_token_start=0), dict(len=7, dst_token_start=6)]])


@pytest.mark.parametrize("layout", ["NHD", "HND"])
@pytest.mark.parametrize("pairing,D,R", [("neox", 32, 32), ("gptj", 32, 16), ("neox", 32, 16), ("gptj", 16, 16)])
def test_inplace_brute_force_bf16(layout, pairing, D, R):
    """Every addressed row becomes the exactly rounded numpy rotation of its OWN prior bytes; every other byte of
    the pool (other slots, pass-through dims, padding) keeps its value.  Deltas: 161, negative, 0."""
    w = _edge_workload(layout, pairing, D, R)
    before = _random_pool(w, 1)
    kc = before.copy()
    deltas = [161, -37, 100000, 0, 2000]
    for si, d in enumerate(deltas):
        assert _inplace(w, kc, si, 50, 50 + d) == orc.OK
    offs = brute_force_offsets(w)
    expect = before.copy()
    for (si, l, h, t), o in offs.items():
        d = deltas[si]
        if d == 0:
            continue
        x = before[o:o + D].view(ml_dtypes.bfloat16).astype(np.float64)[None, :]
        y = rope_direct_np(x, [d], w.inv_freq, R, pairing)[0]
        expect[o:o + R] = [bf16_exact(float(v)) for v in y[:R]]
    assert np.array_equal(kc, expect)


@pytest.mark.parametrize("pairing,R", [("neox", 32), ("gptj", 16)])
def test_inplace_fp8_exact_rational(pairing, R):
    D = 32
    w = _edge_workload("NHD", pairing, D, R, dtype="fp8")
    before = _random_pool(w, 2)
    kc = before.copy()
    deltas = [7, 777, 0, -5, 161]
    for si, d in enumerate(deltas):
        assert _inplace(w, kc, si, 0, d) == orc.OK if d >= 0 else _inplace(w, kc, si, 5, 0) == orc.OK
    offs = brute_force_offsets(w)
    expect = before.copy()
    for (si, l, h, t), o in offs.items():
        d = deltas[si]
        if d == 0:
            continue
        sc = float(w.k_scale[l * w.kv_heads + h])
        x = before[o:o + D].view(ml_dtypes.float8_e4m3fn).astype(np.float64) * sc
        y = rope_direct_np(x[None], [d], w.inv_freq, R, pairing)[0]
        for i in range(R):
            exact = Fraction(float(y[i])) / Fraction(sc)
            expect[o + i] = e4m3_exact_sat(exact, negative_zero=(exact == 0 and math.copysign(1.0, y[i]) < 0))
    assert np.array_equal(kc, expect)


@pytest.mark.parametrize("pairing", ["neox", "gptj"])
def test_inplace_closed_form_quarter_turns(pairing):
    """inv_freq = pi/2: Delta = 1 maps (a, b) -> (-b, a), Delta = 2 -> (-a, -b), Delta = 4 -> identity, bit-exactly."""
    D, R = 16, 8
    w = make_workload(name="q", layers=1, kv_heads=2, head_dim=D, rotary_dim=R, pairing=pairing, block_size=4,
                      inv_freq=np.full(R // 2, np.pi / 2), seed=3,
                      seq_segments=[[dict(len=6, dst_token_start=5)]])
    before = _random_pool(w, 4)
    offs = brute_force_offsets(w)
    ia = np.arange(R // 2) if pairing == "neox" else np.arange(0, R, 2)
    ib = ia + R // 2 if pairing == "neox" else ia + 1
    neg = lambda u: u ^ 0x8000
    for delta, f in [(1, lambda a, b: (neg(b), a)), (2, lambda a, b: (neg(a), neg(b))), (4, lambda a, b: (a, b)),
                     (-1, lambda a, b: (b, neg(a)))]:
        kc = before.copy()
        assert _inplace(w, kc, 0, 10, 10 + delta) == orc.OK
        expect = before.copy()
        for o in offs.values():
            a, b = before[o + ia], before[o + ib]
            expect[o + ia], expect[o + ib] = f(a, b)
        assert np.array_equal(kc, expect), delta


def test_inplace_pos_map_and_zero_delta_tokens():
    D, R = 16, 8
    pm = pos_map_with_gaps(23, 500, 0.3, 64, 5)
    pm[4] = 104                                   # old_start 100, t = 4: Delta_t = 0
    w = make_workload(name="map", layers=1, kv_heads=2, head_dim=D, rotary_dim=R, pairing="gptj", theta=1e4,
                      block_size=8, seed=5, seq_segments=[[dict(len=23, dst_token_start=13)]])
    before = _random_pool(w, 6)
    kc = before.copy()
    assert _inplace(w, kc, 0, 100, 0, pos_map=pm) == orc.OK
    expect = before.copy()
    for (si, l, h, t), o in brute_force_offsets(w).items():
        d = int(pm[t]) - (100 + t)
        if d == 0:
            continue
        x = before[o:o + D].view(ml_dtypes.bfloat16).astype(np.float64)[None, :]
        expect[o:o + R] = [bf16_exact(float(v)) for v in rope_direct_np(x, [d], w.inv_freq, R, "gptj")[0][:R]]
    assert np.array_equal(kc, expect)


def test_inplace_identity_through_the_pool_and_roundtrip():
    """Keys RoPE'd at p and stored in bf16 in the pool, re-floated in place by Delta, are the direct RoPE at
    p + Delta up to the two bf16 roundings (<= 2^-6 of the pair norm); Delta then -Delta returns within 2^-6."""
    D, L = 64, 48
    w = make_workload(name="id", layers=1, kv_heads=2, head_dim=D, pairing="neox", theta=1e6, block_size=16, seed=11,
                      seq_segments=[[dict(len=L, dst_token_start=9)]])
    rng = np.random.default_rng(12)
    offs = brute_force_offsets(w)
    keys = {k: rng.standard_normal(D) for k in offs}
    kc = np.zeros(w.pool_elems(), dtype=np.uint16)
    for (si, l, h, t), o in offs.items():
        kc[o:o + D] = orc.bf16_encode(rope_direct_np(keys[(si, l, h, t)][None], [50 + t], w.inv_freq, D, "neox")[0])
    stored = kc.copy()
    for delta in [161, 2000]:
        kc[:] = stored
        assert _inplace(w, kc, 0, 50, 50 + delta) == orc.OK
        worst = 0.0
        for (si, l, h, t), o in offs.items():
            got = kc[o:o + D].view(ml_dtypes.bfloat16).astype(np.float64)
            direct = rope_direct_np(keys[(si, l, h, t)][None], [50 + t + delta], w.inv_freq, D, "neox")[0]
            k = keys[(si, l, h, t)]
            norm = np.hypot(k[:D // 2], k[D // 2:])
            worst = max(worst, np.max(np.hypot(got[:D // 2] - direct[:D // 2], got[D // 2:] - direct[D // 2:]) / norm))
        assert worst <= 2.0 ** -6
        assert not np.array_equal(kc, stored)                      # rotation is not a no-op
        assert _inplace(w, kc, 0, 50 + delta, 50) == orc.OK
        worst = 0.0
        for (si, l, h, t), o in offs.items():
            back = kc[o:o + D].view(ml_dtypes.bfloat16).astype(np.float64)
            orig = stored[o:o + D].view(ml_dtypes.bfloat16).astype(np.float64)
            k = keys[(si, l, h, t)]
            norm = np.hypot(k[:D // 2], k[D // 2:])
            worst = max(worst, np.max(np.hypot(back[:D // 2] - orig[:D // 2], back[D // 2:] - orig[D // 2:]) / norm))
        assert worst <= 2.0 ** -6 and np.mean(kc == stored) > 0.4


def test_inplace_refuses_bad_blocks_and_bad_args():
    w = make_workload(name="bad", layers=1, kv_heads=1, head_dim=16, theta=1e4, block_size=4, seed=2,
                      seq_segments=[[dict(len=10, dst_token_start=2)]])
    before = _random_pool(w, 8)
    kc = before.copy()
    w.block_table[0, 2] = -1
    assert _inplace(w, kc, 0, 0, 5) == orc.ERR_OUT_OF_RANGE
    assert np.array_equal(kc, before)
    w.block_table[0, 2] = w.num_blocks
    assert _inplace(w, kc, 0, 0, 5) == orc.ERR_OUT_OF_RANGE
    w.block_table[0, 2] = 0
    w.segments[0].dst_token_start = w.block_table.shape[1] * 4 - 9
    assert _inplace(w, kc, 0, 0, 5) == orc.ERR_INVALID_ARG
    assert np.array_equal(kc, before)
