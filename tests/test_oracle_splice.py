"""Pins of the oracle's splice (slot indexing, V copy, untouched bytes) and of the rotation THROUGH the
storage formats, on tiny inputs, against brute force and exact rational rounding (SURVEY 8(c) 'Pins')."""
import math
from fractions import Fraction

import ml_dtypes
import numpy as np
import pytest

from oracle import kvr_oracle as orc
from tests.helpers import (PAIRING, brute_force_offsets, materialize_cpu, ord_bf16, rope_direct_np,
                           run_oracle)
from workloads import SENTINEL_BF16, SENTINEL_FP8, config, inv_freq_standard, make_workload, pos_map_with_gaps


# ---- exact (rational) single-rounding encoders, independent of the C code ----
def _round_half_even(q: Fraction) -> int:
    fl = q.numerator // q.denominator
    rem = q - fl
    return fl + 1 if (rem > Fraction(1, 2) or (rem == Fraction(1, 2) and fl & 1)) else fl


def bf16_exact(v: float) -> int:
    sign = 0x8000 if math.copysign(1.0, v) < 0 else 0
    a = abs(v)
    if a == 0:
        return sign
    e = max(math.frexp(a)[1] - 1, -126)
    fl = _round_half_even(Fraction(a) / Fraction(2) ** (e - 7))
    if fl == 256:
        fl, e = 128, e + 1
    assert e <= 127
    return sign | (fl if fl < 128 else ((e + 127) << 7) | (fl - 128))


def e4m3_exact_sat(v: Fraction, negative_zero=False) -> int:
    sign = 0x80 if (v < 0 or negative_zero) else 0
    a = min(abs(v), Fraction(448))
    if a == 0:
        return sign
    e = max(math.frexp(float(a))[1] - 1, -6)
    if Fraction(2) ** e > a:          # float(a) rounded up across a binade
        e = max(e - 1, -6)
    fl = _round_half_even(a / Fraction(2) ** (e - 3))
    if fl == 16:
        fl, e = 8, e + 1
    if fl == 0:
        return sign
    return sign | (fl if fl < 8 else ((e + 7) << 3) | (fl - 8))


def _expected_k_row_bf16(w, seg, k_row_bits, t):
    """Expected bf16 K row after reposition: numpy fp64 rotation + exact rational rounding."""
    delta = (int(seg.pos_map[t]) - (seg.old_start + t)) if seg.pos_map is not None else seg.new_start - seg.old_start
    if delta == 0:
        return k_row_bits.copy()
    x = k_row_bits.view(ml_dtypes.bfloat16).astype(np.float64)[None, :]
    y = rope_direct_np(x, [delta], w.inv_freq, w.rotary_dim, w.pairing)[0]
    out = np.array([bf16_exact(float(v)) for v in y], dtype=np.uint16)
    out[w.rotary_dim:] = k_row_bits[w.rotary_dim:]
    return out


def _check_against_brute_force(w, check_values=True):
    srcs, kc, vc = materialize_cpu(w)
    sentinel = SENTINEL_BF16 if w.dtype == "bf16" else SENTINEL_FP8
    run_oracle(w, srcs, kc, vc)
    offs = brute_force_offsets(w)
    D = w.head_dim
    touched = np.zeros(kc.shape, dtype=bool)
    starts = sorted(offs.values())
    assert len(set(starts)) == len(starts)                     # slots pairwise disjoint
    assert all(b - a >= D for a, b in zip(starts, starts[1:]))   # sorted row starts are at least a row apart
    for (si, l, h, t), o in offs.items():
        assert not touched[o:o + D].any()                      # rows never overlap
        touched[o:o + D] = True
        k_src, v_src = srcs[si]
        assert np.array_equal(vc[o:o + D], v_src[l, h, t, :D])                 # V: byte copy
        if check_values and w.dtype == "bf16":
            exp = _expected_k_row_bf16(w, w.segments[si], k_src[l, h, t, :D], t)
            assert np.array_equal(kc[o:o + D], exp), (si, l, h, t)
    assert np.all(kc[~touched] == sentinel) and np.all(vc[~touched] == sentinel)   # nothing else written
    assert touched.sum() == w.tokens * w.layers * w.kv_heads * D
    return srcs, kc, vc


def test_cfg0_tiny_brute_force():
    """BASELINE.json configs[0]: 128-token skill, new_start 37, block 16, shuffled table:
    offset-5 start, 7 full blocks, 5-token tail."""
    w = config(0)
    assert w.segments[0].dst_token_start % w.block_size == 5
    assert (w.segments[0].dst_token_start + w.segments[0].len) % w.block_size == 5
    _check_against_brute_force(w)


@pytest.mark.parametrize("layout", ["NHD", "HND"])
@pytest.mark.parametrize("pairing,D,R", [("neox", 32, 32), ("gptj", 32, 16), ("neox", 32, 16), ("gptj", 16, 16)])
def test_edge_cases_brute_force(layout, pairing, D, R):
    """1-token segment, segment ending on a block edge, dst_token_start != new_start, old_start != 0,
    negative Delta, two sequences, padded source rows and padded pool rows."""
    w = make_workload(name="edge", layers=2, kv_heads=3, head_dim=D, rotary_dim=R, pairing=pairing,
                      theta=1e4, block_size=4, layout=layout, seed=99, dst_head_pad=8, slack=1.5,
                      seq_segments=[
                          [dict(len=1, dst_token_start=3, new_start=3),
                           dict(len=9, dst_token_start=7, new_start=1000, old_start=17),       # ends on a block edge
                           dict(len=6, dst_token_start=17, new_start=5, old_start=4000, src_row_pad=8)],  # Delta < 0
                          [dict(len=5, dst_token_start=0, new_start=0),                        # Delta = 0
                           dict(len=7, dst_token_start=6, new_start=161)]])                    # PAPER.md:205 Delta=161
    _check_against_brute_force(w)


def test_pos_map_brute_force():
    pm = pos_map_with_gaps(23, 500, 0.3, 64, 5)
    pm[4] = 4                                   # one token with Delta_t = 0 (old_start 0, t = 4)
    w = make_workload(name="map", layers=1, kv_heads=2, head_dim=16, rotary_dim=8, pairing="gptj", theta=1e4,
                      block_size=8, layout="NHD", seed=5,
                      seq_segments=[[dict(len=23, dst_token_start=13, new_start=500, pos_map=pm)]])
    _check_against_brute_force(w)


def test_delta_zero_is_byte_copy_including_negative_zero_and_nan():
    w = make_workload(name="d0", layers=1, kv_heads=1, head_dim=16, theta=1e4, block_size=4, seed=1,
                      seq_segments=[[dict(len=4, dst_token_start=0, new_start=0)]])
    srcs, kc, vc = materialize_cpu(w)
    k = srcs[0][0]
    k[0, 0, 0, :4] = [0x8000, 0x0000, 0x7FC5, 0xFFC1]        # -0, +0, NaN payloads
    k[0, 0, 1, :2] = [0x0001, 0x8001]                        # subnormals
    run_oracle(w, srcs, kc, vc)
    offs = brute_force_offsets(w)
    for (si, l, h, t), o in offs.items():
        assert np.array_equal(kc[o:o + 16], k[l, h, t])


def test_unallocated_block_refused_and_nothing_written():
    w = make_workload(name="bad", layers=1, kv_heads=1, head_dim=16, theta=1e4, block_size=4, seed=2,
                      seq_segments=[[dict(len=10, dst_token_start=2, new_start=2)]])
    w.block_table[0, 2] = -1
    srcs, kc, vc = materialize_cpu(w)
    k_src, v_src = srcs[0]
    sl, sh, st = w.src_strides(w.segments[0])
    s_l, s_b, s_t, s_h = w.dst_strides()
    args = dict(layers=1, kv_heads=1, head_dim=16, rotary_dim=16, pairing=orc.NEOX_HALF, dtype=orc.BF16,
                inv_freq=w.inv_freq, k_cache=kc, v_cache=vc, stride_layer=s_l, stride_block=s_b,
                stride_token=s_t, stride_head=s_h, num_blocks=w.num_blocks, block_size=4,
                block_table=w.block_table, k_src=k_src.reshape(-1), v_src=v_src.reshape(-1),
                src_stride_layer=sl, src_stride_head=sh, src_stride_token=st, len=10, old_start=0,
                new_start=2, dst_seq=0, dst_token_start=2)
    assert orc.reposition_splice(**args) == orc.ERR_OUT_OF_RANGE
    assert np.all(kc == SENTINEL_BF16) and np.all(vc == SENTINEL_BF16)
    w.block_table[0, 2] = w.num_blocks
    assert orc.reposition_splice(**args) == orc.ERR_OUT_OF_RANGE
    args["dst_token_start"] = w.block_table.shape[1] * 4 - 9              # runs past the table row
    assert orc.reposition_splice(**args) == orc.ERR_INVALID_ARG


def _pairs(w, x):
    R, h = w.rotary_dim, w.rotary_dim // 2
    return (x[..., :h], x[..., h:R]) if w.pairing == "neox" else (x[..., 0:R:2], x[..., 1:R:2])


@pytest.mark.parametrize("pairing", ["neox", "gptj"])
def test_identity_through_bf16_and_roundtrip_and_norm(pairing):
    """K stored in bf16 at p, oracle-repositioned by Delta, vs direct RoPE at p+Delta rounded to bf16:
    within 2^-6 of the pair norm; Delta then -Delta returns within 2^-6; norms within 2^-7 relative."""
    L, D = 64, 64
    for delta in [161, 2000, -37, 100000]:
        w = make_workload(name="id", layers=1, kv_heads=2, head_dim=D, pairing=pairing, theta=1e6, block_size=16,
                          seed=11, seq_segments=[[dict(len=L, dst_token_start=16, old_start=50, new_start=50 + delta)]])
        rng = np.random.default_rng(12)
        k_pre = rng.standard_normal((2 * L, D))
        pos = np.tile(np.arange(50, 50 + L), 2)
        stored = orc.bf16_encode(rope_direct_np(k_pre, pos, w.inv_freq, D, pairing)).reshape(1, 2, L, D)
        srcs, kc, vc = materialize_cpu(w)
        srcs = [(stored, srcs[0][1])]
        run_oracle(w, srcs, kc, vc)
        offs = brute_force_offsets(w)
        got = np.stack([kc[offs[(0, 0, h, t)]:offs[(0, 0, h, t)] + D] for h in range(2) for t in range(L)])
        gotf = got.view(ml_dtypes.bfloat16).astype(np.float64)
        direct = rope_direct_np(k_pre, pos + delta, w.inv_freq, D, pairing)
        ga, gb = _pairs(w, gotf)
        da, db = _pairs(w, direct)
        ka, kb = _pairs(w, k_pre)
        norm = np.hypot(ka, kb)
        assert np.max(np.hypot(ga - da, gb - db) / norm) <= 2.0 ** -6
        assert np.max(np.abs(ga ** 2 + gb ** 2 - norm ** 2) / norm ** 2) <= 2.0 ** -6   # two roundings
        # negative control: NOT rotating is far from the target
        sa, sb = _pairs(w, stored.reshape(2 * L, D).view(ml_dtypes.bfloat16).astype(np.float64))
        assert np.median((np.hypot(sa - da, sb - db) / norm)[:, 0]) > 0.5       # pair 0: 2|sin(Delta/2)|
        # Delta then -Delta through bf16
        w2 = make_workload(name="back", layers=1, kv_heads=2, head_dim=D, pairing=pairing, theta=1e6, block_size=16,
                           seed=11, seq_segments=[[dict(len=L, dst_token_start=0, old_start=50 + delta, new_start=50)]])
        _, kc2, vc2 = materialize_cpu(w2)
        run_oracle(w2, [(got.reshape(1, 2, L, D).copy(), srcs[0][1])], kc2, vc2)
        offs2 = brute_force_offsets(w2)
        back = np.stack([kc2[offs2[(0, 0, h, t)]:offs2[(0, 0, h, t)] + D] for h in range(2) for t in range(L)])
        backf = back.view(ml_dtypes.bfloat16).astype(np.float64)
        ba, bb = _pairs(w, backf)
        assert np.max(np.hypot(ba - sa, bb - sb) / norm) <= 2.0 ** -6
        assert np.mean(back == stored.reshape(2 * L, D)) > 0.4          # most elements return bit-exactly


@pytest.mark.parametrize("scales_differ", [False, True])
@pytest.mark.parametrize("pairing,R", [("neox", 32), ("gptj", 16)])
def test_fp8_values_exact_rational(scales_differ, pairing, R):
    """fp8 mode: q -> q*s_src -> rotate -> /s_dst -> saturating RNE, against exact rational rounding of the
    numpy fp64 rotation; Delta = 0 with equal scales is a byte copy, with different scales a requantisation."""
    D = 32
    w = make_workload(name="fp8", layers=2, kv_heads=2, head_dim=D, rotary_dim=R, pairing=pairing, dtype="fp8",
                      theta=1e4, block_size=4, seed=21, scales_differ=scales_differ,
                      seq_segments=[[dict(len=11, dst_token_start=2, new_start=777),
                                     dict(len=6, dst_token_start=14, new_start=14)]])      # second: Delta = 0
    srcs, kc, vc = materialize_cpu(w)
    srcs[0][0][0, 0, 0, :3] = [0x7E, 0xFE, 0x7F]                   # +-448 (will saturate after rotation) and NaN
    run_oracle(w, srcs, kc, vc)
    offs = brute_force_offsets(w)
    s_src_all = w.k_scale_src if w.k_scale_src is not None else w.k_scale
    n_ambiguous = 0
    for (si, l, h, t), o in offs.items():
        seg = w.segments[si]
        q = srcs[si][0][l, h, t]
        assert np.array_equal(vc[o:o + D], srcs[si][1][l, h, t])
        delta = seg.new_start - seg.old_start
        s_src, s_dst = float(s_src_all[l * 2 + h]), float(w.k_scale[l * 2 + h])
        if delta == 0 and s_src == s_dst:
            assert np.array_equal(kc[o:o + D], q)
            continue
        x = q.view(ml_dtypes.float8_e4m3fn).astype(np.float64) * s_src
        y = rope_direct_np(x[None], [delta], w.inv_freq, R, pairing)[0] if delta else x
        for d in range(D):
            if np.isnan(y[d]):
                assert kc[o + d] & 0x7F == 0x7F
                continue
            if d >= R and s_src == s_dst:
                assert kc[o + d] == q[d]
                continue
            exact = Fraction(float(y[d])) / Fraction(s_dst)
            # the oracle divides in fp64 (one extra 2^-53 rounding); it can only differ from the exact
            # rational quotient on a tie, which float(y)/s_dst hits with negligible probability
            exp = e4m3_exact_sat(exact, negative_zero=(exact == 0 and math.copysign(1.0, y[d]) < 0))
            if kc[o + d] != exp:
                n_ambiguous += 1
    assert n_ambiguous == 0


def test_bytes_moved_is_linear():
    assert orc.bytes_moved(36, 8, 128, orc.BF16, 4096) == 1207959552          # SURVEY 8(d) cfg 1: 1.208 GB
    assert orc.bytes_moved(32, 8, 128, orc.FP8_E4M3, 1) == 131072
    assert orc.bytes_moved(48, 4, 128, orc.BF16, 65536) == 12884901888
    assert orc.bytes_moved(2, 2, 64, orc.BF16, 128) == 262144
