"""NEXT-3 representation adapters (Fig. 22b): M-RoPE 'rotate only the temporal
channels' is expressed through the caller's frequency table (zero frequency on height/width pairs; R22).
Pins: section membership against a brute-force enumeration, and the oracle's output on such a table against an
independent numpy rotation restricted to the temporal pairs."""
import ml_dtypes
import numpy as np
import pytest

from tests.helpers import brute_force_offsets, materialize_cpu, ord_bf16, rope_direct_np, run_oracle
from tests.test_oracle_splice import bf16_exact
from workloads import inv_freq_mrope_temporal, inv_freq_standard, make_workload


def _axis_brute(i, sections, interleaved):
    s_t, s_h, s_w = sections
    if not interleaved:
        return 0 if i < s_t else (1 if i < s_t + s_h else 2)
    # t h w t h w ... while height / width still have pairs left, temporal afterwards
    if i % 3 == 1 and i // 3 < s_h:
        return 1
    if i % 3 == 2 and i // 3 < s_w:
        return 2
    return 0


@pytest.mark.parametrize("interleaved", [False, True])
@pytest.mark.parametrize("sections", [(22, 21, 21), (24, 20, 20), (4, 2, 2)])
def test_mrope_table_membership(sections, interleaved):
    R = 2 * sum(sections)
    f = inv_freq_mrope_temporal(1e6, R, sections, interleaved)
    std = inv_freq_standard(1e6, R)
    for i in range(R // 2):
        assert f[i] == (std[i] if _axis_brute(i, sections, interleaved) == 0 else 0.0)
    assert int((f != 0).sum()) == sections[0]


@pytest.mark.parametrize("interleaved", [False, True])
@pytest.mark.parametrize("pairing", ["neox", "gptj"])
def test_mrope_splice_rotates_only_temporal_pairs(pairing, interleaved):
    """Delta = 161: temporal pairs equal the exactly rounded numpy rotation; height/width pairs
    keep their VALUE (the angle is 0; -0 may become +0, which the ulp metric merges)."""
    D = R = 32
    sections = (6, 5, 5)
    inv = inv_freq_mrope_temporal(1e6, R, sections, interleaved)
    w = make_workload(name="mrope", layers=2, kv_heads=2, head_dim=D, rotary_dim=R, pairing=pairing, inv_freq=inv,
                      block_size=4, seed=31, seq_segments=[[dict(len=13, dst_token_start=3, new_start=161)]])
    srcs, kc, vc = materialize_cpu(w)
    run_oracle(w, srcs, kc, vc)
    temporal = inv != 0
    half = R // 2
    for (si, l, h, t), o in brute_force_offsets(w).items():
        src = srcs[si][0][l, h, t, :D]
        x = src.view(ml_dtypes.bfloat16).astype(np.float64)[None, :]
        y = rope_direct_np(x, [161], inv_freq_standard(1e6, R), R, pairing)[0]
        for i in range(half):
            ia, ib = (i, i + half) if pairing == "neox" else (2 * i, 2 * i + 1)
            if temporal[i]:
                assert kc[o + ia] == bf16_exact(float(y[ia])) and kc[o + ib] == bf16_exact(float(y[ib]))
            else:
                assert ord_bf16(kc[o + ia]) == ord_bf16(src[ia]) and ord_bf16(kc[o + ib]) == ord_bf16(src[ib])
        assert np.array_equal(vc[o:o + D], srcs[si][1][l, h, t, :D])


# ------------------------------------------------------------------ MLA: [latent | k_pe] rows, K-only (reading R23)
from fractions import Fraction  # noqa: E402
import math  # noqa: E402

from oracle import kvr_oracle as orc  # noqa: E402
from tests.test_oracle_splice import e4m3_exact_sat  # noqa: E402


def _mla(pairing, dtype="bf16", inv_freq=None, new_start=161, scales_differ=False, layout="NHD", D=48, off=32, R=16):
    return make_workload(name="mla", layers=2, kv_heads=1, head_dim=D, rotary_dim=R, rotary_offset=off, pairing=pairing,
                         dtype=dtype, theta=1e4, inv_freq=inv_freq, block_size=4, seed=41, has_v=False, layout=layout,
                         scales_differ=scales_differ,
                         seq_segments=[[dict(len=13, dst_token_start=3, new_start=new_start),
                                        dict(len=5, dst_token_start=17, new_start=17)]])     # second: Delta = 0


def _window_pairs(pairing, off, R):
    h = R // 2
    return [((off + i, off + i + h) if pairing == "neox" else (off + 2 * i, off + 2 * i + 1)) for i in range(h)]


@pytest.mark.parametrize("layout", ["NHD", "HND"])
@pytest.mark.parametrize("pairing", ["neox", "gptj"])
def test_mla_rotates_only_the_kpe_window_and_copies_the_latent(pairing, layout):
    """PAPER.md:514 (Fig. 22a): 'repositioning re-rotates only k_pe and copies the latent as-is'.  k_pe pairs equal the
    exactly rounded numpy rotation of the 16-dim sub-vector; the 32 latent dims are byte-equal; slots by brute force;
    the pool has no V tensor; untouched slots keep the sentinel."""
    w = _mla(pairing, layout=layout)
    D, off, R = w.head_dim, w.rotary_offset, w.rotary_dim
    srcs, kc, vc = materialize_cpu(w)
    assert vc is None and srcs[0][1] is None
    before = kc.copy()
    run_oracle(w, srcs, kc, vc)
    touched = np.zeros(kc.shape, dtype=bool)
    for (si, l, h, t), o in brute_force_offsets(w).items():
        seg, src = w.segments[si], srcs[si][0][l, h, t, :D]
        touched[o:o + D] = True
        delta = seg.new_start - seg.old_start
        assert np.array_equal(kc[o:o + off], src[:off])                       # latent c_t: bytes
        assert np.array_equal(kc[o + off + R:o + D], src[off + R:])
        if delta == 0:
            assert np.array_equal(kc[o:o + D], src)
            continue
        kpe = src[off:off + R].view(ml_dtypes.bfloat16).astype(np.float64)[None, :]
        y = rope_direct_np(kpe, [delta], w.inv_freq, R, pairing)[0]           # independent numpy RoPE of the sub-vector
        exp = np.array([bf16_exact(float(v)) for v in y], dtype=np.uint16)
        assert np.array_equal(kc[o + off:o + off + R], exp)
    assert np.array_equal(kc[~touched], before[~touched])


@pytest.mark.parametrize("pairing", ["neox", "gptj"])
def test_mla_closed_form_quarter_turns(pairing):
    """inv_freq = pi/2: Delta = 1 maps a k_pe pair (a, b) -> (-b, a), Delta = 2 -> (-a, -b), Delta = 4 -> identity, at the
    window's OFFSET pair indices (a wrong offset or a pairing laid over the whole row fails)."""
    for delta, f in [(1, lambda a, b: (-b, a)), (2, lambda a, b: (-a, -b)), (4, lambda a, b: (a, b))]:
        w = _mla(pairing, inv_freq=np.full(8, math.pi / 2), new_start=delta)
        for s in w.segments:
            s.new_start = s.old_start + delta
        srcs, kc, vc = materialize_cpu(w)
        run_oracle(w, srcs, kc, vc)
        for (si, l, h, t), o in brute_force_offsets(w).items():
            x = srcs[si][0][l, h, t, :w.head_dim].view(ml_dtypes.bfloat16).astype(np.float64)
            got = kc[o:o + w.head_dim].view(ml_dtypes.bfloat16).astype(np.float64)
            exp = x.copy()
            for ia, ib in _window_pairs(pairing, w.rotary_offset, w.rotary_dim):
                exp[ia], exp[ib] = f(x[ia], x[ib])
            assert np.array_equal(got, exp)


def test_mla_identity_rope_at_p_then_shift_equals_rope_at_p_plus_delta():
    """rot(RoPE(k_pe, p), Delta) = RoPE(k_pe, p + Delta) through bf16, latent carried along untouched."""
    w = _mla("gptj", new_start=2000)
    D, off, R = w.head_dim, w.rotary_offset, w.rotary_dim
    srcs, kc, vc = materialize_cpu(w)
    seg = w.segments[0]
    raw = srcs[0][0][..., :D].view(ml_dtypes.bfloat16).astype(np.float64)          # pre-RoPE rows [L, 1, len, D]
    pos = np.arange(seg.len) + seg.old_start
    for l in range(w.layers):
        roped = rope_direct_np(raw[l, 0][:, off:off + R], pos, w.inv_freq, R, "gptj")
        srcs[0][0][l, 0, :, off:off + R] = roped.astype(ml_dtypes.bfloat16).view(np.uint16)
    run_oracle(w, srcs, kc, vc)
    worst = 0.0
    for (si, l, h, t), o in brute_force_offsets(w).items():
        if si != 0:
            continue
        direct = rope_direct_np(raw[l, 0, t:t + 1, off:off + R], [seg.new_start + t], w.inv_freq, R, "gptj")[0]
        got = kc[o + off:o + off + R].view(ml_dtypes.bfloat16).astype(np.float64)
        for i in range(R // 2):
            n = math.hypot(direct[2 * i], direct[2 * i + 1])
            worst = max(worst, max(abs(got[2 * i] - direct[2 * i]), abs(got[2 * i + 1] - direct[2 * i + 1])) / n)
    assert worst <= 2.0 ** -6


def test_mla_fp8_latent_requantised_under_a_scale_change():
    """fp8 with differing scales: k_pe = dequantise, rotate, requantise; the latent is re-expressed in the new scale
    (reading R8 applied outside the window), against exact rational rounding."""
    w = _mla("gptj", dtype="fp8", scales_differ=True, new_start=777)
    D, off, R = w.head_dim, w.rotary_offset, w.rotary_dim
    srcs, kc, vc = materialize_cpu(w)
    run_oracle(w, srcs, kc, vc)
    for (si, l, h, t), o in brute_force_offsets(w).items():
        seg, q = w.segments[si], srcs[si][0][l, h, t, :D]
        s_src, s_dst = float(w.k_scale_src[l]), float(w.k_scale[l])
        x = q.view(ml_dtypes.float8_e4m3fn).astype(np.float64) * s_src
        y = x.copy()
        delta = seg.new_start - seg.old_start
        if delta:
            y[off:off + R] = rope_direct_np(x[None, off:off + R], [delta], w.inv_freq, R, "gptj")[0]
        for d in range(D):
            exact = Fraction(float(y[d])) / Fraction(s_dst)
            assert kc[o + d] == e4m3_exact_sat(exact, negative_zero=(exact == 0 and math.copysign(1.0, y[d]) < 0))


def test_mla_inplace_equals_splice_of_the_same_rows():
    """kvr_oracle_reposition_inplace_ex on a resident [latent | k_pe] chunk = the K-only splice of the same rows by the
    same Delta (composition identity), and leaves the latent and every other slot alone."""
    w = _mla("neox", new_start=161)
    srcs, kc, vc = materialize_cpu(w)
    for s in w.segments:                      # first lay the rows down unrotated (Delta = 0) ...
        s.old_start, s.new_start = s.dst_token_start, s.dst_token_start
    run_oracle(w, srcs, kc, None)
    resident = kc.copy()
    orc.inplace_workload(w, resident, deltas=[161, 0])     # ... then re-float them in place
    for s, d in zip(w.segments, [161, 0]):
        s.new_start = s.old_start + d
    run_oracle(w, srcs, kc, None)                           # the same move as a splice
    assert np.array_equal(resident, kc)


def test_k_only_bytes_and_arg_rules():
    w = _mla("gptj")
    srcs, kc, vc = materialize_cpu(w)
    s_l, s_b, s_t, s_h = w.dst_strides()
    seg = w.segments[0]
    sl, sh, st = w.src_strides(seg)
    common = dict(layers=2, kv_heads=1, head_dim=48, rotary_dim=16, pairing=orc.GPTJ_INTERLEAVED, dtype=orc.BF16,
                  inv_freq=w.inv_freq, k_cache=kc, stride_layer=s_l, stride_block=s_b, stride_token=s_t, stride_head=s_h,
                  num_blocks=w.num_blocks, block_size=4, block_table=w.block_table, k_src=srcs[0][0].reshape(-1),
                  src_stride_layer=sl, src_stride_head=sh, src_stride_token=st, len=seg.len, old_start=0, new_start=5,
                  dst_seq=0, dst_token_start=3)
    assert orc.reposition_splice(**common, v_cache=None, v_src=None, rotary_offset=32) == orc.OK
    assert orc.reposition_splice(**common, v_cache=kc.copy(), v_src=None, rotary_offset=32) != orc.OK   # all-or-none
    assert orc.reposition_splice(**common, v_cache=None, v_src=None, rotary_offset=40) != orc.OK       # window past row


# ------------------------------------------------------------------ NEXT-4: fresh suffix keys (pre-RoPE) in the same call (R24)
@pytest.mark.parametrize("with_map", [False, True])
@pytest.mark.parametrize("pairing", ["neox", "gptj"])
def test_pre_rope_segment_is_rope_at_the_target_positions(pairing, with_map):
    """A KVR_SEG_PRE_ROPE segment holds keys that are not position-encoded yet; the splice must leave, in the slots,
    exactly RoPE(k, target_t) -- the textbook formula in numpy, rounded once (exact rational rounding) -- with
    target_t = new_start + t or pos_map[t].  A plain segment in the same workload keeps its ordinary meaning."""
    D, R = 32, 16
    pm = np.array([700, 701, 705, 706, 900, 901, 902], dtype=np.int32) if with_map else None
    w = make_workload(name="pre", layers=2, kv_heads=2, head_dim=D, rotary_dim=R, pairing=pairing, theta=1e4,
                      block_size=4, seed=51,
                      seq_segments=[[dict(len=9, dst_token_start=2, new_start=161),                       # a skill
                                     dict(len=7, dst_token_start=11, new_start=170, pre_rope=True, pos_map=pm)]])
    srcs, kc, vc = materialize_cpu(w)
    run_oracle(w, srcs, kc, vc)
    for (si, l, h, t), o in brute_force_offsets(w).items():
        seg, src = w.segments[si], srcs[si][0][l, h, t, :D]
        x = src.view(ml_dtypes.bfloat16).astype(np.float64)[None, :]
        if seg.pre_rope:
            target = int(pm[t]) if with_map else seg.new_start + t
            y = rope_direct_np(x, [target], w.inv_freq, R, pairing)[0]              # RoPE of the raw key at its position
        else:
            y = rope_direct_np(x, [seg.new_start - seg.old_start], w.inv_freq, R, pairing)[0]
        exp = np.array([bf16_exact(float(v)) for v in y], dtype=np.uint16)
        exp[R:] = src[R:]
        assert np.array_equal(kc[o:o + D], exp), (si, l, h, t)
        assert np.array_equal(vc[o:o + D], srcs[si][1][l, h, t, :D])


def test_pre_rope_equals_per_token_map_of_an_ordinary_segment():
    """Delta_t = target_t - old_start: the same bytes as an ordinary segment whose position map is target_t + t
    (old_start = 0), i.e. the flag is only a convenience over the per-token map."""
    w1 = make_workload(name="a", layers=1, kv_heads=2, head_dim=32, theta=1e4, block_size=4, seed=52,
                       seq_segments=[[dict(len=10, dst_token_start=3, new_start=40, pre_rope=True)]])
    w2 = make_workload(name="a", layers=1, kv_heads=2, head_dim=32, theta=1e4, block_size=4, seed=52,
                       seq_segments=[[dict(len=10, dst_token_start=3, new_start=40,
                                           pos_map=(40 + 2 * np.arange(10)).astype(np.int32))]])
    s1, k1, v1 = materialize_cpu(w1)
    s2, k2, v2 = materialize_cpu(w2)
    assert np.array_equal(s1[0][0], s2[0][0])
    run_oracle(w1, s1, k1, v1)
    run_oracle(w2, s2, k2, v2)
    assert np.array_equal(k1, k2) and np.array_equal(v1, v2)
