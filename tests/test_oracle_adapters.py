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
