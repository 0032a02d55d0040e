"""Pins of the oracle's rotation against what the paper and the mathematics fix
(SURVEY 8(c) 'Pins'; PAPER.md:131 'post-RoPE keys ... re-rotate ... to the target positions')."""
import numpy as np
import pytest

from oracle import kvr_oracle as orc
from tests.helpers import PAIRING, rope_direct_np
from workloads import inv_freq_llama3, inv_freq_standard

THETAS = [1e4, 5e5, 1e6]


def _tables(R):
    out = [inv_freq_standard(t, R) for t in THETAS]
    out.append(inv_freq_llama3(5e5, R, 8.0, 1.0, 4.0, 8192))
    return out


@pytest.mark.parametrize("pairing", ["neox", "gptj"])
@pytest.mark.parametrize("D,R", [(128, 128), (128, 64), (64, 64), (16, 6)])
def test_rope_identity_fp64(pairing, D, R):
    """rot(RoPE(k, p), Delta) == RoPE(k, p + Delta): the statement that makes the splice exact.
    The left side uses the ORACLE twice, the right side the independent numpy direct RoPE."""
    rng = np.random.default_rng(3)
    n = 4000
    for inv in _tables(R):
        k = rng.standard_normal((n, D))
        p = rng.integers(0, 4096, n)
        d = rng.integers(-4096, 131073, n)
        stored = orc.rotate_f64(k, p, inv, R, PAIRING[pairing])          # RoPE at p (oracle as RoPE)
        assert np.max(np.abs(stored - rope_direct_np(k, p, inv, R, pairing))) < 1e-12
        moved = orc.rotate_f64(stored, d, inv, R, PAIRING[pairing])      # reposition by Delta
        direct = rope_direct_np(k, p + d, inv, R, pairing)               # RoPE at p + Delta
        h = R // 2
        if pairing == "neox":
            norm = np.hypot(k[:, :h], k[:, h:R])
            err = np.hypot(moved[:, :h] - direct[:, :h], moved[:, h:R] - direct[:, h:R])
        else:
            norm = np.hypot(k[:, 0:R:2], k[:, 1:R:2])
            err = np.hypot(moved[:, 0:R:2] - direct[:, 0:R:2], moved[:, 1:R:2] - direct[:, 1:R:2])
        assert np.max(err / norm) <= 1e-9
        assert np.array_equal(moved[:, R:], k[:, R:])                    # pass-through dims untouched


def test_direct_rope_helper_vs_transformers():
    """The numpy direct-RoPE helper the identity test leans on reduces, for NeoX pairing and a full
    rotary dim, to the transformers library's rotary application (test-only import)."""
    tf = pytest.importorskip("transformers.models.llama.modeling_llama")
    import torch
    rng = np.random.default_rng(4)
    n, D = 257, 128
    inv = inv_freq_standard(5e5, D)
    k = rng.standard_normal((n, D))
    pos = rng.integers(0, 100000, n)
    ang = torch.from_numpy(pos.astype(np.float64))[:, None] * torch.from_numpy(inv)[None, :]
    emb = torch.cat([ang, ang], dim=-1)
    cos, sin = emb.cos()[None], emb.sin()[None]                          # [1, n, D]
    kt = torch.from_numpy(k)[None, None]                                 # [1, 1, n, D]
    _, k_rot = tf.apply_rotary_pos_emb(kt, kt, cos, sin)
    ref = k_rot[0, 0].numpy()
    assert np.max(np.abs(rope_direct_np(k, pos, inv, D, "neox") - ref)) <= 1e-12
    assert np.max(np.abs(orc.rotate_f64(k, pos, inv, D, orc.NEOX_HALF) - ref)) <= 1e-12


def test_gptj_helper_vs_transformers_gptj():
    """Interleaved pairing against the library's GPT-J rotary application (test-only import)."""
    tf = pytest.importorskip("transformers.models.gptj.modeling_gptj")
    import torch
    rng = np.random.default_rng(5)
    n, D, R = 65, 128, 64
    inv = inv_freq_standard(1e4, R)
    k = rng.standard_normal((n, D))
    pos = rng.integers(0, 100000, n)
    ang = torch.from_numpy(pos.astype(np.float64))[:, None] * torch.from_numpy(inv)[None, :]   # [n, R/2]
    sin, cos = ang.sin()[None, :, None, :], ang.cos()[None, :, None, :]
    sin = torch.repeat_interleave(sin, 2, dim=3)
    cos = torch.repeat_interleave(cos, 2, dim=3)
    kt = torch.from_numpy(k[:, :R])[None, :, None, :]                    # [1, n, 1, R]
    ref = ((kt * cos) + (tf.rotate_every_two(kt) * sin))[0, :, 0].numpy()
    got = orc.rotate_f64(k, pos, inv, R, orc.GPTJ_INTERLEAVED)
    assert np.max(np.abs(got[:, :R] - ref)) <= 1e-12
    assert np.array_equal(got[:, R:], k[:, R:])


@pytest.mark.parametrize("pairing", ["neox", "gptj"])
def test_delta_then_minus_delta_and_norm_fp64(pairing):
    rng = np.random.default_rng(6)
    n, D, R = 3000, 128, 128
    inv = inv_freq_standard(1e6, R)
    k = rng.standard_normal((n, D))
    d = rng.integers(-4096, 131073, n)
    fwd = orc.rotate_f64(k, d, inv, R, PAIRING[pairing])
    back = orc.rotate_f64(fwd, -d, inv, R, PAIRING[pairing])
    assert np.max(np.abs(back - k)) <= 1e-9
    if pairing == "neox":
        n0 = k[:, :64] ** 2 + k[:, 64:] ** 2
        n1 = fwd[:, :64] ** 2 + fwd[:, 64:] ** 2
    else:
        n0 = k[:, 0::2] ** 2 + k[:, 1::2] ** 2
        n1 = fwd[:, 0::2] ** 2 + fwd[:, 1::2] ** 2
    assert np.max(np.abs(n1 - n0) / n0) <= 1e-12
    # Delta = 0 is the identity on values
    assert np.array_equal(orc.rotate_f64(k, np.zeros(n, dtype=np.int64), inv, R, PAIRING[pairing]), k)
    # negative control (the no-rotation control collapses): Delta != 0 really moves keys
    assert np.max(np.abs(fwd - k)) > 0.5


@pytest.mark.parametrize("pairing", ["neox", "gptj"])
@pytest.mark.parametrize("D,R", [(8, 8), (12, 8)])
def test_closed_form_quarter_turns(pairing, D, R):
    """inv_freq = pi/2 for every pair: Delta=1 -> (a,b)->(-b,a); Delta=2 -> (-a,-b); Delta=4 -> identity.
    Fixes the pairing AND the sign of the rotation (a transposed operand or a flipped sign fails)."""
    rng = np.random.default_rng(7)
    n = 50
    k = rng.integers(1, 9, (n, D)).astype(np.float64) * rng.choice([-1.0, 1.0], (n, D))
    inv = np.full(R // 2, np.pi / 2)
    ia = np.arange(R // 2) if pairing == "neox" else 2 * np.arange(R // 2)
    ib = ia + R // 2 if pairing == "neox" else ia + 1
    for delta, fa, fb in [(1, lambda a, b: -b, lambda a, b: a),
                          (2, lambda a, b: -a, lambda a, b: -b),
                          (3, lambda a, b: b, lambda a, b: -a),
                          (4, lambda a, b: a, lambda a, b: b),
                          (-1, lambda a, b: b, lambda a, b: -a)]:
        out = orc.rotate_f64(k, np.full(n, delta), inv, R, PAIRING[pairing])
        exp = k.copy()
        exp[:, ia] = fa(k[:, ia], k[:, ib])
        exp[:, ib] = fb(k[:, ia], k[:, ib])
        assert np.max(np.abs(out - exp)) <= 1e-14          # cos(pi/2) residue ~6e-17 * 8
        assert np.array_equal(out[:, R:], k[:, R:])
        # through the storage format the residue cannot move a rounding: bit-exact
        assert np.array_equal(orc.bf16_encode(out), orc.bf16_encode(exp))
