"""Test-side helpers: independent restatements used to PIN the oracle, adapters from a
workloads.Workload to the oracle's flat call, and the distance functions of the tolerances."""
import numpy as np
import torch

from oracle import kvr_oracle as orc

PAIRING = {"neox": orc.NEOX_HALF, "gptj": orc.GPTJ_INTERLEAVED}
DTYPE = {"bf16": orc.BF16, "fp8": orc.FP8_E4M3}


# ---------------------------------------------------------------- direct RoPE (numpy, fp64)
def rope_direct_np(k, pos, inv_freq, rotary_dim, pairing):
    """Textbook RoPE (RoFormer) of pre-RoPE keys k[n, D] at integer positions pos[n], written
    independently of the oracle: out[ia] = k[ia] cos - k[ib] sin ; out[ib] = k[ib] cos + k[ia] sin."""
    k = np.asarray(k, dtype=np.float64)
    pos = np.asarray(pos, dtype=np.float64).reshape(-1, 1)
    ang = pos * np.asarray(inv_freq, dtype=np.float64).reshape(1, -1)      # [n, R/2]
    c, s = np.cos(ang), np.sin(ang)
    out = k.copy()
    h = rotary_dim // 2
    if pairing == "neox":
        a, b = k[:, :h], k[:, h:rotary_dim]
        out[:, :h] = a * c - b * s
        out[:, h:rotary_dim] = b * c + a * s
    else:
        a, b = k[:, 0:rotary_dim:2], k[:, 1:rotary_dim:2]
        out[:, 0:rotary_dim:2] = a * c - b * s
        out[:, 1:rotary_dim:2] = b * c + a * s
    return out


# ---------------------------------------------------------------- distances of the tolerances
def ord_bf16(u):
    """Ordered-integer lattice of bf16 (+-0 coincide): reading R14 / SURVEY Q14."""
    u = np.asarray(u).view(np.uint16).astype(np.int32)
    return np.where(u & 0x8000, -(u & 0x7FFF), u)


def _e4m3_rank_table():
    # rank on the sorted list of the distinct finite e4m3fn values, +-0 merged (reading R15)
    rank = np.zeros(256, dtype=np.int32)
    for b in range(256):
        mag = b & 0x7F
        rank[b] = -mag if (b & 0x80) else mag       # magnitude codes 0..0x7E are monotone in value
    return rank


_E4M3_RANK = _e4m3_rank_table()


def rank_e4m3(u):
    return _E4M3_RANK[np.asarray(u).view(np.uint8)]


def is_nan_e4m3(u):
    return (np.asarray(u).view(np.uint8) & 0x7F) == 0x7F


def k_distance(w, got, ref):
    """Per-element distance in the unit the tolerance is stated in (bf16 ulps or e4m3 steps)."""
    if w.dtype == "bf16":
        return np.abs(ord_bf16(got) - ord_bf16(ref))
    d = np.abs(rank_e4m3(got) - rank_e4m3(ref))
    both_nan = is_nan_e4m3(got) & is_nan_e4m3(ref)
    one_nan = is_nan_e4m3(got) ^ is_nan_e4m3(ref)
    return np.where(both_nan, 0, np.where(one_nan, 255, d))


K_TOL = {"bf16": 2, "fp8": 1}   # BASELINE.json north_star: 2 bf16 ulps / 1 e4m3 step


# ---------------------------------------------------------------- bits <-> numpy
def np_bits(t: torch.Tensor) -> np.ndarray:
    a = t.detach().cpu().contiguous().numpy()
    return a.view(np.uint16) if a.dtype == np.int16 else a


def torch_bits(a: np.ndarray) -> torch.Tensor:
    return torch.from_numpy(a.view(np.int16) if a.dtype == np.uint16 else a)


# ---------------------------------------------------------------- materialise a workload on the CPU
def materialize_cpu(w):
    """(sources, k_cache, v_cache) as numpy bit arrays.  Config 0's keys are RoPE'd at
    old_start + t by the harness (BASELINE.json configs[0]) via the ORACLE's fp64 rotation."""
    from workloads import make_pool, make_sources
    srcs = [(np_bits(k), None if v is None else np_bits(v)) for k, v in make_sources(w, "cpu")]
    if w.pre_rope_theta is not None:
        assert w.dtype == "bf16"
        out = []
        for seg, (k, v) in zip(w.segments, srcs):
            raw = orc.bf16_decode(k[..., :w.head_dim].reshape(-1, w.head_dim))     # pre-RoPE keys
            pos = np.tile(np.arange(seg.old_start, seg.old_start + seg.len), w.layers * w.kv_heads)
            from workloads import inv_freq_standard
            roped = orc.rotate_f64(raw, pos, inv_freq_standard(w.pre_rope_theta, w.rotary_dim),
                                   w.rotary_dim, PAIRING[w.pairing])
            k = k.copy()
            k[..., :w.head_dim] = orc.bf16_encode(roped).reshape(k[..., :w.head_dim].shape)
            out.append((k, v))
        srcs = out
    kc, vc = make_pool(w, "cpu")
    return srcs, np_bits(kc).copy(), None if vc is None else np_bits(vc).copy()


def run_oracle(w, srcs, k_cache, v_cache, n_threads=1, layer_begin=0, layer_end=None, segments=None):
    """Splices every segment of w into (k_cache, v_cache) in place with the oracle."""
    orc.splice_workload(w, srcs, k_cache, v_cache, n_threads=n_threads, layer_begin=layer_begin,
                        layer_end=layer_end, segments=segments)


# ---------------------------------------------------------------- brute-force slot enumeration
def brute_force_offsets(w):
    """Independent enumeration {(seg, layer, head, t): element offset of dim 0 in the pool}, in
    plain Python from the block table (PAPER.md:131 'concatenating'; DESIGN.md boundary)."""
    s_l, s_b, s_t, s_h = w.dst_strides()
    out = {}
    for si, seg in enumerate(w.segments):
        row = w.block_table[seg.dst_seq]
        for t in range(seg.len):
            j = seg.dst_token_start + t
            blk, off = int(row[j // w.block_size]), j % w.block_size
            assert 0 <= blk < w.num_blocks
            for l in range(w.layers):
                for h in range(w.kv_heads):
                    out[(si, l, h, t)] = l * s_l + blk * s_b + off * s_t + h * s_h
    return out
