"""Workload descriptions and seeded value generators.  NO method arithmetic here.

Recipe: base seed S0 = 17107, config c
uses S0 + c; sub-streams by fixed offsets (+1000 K values, +2000 V values, +3000
block tables, +4000 lengths/offsets, +5000 scales, +6000 pos_map).  K, V ~ N(0,1)
drawn in fp32 by a seeded torch.Generator on the device that will hold them and
cast to the cache dtype (bf16, or e4m3fn after division by the per-head scale).
The very same bytes are handed to the oracle (copied device -> host), so the two
sides never depend on reproducing a random stream across machines.

The paper's real inputs (skills, LoCoMo memories, the tau^2-bench policy, images;
PAPER.md:143, :191, :199, :532) need its models and datasets, which are not
available; only their SHAPES are used: skill lengths 2k/8k/32k, N = 1-4 skills,
~2k and ~19.7k memories, 8B-class model shapes.

Raw bits convention: every K/V tensor returned here is an integer tensor of bit
patterns -- torch.int16 for bf16, torch.uint8 for e4m3fn.
"""
from dataclasses import dataclass, field
from typing import List, Optional

import numpy as np
import torch

S0 = 17107
SENTINEL_BF16 = 0x7FC1  # a bf16 NaN pattern no computation here produces
SENTINEL_FP8 = 0x7F     # the e4m3fn NaN


# ------------------------------------------------------------ frequency tables
# inv_freq is an INPUT of the kvr_* calls (the caller applies any scaling; R2/R3).

def inv_freq_standard(theta: float, rotary_dim: int) -> np.ndarray:
    i = np.arange(rotary_dim // 2, dtype=np.float64)
    return np.float64(theta) ** (-(2.0 * i) / np.float64(rotary_dim))


def inv_freq_llama3(theta: float, rotary_dim: int, factor: float, low_freq_factor: float,
                    high_freq_factor: float, original_max_position: int) -> np.ndarray:
    """llama3 rope scaling of the standard table (Llama-3.1 config: 8, 1, 4, 8192)."""
    f = inv_freq_standard(theta, rotary_dim)
    wavelen = 2.0 * np.pi / f
    low_wl = original_max_position / low_freq_factor
    high_wl = original_max_position / high_freq_factor
    smooth = (original_max_position / wavelen - low_freq_factor) / (high_freq_factor - low_freq_factor)
    mid = (1.0 - smooth) * f / factor + smooth * f
    return np.where(wavelen < high_wl, f, np.where(wavelen > low_wl, f / factor, mid))


def inv_freq_mrope_temporal(theta: float, rotary_dim: int, sections, interleaved: bool = False) -> np.ndarray:
    """M-RoPE adapter table (Fig. 22b: "re-rotate only the temporal channels"; R22).
    The rotary_dim/2 pairs are divided among the (temporal, height, width) axes: `sections` = pairs per axis.
    sectioned layout (Qwen2.5-VL-like): pairs [0, s_t) temporal, [s_t, s_t+s_h) height, the rest width;
    interleaved layout (Qwen3-VL-like): pair i is height if i % 3 == 1 and i < 3*s_h, width if i % 3 == 2 and
    i < 3*s_w, temporal otherwise.  A text-position shift moves only the temporal axis, so the table handed to
    kvr_create is the standard one with ZERO frequency on the height/width pairs (angle 0: unrotated)."""
    s_t, s_h, s_w = sections
    half = rotary_dim // 2
    assert s_t + s_h + s_w == half
    i = np.arange(half)
    if interleaved:
        temporal = ~(((i % 3 == 1) & (i < 3 * s_h)) | ((i % 3 == 2) & (i < 3 * s_w)))
    else:
        temporal = i < s_t
    assert int(temporal.sum()) == s_t
    return np.where(temporal, inv_freq_standard(theta, rotary_dim), 0.0)


def pos_map_with_gaps(length: int, first: int, gap_prob: float, max_gap: int, seed: int) -> np.ndarray:
    """pos[0] = first; pos[t+1] - pos[t] = 1 w.p. 1-gap_prob else 1 + U{1..max_gap} (R5)."""
    rng = np.random.default_rng(seed)
    step = np.ones(length, dtype=np.int64)
    gaps = rng.random(length) < gap_prob
    step[gaps] += rng.integers(1, max_gap + 1, size=int(gaps.sum()))
    step[0] = 0
    pos = first + np.cumsum(step)
    assert pos[-1] < 2 ** 31
    return pos.astype(np.int32)


# ------------------------------------------------------------------ dataclasses

@dataclass
class SegmentSpec:
    len: int
    old_start: int
    new_start: int
    dst_seq: int
    dst_token_start: int
    pos_map: Optional[np.ndarray] = None   # int32 [len]: new position of token t
    src_row_pad: int = 0                   # extra elements after each source token row (stride tests)
    pre_rope: bool = False                 # keys not yet position-encoded (fresh suffix keys): all tokens at old_start
    src_stable: bool = True                # a precompiled skill: nothing earlier on the stream writes its K / V (kvr.h)


@dataclass
class Workload:
    name: str
    layers: int
    kv_heads: int
    head_dim: int
    rotary_dim: int
    pairing: str                 # "neox" | "gptj"
    dtype: str                   # "bf16" | "fp8"
    inv_freq: np.ndarray         # float64 [rotary_dim/2]
    block_size: int
    num_blocks: int
    layout: str                  # "NHD": [layer][block][token][head][dim]; "HND": [layer][block][head][token][dim]
    block_table: np.ndarray      # int32 [num_seqs, max_blocks_per_seq]; < 0 = unallocated
    segments: List[SegmentSpec]
    seed: int
    k_scale: Optional[np.ndarray] = None       # float32 [layers*kv_heads], destination K scales (fp8)
    k_scale_src: Optional[np.ndarray] = None   # None = same as k_scale
    dst_head_pad: int = 0        # extra elements after each (token, head) row in the pool (stride tests)
    pre_rope_theta: Optional[float] = None     # config 0: K is RoPE'd at old_start + t by the harness
    rotary_offset: int = 0       # first rotary dim of a row ([latent | k_pe] caches: the latent width)
    has_v: bool = True           # False: a single cached tensor per token (MLA latent cache), no V pool
    notes: dict = field(default_factory=dict)

    @property
    def elt_bytes(self) -> int:
        return 2 if self.dtype == "bf16" else 1

    @property
    def tokens(self) -> int:
        return sum(s.len for s in self.segments)

    def dst_strides(self):
        """(stride_layer, stride_block, stride_token, stride_head) in elements."""
        row = self.head_dim + self.dst_head_pad
        if self.layout == "NHD":
            s_h, s_t = row, self.kv_heads * row
        elif self.layout == "HND":
            s_t, s_h = row, self.block_size * row
        else:
            raise ValueError(self.layout)
        s_b = self.block_size * self.kv_heads * row
        s_l = self.num_blocks * s_b
        return s_l, s_b, s_t, s_h

    def pool_elems(self) -> int:
        return self.layers * self.dst_strides()[0]

    def src_strides(self, seg: SegmentSpec):
        """(stride_layer, stride_head, stride_token) in elements for [layers][heads][len][dim]."""
        s_t = self.head_dim + seg.src_row_pad
        s_h = seg.len * s_t
        return self.kv_heads * s_h, s_h, s_t

    def src_elems(self, seg: SegmentSpec) -> int:
        return self.layers * self.src_strides(seg)[0]


def _torch_bits_dtype(w: Workload):
    return torch.int16 if w.dtype == "bf16" else torch.uint8


def _draw(w: Workload, seg: SegmentSpec, seg_idx: int, which: str, device) -> torch.Tensor:
    """[layers, heads, len, dim(+pad)] bit patterns of N(0,1) values in the cache dtype."""
    gen = torch.Generator(device=device)
    gen.manual_seed(w.seed + (1000 if which == "k" else 2000) + 7919 * seg_idx)
    row = w.head_dim + seg.src_row_pad
    out = torch.empty((w.layers, w.kv_heads, seg.len, row), dtype=_torch_bits_dtype(w), device=device)
    scale = None
    if w.dtype == "fp8" and which == "k":
        s = w.k_scale_src if w.k_scale_src is not None else w.k_scale
        scale = torch.from_numpy(np.asarray(s, dtype=np.float32)).to(device).view(w.layers, w.kv_heads)
    for l in range(w.layers):                      # layer by layer: bounded fp32 temporaries
        x = torch.randn((w.kv_heads, seg.len, row), generator=gen, device=device, dtype=torch.float32)
        if w.dtype == "bf16":
            out[l] = x.to(torch.bfloat16).view(torch.int16)
        else:
            if scale is not None:
                x = x / scale[l].view(-1, 1, 1)
            out[l] = x.clamp_(-448.0, 448.0).to(torch.float8_e4m3fn).view(torch.uint8)
    return out


def make_sources(w: Workload, device="cpu"):
    """[(k_src, v_src)] per segment, each [layers, heads, len, dim(+pad)] of bit patterns."""
    return [(_draw(w, s, i, "k", device), _draw(w, s, i, "v", device) if w.has_v else None)
            for i, s in enumerate(w.segments)]


def make_pool(w: Workload, device="cpu"):
    """Sentinel-filled (k_cache, v_cache), flat [pool_elems] of bit patterns."""
    if w.dtype == "bf16":
        val = int(np.array(SENTINEL_BF16, dtype=np.uint16).view(np.int16))
    else:
        val = SENTINEL_FP8
    n = w.pool_elems()
    return (torch.full((n,), val, dtype=_torch_bits_dtype(w), device=device),
            torch.full((n,), val, dtype=_torch_bits_dtype(w), device=device) if w.has_v else None)


# --------------------------------------------------------------------- builders

def _table_rows(num_blocks: int, rows: List[int], seed: int, unallocated_prefix: Optional[List[int]] = None):
    """Rows of distinct physical blocks: disjoint slices of one seeded permutation."""
    rng = np.random.default_rng(seed)
    perm = rng.permutation(num_blocks).astype(np.int32)
    need = sum(rows)
    assert need <= num_blocks, (need, num_blocks)
    width = max(r + (unallocated_prefix[i] if unallocated_prefix else 0) for i, r in enumerate(rows))
    table = np.full((len(rows), width), -1, dtype=np.int32)
    at = 0
    for i, r in enumerate(rows):
        pre = unallocated_prefix[i] if unallocated_prefix else 0
        table[i, pre:pre + r] = perm[at:at + r]
        at += r
    return table


def make_workload(*, name, layers, kv_heads, head_dim, rotary_dim=None, pairing="neox", dtype="bf16",
                  theta=1e4, inv_freq=None, block_size=16, layout="NHD", seed=S0,
                  seq_segments, num_blocks=None, slack=1.25, scales_differ=False,
                  dst_head_pad=0, pre_rope_theta=None, rotary_offset=0, has_v=True) -> Workload:
    """seq_segments: list (one per destination sequence) of lists of dicts with keys
    len, dst_token_start and optionally old_start, new_start, pos_map, src_row_pad.
    new_start defaults to dst_token_start, old_start to 0."""
    rotary_dim = rotary_dim or (head_dim - rotary_offset)
    if inv_freq is None:
        inv_freq = inv_freq_standard(theta, rotary_dim)
    segs, rows, prefix = [], [], []
    for q, lst in enumerate(seq_segments):
        lo = min(d["dst_token_start"] for d in lst) // block_size
        hi = max(d["dst_token_start"] + d["len"] for d in lst)
        prefix.append(lo if any(d.get("_skip_prefix") for d in lst) else 0)
        nblk = -(-hi // block_size) - prefix[-1]
        rows.append(nblk)
        for d in lst:
            segs.append(SegmentSpec(len=d["len"], old_start=d.get("old_start", 0),
                                    new_start=d.get("new_start", d["dst_token_start"]), dst_seq=q,
                                    dst_token_start=d["dst_token_start"], pos_map=d.get("pos_map"),
                                    src_row_pad=d.get("src_row_pad", 0), pre_rope=d.get("pre_rope", False),
                                    src_stable=d.get("src_stable", not d.get("pre_rope", False))))
    if num_blocks is None:
        num_blocks = int(np.ceil(slack * sum(rows)))
    table = _table_rows(num_blocks, rows, seed + 3000, prefix)
    k_scale = k_scale_src = None
    if dtype == "fp8":
        rng = np.random.default_rng(seed + 5000)
        k_scale = rng.uniform(0.5, 2.0, size=layers * kv_heads).astype(np.float32)
        if scales_differ:
            k_scale_src = rng.uniform(0.5, 2.0, size=layers * kv_heads).astype(np.float32)
    return Workload(name=name, layers=layers, kv_heads=kv_heads, head_dim=head_dim, rotary_dim=rotary_dim,
                    pairing=pairing, dtype=dtype, inv_freq=np.asarray(inv_freq, dtype=np.float64),
                    block_size=block_size, num_blocks=num_blocks, layout=layout, block_table=table,
                    segments=segs, seed=seed, k_scale=k_scale, k_scale_src=k_scale_src,
                    dst_head_pad=dst_head_pad, pre_rope_theta=pre_rope_theta, rotary_offset=rotary_offset,
                    has_v=has_v)


def _compose_offsets(lengths, total, seed):
    """Non-overlapping starts: the slack (total - sum) split into len+1 gaps by a seeded uniform composition."""
    rng = np.random.default_rng(seed)
    slack = total - sum(lengths)
    assert slack >= 0
    cuts = np.sort(rng.integers(0, slack + 1, size=len(lengths)))
    gaps = np.diff(np.concatenate([[0], cuts]))          # gap before each segment (last gap implied)
    starts, at = [], 0
    for g, n in zip(gaps, lengths):
        at += int(g)
        starts.append(at)
        at += n
    assert at <= total
    return starts


def config(c: int, layout: str = "NHD", layers: Optional[int] = None, shrink: int = 1) -> Workload:
    """BASELINE.json configs[c].  layers / shrink (divide every length) give reduced
    variants with the same structure (used by config_small and by sampled parity)."""
    seed = S0 + c
    if c == 0:
        return make_workload(name="cfg0-tiny", layers=layers or 2, kv_heads=2, head_dim=64, theta=1e4,
                             pairing="neox", dtype="bf16", block_size=16, layout=layout, seed=seed,
                             seq_segments=[[dict(len=128, dst_token_start=37, new_start=37)]],
                             num_blocks=16, pre_rope_theta=1e4)
    if c == 1:
        n = 4096 // shrink
        w = make_workload(name="cfg1-qwen3-8b", layers=layers or 36, kv_heads=8, head_dim=128, theta=1e6,
                          block_size=16, layout=layout, seed=seed, num_blocks=1024,
                          seq_segments=[[dict(len=n, dst_token_start=2000, new_start=2000)]])
        return w
    if c == 2:
        lens = [2048 // shrink, 8192 // shrink, 512 // shrink, 16384 // shrink]
        rng = np.random.default_rng(seed + 4000)
        order = rng.permutation(4)
        lens = [lens[i] for i in order]
        total = 32768 // shrink
        starts = _compose_offsets(lens, total, seed + 4001)
        inv = inv_freq_llama3(5e5, 128, 8.0, 1.0, 4.0, 8192)
        return make_workload(name="cfg2-llama31-8b", layers=layers or 32, kv_heads=8, head_dim=128,
                             inv_freq=inv, block_size=16, layout=layout, seed=seed,
                             num_blocks=2 * (total // 16),
                             seq_segments=[[dict(len=n, dst_token_start=s, new_start=s) for n, s in zip(lens, starts)]])
    if c == 3:
        rng = np.random.default_rng(seed + 4000)
        n_req = 64 if shrink == 1 else max(2, 64 // shrink)
        seqs = []
        for _ in range(n_req):
            at, lst = 0, []
            for _ in range(3):
                at += int(rng.integers(0, 513))
                n = int(rng.integers(256, 4097)) // shrink
                lst.append(dict(len=n, dst_token_start=at, new_start=at))
                at += n
            seqs.append(lst)
        return make_workload(name="cfg3-serving-fp8", layers=layers or 32, kv_heads=8, head_dim=128, theta=1e6,
                             dtype="fp8", block_size=16, layout=layout, seed=seed, slack=1.25, seq_segments=seqs)
    if c == 4:
        n = 65536 // shrink
        pm = pos_map_with_gaps(n, 100000, 0.05, 64, seed + 6000)
        w = make_workload(name="cfg4-long-partial-rotary", layers=layers or 48, kv_heads=4, head_dim=128,
                          rotary_dim=64, pairing="gptj", theta=1e4, block_size=16, layout=layout, seed=seed,
                          num_blocks=2 * (n // 16),
                          seq_segments=[[dict(len=n, dst_token_start=100000, new_start=100000, pos_map=pm,
                                              _skip_prefix=True)]])
        return w
    raise ValueError(c)


def config_small(c: int, layout: str = "NHD") -> Workload:
    """Reduced variants the oracle finishes in seconds; still several tiles and ragged tails."""
    if c == 0:
        return config(0, layout)
    return config(c, layout, layers={1: 3, 2: 2, 3: 2, 4: 3}[c], shrink={1: 8, 2: 16, 3: 16, 4: 32}[c])


# ------------------------------------------------------------- NEXT-3 / NEXT-4 adapter workloads

ADAPTERS = ("mla-dsv2-lite", "image-kv-qwen25vl-7b", "image-kv-qwen3vl-8b", "compose-qwen3-8b")


def adapter_config(name: str, layout: str = "NHD", layers: Optional[int] = None, shrink: int = 1) -> Workload:
    """Shapes of the paper's attention-variant adapters (PAPER.md:205, :215, :514 Fig. 22; Table 2 :306, :308).
    Synthetic, seeded; only shapes are taken from the models the paper names.

    mla-dsv2-lite         DeepSeek-V2-Lite-shaped latent cache: 27 layers, one cached row per token =
                          [latent c_t (512) | k_pe (64)], no V tensor; only k_pe rotates (interleaved pairs,
                          theta 1e4); one 8192-token skill precompiled at 0 and spliced at 2000; block_size 64.
    image-kv-qwen25vl-7b  Qwen2.5-VL-7B-shaped image KV: 28 layers, 4 kv heads, D 128, SECTIONED M-RoPE (16, 24, 24),
                          theta 1e6; 32 cached images of 1296 soft tokens each moved by Delta = 161 temporal positions
                           into 32 sequences; only the 16 temporal pairs rotate.
    image-kv-qwen3vl-8b   Qwen3-VL-8B-shaped: 36 layers, 8 kv heads, D 128, INTERLEAVED M-RoPE (24, 20, 20), theta 5e6;
                          same 32 images.
    compose-qwen3-8b      NEXT-4, one call per composed context ("a re-rotation pass plus the suffix"),
                          configs[1]'s shape: 16 requests, each = a 4096-token precompiled skill moved to 2000, one
                          repaired seam token (Delta = 0 row) and a 512-token task suffix whose freshly
                          projected keys are not position-encoded yet (pre_rope: RoPE applied on the way in).
    """
    seed = S0 + 100 + ADAPTERS.index(name)
    if name == "mla-dsv2-lite":
        n = 8192 // shrink
        return make_workload(name=name, layers=layers or 27, kv_heads=1, head_dim=576, rotary_dim=64, rotary_offset=512,
                             pairing="gptj", theta=1e4, block_size=64, layout=layout, seed=seed, has_v=False,
                             num_blocks=2 * ((2000 + n + 63) // 64),
                             seq_segments=[[dict(len=n, dst_token_start=2000, new_start=2000)]])
    if name in ("image-kv-qwen25vl-7b", "image-kv-qwen3vl-8b"):
        q3 = name.endswith("qwen3vl-8b")
        sections, theta = ((24, 20, 20), 5e6) if q3 else ((16, 24, 24), 1e6)
        inv = inv_freq_mrope_temporal(theta, 128, sections, interleaved=q3)
        n_img = 32 if shrink == 1 else max(2, 32 // shrink)
        n_tok = 1296 // shrink
        rng = np.random.default_rng(seed + 4000)
        seqs = []
        for _ in range(n_img):
            at = int(rng.integers(0, 2048 // shrink + 1))          # text before the image in its new trajectory
            seqs.append([dict(len=n_tok, dst_token_start=at, old_start=at, new_start=at + 161)])
        return make_workload(name=name, layers=layers or (36 if q3 else 28), kv_heads=8 if q3 else 4, head_dim=128,
                             inv_freq=inv, block_size=16, layout=layout, seed=seed, seq_segments=seqs)
    if name == "compose-qwen3-8b":
        n_req = 16 if shrink == 1 else max(2, 16 // shrink)
        n, suf = 4096 // shrink, 512 // shrink
        seqs = [[dict(len=n, dst_token_start=2000, new_start=2000),
                 dict(len=1, dst_token_start=2000 + n, new_start=0),
                 dict(len=suf, dst_token_start=2001 + n, new_start=2001 + n, pre_rope=True)] for _ in range(n_req)]
        return make_workload(name=name, layers=layers or 36, kv_heads=8, head_dim=128, theta=1e6, block_size=16,
                             layout=layout, seed=seed, seq_segments=seqs)
    raise ValueError(name)


def adapter_small(name: str, layout: str = "NHD") -> Workload:
    return adapter_config(name, layout, layers=2, shrink=8)
