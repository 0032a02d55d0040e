"""Seeded synthetic inputs for rotate-on-read attention (kvr_rotate_on_read_attention; R25).  NO method
arithmetic here: shapes, segment lists, frequency tables and N(0,1) values only.

Shapes are those of the paper's workloads, nothing else of them: skills of 2k / 8k / 32k tokens,
N = 1-4 skills composed into one context, a serving batch of requests each reading a few skills
(BASELINE.json configs[3]'s length law), on the Qwen3-8B attention shape (32 query heads / 8 kv heads, head_dim 128,
rope_theta 1e6, NeoX).  Seed recipe as in configs.py: base 17107 + 100 + index; sub-streams +1000 K,
+2000 V, +4000 lengths / offsets, +7000 queries.  Values are bf16 bit patterns (torch.int16).
"""
from dataclasses import dataclass, field
from typing import List

import numpy as np
import torch

from .configs import S0, inv_freq_standard


@dataclass
class ReadSegmentSpec:
    len: int
    delta: int           # new_start - old_start of the skill in this request's context
    request: int
    src_row_pad: int = 0
    src_stable: bool = True   # a precompiled skill: nothing earlier on the stream writes its K / V (kvr.h)


@dataclass
class ReadWorkload:
    name: str
    layers: int          # layers the source tensors hold
    layer: int           # the layer one call attends
    q_heads: int
    kv_heads: int
    head_dim: int
    rotary_dim: int
    pairing: str
    inv_freq: np.ndarray
    n_req: int
    segments: List[ReadSegmentSpec]
    seed: int
    rotary_offset: int = 0
    dtype: str = "bf16"
    notes: dict = field(default_factory=dict)

    @property
    def tokens(self) -> int:
        return sum(s.len for s in self.segments)

    @property
    def scale(self) -> float:
        return float(self.head_dim) ** -0.5

    def src_strides(self, seg: ReadSegmentSpec):
        s_t = self.head_dim + seg.src_row_pad
        s_h = seg.len * s_t
        return self.kv_heads * s_h, s_h, s_t

    def bytes_read(self) -> int:
        return 2 * self.kv_heads * self.head_dim * 2 * self.tokens


def _draw(shape, seed, device):
    gen = torch.Generator(device=device)
    gen.manual_seed(seed)
    return torch.randn(shape, generator=gen, device=device, dtype=torch.float32).to(torch.bfloat16).view(torch.int16)


def make_read_sources(w: ReadWorkload, device="cpu"):
    """[(k, v)] per segment: int16 bf16 bits [layers, kv_heads, len, head_dim (+ pad)]."""
    out = []
    for i, s in enumerate(w.segments):
        shape = (w.layers, w.kv_heads, s.len, w.head_dim + s.src_row_pad)
        out.append((_draw(shape, w.seed + 1000 + 7919 * i, device), _draw(shape, w.seed + 2000 + 7919 * i, device)))
    return out


def make_queries(w: ReadWorkload, device="cpu"):
    """int16 bf16 bits [n_req, q_heads, head_dim]: the query rows as a model would hand them over (post-RoPE; RoPE does
    not change the distribution of iid Gaussian pairs, so N(0,1) is stored directly -- DESIGN.md 4)."""
    return _draw((w.n_req, w.q_heads, w.head_dim), w.seed + 7000, device)


def read_workload(name, *, q_heads=32, kv_heads=8, head_dim=128, rotary_dim=None, rotary_offset=0, pairing="neox",
                  theta=1e6, layers=2, layer=1, requests, seed, pad=0, inv_freq=None) -> ReadWorkload:
    """requests: list (one entry per request) of lists of (len, delta)."""
    R = head_dim if rotary_dim is None else rotary_dim
    segs = [ReadSegmentSpec(int(L), int(d), r, pad) for r, lst in enumerate(requests) for (L, d) in lst]
    return ReadWorkload(name, layers, layer, q_heads, kv_heads, head_dim, R, pairing,
                        inv_freq_standard(theta, R) if inv_freq is None else inv_freq, len(requests), segs, seed,
                        rotary_offset=rotary_offset)


READ_WORKLOADS = ("attend-tiny", "attend-compose4", "attend-32k-x8", "attend-serving")


def attention_config(name: str, shrink: int = 1) -> ReadWorkload:
    """The rotate-on-read workloads.  shrink > 1 divides every length (the parity cases the oracle finishes in seconds;
    they still span several 128-key tiles, ragged tails and several work items per (request, kv head))."""
    idx = READ_WORKLOADS.index(name)
    seed = S0 + 100 + idx
    rng = np.random.default_rng(seed + 4000)
    sh = lambda L: max(1, int(L) // shrink)
    if name == "attend-tiny":            # one 128-token skill read at offset 37, 4 query heads over 2 kv heads
        return read_workload(name, q_heads=4, kv_heads=2, theta=1e4, requests=[[(sh(128), 37)]], seed=seed)
    if name == "attend-compose4":        # N = 4 skills composed into one context (configs[2]'s lengths)
        lens = [2048, 8192, 512, 16384]
        starts = np.sort(rng.integers(0, 32768 - sum(lens), size=4)) + np.concatenate([[0], np.cumsum(lens)[:-1]])
        return read_workload(name, requests=[[(sh(L), int(s)) for L, s in zip(lens, starts)]], seed=seed)
    if name == "attend-32k-x8":          # a 32k-token skill; eight concurrent requests reading it at 2000
        return read_workload(name, requests=[[(sh(32768), 2000)] for _ in range(8)], seed=seed)
    if name == "attend-serving":         # BASELINE.json configs[3]'s law: 64 requests x 3 skills of U{256..4096} tokens
        reqs = []
        for _ in range(64):
            lens = rng.integers(256, 4097, size=3)
            gaps = rng.integers(0, 513, size=3)
            pos, lst = 0, []
            for L, g in zip(lens, gaps):
                pos += int(g)
                lst.append((sh(L), pos))       # compiled at 0, placed at pos: delta = pos
                pos += int(L)
            reqs.append(lst)
        return read_workload(name, requests=reqs, seed=seed)
    raise ValueError(name)
