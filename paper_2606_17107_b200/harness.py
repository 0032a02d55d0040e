"""Device-side materialisation of a workloads.Workload and its marshalling into the kvr C ABI.

Used by tests/, bench.py and __graft_entry__.smoke().  torch is plumbing here: device memory, streams.
Nothing in this module computes any part of the method, and nothing here touches oracle/.
"""
import numpy as np
import torch

from . import kvr

_PAIRING = {"neox": kvr.KVR_PAIR_NEOX_HALF, "gptj": kvr.KVR_PAIR_GPTJ_INTERLEAVED}
_DTYPE = {"bf16": kvr.KVR_BF16, "fp8": kvr.KVR_FP8_E4M3}


def model_of(w):
    return kvr.model_desc(w.layers, w.kv_heads, w.head_dim, w.rotary_dim, _PAIRING[w.pairing],
                          _DTYPE[w.dtype], w.inv_freq, rotary_offset=getattr(w, "rotary_offset", 0))


def _seg_flags(s):
    return ((kvr.KVR_SEG_PRE_ROPE if getattr(s, "pre_rope", False) else 0) |
            (kvr.KVR_SEG_SRC_STABLE if getattr(s, "src_stable", False) else 0))


GUARD_BYTE = 0xA5


class DeviceWorkload:
    """Sources, sentinel-filled pool, block table, position maps and scales of `w` resident on `device`,
    plus the ctypes structs of one kvr_reposition_splice call over all segments.

    guard_bytes > 0 (the GPU tests): every device buffer a call may touch -- pools, sources, block table, position
    maps, scales -- is a window inside a larger allocation whose first and last `guard_bytes` bytes hold a canary
    pattern; check_guards() asserts that no kernel wrote outside a window (compute-sanitizer is closed on the GPU
    pool, and the pool's own sentinel only guards bytes INSIDE it)."""

    def __init__(self, w, device="cuda:0", sources=None, make_pool=True, guard_bytes=0):
        from workloads import make_pool as _make_pool, make_sources
        self.w = w
        self.device = torch.device(device)
        self.guard_bytes = int(guard_bytes)
        self._guarded = []                         # (name, whole uint8 allocation, payload bytes)
        self.model, self._inv_keep = model_of(w)
        if sources is None:
            sources = make_sources(w, self.device)
        self.sources = [(self._dev(k, f"k_src[{i}]"), None if v is None else self._dev(v, f"v_src[{i}]"))
                        for i, (k, v) in enumerate(sources)]   # v is None for a K-only [latent | k_pe] cache (kvr.h, NEXT-3)
        self.block_table = self._dev(torch.from_numpy(np.ascontiguousarray(w.block_table)), "block_table")
        self.k_scale = self.k_scale_src = None
        if w.k_scale is not None:
            self.k_scale = self._dev(torch.from_numpy(w.k_scale), "k_scale")
        if w.k_scale_src is not None:
            self.k_scale_src = self._dev(torch.from_numpy(w.k_scale_src), "k_scale_src")
        self.pos_maps = [None if s.pos_map is None else self._dev(torch.from_numpy(s.pos_map), f"pos_map[{i}]")
                         for i, s in enumerate(w.segments)]
        self.k_cache = self.v_cache = None
        if make_pool:
            kc, vc = _make_pool(w, "cpu" if self.guard_bytes else self.device)
            self.k_cache = self._dev(kc, "k_cache")
            self.v_cache = None if vc is None else self._dev(vc, "v_cache")
        self.segs = kvr.segment_array([
            kvr.segment(k, v, w.src_strides(s), s.len, s.old_start, s.new_start, s.dst_seq, s.dst_token_start,
                        pos_map=pm, k_scale_src=self.k_scale_src,
                        flags=_seg_flags(s))
            for s, (k, v), pm in zip(w.segments, self.sources, self.pos_maps)])
        self.dst = self.dst_for(self.k_cache, self.v_cache) if make_pool else None

    def _dev(self, t, name):
        """`t` on the device; with guards, as a window between two canary regions of one larger allocation."""
        if not self.guard_bytes:
            return t.to(self.device).contiguous()
        t = t.contiguous()
        g, n = self.guard_bytes, t.numel() * t.element_size()
        whole = torch.full((2 * g + n,), GUARD_BYTE, dtype=torch.uint8, device=self.device)
        win = whole[g:g + n].view(t.dtype).view(t.shape)
        win.copy_(t)
        self._guarded.append((name, whole, n))
        return win

    def check_guards(self):
        """Every canary byte before and after every guarded window still holds GUARD_BYTE."""
        assert self.guard_bytes and self._guarded, "built without guard_bytes"
        g = self.guard_bytes
        for name, whole, n in self._guarded:
            for side, region in (("before", whole[:g]), ("after", whole[g + n:])):
                bad = torch.nonzero(region != GUARD_BYTE)
                assert bad.numel() == 0, (f"{name}: {bad.numel()} byte(s) written {side} the buffer, "
                                          f"first at offset {int(bad[0])} of the guard region")
        return len(self._guarded)

    def dst_for(self, k_cache, v_cache):
        w = self.w
        return kvr.paged_dst(k_cache, v_cache, w.dst_strides(), w.num_blocks, w.block_size, self.block_table,
                             w.block_table.shape[0], w.block_table.shape[1], k_scale=self.k_scale)

    def bytes_moved(self):
        return kvr.kvr_bytes_moved(self.model, self.segs)

    def run(self, ctx, stream=None, dst=None):
        return ctx.reposition_splice(dst if dst is not None else self.dst, self.segs, stream=stream)

    # ---- NEXT-1: re-float the resident chunks in place (kvr_reposition_inplace) ----
    def inplace_spans(self, deltas, with_pos_map=False):
        """One resident span per segment of w: the slots the splice wrote, moved by deltas[i] more positions.
        with_pos_map: express the same shift as a per-token position map (device int32) instead of old/new start."""
        spans, self._ip_keep = [], []
        for s, d in zip(self.w.segments, deltas):
            d = int(d)
            old, new = max(0, -d), max(0, d)             # positions are non-negative; new - old = d
            pm = None
            if with_pos_map:
                pm = (torch.arange(s.len, dtype=torch.int32, device=self.device) + new)
                self._ip_keep.append(pm)
            spans.append(kvr.resident_span(s.dst_seq, s.dst_token_start, s.len, old, new, pos_map=pm))
        return kvr.resident_span_array(spans)

    def run_inplace(self, ctx, spans, stream=None, dst=None):
        return ctx.reposition_inplace(dst if dst is not None else self.dst, spans, stream=stream)

    # ---- NEXT-2: span overwrite (kvr_write_span) of every segment's rows, unrotated ----
    def write_spans(self):
        w = self.w
        return kvr.span_array([kvr.span(k, v, w.src_strides(s), s.len, s.dst_seq, s.dst_token_start)
                               for s, (k, v) in zip(w.segments, self.sources)])

    # ---- host-resident sources (kvr_reposition_splice_host) ----
    def make_host_sources(self):
        """Pinned host copies of the sources, position maps and source scales, and the segment array that
        points at them.  Dense [layers][heads][len][dim] only (the host entry point requires it)."""
        w = self.w
        assert all(s.src_row_pad == 0 for s in w.segments)
        self.host_sources = [(k.cpu().pin_memory(), None if v is None else v.cpu().pin_memory())
                             for k, v in self.sources]
        self.host_pos_maps = [None if pm is None else pm.cpu().pin_memory() for pm in self.pos_maps]
        self.host_k_scale_src = None if self.k_scale_src is None else self.k_scale_src.cpu().pin_memory()
        self.host_segs = kvr.segment_array([
            kvr.segment(k, v, w.src_strides(s), s.len, s.old_start, s.new_start, s.dst_seq, s.dst_token_start,
                        pos_map=pm, k_scale_src=self.host_k_scale_src,
                        flags=_seg_flags(s))
            for s, (k, v), pm in zip(w.segments, self.host_sources, self.host_pos_maps)])
        return self.host_segs

    def run_host(self, ctx, stream=None, dst=None):
        return ctx.reposition_splice_host(dst if dst is not None else self.dst, self.host_segs, stream=stream)


def bits_to_numpy(t):
    """Bit-pattern tensor (int16 for bf16, uint8 for fp8) -> contiguous numpy array (uint16 / uint8) on the host."""
    a = t.detach().cpu().contiguous().numpy()
    return a.view(np.uint16) if a.dtype == np.int16 else a


class DeviceReadWorkload:
    """Sources, queries and outputs of a workloads.ReadWorkload resident on `device`, plus the ctypes structs of one
    kvr_rotate_on_read_attention call (one layer) over all segments.  guard_bytes as in DeviceWorkload."""

    def __init__(self, w, device="cuda:0", sources=None, queries=None, guard_bytes=0):
        from workloads import make_queries, make_read_sources
        self.w = w
        self.device = torch.device(device)
        self.guard_bytes = int(guard_bytes)
        self._guarded = []
        self.model, self._inv_keep = kvr.model_desc(w.layers, w.kv_heads, w.head_dim, w.rotary_dim, _PAIRING[w.pairing],
                                                    kvr.KVR_BF16, w.inv_freq, rotary_offset=w.rotary_offset)
        if sources is None:
            sources = make_read_sources(w, self.device)
        if queries is None:
            queries = make_queries(w, self.device)
        self.sources = [(self._dev(k, f"k_src[{i}]"), self._dev(v, f"v_src[{i}]")) for i, (k, v) in enumerate(sources)]
        self.q = self._dev(queries, "q")
        self.o = self._dev(torch.full((w.n_req, w.q_heads, w.head_dim), float("nan"), dtype=torch.float32), "o")
        self.lse = self._dev(torch.full((w.n_req, w.q_heads), float("nan"), dtype=torch.float32), "lse")
        self.segs = kvr.read_segment_array([kvr.read_segment(k, v, w.src_strides(s), s.len, s.delta, s.request,
                                                             flags=kvr.KVR_SEG_SRC_STABLE if getattr(s, "src_stable", True) else 0)
                                            for s, (k, v) in zip(w.segments, self.sources)])

    _dev = DeviceWorkload._dev
    check_guards = DeviceWorkload.check_guards

    def bytes_read(self):
        return kvr.kvr_attention_bytes_read(self.model, self.segs)

    def run(self, ctx, stream=None, layer=None):
        w = self.w
        return ctx.rotate_on_read_attention(self.q, w.n_req, w.q_heads, w.layer if layer is None else layer, w.scale,
                                            self.segs, self.o, self.lse, stream=stream)
