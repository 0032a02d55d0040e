"""ctypes wrapper around oracle/libkvr_oracle.so -- ORACLE, test infrastructure.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
reference legs may import this module.  It imports nothing from the product
package and the product package imports nothing from here.  All arrays are
numpy arrays in HOST memory: uint16 holds bf16 bit patterns, uint8 holds
e4m3fn bit patterns.  See kvr_oracle.c for the definition and its citations
(PAPER.md:131, :393, :143).
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

BF16, FP8_E4M3 = 0, 1
NEOX_HALF, GPTJ_INTERLEAVED = 0, 1
OK, ERR_INVALID_ARG, ERR_OUT_OF_RANGE = 0, -1, -4
SEG_PRE_ROPE = 1

_lib = None


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        _lib = C.CDLL(path)
        _lib.kvr_oracle_bf16_decode.restype = C.c_double
        _lib.kvr_oracle_bf16_decode.argtypes = [C.c_uint16]
        _lib.kvr_oracle_bf16_encode.restype = C.c_uint16
        _lib.kvr_oracle_bf16_encode.argtypes = [C.c_double]
        _lib.kvr_oracle_e4m3_decode.restype = C.c_double
        _lib.kvr_oracle_e4m3_decode.argtypes = [C.c_uint8]
        _lib.kvr_oracle_e4m3_encode_sat.restype = C.c_uint8
        _lib.kvr_oracle_e4m3_encode_sat.argtypes = [C.c_double]
        _lib.kvr_oracle_rotate_f64.restype = C.c_int
        _lib.kvr_oracle_rotate_f64.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_int, C.c_int,
                                               C.c_int, C.c_void_p, C.c_void_p]
        _lib.kvr_oracle_reposition_splice.restype = C.c_int
        _lib.kvr_oracle_reposition_splice.argtypes = (
            [C.c_int] * 6 + [C.c_void_p] +                      # model
            [C.c_void_p, C.c_void_p] + [C.c_int64] * 4 + [C.c_int, C.c_int] +
            [C.c_void_p, C.c_int, C.c_int, C.c_void_p] +          # pool
            [C.c_void_p, C.c_void_p] + [C.c_int64] * 3 + [C.c_int] * 5 +
            [C.c_void_p, C.c_void_p] +                            # segment
            [C.c_int] * 3)                                        # control
        _lib.kvr_oracle_reposition_splice_ex.restype = C.c_int
        _lib.kvr_oracle_reposition_splice_ex.argtypes = (
            [C.c_int] * 7 + [C.c_void_p] +                      # model (+ rotary_offset)
            [C.c_void_p, C.c_void_p] + [C.c_int64] * 4 + [C.c_int, C.c_int] +
            [C.c_void_p, C.c_int, C.c_int, C.c_void_p] +
            [C.c_void_p, C.c_void_p] + [C.c_int64] * 3 + [C.c_int] * 5 +
            [C.c_void_p, C.c_void_p, C.c_int] +                   # pos_map, k_scale_src, seg_flags
            [C.c_int] * 3)
        _lib.kvr_oracle_reposition_inplace_ex.restype = C.c_int
        _lib.kvr_oracle_reposition_inplace_ex.argtypes = (
            [C.c_int] * 7 + [C.c_void_p] +
            [C.c_void_p] + [C.c_int64] * 4 + [C.c_int, C.c_int] +
            [C.c_void_p, C.c_int, C.c_int, C.c_void_p] +
            [C.c_int] * 5 + [C.c_void_p] +
            [C.c_int] * 3)
        _lib.kvr_oracle_reposition_inplace.restype = C.c_int
        _lib.kvr_oracle_reposition_inplace.argtypes = (
            [C.c_int] * 6 + [C.c_void_p] +                      # model
            [C.c_void_p] + [C.c_int64] * 4 + [C.c_int, C.c_int] +
            [C.c_void_p, C.c_int, C.c_int, C.c_void_p] +          # pool (K only)
            [C.c_int] * 5 + [C.c_void_p] +                        # the resident span
            [C.c_int] * 3)                                        # control
        _lib.kvr_oracle_bytes_moved.restype = C.c_uint64
        _lib.kvr_oracle_bytes_moved.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, C.c_int64]
        _lib.kvr_oracle_rotate_on_read_attention.restype = C.c_int
        _lib.kvr_oracle_rotate_on_read_attention.argtypes = (
            [C.c_void_p] + [C.c_int] * 6 + [C.c_void_p, C.c_double] +     # q, shapes, inv_freq, scale
            [C.c_int] + [C.c_void_p] * 6 +                                  # segments
            [C.c_void_p, C.c_void_p, C.c_int])                              # o, lse, n_threads
        _lib.kvr_oracle_attention_bytes_read.restype = C.c_uint64
        _lib.kvr_oracle_attention_bytes_read.argtypes = [C.c_int, C.c_int, C.c_int64]
    return _lib


def _ptr(a, dtype=None, writable=False):
    if a is None:
        return None
    assert isinstance(a, np.ndarray), type(a)
    if dtype is not None:
        assert a.dtype == dtype, (a.dtype, dtype)
    assert a.flags["C_CONTIGUOUS"]
    if writable:
        assert a.flags["WRITEABLE"]
    return a.ctypes.data


# ---- codecs (scalar, and vectorised by plain loops over the C scalar routine) ----

def bf16_decode(bits):
    f = lib().kvr_oracle_bf16_decode
    b = np.asarray(bits, dtype=np.uint16)
    return np.array([f(int(x)) for x in b.ravel()], dtype=np.float64).reshape(b.shape)


def bf16_encode(x):
    f = lib().kvr_oracle_bf16_encode
    v = np.asarray(x, dtype=np.float64)
    return np.array([f(float(t)) for t in v.ravel()], dtype=np.uint16).reshape(v.shape)


def e4m3_decode(bits):
    f = lib().kvr_oracle_e4m3_decode
    b = np.asarray(bits, dtype=np.uint8)
    return np.array([f(int(x)) for x in b.ravel()], dtype=np.float64).reshape(b.shape)


def e4m3_encode_sat(x):
    f = lib().kvr_oracle_e4m3_encode_sat
    v = np.asarray(x, dtype=np.float64)
    return np.array([f(float(t)) for t in v.ravel()], dtype=np.uint8).reshape(v.shape)


# ---- pure fp64 rotation (the arithmetic core; RoPE itself when applied to a pre-RoPE key) ----

def rotate_f64(x, delta, inv_freq, rotary_dim, pairing):
    """x: [n, head_dim] float64; delta: [n] int64 position shift per row."""
    x = np.ascontiguousarray(x, dtype=np.float64)
    n, head_dim = x.shape
    delta = np.ascontiguousarray(np.broadcast_to(np.asarray(delta, dtype=np.int64), (n,)))
    inv_freq = np.ascontiguousarray(inv_freq, dtype=np.float64)
    assert inv_freq.shape == (rotary_dim // 2,)
    out = np.empty_like(x)
    st = lib().kvr_oracle_rotate_f64(_ptr(x), _ptr(out, writable=True), n, head_dim, rotary_dim,
                                     pairing, _ptr(inv_freq), _ptr(delta))
    if st != OK:
        raise ValueError(f"kvr_oracle_rotate_f64 -> {st}")
    return out


# ---- the oracle proper ----

def reposition_splice(*, layers, kv_heads, head_dim, rotary_dim, pairing, dtype, inv_freq,
                      k_cache, v_cache, stride_layer, stride_block, stride_token, stride_head,
                      num_blocks, block_size, block_table, k_scale_dst=None,
                      k_src, v_src, src_stride_layer, src_stride_head, src_stride_token,
                      len, old_start, new_start, dst_seq, dst_token_start,
                      pos_map=None, k_scale_src=None,
                      layer_begin=0, layer_end=None, n_threads=1, rotary_offset=0, pre_rope=False):
    """Splices ONE segment into (k_cache, v_cache) in place.  Returns the status code.
    rotary_offset != 0 or v_cache is None / v_src is None (a [latent | k_pe] cache, reading R23) go through
    kvr_oracle_reposition_splice_ex."""
    edt = np.uint16 if dtype == BF16 else np.uint8
    inv_freq = np.ascontiguousarray(inv_freq, dtype=np.float64)
    assert inv_freq.shape == (rotary_dim // 2,)
    assert block_table.dtype == np.int32 and block_table.ndim == 2
    num_seqs, max_blocks = block_table.shape
    if layer_end is None:
        layer_end = layers
    if rotary_offset != 0 or v_cache is None or v_src is None or pre_rope:
        return lib().kvr_oracle_reposition_splice_ex(
            layers, kv_heads, head_dim, rotary_dim, rotary_offset, pairing, dtype, _ptr(inv_freq),
            _ptr(k_cache, edt, True), _ptr(v_cache, edt, True),
            stride_layer, stride_block, stride_token, stride_head, num_blocks, block_size,
            _ptr(block_table, np.int32), num_seqs, max_blocks, _ptr(k_scale_dst, np.float32),
            _ptr(k_src, edt), _ptr(v_src, edt), src_stride_layer, src_stride_head, src_stride_token,
            len, old_start, new_start, dst_seq, dst_token_start,
            _ptr(pos_map, np.int32), _ptr(k_scale_src, np.float32), SEG_PRE_ROPE if pre_rope else 0,
            layer_begin, layer_end, n_threads)
    return lib().kvr_oracle_reposition_splice(
        layers, kv_heads, head_dim, rotary_dim, pairing, dtype, _ptr(inv_freq),
        _ptr(k_cache, edt, True), _ptr(v_cache, edt, True),
        stride_layer, stride_block, stride_token, stride_head, num_blocks, block_size,
        _ptr(block_table, np.int32), num_seqs, max_blocks, _ptr(k_scale_dst, np.float32),
        _ptr(k_src, edt), _ptr(v_src, edt), src_stride_layer, src_stride_head, src_stride_token,
        len, old_start, new_start, dst_seq, dst_token_start,
        _ptr(pos_map, np.int32), _ptr(k_scale_src, np.float32),
        layer_begin, layer_end, n_threads)


def reposition_inplace(*, layers, kv_heads, head_dim, rotary_dim, pairing, dtype, inv_freq,
                       k_cache, stride_layer, stride_block, stride_token, stride_head,
                       num_blocks, block_size, block_table, k_scale=None,
                       seq, token_start, len, old_start, new_start, pos_map=None,
                       layer_begin=0, layer_end=None, n_threads=1, rotary_offset=0):
    """Re-rotates ONE resident span of k_cache in place (kvr_oracle_reposition_inplace).  Returns the status."""
    edt = np.uint16 if dtype == BF16 else np.uint8
    inv_freq = np.ascontiguousarray(inv_freq, dtype=np.float64)
    assert inv_freq.shape == (rotary_dim // 2,)
    assert block_table.dtype == np.int32 and block_table.ndim == 2
    num_seqs, max_blocks = block_table.shape
    if layer_end is None:
        layer_end = layers
    if rotary_offset != 0:
        return lib().kvr_oracle_reposition_inplace_ex(
            layers, kv_heads, head_dim, rotary_dim, rotary_offset, pairing, dtype, _ptr(inv_freq),
            _ptr(k_cache, edt, True), stride_layer, stride_block, stride_token, stride_head,
            num_blocks, block_size, _ptr(block_table, np.int32), num_seqs, max_blocks, _ptr(k_scale, np.float32),
            seq, token_start, len, old_start, new_start, _ptr(pos_map, np.int32),
            layer_begin, layer_end, n_threads)
    return lib().kvr_oracle_reposition_inplace(
        layers, kv_heads, head_dim, rotary_dim, pairing, dtype, _ptr(inv_freq),
        _ptr(k_cache, edt, True), stride_layer, stride_block, stride_token, stride_head,
        num_blocks, block_size, _ptr(block_table, np.int32), num_seqs, max_blocks, _ptr(k_scale, np.float32),
        seq, token_start, len, old_start, new_start, _ptr(pos_map, np.int32),
        layer_begin, layer_end, n_threads)


def bytes_moved(layers, kv_heads, head_dim, dtype, tokens):
    return int(lib().kvr_oracle_bytes_moved(layers, kv_heads, head_dim, dtype, tokens))


def rotate_on_read_attention(*, q, kv_heads, rotary_dim, pairing, inv_freq, scale, segments, rotary_offset=0,
                             n_threads=1):
    """kvr_oracle_rotate_on_read_attention (kvr_attention_oracle.c; reading R25) for ONE request at ONE layer.
    q: uint16 [q_heads, head_dim] bf16 bits (post-RoPE at the query's position).  segments: list of
    (k_bits, v_bits, delta) with k_bits / v_bits uint16 arrays [kv_heads, len, head_dim] AT THAT LAYER (any strides
    numpy can express with head_dim contiguous).  Returns (o float64 [q_heads, head_dim], lse float64 [q_heads])."""
    q = np.ascontiguousarray(q, dtype=np.uint16)
    q_heads, head_dim = q.shape
    inv_freq = np.ascontiguousarray(inv_freq, dtype=np.float64)
    assert inv_freq.shape == (rotary_dim // 2,)
    n = len(segments)
    keep, kp, vp = [], (C.c_void_p * n)(), (C.c_void_p * n)()
    sh, st = np.empty(n, np.int64), np.empty(n, np.int64)
    ln, dl = np.empty(n, np.int32), np.empty(n, np.int32)
    for i, (k, v, delta) in enumerate(segments):
        assert k.dtype == np.uint16 and v.dtype == np.uint16 and k.shape == v.shape and k.shape[0] == kv_heads
        assert k.shape[2] == head_dim and k.strides[2] == 2 and v.strides == k.strides, (k.shape, k.strides, v.strides)
        keep.append((k, v))
        kp[i], vp[i] = k.ctypes.data, v.ctypes.data
        sh[i], st[i], ln[i], dl[i] = k.strides[0] // 2, k.strides[1] // 2, k.shape[1], delta
    o = np.empty((q_heads, head_dim), np.float64)
    lse = np.empty(q_heads, np.float64)
    status = lib().kvr_oracle_rotate_on_read_attention(
        _ptr(q), q_heads, kv_heads, head_dim, rotary_dim, rotary_offset, pairing, _ptr(inv_freq), float(scale),
        n, C.cast(kp, C.c_void_p), C.cast(vp, C.c_void_p), _ptr(sh), _ptr(st), _ptr(ln), _ptr(dl),
        _ptr(o, writable=True), _ptr(lse, writable=True), n_threads)
    if status != OK:
        raise ValueError(f"kvr_oracle_rotate_on_read_attention -> {status}")
    return o, lse


def attention_bytes_read(kv_heads, head_dim, tokens):
    return int(lib().kvr_oracle_attention_bytes_read(kv_heads, head_dim, tokens))


def host_threads():
    """Threads the OpenMP timing variant can use = cores this process may run on."""
    return len(os.sched_getaffinity(0))


# ---- adapter: a workloads.Workload (duck-typed: only attributes are read) -> one oracle call per segment ----

_PAIRING = {"neox": NEOX_HALF, "gptj": GPTJ_INTERLEAVED}
_DTYPE = {"bf16": BF16, "fp8": FP8_E4M3}


def splice_workload(w, srcs, k_cache, v_cache, n_threads=1, layer_begin=0, layer_end=None, segments=None):
    """Splices every segment of w (sources srcs[i] = (k_bits, v_bits) numpy arrays) into the numpy pools
    (k_cache, v_cache) in place.  Pure marshalling; the arithmetic is kvr_oracle.c."""
    s_l, s_b, s_t, s_h = w.dst_strides()
    for i, seg in enumerate(w.segments):
        if segments is not None and i not in segments:
            continue
        k_src, v_src = srcs[i]
        no_v = v_src is None or v_cache is None      # a [latent | k_pe] cache has no V tensor (R23)
        sl, sh, st = w.src_strides(seg)
        status = reposition_splice(
            layers=w.layers, kv_heads=w.kv_heads, head_dim=w.head_dim, rotary_dim=w.rotary_dim,
            pairing=_PAIRING[w.pairing], dtype=_DTYPE[w.dtype], inv_freq=w.inv_freq,
            k_cache=k_cache, v_cache=None if no_v else v_cache, stride_layer=s_l, stride_block=s_b, stride_token=s_t,
            stride_head=s_h, num_blocks=w.num_blocks, block_size=w.block_size, block_table=w.block_table,
            k_scale_dst=w.k_scale, k_src=np.ascontiguousarray(k_src).reshape(-1),
            v_src=None if no_v else np.ascontiguousarray(v_src).reshape(-1),
            src_stride_layer=sl, src_stride_head=sh, src_stride_token=st,
            len=seg.len, old_start=seg.old_start, new_start=seg.new_start, dst_seq=seg.dst_seq,
            dst_token_start=seg.dst_token_start, pos_map=seg.pos_map, k_scale_src=w.k_scale_src,
            layer_begin=layer_begin, layer_end=layer_end, n_threads=n_threads,
            rotary_offset=getattr(w, "rotary_offset", 0), pre_rope=getattr(seg, "pre_rope", False))
        if status != OK:
            raise RuntimeError(f"oracle: segment {i} -> status {status}")


def inplace_workload(w, k_cache, n_threads=1, layer_begin=0, layer_end=None, deltas=None):
    """Re-rotates, in place, the span every segment of w occupies in k_cache: segment i moves from the positions
    it was spliced at (new_start.., or its pos_map) by deltas[i] more positions.  Pure marshalling."""
    s_l, s_b, s_t, s_h = w.dst_strides()
    for i, seg in enumerate(w.segments):
        d = int(deltas[i])
        status = reposition_inplace(
            layers=w.layers, kv_heads=w.kv_heads, head_dim=w.head_dim, rotary_dim=w.rotary_dim,
            pairing=_PAIRING[w.pairing], dtype=_DTYPE[w.dtype], inv_freq=w.inv_freq, k_cache=k_cache,
            stride_layer=s_l, stride_block=s_b, stride_token=s_t, stride_head=s_h, num_blocks=w.num_blocks,
            block_size=w.block_size, block_table=w.block_table, k_scale=w.k_scale,
            seq=seg.dst_seq, token_start=seg.dst_token_start, len=seg.len, old_start=max(0, -d), new_start=max(0, d),
            layer_begin=layer_begin, layer_end=layer_end, n_threads=n_threads,
            rotary_offset=getattr(w, "rotary_offset", 0))
        if status != OK:
            raise RuntimeError(f"oracle in-place: segment {i} -> status {status}")
