"""Thin ctypes binding of libkvr.so -- argument marshalling only; every step of the path runs in the
CUDA kernels behind the C ABI (include/kvr.h).  torch is used by callers for device memory and streams;
this module only needs `.data_ptr()`-style integers.

Names mirror the C ABI: kvr_create / kvr_destroy / kvr_reposition_splice / kvr_bytes_moved /
kvr_validate / kvr_last_device_status / ...  `Context` is a small RAII convenience on top of them.
"""
import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libkvr.so")

KVR_OK, KVR_ERR_INVALID_ARG, KVR_ERR_UNSUPPORTED, KVR_ERR_ALIGNMENT = 0, -1, -2, -3
KVR_ERR_OUT_OF_RANGE, KVR_ERR_CUDA, KVR_ERR_NOMEM = -4, -5, -6
KVR_BF16, KVR_FP8_E4M3 = 0, 1
KVR_PAIR_NEOX_HALF, KVR_PAIR_GPTJ_INTERLEAVED = 0, 1
KVR_SEG_PRE_ROPE, KVR_SEG_SRC_STABLE = 1, 2
KVR_NOALLOC_MAX_SEGMENTS, KVR_NOALLOC_MAX_ROTARY_DIM, KVR_NOALLOC_SCRATCH_BYTES = 8, 1024, 4352
PATH_AUTO, PATH_GENERIC, PATH_RING, PATH_ATTEND, PATH_WINDOW, PATH_GENERIC_VEC = 0, 1, 2, 3, 4, 5


class kvr_model_desc(C.Structure):
    _fields_ = [("layers", C.c_int32), ("kv_heads", C.c_int32), ("head_dim", C.c_int32),
                ("rotary_dim", C.c_int32), ("pairing", C.c_int32), ("dtype", C.c_int32),
                ("inv_freq", C.POINTER(C.c_double)),
                ("rotary_offset", C.c_int32), ("reserved_", C.c_int32)]


class kvr_paged_dst(C.Structure):
    _fields_ = [("k_cache", C.c_void_p), ("v_cache", C.c_void_p),
                ("stride_layer", C.c_int64), ("stride_block", C.c_int64),
                ("stride_token", C.c_int64), ("stride_head", C.c_int64),
                ("num_blocks", C.c_int32), ("block_size", C.c_int32),
                ("block_table", C.c_void_p),
                ("num_seqs", C.c_int32), ("max_blocks_per_seq", C.c_int32),
                ("k_scale", C.c_void_p)]


class kvr_segment(C.Structure):
    _fields_ = [("k_src", C.c_void_p), ("v_src", C.c_void_p),
                ("src_stride_layer", C.c_int64), ("src_stride_head", C.c_int64),
                ("src_stride_token", C.c_int64),
                ("len", C.c_int32), ("old_start", C.c_int32), ("new_start", C.c_int32),
                ("dst_seq", C.c_int32), ("dst_token_start", C.c_int32), ("flags", C.c_int32),
                ("pos_map", C.c_void_p), ("k_scale_src", C.c_void_p)]


class kvr_tuning(C.Structure):
    _fields_ = [("path", C.c_int32), ("ctas_per_sm", C.c_int32), ("consumer_warps", C.c_int32),
                ("stages", C.c_int32), ("layers_per_unit", C.c_int32), ("v_bulk_store", C.c_int32),
                ("max_ctas", C.c_int32), ("grab", C.c_int32), ("pdl", C.c_int32), ("hsplit", C.c_int32),
                ("chunk_tokens", C.c_int32), ("tile_bytes", C.c_int32), ("gather", C.c_int32),
                ("warps_per_stage", C.c_int32), ("lanes_over_heads", C.c_int32), ("transpose_load", C.c_int32)]


class kvr_resident_span(C.Structure):
    _fields_ = [("seq", C.c_int32), ("token_start", C.c_int32), ("len", C.c_int32),
                ("old_start", C.c_int32), ("new_start", C.c_int32), ("pos_map", C.c_void_p)]


class kvr_span(C.Structure):
    _fields_ = [("k_src", C.c_void_p), ("v_src", C.c_void_p),
                ("src_stride_layer", C.c_int64), ("src_stride_head", C.c_int64), ("src_stride_token", C.c_int64),
                ("len", C.c_int32), ("dst_seq", C.c_int32), ("dst_token_start", C.c_int32)]


class kvr_read_segment(C.Structure):
    _fields_ = [("k_src", C.c_void_p), ("v_src", C.c_void_p),
                ("src_stride_layer", C.c_int64), ("src_stride_head", C.c_int64), ("src_stride_token", C.c_int64),
                ("len", C.c_int32), ("delta", C.c_int32), ("request", C.c_int32), ("flags", C.c_int32)]


EXPORTS = ["kvr_rotate_on_read_attention", "kvr_attention_bytes_read", "kvr_validate_read", "kvr_reposition_inplace", "kvr_inplace_bytes_moved", "kvr_write_span",
           "kvr_create", "kvr_destroy", "kvr_set_tuning", "kvr_validate", "kvr_reposition_splice",
           "kvr_reposition_splice_noalloc",
           "kvr_reposition_splice_host", "kvr_last_h2d_bytes",
           "kvr_bytes_moved", "kvr_last_device_status", "kvr_launch_count", "kvr_last_launch_info",
           "kvr_status_string", "kvr_last_cuda_error", "kvr_version"]


def _load():
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2606_17107_b200.build` "
                          "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    P = C.POINTER
    lib.kvr_create.restype = C.c_int
    lib.kvr_create.argtypes = [P(C.c_void_p), P(kvr_model_desc), C.c_int]
    lib.kvr_destroy.restype = C.c_int
    lib.kvr_destroy.argtypes = [C.c_void_p]
    lib.kvr_set_tuning.restype = C.c_int
    lib.kvr_set_tuning.argtypes = [C.c_void_p, P(kvr_tuning)]
    lib.kvr_validate.restype = C.c_int
    lib.kvr_validate.argtypes = [P(kvr_model_desc), P(kvr_paged_dst), P(kvr_segment), C.c_int32]
    lib.kvr_reposition_splice.restype = C.c_int
    lib.kvr_reposition_splice.argtypes = [C.c_void_p, P(kvr_paged_dst), P(kvr_segment), C.c_int32, C.c_void_p]
    lib.kvr_reposition_splice_noalloc.restype = C.c_int
    lib.kvr_reposition_splice_noalloc.argtypes = [P(kvr_model_desc), C.c_int, P(kvr_paged_dst), P(kvr_segment), C.c_int32,
                                                  C.c_void_p, C.c_void_p, C.c_char_p, C.c_int32]
    lib.kvr_reposition_splice_host.restype = C.c_int
    lib.kvr_reposition_splice_host.argtypes = lib.kvr_reposition_splice.argtypes
    lib.kvr_reposition_inplace.restype = C.c_int
    lib.kvr_reposition_inplace.argtypes = [C.c_void_p, P(kvr_paged_dst), P(kvr_resident_span), C.c_int32, C.c_void_p]
    lib.kvr_inplace_bytes_moved.restype = C.c_uint64
    lib.kvr_inplace_bytes_moved.argtypes = [P(kvr_model_desc), P(kvr_resident_span), C.c_int32]
    lib.kvr_write_span.restype = C.c_int
    lib.kvr_write_span.argtypes = [C.c_void_p, P(kvr_paged_dst), P(kvr_span), C.c_int32, C.c_void_p]
    lib.kvr_rotate_on_read_attention.restype = C.c_int
    lib.kvr_rotate_on_read_attention.argtypes = [C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.c_int32, C.c_float,
                                                 P(kvr_read_segment), C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p]
    lib.kvr_validate_read.restype = C.c_int
    lib.kvr_validate_read.argtypes = [P(kvr_model_desc), C.c_void_p, C.c_int32, C.c_int32, C.c_int32, C.c_float,
                                      P(kvr_read_segment), C.c_int32, C.c_void_p, C.c_void_p]
    lib.kvr_attention_bytes_read.restype = C.c_uint64
    lib.kvr_attention_bytes_read.argtypes = [P(kvr_model_desc), P(kvr_read_segment), C.c_int32]
    lib.kvr_last_h2d_bytes.restype = C.c_uint64
    lib.kvr_last_h2d_bytes.argtypes = [C.c_void_p]
    lib.kvr_bytes_moved.restype = C.c_uint64
    lib.kvr_bytes_moved.argtypes = [P(kvr_model_desc), P(kvr_segment), C.c_int32]
    lib.kvr_last_device_status.restype = C.c_int
    lib.kvr_last_device_status.argtypes = [C.c_void_p, P(C.c_int32), P(C.c_int32)]
    lib.kvr_launch_count.restype = C.c_uint64
    lib.kvr_launch_count.argtypes = [C.c_void_p]
    lib.kvr_last_launch_info.restype = C.c_int
    lib.kvr_last_launch_info.argtypes = [C.c_void_p] + [P(C.c_int32)] * 4
    lib.kvr_status_string.restype = C.c_char_p
    lib.kvr_status_string.argtypes = [C.c_int]
    lib.kvr_last_cuda_error.restype = C.c_char_p
    lib.kvr_last_cuda_error.argtypes = [C.c_void_p]
    lib.kvr_version.restype = C.c_char_p
    lib.kvr_version.argtypes = []
    return lib


lib = _load()


class KvrError(RuntimeError):
    def __init__(self, status, detail=""):
        self.status = status
        super().__init__(f"{lib.kvr_status_string(status).decode()}{(': ' + detail) if detail else ''}")


def _ptr(x):
    """int address from a torch tensor / numpy array / int / None."""
    if x is None:
        return None
    if isinstance(x, int):
        return x
    if hasattr(x, "data_ptr"):
        return x.data_ptr()
    if hasattr(x, "ctypes"):
        return x.ctypes.data
    raise TypeError(type(x))


def model_desc(layers, kv_heads, head_dim, rotary_dim, pairing, dtype, inv_freq, rotary_offset=0):
    """inv_freq: sequence / numpy array of rotary_dim/2 doubles (HOST).  Returns (desc, keepalive)."""
    arr = (C.c_double * len(inv_freq))(*[float(f) for f in inv_freq])
    return kvr_model_desc(layers, kv_heads, head_dim, rotary_dim, pairing, dtype, arr, rotary_offset, 0), arr


def paged_dst(k_cache, v_cache, strides, num_blocks, block_size, block_table, num_seqs, max_blocks_per_seq,
              k_scale=None):
    s_l, s_b, s_t, s_h = strides
    return kvr_paged_dst(_ptr(k_cache), _ptr(v_cache), s_l, s_b, s_t, s_h, num_blocks, block_size,
                         _ptr(block_table), num_seqs, max_blocks_per_seq, _ptr(k_scale))


def segment(k_src, v_src, src_strides, len, old_start, new_start, dst_seq, dst_token_start, pos_map=None,
            k_scale_src=None, flags=0):
    sl, sh, st = src_strides
    return kvr_segment(_ptr(k_src), _ptr(v_src), sl, sh, st, len, old_start, new_start, dst_seq,
                       dst_token_start, flags, _ptr(pos_map), _ptr(k_scale_src))


def resident_span(seq, token_start, len, old_start, new_start, pos_map=None):
    return kvr_resident_span(seq, token_start, len, old_start, new_start, _ptr(pos_map))


def resident_span_array(spans):
    return (kvr_resident_span * len(spans))(*spans)


def span(k_src, v_src, src_strides, len, dst_seq, dst_token_start):
    sl, sh, st = src_strides
    return kvr_span(_ptr(k_src), _ptr(v_src), sl, sh, st, len, dst_seq, dst_token_start)


def span_array(spans):
    return (kvr_span * len(spans))(*spans)


def read_segment(k_src, v_src, src_strides, len, delta, request, flags=0):
    sl, sh, st = src_strides
    return kvr_read_segment(_ptr(k_src), _ptr(v_src), sl, sh, st, len, delta, request, flags)


def read_segment_array(segs):
    return (kvr_read_segment * len(segs))(*segs)


def kvr_validate_read(model, q, n_req, q_heads, layer, softmax_scale, segs, o, lse):
    arr = segs if not isinstance(segs, (list, tuple)) else read_segment_array(segs)
    return lib.kvr_validate_read(C.byref(model), _ptr(q), n_req, q_heads, layer, softmax_scale, arr, len(arr), _ptr(o), _ptr(lse))


def kvr_attention_bytes_read(model, segs):
    arr = segs if not isinstance(segs, (list, tuple)) else read_segment_array(segs)
    return int(lib.kvr_attention_bytes_read(C.byref(model), arr, len(arr)))


def kvr_inplace_bytes_moved(model, spans):
    arr = spans if not isinstance(spans, (list, tuple)) else resident_span_array(spans)
    return int(lib.kvr_inplace_bytes_moved(C.byref(model), arr, len(arr)))


def segment_array(segs):
    return (kvr_segment * len(segs))(*segs)


def kvr_validate(model, dst, segs):
    arr = segs if not isinstance(segs, (list, tuple)) else segment_array(segs)
    return lib.kvr_validate(C.byref(model), C.byref(dst), arr, len(arr))


def kvr_bytes_moved(model, segs):
    arr = segs if not isinstance(segs, (list, tuple)) else segment_array(segs)
    return int(lib.kvr_bytes_moved(C.byref(model), arr, len(arr)))


def kvr_reposition_splice_noalloc(model, dst, segs, device=0, device_status=None, stream=None, check=True):
    """kvr_reposition_splice_noalloc (kvr.h): the reposition + splice for hosts that cannot let this library allocate
    CUDA memory (an engine that gave all free HBM to its KV pool, a process with a graph capture in flight on another
    thread, a plug-in under a no-driver-allocations policy).  No Context: the scheduler counters, status word and
    inv_freq table sit in a fixed 4352-byte array inside the library's device image, shared by every call on the device,
    so calls must not overlap on the GPU.  At most 8 segments and rotary_dim <= 1024 per call (KvrError otherwise).
    device_status: optional device int32[4] that receives {flag, segment, token, -} for a bad block-table entry.
    Make the first call on a device outside any stream capture."""
    arr = segs if not isinstance(segs, (list, tuple)) else segment_array(segs)
    s = None if stream is None else (stream if isinstance(stream, int) else stream.cuda_stream)
    msg = C.create_string_buffer(256)
    st = lib.kvr_reposition_splice_noalloc(C.byref(model), device, C.byref(dst), arr, len(arr), _ptr(device_status), s,
                                           msg, len(msg))
    if check and st != KVR_OK:
        raise KvrError(st, msg.value.decode())
    return st


def kvr_version():
    return lib.kvr_version().decode()


class Context:
    """kvr_create / kvr_destroy with the other calls as methods."""

    def __init__(self, model: kvr_model_desc, device: int = 0):
        self._h = C.c_void_p()
        self._model = model
        st = lib.kvr_create(C.byref(self._h), C.byref(model), device)
        if st != KVR_OK:
            self._h = C.c_void_p()
            raise KvrError(st, "kvr_create (no usable sm_100 CUDA device?)")

    def close(self):
        if self._h:
            lib.kvr_destroy(self._h)
            self._h = C.c_void_p()

    __del__ = close

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def set_tuning(self, **kw):
        t = kvr_tuning()
        for k, v in kw.items():
            setattr(t, k, v)
        st = lib.kvr_set_tuning(self._h, C.byref(t))
        if st != KVR_OK:
            raise KvrError(st)

    def reposition_splice(self, dst: kvr_paged_dst, segs, stream=None, check=True):
        """segs: ctypes array from segment_array() (preferred: no per-call marshalling) or a list.
        stream: an int cudaStream_t, a torch.cuda.Stream, or None (legacy default stream)."""
        arr = segs if not isinstance(segs, (list, tuple)) else segment_array(segs)
        s = None if stream is None else (stream if isinstance(stream, int) else stream.cuda_stream)
        st = lib.kvr_reposition_splice(self._h, C.byref(dst), arr, len(arr), s)
        if check and st != KVR_OK:
            raise KvrError(st, lib.kvr_last_cuda_error(self._h).decode())
        return st

    def reposition_splice_host(self, dst: kvr_paged_dst, segs, stream=None, check=True):
        """kvr_reposition_splice_host: the segments' k_src / v_src / pos_map / k_scale_src are HOST pointers."""
        arr = segs if not isinstance(segs, (list, tuple)) else segment_array(segs)
        s = None if stream is None else (stream if isinstance(stream, int) else stream.cuda_stream)
        st = lib.kvr_reposition_splice_host(self._h, C.byref(dst), arr, len(arr), s)
        if check and st != KVR_OK:
            raise KvrError(st, lib.kvr_last_cuda_error(self._h).decode())
        return st

    def reposition_inplace(self, pool: kvr_paged_dst, spans, stream=None, check=True):
        """kvr_reposition_inplace: spans = ctypes array from resident_span_array() or a list of kvr_resident_span."""
        arr = spans if not isinstance(spans, (list, tuple)) else resident_span_array(spans)
        s = None if stream is None else (stream if isinstance(stream, int) else stream.cuda_stream)
        st = lib.kvr_reposition_inplace(self._h, C.byref(pool), arr, len(arr), s)
        if check and st != KVR_OK:
            raise KvrError(st, lib.kvr_last_cuda_error(self._h).decode())
        return st

    def write_span(self, dst: kvr_paged_dst, spans, stream=None, check=True):
        """kvr_write_span: spans = ctypes array from span_array() or a list of kvr_span."""
        arr = spans if not isinstance(spans, (list, tuple)) else span_array(spans)
        s = None if stream is None else (stream if isinstance(stream, int) else stream.cuda_stream)
        st = lib.kvr_write_span(self._h, C.byref(dst), arr, len(arr), s)
        if check and st != KVR_OK:
            raise KvrError(st, lib.kvr_last_cuda_error(self._h).decode())
        return st

    def rotate_on_read_attention(self, q, n_req, q_heads, layer, softmax_scale, segs, o, lse, stream=None, check=True):
        """kvr_rotate_on_read_attention: q bf16 [n_req, q_heads, head_dim], o fp32 [n_req, q_heads, head_dim],
        lse fp32 [n_req, q_heads] (device tensors or addresses); segs = read_segment_array() or a list."""
        arr = segs if not isinstance(segs, (list, tuple)) else read_segment_array(segs)
        s = None if stream is None else (stream if isinstance(stream, int) else stream.cuda_stream)
        st = lib.kvr_rotate_on_read_attention(self._h, _ptr(q), n_req, q_heads, layer, softmax_scale, arr, len(arr),
                                              _ptr(o), _ptr(lse), s)
        if check and st != KVR_OK:
            raise KvrError(st, lib.kvr_last_cuda_error(self._h).decode())
        return st

    def last_h2d_bytes(self):
        return int(lib.kvr_last_h2d_bytes(self._h))

    def last_device_status(self):
        seg, tok = C.c_int32(-1), C.c_int32(-1)
        st = lib.kvr_last_device_status(self._h, C.byref(seg), C.byref(tok))
        return st, seg.value, tok.value

    def launch_count(self):
        return int(lib.kvr_launch_count(self._h))

    def last_launch_info(self):
        v = [C.c_int32() for _ in range(4)]
        lib.kvr_last_launch_info(self._h, *[C.byref(x) for x in v])
        return dict(path=v[0].value, grid=v[1].value, block=v[2].value, smem=v[3].value)
