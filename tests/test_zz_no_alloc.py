"""kvr_reposition_splice_noalloc (include/kvr.h): the reposition + splice for hosts of this library that cannot let it
allocate CUDA memory -- a serving engine that handed every free byte of HBM to its KV pool (a late cudaMalloc fails
there, or escapes the engine's accounting), a process in which another thread is recording a CUDA graph (cudaMalloc from
any thread breaks that recording), a plug-in under a "no driver allocations" policy.  The call needs no context; its
scheduler counters, status word and inv_freq table live in one fixed 4352-byte array inside the library's device image,
shared by every call on the device and holding whatever the previous call left there.

What is checked: the pools it writes are the pools the ordinary path (kvr_create + kvr_reposition_splice) writes, at the
tolerance of every other GPU test here (V and untouched bytes bit-exact, K within K_TOL lattice steps -- the kernels are
the same, so in fact 0), for several calls IN A ROW on one stream with different models, so that a stale counter, status
word or frequency table from the previous call would show; and that a call beyond the fixed limits is refused with a
message before anything runs.

This file is named to be collected last: `pytest -x` stops at the first failure, and a failure here must not hide the
parity tests.  It passes alone in a fresh process (the first call on the device does the set-up) and after the others."""
import ctypes as C

import numpy as np
import pytest
import torch

from tests.helpers import K_TOL, k_distance, np_bits
from workloads import config_small

GUARD = 1 << 16


def _pair(w):
    """Two device copies of the same seeded workload: one for the ordinary path, one for the no-allocation call."""
    from paper_2606_17107_b200.harness import DeviceWorkload
    return DeviceWorkload(w, "cuda:0", guard_bytes=GUARD), DeviceWorkload(w, "cuda:0", guard_bytes=GUARD)


def _same_pools(w, ref, got):
    torch.cuda.synchronize()
    got.check_guards()
    if ref.v_cache is not None:
        assert torch.equal(ref.v_cache, got.v_cache), f"{w.name}: V / untouched V bytes differ"
    rk, gk = np_bits(ref.k_cache), np_bits(got.k_cache)
    d = k_distance(w, gk, rk)
    assert d.max() <= K_TOL[w.dtype], (w.name, int(d.max()), int((d > K_TOL[w.dtype]).sum()))
    assert np.array_equal(gk, rk), f"{w.name}: same kernels, same inputs: the K pools should be identical"


def _chunks(arr, n):
    from paper_2606_17107_b200 import kvr
    return [(kvr.kvr_segment * len(arr[i:i + n]))(*arr[i:i + n]) for i in range(0, len(arr), n)]


@pytest.mark.gpu
def test_calls_in_a_row_match_the_ordinary_path():
    """cfg2 (bf16, 4 segments, rotary 128) -> cfg4 (bf16, position map, rotary 64 of 128) -> cfg2 again -> cfg3 (fp8, 12
    segments = two calls of <= 8): every call follows the previous one on the same stream with no synchronisation, each
    with another model, table length and kernel instantiation."""
    from paper_2606_17107_b200 import kvr
    stream = torch.cuda.current_stream()
    cases = []
    for c, layout in ((2, "NHD"), (4, "HND"), (2, "NHD"), (3, "HND")):
        w = config_small(c, layout)
        ref, got = _pair(w)
        with kvr.Context(ref.model) as ctx:                       # the ordinary path: context-owned scratch
            ref.run(ctx, stream=stream)
            assert ctx.last_device_status()[0] == kvr.KVR_OK
        cases.append((w, ref, got))
    torch.cuda.synchronize()
    for w, ref, got in cases:                                     # no synchronisation between these calls
        for part in _chunks(got.segs, kvr.KVR_NOALLOC_MAX_SEGMENTS):
            kvr.kvr_reposition_splice_noalloc(got.model, got.dst, part, device=0, stream=stream)
    for w, ref, got in cases:
        _same_pools(w, ref, got)


@pytest.mark.gpu
def test_twice_into_the_same_pool_and_status_word():
    """The same call twice in a row gives the same pool as once (the counters the first call used are clear again);
    a bad block-table entry is reported through device_status exactly as the context reports it, and a clean call that
    follows does not inherit the flag."""
    from paper_2606_17107_b200 import kvr
    w = config_small(1, "NHD")
    ref, got = _pair(w)
    with kvr.Context(ref.model) as ctx:
        ref.run(ctx)
    status = torch.full((4,), 7, dtype=torch.int32, device="cuda:0")
    kvr.kvr_reposition_splice_noalloc(got.model, got.dst, got.segs, device_status=status)
    kvr.kvr_reposition_splice_noalloc(got.model, got.dst, got.segs, device_status=status)
    _same_pools(w, ref, got)
    assert status.tolist()[0] == 0

    seg = w.segments[0]
    col = (seg.dst_token_start + seg.len // 2) // w.block_size
    for dw in (ref, got):
        dw.block_table[seg.dst_seq, col] = w.num_blocks + 5        # a block id past the pool
    with kvr.Context(ref.model) as ctx:
        ref.run(ctx)
        st, bad_seg, bad_tok = ctx.last_device_status()
    assert st == kvr.KVR_ERR_OUT_OF_RANGE
    kvr.kvr_reposition_splice_noalloc(got.model, got.dst, got.segs, device_status=status)
    torch.cuda.synchronize()
    flag, s, t, _ = status.tolist()
    assert flag != 0 and s == bad_seg == 0
    assert max(0, col * w.block_size - seg.dst_token_start) <= t < (col + 1) * w.block_size - seg.dst_token_start
    _same_pools(w, ref, got)                                      # the bad block's tokens are skipped on both paths
    w0 = config_small(0, "NHD")
    r0, g0 = _pair(w0)
    with kvr.Context(r0.model) as ctx:
        r0.run(ctx)
    kvr.kvr_reposition_splice_noalloc(g0.model, g0.dst, g0.segs, device_status=status)
    _same_pools(w0, r0, g0)
    assert status.tolist()[0] == 0


def test_limits_are_refused_with_a_message_before_anything_runs():
    """More than KVR_NOALLOC_MAX_SEGMENTS segments, or a rotary_dim whose inv_freq table does not fit the fixed array:
    KVR_ERR_UNSUPPORTED plus a message, decided on the host (this test needs no GPU)."""
    from paper_2606_17107_b200 import kvr
    base = 1 << 20
    m, keep = kvr.model_desc(2, 2, 64, 64, 0, 0, [1.0] * 32)
    d = kvr.paged_dst(base, base * 2, (16 * 4 * 2 * 64, 4 * 2 * 64, 2 * 64, 64), 16, 4, base * 3, 1, 16)
    seg = lambda i: kvr.segment(base * 4, base * 5, (2 * 4 * 64, 4 * 64, 64), 4, 0, 7, 0, 4 * i)
    assert kvr.kvr_validate(m, d, [seg(i) for i in range(9)]) == kvr.KVR_OK
    with pytest.raises(kvr.KvrError) as e:
        kvr.kvr_reposition_splice_noalloc(m, d, [seg(i) for i in range(kvr.KVR_NOALLOC_MAX_SEGMENTS + 1)])
    assert e.value.status == kvr.KVR_ERR_UNSUPPORTED and "at most 8" in str(e.value)

    R = kvr.KVR_NOALLOC_MAX_ROTARY_DIM + 32
    big, keep2 = kvr.model_desc(1, 1, R, R, 0, 0, [1.0] * (R // 2))
    d2 = kvr.paged_dst(base, base * 2, (16 * 4 * R, 4 * R, R, R), 16, 4, base * 3, 1, 16)
    s2 = kvr.segment(base * 4, base * 5, (4 * R, 4 * R, R), 4, 0, 7, 0, 0)
    assert kvr.kvr_validate(big, d2, [s2]) == kvr.KVR_OK
    with pytest.raises(kvr.KvrError) as e:
        kvr.kvr_reposition_splice_noalloc(big, d2, [s2])
    assert e.value.status == kvr.KVR_ERR_UNSUPPORTED and "rotary_dim" in str(e.value)

    with pytest.raises(kvr.KvrError) as e:                          # the ordinary validation comes first
        kvr.kvr_reposition_splice_noalloc(m, d, [kvr.segment(base * 4 + 8, base * 5, (2 * 4 * 64, 4 * 64, 64), 4, 0, 7, 0, 0)])
    assert e.value.status == kvr.KVR_ERR_ALIGNMENT
    assert kvr.KVR_NOALLOC_SCRATCH_BYTES == 4352 and C.sizeof(C.c_double) * kvr.KVR_NOALLOC_MAX_ROTARY_DIM // 2 + 64 <= 4352
