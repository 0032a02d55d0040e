"""Host-side checks of the C-ABI boundary that need no GPU: the library loads, exports every symbol
include/kvr.h declares, validates arguments, counts bytes, and refuses to run without a device."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def kvr():
    from paper_2606_17107_b200 import build
    build.build()
    from paper_2606_17107_b200 import kvr as k
    return k


def test_exports_match_header(kvr):
    header = open(os.path.join(ROOT, "include", "kvr.h")).read()
    declared = set(re.findall(r"KVR_API\s+[\w\s\*]+?\b(kvr_\w+)\s*\(", header))
    assert declared == set(kvr.EXPORTS), declared ^ set(kvr.EXPORTS)
    for name in declared:
        assert hasattr(kvr.lib, name), name
    assert kvr.kvr_version().startswith("kvr ")


def test_struct_layouts_match_header(kvr):
    # sizes implied by the field lists in include/kvr.h on LP64
    assert C.sizeof(kvr.kvr_model_desc) == 32 + 8      # + rotary_offset, reserved_ (NEXT-3 adapters)
    assert C.sizeof(kvr.kvr_paged_dst) == 16 + 32 + 8 + 8 + 8 + 8
    assert C.sizeof(kvr.kvr_segment) == 16 + 24 + 20 + 4 + 16
    assert C.sizeof(kvr.kvr_tuning) == 64
    assert C.sizeof(kvr.kvr_resident_span) == 32
    assert C.sizeof(kvr.kvr_span) == 16 + 24 + 12 + 4


def _call(kvr, **over):
    m, keep = kvr.model_desc(over.get("layers", 2), 2, over.get("head_dim", 64), over.get("rotary_dim", 64),
                             over.get("pairing", 0), over.get("dtype", 0), [1.0] * (over.get("rotary_dim", 64) // 2),
                             rotary_offset=over.get("rotary_offset", 0))
    base = 1 << 20
    d = kvr.paged_dst(base, over.get("v_cache", base * 2), over.get("strides", (16 * 4 * 2 * 64, 4 * 2 * 64, 2 * 64, 64)), 16, 4, base * 3, 1,
                      over.get("max_blocks", 8), k_scale=over.get("k_scale"))
    s = kvr.segment(over.get("k_src", base * 4), over.get("v_src", base * 5), over.get("src_strides", (2 * 10 * 64, 10 * 64, 64)),
                    over.get("len", 10), 0, over.get("new_start", 7), over.get("dst_seq", 0),
                    over.get("dst_token_start", 3), flags=over.get("flags", 0))
    return kvr.kvr_validate(m, d, [s]), keep


def test_validation(kvr):
    assert _call(kvr)[0] == kvr.KVR_OK
    assert _call(kvr, rotary_dim=63)[0] == kvr.KVR_ERR_INVALID_ARG
    assert _call(kvr, rotary_dim=66)[0] == kvr.KVR_ERR_INVALID_ARG
    assert _call(kvr, pairing=2)[0] == kvr.KVR_ERR_INVALID_ARG
    assert _call(kvr, dtype=1)[0] == kvr.KVR_ERR_INVALID_ARG            # fp8 without k_scale
    assert _call(kvr, dtype=1, k_scale=1 << 22)[0] == kvr.KVR_OK
    assert _call(kvr, head_dim=60, rotary_dim=60)[0] == kvr.KVR_ERR_ALIGNMENT
    assert _call(kvr, len=0)[0] == kvr.KVR_ERR_INVALID_ARG
    assert _call(kvr, dst_seq=1)[0] == kvr.KVR_ERR_INVALID_ARG
    assert _call(kvr, dst_token_start=23)[0] == kvr.KVR_ERR_OUT_OF_RANGE  # 23 + 10 > 8 * 4
    assert _call(kvr, dst_token_start=22)[0] == kvr.KVR_OK
    assert _call(kvr, k_src=(1 << 22) + 8)[0] == kvr.KVR_ERR_ALIGNMENT
    assert _call(kvr, src_strides=(2 * 10 * 64, 10 * 64, 68))[0] == kvr.KVR_ERR_ALIGNMENT
    assert _call(kvr, src_strides=(2 * 10 * 64, 10 * 64, 32))[0] == kvr.KVR_ERR_INVALID_ARG
    assert _call(kvr, strides=(16 * 4 * 2 * 64, 4 * 2 * 64, 2 * 64, 68))[0] == kvr.KVR_ERR_ALIGNMENT
    assert _call(kvr, new_start=-1)[0] == kvr.KVR_ERR_INVALID_ARG
    # NEXT-3 adapters (kvr.h): rotary window inside the row; K-only calls are all-or-none
    assert _call(kvr, rotary_dim=32, rotary_offset=32)[0] == kvr.KVR_OK
    assert _call(kvr, rotary_dim=32, rotary_offset=40)[0] == kvr.KVR_ERR_INVALID_ARG   # window past the row
    assert _call(kvr, rotary_dim=32, rotary_offset=-8)[0] == kvr.KVR_ERR_INVALID_ARG
    assert _call(kvr, rotary_dim=32, rotary_offset=4)[0] == kvr.KVR_ERR_ALIGNMENT      # 8 bytes
    assert _call(kvr, v_cache=None, v_src=None)[0] == kvr.KVR_OK
    assert _call(kvr, v_cache=None)[0] == kvr.KVR_ERR_INVALID_ARG
    assert _call(kvr, v_src=None)[0] == kvr.KVR_ERR_INVALID_ARG
    # NEXT-4: segment flags (the field sits in former padding: the struct size asserted above is unchanged)
    assert _call(kvr, flags=kvr.KVR_SEG_PRE_ROPE)[0] == kvr.KVR_OK
    assert _call(kvr, flags=kvr.KVR_SEG_SRC_STABLE | kvr.KVR_SEG_PRE_ROPE)[0] == kvr.KVR_OK
    assert _call(kvr, flags=4)[0] == kvr.KVR_ERR_INVALID_ARG


def test_bytes_moved_is_linear(kvr):
    """O(L) of PAPER.md:143: 4 * layers * kv_heads * head_dim * esz bytes per token."""
    m, keep = kvr.model_desc(36, 8, 128, 128, 0, 0, [1.0] * 64)
    seg = lambda n: kvr.segment(16, 16, (0, 0, 128), n, 0, 0, 0, 0)
    assert kvr.kvr_bytes_moved(m, [seg(4096)]) == 1207959552
    assert kvr.kvr_bytes_moved(m, [seg(1), seg(2), seg(3)]) == 6 * 294912
    m8, keep8 = kvr.model_desc(32, 8, 128, 128, 0, 1, [1.0] * 64)
    assert kvr.kvr_bytes_moved(m8, [seg(1)]) == 131072
    assert kvr.kvr_bytes_moved(m, []) == 0


def test_inplace_bytes_moved_is_half_of_a_splice(kvr):
    """NEXT-1: K read + K write only = 2 * layers * kv_heads * head_dim * esz bytes per token."""
    m, keep = kvr.model_desc(36, 8, 128, 128, 0, 0, [1.0] * 64)
    sp = [kvr.resident_span(0, 0, 4096, 0, 161)]
    assert kvr.kvr_inplace_bytes_moved(m, sp) == 1207959552 // 2
    assert kvr.kvr_inplace_bytes_moved(m, []) == 0


def test_no_cpu_fallback(kvr):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    m, keep = kvr.model_desc(2, 2, 64, 64, 0, 0, [1.0] * 32)
    with pytest.raises(kvr.KvrError):
        kvr.Context(m)


def test_status_strings(kvr):
    names = {0: "KVR_OK", -1: "KVR_ERR_INVALID_ARG", -2: "KVR_ERR_UNSUPPORTED", -3: "KVR_ERR_ALIGNMENT",
             -4: "KVR_ERR_OUT_OF_RANGE", -5: "KVR_ERR_CUDA", -6: "KVR_ERR_NOMEM"}
    for k, v in names.items():
        assert kvr.lib.kvr_status_string(k).decode() == v


def test_product_does_not_import_oracle():
    """The product path must never route through the oracle."""
    pkg = os.path.join(ROOT, "paper_2606_17107_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle", text, re.M), f
                assert "kvr_oracle" not in text, f
    orc = open(os.path.join(ROOT, "oracle", "kvr_oracle.c")).read() + open(os.path.join(ROOT, "oracle", "kvr_oracle.py")).read()
    assert "kvr.h" not in orc.replace("include/kvr.h)", "") and "paper_2606_17107_b200 import" not in orc


def test_header_is_valid_c99_and_struct_sizes_match_the_binding(kvr, tmp_path):
    """include/kvr.h is a C header (extern "C" only under C++): it must compile as strict C99 on its own, and the
    struct sizes the C compiler sees must be the ones the ctypes binding marshals."""
    import os
    import shutil
    import subprocess
    gcc = shutil.which("gcc")
    if gcc is None:
        pytest.skip("no gcc")
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    src = tmp_path / "abi.c"
    src.write_text(
        '#include "kvr.h"\n#include <stdio.h>\n'
        'int main(void) { printf("%zu %zu %zu %zu %zu %zu\\n", sizeof(kvr_model_desc), sizeof(kvr_paged_dst), '
        'sizeof(kvr_segment), sizeof(kvr_tuning), sizeof(kvr_resident_span), sizeof(kvr_span)); return 0; }\n')
    exe = tmp_path / "abi"
    subprocess.run([gcc, "-std=c99", "-pedantic", "-Wall", "-Werror", "-I", os.path.join(root, "include"),
                    str(src), "-o", str(exe)], check=True)
    sizes = [int(x) for x in subprocess.run([str(exe)], check=True, capture_output=True, text=True).stdout.split()]
    assert sizes == [C.sizeof(t) for t in (kvr.kvr_model_desc, kvr.kvr_paged_dst, kvr.kvr_segment, kvr.kvr_tuning,
                                           kvr.kvr_resident_span, kvr.kvr_span)]


def test_validate_read_without_a_gpu(kvr):
    """kvr_validate_read: host-only argument checks of kvr_rotate_on_read_attention (kvr.h), no CUDA call."""
    inv = [1.0] * 64
    m, keep = kvr.model_desc(4, 8, 128, 128, kvr.KVR_PAIR_NEOX_HALF, kvr.KVR_BF16, inv)
    A = 0x10000                                     # any 16-byte aligned, non-NULL address: nothing is dereferenced
    seg = lambda **kw: kvr.read_segment(kw.get("k", A), kw.get("v", A), kw.get("strides", (8 * 100 * 128, 100 * 128, 128)),
                                        kw.get("len", 100), kw.get("delta", 7), kw.get("request", 0), kw.get("flags", 0))
    ok = lambda segs, **kw: kvr.kvr_validate_read(kw.get("model", m), kw.get("q", A), kw.get("n_req", 1), kw.get("q_heads", 32),
                                                  kw.get("layer", 0), kw.get("scale", 0.088), segs, kw.get("o", A), kw.get("lse", A))
    assert ok([seg()]) == kvr.KVR_OK
    assert ok([seg(flags=kvr.KVR_SEG_SRC_STABLE), seg(delta=-5)]) == kvr.KVR_OK
    assert ok([seg()], layer=4) == kvr.KVR_ERR_INVALID_ARG and ok([seg()], layer=-1) == kvr.KVR_ERR_INVALID_ARG
    assert ok([seg()], q_heads=12) == kvr.KVR_ERR_INVALID_ARG                 # not a multiple of kv_heads
    assert ok([seg()], scale=0.0) == kvr.KVR_ERR_INVALID_ARG and ok([seg()], scale=float("inf")) == kvr.KVR_ERR_INVALID_ARG
    assert ok([seg()], q=None) == kvr.KVR_ERR_INVALID_ARG and ok([seg()], o=None) == kvr.KVR_ERR_INVALID_ARG
    assert ok([seg()], n_req=2) == kvr.KVR_ERR_INVALID_ARG                    # request 1 owns no segment
    assert ok([seg(request=1)]) == kvr.KVR_ERR_INVALID_ARG
    assert ok([seg(len=0)]) == kvr.KVR_ERR_INVALID_ARG and ok([seg(flags=1)]) == kvr.KVR_ERR_INVALID_ARG
    assert ok([seg(strides=(8 * 100 * 128, 100 * 128, 64))]) == kvr.KVR_ERR_INVALID_ARG      # rows overlap
    assert ok([seg(k=A + 8)]) == kvr.KVR_ERR_ALIGNMENT and ok([seg()], q=A + 2) == kvr.KVR_ERR_ALIGNMENT
    assert ok([seg(strides=(8 * 100 * 132, 100 * 132, 132))]) == kvr.KVR_ERR_ALIGNMENT        # 264-byte rows
    assert ok([seg()], q_heads=256) == kvr.KVR_ERR_UNSUPPORTED                # 32 query heads per kv head
    m64, keep64 = kvr.model_desc(4, 8, 64, 64, kvr.KVR_PAIR_NEOX_HALF, kvr.KVR_BF16, [1.0] * 32)
    assert ok([seg(strides=(8 * 100 * 64, 100 * 64, 64))], model=m64) == kvr.KVR_ERR_UNSUPPORTED
    m8, keep8 = kvr.model_desc(4, 8, 128, 128, kvr.KVR_PAIR_NEOX_HALF, kvr.KVR_FP8_E4M3, inv)
    assert ok([seg()], model=m8) == kvr.KVR_ERR_UNSUPPORTED
    assert kvr.kvr_attention_bytes_read(m, [seg(), seg(len=28)]) == 2 * 8 * 128 * 2 * 128
    # what a TMA tensor map cannot describe is refused here, before the call would touch its descriptor cache
    assert ok([seg(strides=(0, 100 * 128, 128))]) == kvr.KVR_ERR_UNSUPPORTED                  # 4 layers on a zero stride
    assert ok([seg(strides=(1 << 39, 100 * 128, 128))]) == kvr.KVR_ERR_UNSUPPORTED            # 2^40 bytes
    m1, keep1 = kvr.model_desc(1, 8, 128, 128, kvr.KVR_PAIR_NEOX_HALF, kvr.KVR_BF16, inv)
    assert ok([seg(strides=(0, 100 * 128, 128))], model=m1) == kvr.KVR_OK                     # one layer never uses its stride
    assert ok([seg()], n_req=1 << 30) == kvr.KVR_ERR_INVALID_ARG                              # more requests than segments
