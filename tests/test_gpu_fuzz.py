"""Seeded random workloads against the oracle: shapes, pairings, dtypes, layouts, block sizes, segment mixes (constant
shift, Delta = 0, position maps, pre-RoPE keys, padded rows, K-only window rows) and launch shapes drawn at random.
Every case is small enough for the oracle to finish in well under a second; the bar is the one of
tests/test_gpu_parity.py."""
import numpy as np
import pytest

from tests.test_gpu_parity import check_parity
from workloads import make_workload, pos_map_with_gaps

pytestmark = pytest.mark.gpu


def _random_case(seed):
    rng = np.random.default_rng(1000 + seed)
    dtype = "fp8" if rng.random() < 0.3 else "bf16"
    E = 2 if dtype == "bf16" else 1
    D = int(rng.choice([32, 48, 64, 96, 128, 256] if dtype == "bf16" else [64, 128, 192, 256]))
    window = rng.random() < 0.25
    if window:
        R = int(rng.choice([r for r in (16, 32, 64) if r <= D and (r * E) % 32 == 0]))
        off = int(rng.choice([o for o in range(0, D - R + 1, 16 // E * 1) if (o * E) % 16 == 0]))
    else:
        R = int(rng.choice([r for r in (D, D // 2) if (r * E) % 32 == 0]))
        off = 0
    heads = int(rng.choice([1, 2, 3, 4, 8]))
    has_v = not (window and rng.random() < 0.5)
    bs = int(rng.choice([1, 4, 8, 16, 32, 64]))
    pad = int(rng.choice([0, 0, 16 // E]))
    n_seq = int(rng.integers(1, 4))
    seqs = []
    for _ in range(n_seq):
        at, lst = int(rng.integers(0, 40)), []
        for _ in range(int(rng.integers(1, 5))):
            n = int(rng.choice([1, 2, 5, 17, 64, 200, 333]))
            kind = rng.random()
            d = dict(len=n, dst_token_start=at, old_start=int(rng.integers(0, 5000)), src_row_pad=int(rng.choice([0, pad])))
            if kind < 0.15:
                d["new_start"] = d["old_start"]                                    # Delta = 0
            elif kind < 0.35:
                d["pos_map"] = pos_map_with_gaps(n, int(rng.integers(0, 100000)), 0.2, 64, int(rng.integers(1 << 30)))
                d["new_start"] = int(d["pos_map"][0])
            elif kind < 0.5:
                d["pre_rope"] = True
                d["new_start"] = int(rng.integers(0, 100000))
                if rng.random() < 0.5:
                    d["pos_map"] = pos_map_with_gaps(n, d["new_start"], 0.1, 16, int(rng.integers(1 << 30)))
            else:
                d["new_start"] = int(rng.integers(0, 131072))
            lst.append(d)
            at += n + int(rng.integers(0, 9))
        seqs.append(lst)
    w = make_workload(name=f"fuzz{seed}", layers=int(rng.integers(1, 5)), kv_heads=heads, head_dim=D, rotary_dim=R,
                      rotary_offset=off, pairing=str(rng.choice(["neox", "gptj"])), dtype=dtype,
                      theta=float(rng.choice([1e4, 5e5, 1e6])), block_size=bs, layout=str(rng.choice(["NHD", "HND"])),
                      seed=7000 + seed, seq_segments=seqs, slack=1.5, scales_differ=bool(rng.random() < 0.5),
                      dst_head_pad=int(rng.choice([0, pad])), has_v=has_v)
    tuning = {}
    if rng.random() < 0.6:
        tuning = dict(max_ctas=int(rng.integers(1, 6)), stages=int(rng.integers(2, 16)),
                      consumer_warps=int(rng.integers(1, 9)))
        if rng.random() < 0.3:
            tuning["gather"] = int(rng.choice([1, 3]))
        if rng.random() < 0.3:
            tuning["grab"] = int(rng.integers(1, 5))
    rng2 = np.random.default_rng(5000 + seed)          # drawn from a stream of its own: the cases above stay as they were
    if rng2.random() < 0.4 and "gather" not in tuning:
        tuning["transpose_load"] = 1                   # ignored by the library where the pool is not dense token-major
        if rng2.random() < 0.5:
            tuning["tile_bytes"] = int(rng2.choice([512, 2048, 8192]))
    return w, tuning


@pytest.mark.parametrize("seed", range(200))
def test_random_workload_generic_kernel(seed):
    w, _ = _random_case(seed)
    check_parity(w, "generic")


@pytest.mark.parametrize("seed", range(200))
def test_random_workload_generic_vec_kernel(seed):
    """The generic kernel with 16-byte accesses (tuning.path = 5): parity with the oracle, and the very bits the scalar
    generic kernel writes (same table, same per-element arithmetic).  Shapes whose rotary window does not split into
    whole vectors are refused and stay on the scalar kernel."""
    from tests.test_gpu_parity import PATHS, RingDeclined, _gpu
    from tests.helpers import materialize_cpu
    w, _ = _random_case(seed)
    if check_parity(w, "generic_vec", declined_ok=True) is None:
        E = 2 if w.dtype == "bf16" else 1
        assert (w.rotary_dim * E) % (32 if w.pairing == "neox" else 16) != 0, "refused a shape it documents as supported"
        return
    srcs, _, _ = materialize_cpu(w)
    k1, v1, _, _ = _gpu(w, srcs, dict(path=PATHS["generic"]))
    k5, v5, _, info = _gpu(w, srcs, dict(path=PATHS["generic_vec"]))
    assert info["path"] == 5 and np.array_equal(k1, k5) and ((v1 is None and v5 is None) or np.array_equal(v1, v5))


RING_DECLINED = []     # shapes the ring kernel declined (they take the generic kernel, checked above)


@pytest.mark.parametrize("seed", range(200))
def test_random_workload_ring_kernel(seed):
    """Shapes outside the ring kernel's domain (rotary_dim * esz / 32 not a power of two: head_dim 48 / 96 / 192 with
    full rotary) are declined with KVR_ERR_UNSUPPORTED before anything is launched -- that is the expected result for
    them, and auto dispatch must then take the generic kernel."""
    w, tuning = _random_case(seed)
    if check_parity(w, "ring", declined_ok=True, **tuning) is None:
        RING_DECLINED.append((seed, w.dtype, w.head_dim, w.rotary_dim, w.rotary_offset, w.pairing))
        from tests.test_gpu_parity import _gpu
        from tests.helpers import materialize_cpu
        srcs, _, _ = materialize_cpu(w)
        _, _, status, info = _gpu(w, srcs, dict(path=0))
        assert status[0] == 0 and info["path"] in (1, 5), info      # scalar, or with 16-byte accesses where the window allows


def test_report_the_shapes_the_ring_kernel_declined(capsys):
    """Runs after the fuzz cases (file order): the declined shapes are printed, and they are a minority."""
    shapes = sorted({s[1:] for s in RING_DECLINED})
    with capsys.disabled():
        print(f"\nring kernel declined {len(RING_DECLINED)} of 200 fuzz cases; distinct (dtype, D, R, offset, pairing): {shapes}")
    assert len(RING_DECLINED) < 100
