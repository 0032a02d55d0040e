"""GPU parity of kvr_rotate_on_read_attention (include/kvr.h; R25) against the fp64 oracle
(oracle/kvr_attention_oracle.c), through the C ABI.

Two comparisons per case, both element by element:
 (1) against the ORACLE (the definition: every key re-rotated in fp64, exact softmax), within the tolerance DESIGN.md
     derives from the kernel's arithmetic contract: the counter-rotated query is rounded once to bf16, so score j is off
     by at most E_j = scale * sum_d |q'_d - bf16(q'_d)| * |k_jd| (computed here exactly, per query head), the softmax
     weights are rounded to bf16 (relative 2^-9 each, numerator and denominator alike), everything else is fp32:
         |o - o_ref|[g, d] <= first-order term + kappa(E) sum_j w_j |v_jd - o_d| + 2^-7 sum_j w_j |v_jd| + 2^-12 max_j |v_jd|
                              (reference() below and DESIGN.md section 3: per element, a few per cent of |o|, not of max |v|)
         |lse - lse_ref| <= max_j E_j + 2^-8
 (2) against the same definition evaluated with the bf16-rounded counter-rotated query (numpy fp64; "both sides take
     the rounding decision in the same precision"): what is left is the bf16 rounding of the weights and fp32
     accumulation, so the bound is tight enough to see a single wrong key, dim or head:
         |o - o_model| <= 2^-7 * sum_j w_j |v_jd| + 2^-12 * max_j |v_jd| ;  |lse - lse_model| <= 2^-8
"""
import numpy as np
import pytest
import torch

from oracle import kvr_oracle as orc
from tests.helpers import PAIRING, np_bits
from workloads import READ_WORKLOADS, attention_config, inv_freq_llama3, make_queries, make_read_sources, read_workload

pytestmark = pytest.mark.gpu

GUARD = 64 * 1024


def bf16_val(bits):
    return torch.from_numpy(np.ascontiguousarray(bits).view(np.int16)).view(torch.bfloat16).to(torch.float64).numpy()


def bf16_round(x):
    """fp64 -> fp32 -> bf16 (RNE), back as fp64: the rounding kvr.h states for the counter-rotated query."""
    t = torch.from_numpy(np.ascontiguousarray(x, dtype=np.float64)).to(torch.float32).to(torch.bfloat16)
    return t.to(torch.float64).numpy()


def counter_rotate(q, delta, inv_freq, R, pairing, offset):
    """R(-delta) q in fp64 (complex form; independent of oracle and kernel)."""
    q = np.array(q, dtype=np.float64)
    h = R // 2
    if pairing == "neox":
        ia, ib = offset + np.arange(h), offset + h + np.arange(h)
    else:
        ia, ib = offset + 2 * np.arange(h), offset + 2 * np.arange(h) + 1
    z = (q[..., ia] + 1j * q[..., ib]) * np.exp(-1j * float(delta) * np.asarray(inv_freq, dtype=np.float64))
    out = q.copy()
    out[..., ia], out[..., ib] = z.real, z.imag
    return out


def reference(w, srcs, q_bits, n_threads):
    """Per request: oracle (o, lse); the bf16-query model (o, lse, sum_j w_j |v_j|); E = max_j E_j, max_j |v_jd|; and
    tol_ref[g, d], the per-element bound on |o_kernel - o_oracle| that DESIGN.md section 3 derives:
        scale * sum_s sum_c u^(s)_c |C^(s)_cd|  +  kappa(E) * sum_j w_j |v_jd - o_d|  +  2^-7 sum_j w_j |v_jd|  +  2^-12 max_j |v_jd|
    with w, o the ORACLE's weights and output, u^(s) = |q'^(s) - bf16(q'^(s))| the rounding error of the query counter-
    rotated for segment s, C^(s)_cd = sum_{j in s} w_j k_jc (v_jd - o_d)  (first order in the score error: the softmax
    weights sum to one, so only the covariance of keys and values under w is seen), and
    kappa(E) = e^E (2 (e^E - 1 - E)(1 + E) + 2 E^2) the bound on everything beyond first order."""
    D, G = w.head_dim, w.q_heads // w.kv_heads
    out = []
    for r in range(w.n_req):
        segs = [(i, s) for i, s in enumerate(w.segments) if s.request == r]
        o_ref, lse_ref = orc.rotate_on_read_attention(
            q=q_bits[r], kv_heads=w.kv_heads, rotary_dim=w.rotary_dim, pairing=PAIRING[w.pairing], inv_freq=w.inv_freq,
            scale=w.scale, rotary_offset=w.rotary_offset, n_threads=n_threads,
            segments=[(srcs[i][0][w.layer][:, :, :D], srcs[i][1][w.layer][:, :, :D], s.delta) for i, s in segs])
        qv = bf16_val(q_bits[r])                                       # [Hq, D]
        ks = [bf16_val(srcs[i][0][w.layer][:, :, :D]) for i, s in segs]   # per segment [Hkv, L, D]
        vs = [bf16_val(srcs[i][1][w.layer][:, :, :D]) for i, s in segs]
        qps = [counter_rotate(qv, s.delta, w.inv_freq, w.rotary_dim, w.pairing, w.rotary_offset) for i, s in segs]
        qbs = [bf16_round(qp) for qp in qps]
        cuts = np.cumsum([0] + [s.len for i, s in segs])
        R = dict(o_ref=o_ref, lse_ref=lse_ref, o_model=np.zeros((w.q_heads, D)), lse_model=np.zeros(w.q_heads),
                 wabsv=np.zeros((w.q_heads, D)), vmax=np.zeros((w.q_heads, D)), E=np.zeros(w.q_heads),
                 tol_ref=np.zeros((w.q_heads, D)), tol_first_order=np.zeros((w.q_heads, D)))
        for g in range(w.q_heads):
            h = g // G
            v = np.concatenate([v_[h] for v_ in vs], axis=0)                                      # [T, D]
            x_b = np.concatenate([w.scale * (k[h] @ qb[g]) for k, qb in zip(ks, qbs)])            # bf16-query scores
            x = np.concatenate([w.scale * (k[h] @ qp[g]) for k, qp in zip(ks, qps)])              # exact scores
            E = max(float((w.scale * (np.abs(k[h]) @ np.abs(qp[g] - qb[g]))).max()) for k, qp, qb in zip(ks, qps, qbs))
            # the bf16-query model
            m = x_b.max(); p = np.exp(x_b - m); z = p.sum(); wb = p / z
            R["o_model"][g] = wb @ v
            R["lse_model"][g] = m + np.log(z)
            R["wabsv"][g] = wb @ np.abs(v)
            R["vmax"][g] = np.abs(v).max(axis=0)
            R["E"][g] = E
            # the oracle-side bound (weights and output of the definition itself)
            p = np.exp(x - x.max()); wt = p / p.sum()
            o = wt @ v
            dv = v - o
            first = np.zeros(D)
            for si, (k, qp, qb) in enumerate(zip(ks, qps, qbs)):
                a, b = cuts[si], cuts[si + 1]
                C = (k[h] * wt[a:b, None]).T @ dv[a:b]                                             # [D(c), D(d)]
                first += w.scale * (np.abs(qp[g] - qb[g]) @ np.abs(C))
            kappa = np.exp(E) * (2 * (np.expm1(E) - E) * (1 + E) + 2 * E * E)
            R["tol_first_order"][g] = first + kappa * (wt @ np.abs(dv))
            R["tol_ref"][g] = R["tol_first_order"][g] + 2.0 ** -7 * (wt @ np.abs(v)) + 2.0 ** -12 * R["vmax"][g]
        out.append(R)
    return out


def run_and_check(w, tuning=None, n_threads=None, layer=None):
    from paper_2606_17107_b200 import kvr
    from paper_2606_17107_b200.harness import DeviceReadWorkload
    if layer is not None:
        w.layer = layer
    srcs_t = make_read_sources(w, "cpu")
    q_t = make_queries(w, "cpu")
    dw = DeviceReadWorkload(w, "cuda:0", sources=srcs_t, queries=q_t, guard_bytes=GUARD)
    with kvr.Context(dw.model) as ctx:
        if tuning:
            ctx.set_tuning(**tuning)
        dw.run(ctx)
        dw.run(ctx)                                        # twice: tickets and staging slots re-arm themselves
        torch.cuda.synchronize()
        info = ctx.last_launch_info()
        assert ctx.last_device_status()[0] == kvr.KVR_OK
    assert info["path"] == kvr.PATH_ATTEND
    dw.check_guards()
    o, lse = dw.o.cpu().numpy().astype(np.float64), dw.lse.cpu().numpy().astype(np.float64)
    assert np.isfinite(o).all() and np.isfinite(lse).all()
    srcs = [(np_bits(k), np_bits(v)) for k, v in srcs_t]
    ref = reference(w, srcs, np_bits(q_t), n_threads or orc.host_threads())
    worst = 0.0
    for r, R in enumerate(ref):
        tol_o = R["tol_ref"]
        assert (np.abs(o[r] - R["o_ref"]) <= tol_o).all(), (r, float((np.abs(o[r] - R["o_ref"]) / tol_o).max()))
        assert (np.abs(lse[r] - R["lse_ref"]) <= R["E"] + 2.0 ** -8).all(), (r, float(np.abs(lse[r] - R["lse_ref"]).max()))
        tol_m = 2.0 ** -7 * R["wabsv"] + 2.0 ** -12 * R["vmax"]
        d = np.abs(o[r] - R["o_model"])
        assert (d <= tol_m).all(), (r, float((d / tol_m).max()), np.unravel_index(np.argmax(d / tol_m), d.shape))
        assert (np.abs(lse[r] - R["lse_model"]) <= 2.0 ** -8).all(), (r, float(np.abs(lse[r] - R["lse_model"]).max()))
        worst = max(worst, float((d / tol_m).max()))
    return info, worst


@pytest.mark.parametrize("name", READ_WORKLOADS)
def test_attention_workloads_reduced(name):
    """The four rotate-on-read workloads with every length divided (several tiles, ragged tails, several items per group)."""
    shrink = {"attend-tiny": 1, "attend-compose4": 8, "attend-32k-x8": 32, "attend-serving": 16}[name]
    run_and_check(attention_config(name, shrink=shrink))


@pytest.mark.parametrize("q_heads,kv_heads", [(2, 2), (6, 2), (8, 2), (10, 2), (16, 2), (16, 1), (32, 8)])
def test_gqa_group_sizes(q_heads, kv_heads):
    """q_heads / kv_heads = 1, 3, 4, 5, 8, 16: the three instantiations (4, 8, 16 columns) with and without padding rows."""
    w = read_workload("gqa", q_heads=q_heads, kv_heads=kv_heads, requests=[[(300, 1234), (129, -77)], [(515, 40000)]],
                      seed=4242 + q_heads)
    run_and_check(w)


@pytest.mark.parametrize("pairing", ["neox", "gptj"])
@pytest.mark.parametrize("R,off", [(128, 0), (64, 0), (64, 64), (32, 16)])
def test_pairings_partial_rotary_and_window(pairing, R, off):
    inv = inv_freq_llama3(5e5, R, 8.0, 1.0, 4.0, 8192)
    w = read_workload("rot", q_heads=8, kv_heads=2, rotary_dim=R, rotary_offset=off, pairing=pairing, inv_freq=inv,
                      requests=[[(257, 161), (64, 100000)]], seed=99 + R + off)
    run_and_check(w)


@pytest.mark.parametrize("lens", [[1], [127], [128], [129], [1, 1, 1], [255, 1, 384], [4096 + 17]])
def test_ragged_lengths(lens):
    w = read_workload("ragged", q_heads=8, kv_heads=2, requests=[[(L, 37 + 1000 * i) for i, L in enumerate(lens)]], seed=7 + sum(lens))
    run_and_check(w)


@pytest.mark.parametrize("tiles_per_item,max_ctas", [(1, 0), (1, 1), (3, 2), (2, 5), (32, 0)])
def test_item_shapes_and_cta_counts(tiles_per_item, max_ctas):
    """One tile per item (every tile a partial to merge), everything on one CTA (item transitions, every double buffer
    wraps), a handful of CTAs: the decomposition never changes the result beyond the tolerance."""
    w = read_workload("items", q_heads=16, kv_heads=4, requests=[[(1500, 2000), (700, 5)], [(129, -3)], [(2048, 77)]], seed=31337)
    info, _ = run_and_check(w, tuning=dict(layers_per_unit=tiles_per_item, max_ctas=max_ctas))
    if max_ctas:
        assert info["grid"] <= max_ctas


@pytest.mark.parametrize("inline_limit", [1, 3, 64])
def test_merge_in_kernel_and_by_the_merge_kernel(inline_limit):
    """Groups of 1, 2, 5 and 24 partials in one call, merged by the group's last item (few partials) or by
    kvr_attend_merge_kernel after the grid (many): tuning.hsplit overrides the limit between the two."""
    w = read_workload("merge", q_heads=8, kv_heads=2, requests=[[(100, 1)], [(256, 2)], [(640, 3)], [(3000, 4)]], seed=808)
    run_and_check(w, tuning=dict(layers_per_unit=1, hsplit=inline_limit))


def test_descriptor_cache_hits_and_evictions():
    """Twelve different calls through ONE context, round robin, three rounds: more distinct segment arrays than the
    8-entry descriptor cache holds, so entries are rebuilt, reused and evicted while earlier launches are in flight."""
    from paper_2606_17107_b200 import kvr
    from paper_2606_17107_b200.harness import DeviceReadWorkload
    ws = [read_workload(f"c{i}", q_heads=8, kv_heads=2, requests=[[(130 + 37 * i, 10 * i + 1)], [(64 + i, 5)]], seed=900 + i)
          for i in range(12)]
    dws = [DeviceReadWorkload(w, "cuda:0") for w in ws]
    with kvr.Context(dws[0].model) as ctx:
        for _ in range(3):
            for dw in dws:
                dw.run(ctx)
        torch.cuda.synchronize()
    for w, dw in zip(ws, dws):
        srcs = [(np_bits(k), np_bits(v)) for k, v in dw.sources]
        ref = reference(w, srcs, np_bits(dw.q), orc.host_threads())
        o, lse = dw.o.cpu().numpy().astype(np.float64), dw.lse.cpu().numpy().astype(np.float64)
        for r, R in enumerate(ref):
            assert (np.abs(o[r] - R["o_model"]) <= 2.0 ** -7 * R["wabsv"] + 2.0 ** -12 * R["vmax"]).all(), (w.name, r)
            assert (np.abs(lse[r] - R["lse_model"]) <= 2.0 ** -8).all(), (w.name, r)


def test_padded_source_rows_every_layer_and_unsorted_requests():
    w = read_workload("strides", q_heads=8, kv_heads=2, layers=3, pad=8,
                      requests=[[(200, 10)], [(333, 20), (100, 30)], [(64, 40)]], seed=555)
    w.segments = [w.segments[i] for i in (2, 0, 3, 1)]          # segments need not be grouped by request
    for layer in range(3):
        run_and_check(w, layer=layer)


def test_large_scores_move_the_reference_maximum():
    """Scaled-up queries: scores span hundreds of log2 units between tiles, so the lazily moved reference maximum and
    the rescale of O^T in TMEM are exercised (a tile whose maximum exceeds the reference by more than 2^8)."""
    from paper_2606_17107_b200 import kvr
    from paper_2606_17107_b200.harness import DeviceReadWorkload
    w = read_workload("hot", q_heads=8, kv_heads=2, requests=[[(1024, 9)]], seed=2024)
    q = make_queries(w, "cpu")
    q = (q.view(torch.bfloat16).to(torch.float32) * 16).to(torch.bfloat16).view(torch.int16)     # exact in bf16
    srcs = make_read_sources(w, "cpu")
    dw = DeviceReadWorkload(w, "cuda:0", sources=srcs, queries=q, guard_bytes=GUARD)
    with kvr.Context(dw.model) as ctx:
        ctx.set_tuning(max_ctas=1, layers_per_unit=8)
        dw.run(ctx)
        torch.cuda.synchronize()
    o, lse = dw.o.cpu().numpy().astype(np.float64), dw.lse.cpu().numpy().astype(np.float64)
    R = reference(w, [(np_bits(k), np_bits(v)) for k, v in srcs], np_bits(q), orc.host_threads())[0]
    assert (np.abs(lse[0] - R["lse_model"]) <= 2.0 ** -8 + 1e-6 * np.abs(R["lse_model"])).all()
    assert (np.abs(o[0] - R["o_model"]) <= 2.0 ** -7 * R["wabsv"] + 2.0 ** -12 * R["vmax"]).all()
    assert (np.abs(lse[0] - R["lse_ref"]) <= R["E"] + 2.0 ** -8).all()


def test_argument_errors_and_limits():
    from paper_2606_17107_b200 import kvr
    from paper_2606_17107_b200.harness import DeviceReadWorkload
    w = read_workload("err", q_heads=8, kv_heads=2, requests=[[(130, 5)], [(64, 6)]], seed=1)
    dw = DeviceReadWorkload(w, "cuda:0")
    with kvr.Context(dw.model) as ctx:
        call = lambda **kw: ctx.rotate_on_read_attention(
            kw.get("q", dw.q), kw.get("n_req", 2), kw.get("q_heads", 8), kw.get("layer", 1), kw.get("scale", w.scale),
            kw.get("segs", dw.segs), dw.o, dw.lse, check=False)
        assert call() == kvr.KVR_OK
        assert call(layer=2) == kvr.KVR_ERR_INVALID_ARG
        assert call(q_heads=7) == kvr.KVR_ERR_INVALID_ARG
        assert call(scale=0.0) == kvr.KVR_ERR_INVALID_ARG
        assert call(n_req=3) == kvr.KVR_ERR_INVALID_ARG                 # request 2 owns no segment
        assert call(q_heads=64) == kvr.KVR_ERR_UNSUPPORTED              # 32 query heads per kv head
        assert call(q=dw.q.data_ptr() + 2) == kvr.KVR_ERR_ALIGNMENT
        k, v = dw.sources[0]
        bad = [kvr.read_segment(k, v, w.src_strides(w.segments[0]), 130, 5, 5)]
        assert call(segs=bad) == kvr.KVR_ERR_INVALID_ARG                # request out of range
        bad = [kvr.read_segment(k, v, w.src_strides(w.segments[0]), 130, 5, 0, flags=4), dw.segs[1]]
        assert call(segs=bad) == kvr.KVR_ERR_INVALID_ARG                # unknown flag
        g = torch.cuda.CUDAGraph()
        s = torch.cuda.Stream()
        fresh = kvr.read_segment_array([kvr.read_segment(k, v, w.src_strides(w.segments[0]), 129, 5, 0),
                                        kvr.read_segment(k, v, w.src_strides(w.segments[0]), 60, 6, 1)])
        with torch.cuda.stream(s):
            g.capture_begin()
            st = ctx.rotate_on_read_attention(dw.q, 2, 8, 1, w.scale, fresh, dw.o, dw.lse, stream=s, check=False)
            g.capture_end()
        assert st == kvr.KVR_ERR_UNSUPPORTED                            # descriptors not cached yet: refused under capture
        torch.cuda.synchronize()
    w64 = read_workload("d64", q_heads=4, kv_heads=2, head_dim=64, requests=[[(64, 1)]], seed=2)
    d64 = DeviceReadWorkload(w64, "cuda:0")
    with kvr.Context(d64.model) as ctx:
        assert d64.run.__func__ is not None
        st = ctx.rotate_on_read_attention(d64.q, 1, 4, 1, w64.scale, d64.segs, d64.o, d64.lse, check=False)
        assert st == kvr.KVR_ERR_UNSUPPORTED


@pytest.mark.parametrize("name", ["attend-compose4", "attend-32k-x8", "attend-serving"])
def test_full_size_every_request(name):
    """BASELINE-sized calls in the launch configuration bench.py times: the whole call runs on the GPU and EVERY request
    of it (all query heads and dims) is checked against the oracle and against the bf16-query model, at the tolerances of
    the small cases."""
    from paper_2606_17107_b200 import kvr
    from paper_2606_17107_b200.harness import DeviceReadWorkload
    w = attention_config(name)
    dw = DeviceReadWorkload(w, "cuda:0")
    with kvr.Context(dw.model) as ctx:
        dw.run(ctx)
        torch.cuda.synchronize()
        assert ctx.last_launch_info()["grid"] == torch.cuda.get_device_properties(0).multi_processor_count
    o, lse = dw.o.cpu().numpy().astype(np.float64), dw.lse.cpu().numpy().astype(np.float64)
    assert np.isfinite(o).all() and np.isfinite(lse).all()
    q_bits = np_bits(dw.q)
    for r in range(w.n_req):
        idx = [i for i, s in enumerate(w.segments) if s.request == r]
        sub = read_workload("sub", q_heads=w.q_heads, kv_heads=w.kv_heads, layers=w.layers, layer=w.layer,
                            requests=[[(w.segments[i].len, w.segments[i].delta) for i in idx]], seed=0, inv_freq=w.inv_freq)
        # only this request's layer of its sources comes to the host (the other layers stay zero: reference() reads one)
        srcs = []
        for i in idx:
            k, v = dw.sources[i]
            kh, vh = np.zeros(tuple(k.shape), np.uint16), np.zeros(tuple(v.shape), np.uint16)
            kh[w.layer], vh[w.layer] = np_bits(k[w.layer]), np_bits(v[w.layer])
            srcs.append((kh, vh))
        R = reference(sub, srcs, q_bits[r:r + 1], orc.host_threads())[0]
        assert (np.abs(o[r] - R["o_model"]) <= 2.0 ** -7 * R["wabsv"] + 2.0 ** -12 * R["vmax"]).all(), r
        assert (np.abs(lse[r] - R["lse_model"]) <= 2.0 ** -8).all(), r
        assert (np.abs(o[r] - R["o_ref"]) <= R["tol_ref"]).all(), (r, float((np.abs(o[r] - R["o_ref"]) / R["tol_ref"]).max()))
        assert (np.abs(lse[r] - R["lse_ref"]) <= R["E"] + 2.0 ** -8).all(), r


@pytest.mark.parametrize("case", range(40))
def test_fuzz_shapes_and_decompositions(case):
    """Seeded random calls: GQA group 1..16, 1-8 kv heads, 1-5 requests of 1-4 segments of 1-3000 tokens, shifts up to
    +-2^30 (the fp64 sincos slow path), both pairings, partial rotary windows, padded rows, random tiles per item, CTA
    counts and in-kernel merge limits -- every one against the oracle and the bf16-query model."""
    rng = np.random.default_rng(77000 + case)
    kv_heads = int(rng.choice([1, 2, 4, 8]))
    group = int(rng.choice([1, 2, 3, 4, 5, 7, 8, 12, 16]))
    R = int(rng.choice([128, 128, 64, 32]))
    off = int(rng.choice([0, 0, 16, 128 - R])) if R < 128 else 0
    off = min(off, 128 - R)
    reqs = []
    for _ in range(int(rng.integers(1, 6))):
        lst = []
        for _ in range(int(rng.integers(1, 5))):
            L = int(rng.choice([1, int(rng.integers(2, 200)), int(rng.integers(200, 3000))]))
            big = rng.random() < 0.2
            d = int(rng.integers(-(1 << 30), 1 << 30)) if big else int(rng.integers(-5000, 200000))
            lst.append((L, d))
        reqs.append(lst)
    w = read_workload(f"fuzz{case}", q_heads=kv_heads * group, kv_heads=kv_heads, rotary_dim=R, rotary_offset=off,
                      pairing=str(rng.choice(["neox", "gptj"])), theta=float(rng.choice([1e4, 5e5, 1e6])),
                      layers=int(rng.integers(1, 4)), layer=0, pad=int(rng.choice([0, 0, 8, 24])), requests=reqs, seed=88000 + case)
    w.layer = int(rng.integers(0, w.layers))
    perm = rng.permutation(len(w.segments))
    w.segments = [w.segments[i] for i in perm]
    if rng.random() < 0.5:                       # a segment that is not flagged stable: no early loads for the call
        w.segments[0].src_stable = False
    tuning = dict(layers_per_unit=int(rng.choice([0, 1, 2, 3, 5])), max_ctas=int(rng.choice([0, 0, 1, 3, 17])),
                  hsplit=int(rng.choice([0, 1, 2, 100])))
    run_and_check(w, tuning=tuning)


def test_cuda_graph_of_cached_calls_replays_after_cache_churn():
    """A decode step as a CUDA graph: the attention calls of three layers (descriptors cached by one eager call each)
    captured once, replayed after a dozen other calls have churned the descriptor cache and the query has changed; the
    pinned cache entries and the partial buffers the graph points at must still be the ones it was captured with."""
    from paper_2606_17107_b200 import kvr
    from paper_2606_17107_b200.harness import DeviceReadWorkload
    w = read_workload("graph", q_heads=8, kv_heads=2, layers=3, requests=[[(700, 11), (300, -4)], [(2500, 3000)]], seed=4711)
    srcs_t, q_t = make_read_sources(w, "cpu"), make_queries(w, "cpu")
    dw = DeviceReadWorkload(w, "cuda:0", sources=srcs_t, queries=q_t)
    outs = [(torch.empty_like(dw.o), torch.empty_like(dw.lse)) for _ in range(3)]
    others = [DeviceReadWorkload(read_workload(f"o{i}", q_heads=8, kv_heads=2, requests=[[(3000 + 100 * i, i)] * 3], seed=i), "cuda:0")
              for i in range(12)]
    stream = torch.cuda.Stream()
    with kvr.Context(dw.model) as ctx:
        call = lambda l: ctx.rotate_on_read_attention(dw.q, w.n_req, w.q_heads, l, w.scale, dw.segs, outs[l][0], outs[l][1], stream=stream)
        call(0)                                                  # eager once: descriptors cached, buffers sized
        torch.cuda.synchronize()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.stream(stream):
            graph.capture_begin()
            for l in range(3):
                call(l)
            graph.capture_end()
        for od in others:                                        # churn the cache (and grow the partial buffers)
            od.run(ctx, stream=stream)
        for o_, l_ in outs:
            o_.fill_(float("nan")); l_.fill_(float("nan"))
        with torch.cuda.stream(stream):
            graph.replay()
        torch.cuda.synchronize()
        srcs = [(np_bits(k), np_bits(v)) for k, v in srcs_t]
        for l in range(3):
            w.layer = l
            ref = reference(w, srcs, np_bits(q_t), orc.host_threads())
            o, lse = outs[l][0].cpu().numpy().astype(np.float64), outs[l][1].cpu().numpy().astype(np.float64)
            for r, R in enumerate(ref):
                assert (np.abs(o[r] - R["o_model"]) <= 2.0 ** -7 * R["wabsv"] + 2.0 ** -12 * R["vmax"]).all(), (l, r)
                assert (np.abs(lse[r] - R["lse_model"]) <= 2.0 ** -8).all(), (l, r)


def test_cuda_graph_survives_growth_of_tickets_and_partials():
    """After a graph has pinned its cache entry, a call with more than 1024 (request, kv head) groups AND a larger
    partial buffer makes both context buffers grow in one call.  The outgrown buffers are what the graph still points
    at: they must stay allocated until kvr_destroy (freeing them at regrowth handed a later replay freed memory, and
    kvr_destroy then freed them a second time).  Replay twice after the growth and check the outputs."""
    from paper_2606_17107_b200 import kvr
    from paper_2606_17107_b200.harness import DeviceReadWorkload
    w = read_workload("graph-grow", q_heads=8, kv_heads=2, layers=2, requests=[[(900, 5), (200, -3)], [(1500, 777)]], seed=99)
    srcs_t, q_t = make_read_sources(w, "cpu"), make_queries(w, "cpu")
    dw = DeviceReadWorkload(w, "cuda:0", sources=srcs_t, queries=q_t)
    outs = [(torch.empty_like(dw.o), torch.empty_like(dw.lse)) for _ in range(2)]
    big = DeviceReadWorkload(read_workload("many-groups", q_heads=8, kv_heads=2, requests=[[(8, i)] for i in range(640)], seed=5),
                             "cuda:0")                          # 1280 groups > the 1024-ticket floor; 1280 items x 4 x 130 floats > 1 MB
    stream = torch.cuda.Stream()
    with kvr.Context(dw.model) as ctx:
        call = lambda l: ctx.rotate_on_read_attention(dw.q, w.n_req, w.q_heads, l, w.scale, dw.segs, outs[l][0], outs[l][1], stream=stream)
        call(0)
        torch.cuda.synchronize()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.stream(stream):
            graph.capture_begin()
            for l in range(2):
                call(l)
            graph.capture_end()
        big.run(ctx, stream=stream)                              # tickets and partials both outgrown in this call
        torch.cuda.synchronize()
        assert torch.isfinite(big.o).all() and torch.isfinite(big.lse).all()
        srcs = [(np_bits(k), np_bits(v)) for k, v in srcs_t]
        for rep in range(2):
            for o_, l_ in outs:
                o_.fill_(float("nan")); l_.fill_(float("nan"))
            with torch.cuda.stream(stream):
                graph.replay()
            big.run(ctx, stream=stream)                          # the new buffers in use right behind the replay
            torch.cuda.synchronize()
            for l in range(2):
                w.layer = l
                ref = reference(w, srcs, np_bits(q_t), orc.host_threads())
                o, lse = outs[l][0].cpu().numpy().astype(np.float64), outs[l][1].cpu().numpy().astype(np.float64)
                for r, R in enumerate(ref):
                    assert (np.abs(o[r] - R["o_model"]) <= 2.0 ** -7 * R["wabsv"] + 2.0 ** -12 * R["vmax"]).all(), (rep, l, r)
                    assert (np.abs(lse[r] - R["lse_model"]) <= 2.0 ** -8).all(), (rep, l, r)
