#!/usr/bin/env python
"""bench.py -- KV tokens repositioned+spliced per second on B200 (BASELINE.json `metric`).

A "step" is one pass of the whole hot path (SURVEY.md 8(a) a1..a6 = one kvr_reposition_splice call) over one
BASELINE.json configuration of synthetic seeded input.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl kvr|reference] [--config c] [--layout NHD|HND]

Default (no --config): the HEADLINE is configs[4] (cfg4-long-partial-rotary, 12.9 GB per step, bf16 cache: the largest
single-GPU configuration at the paper's cache precision; BASELINE.json's metric is not quoted on one configuration),
token-major (NHD) pool, and the same JSON line carries `per_config`: configs[1..4] x {NHD, HND}, each timed in the
same run (north_star: ">= 80 % of peak HBM bandwidth on configs 1-4").  `--config c` times that one configuration
alone (what the ncu captures under profiles/ run).

* value      whole-job KV tokens/s of the headline: EXACTLY K steps, inputs resident in HBM, CUDA events on the
             launching stream, barrier + synchronize on both sides, max over ranks (N > 1: independent replicas).
* per_config for every (config, layout): blocks of K steps repeated back to back until >= 0.25 s of device time;
             median / best / spread over the blocks, GB/s of algorithmic bytes, fraction of the measured peak,
             NVML clocks sampled during that configuration's timed region.
* roofline   algorithmic bytes (4 * layers*kv_heads*head_dim*esz per KV token) / measured launch time
             against MEASURED_PEAKS.json `hbm_gbs` (the measured copy bandwidth of this pool's B200s).
* e2e        the same metric through kvr_reposition_splice_host: sources in pinned HOST memory, the
             host->device copies and the device->host read of the status word inside the timed region.
* cpu_baseline  the fp64 oracle (oracle/, as it stands) on this box's host cores over a bounded sample.
* --impl reference  times the oracle alone (rank 0 only), same metric/config, JSON line with "impl": "reference".
             That arm imports nothing of the product package (tests/test_bench_arms.py).
"""
import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "KV tokens repositioned+spliced/sec"
UNIT = "KV tokens/s"
HEADLINE_CONFIG = 4                # largest single-GPU configuration with the paper's (bf16) cache precision
SWEEP_CONFIGS = (1, 2, 3, 4)       # north_star: the bandwidth bar is on configs 1-4
SWEEP_LAYOUTS = ("NHD", "HND")
FALLBACK_HBM_GBS = 6650.0          # /opt/skills/guides/B200_PROFILING.md fallback ("of fallback")
CACHE_DTYPE = {"bf16": "bf16", "fp8": "fp8-e4m3"}
L2_BYTES = 126e6
# dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from one `ncu --set full`
# capture of the bench command (profiles/, named per round); None until a capture of that case exists.
# Keys: "<workload>:<layout>" for the splice, "<workload>:<layout>:<op>" for the other ops.
NCU_TRAFFIC_BYTES = {}
try:
    with open(os.path.join(ROOT, "profiles", "traffic.txt")) as _f:     # lines: "<key> <bytes> <source file>"
        for _line in _f:
            _p = _line.split()
            if len(_p) >= 2 and not _line.startswith("#"):
                NCU_TRAFFIC_BYTES[_p[0]] = int(_p[1])
except OSError:
    pass


def traffic_of(name, layout, op):
    return NCU_TRAFFIC_BYTES.get(f"{name}:{layout}" + ("" if op == "splice" else f":{op}"))


def parse_args(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=None)
    ap.add_argument("--config", type=int, default=None,
                    help="index into BASELINE.json configs: time that one alone (default: headline configs[4] + sweep)")
    ap.add_argument("--workload", default="", help="an adapter workload instead of --config (SURVEY.md 8(f) NEXT-3/4): "
                    "mla-dsv2-lite | image-kv-qwen25vl-7b | image-kv-qwen3vl-8b | compose-qwen3-8b; device-timed and e2e only")
    ap.add_argument("--layout", default="NHD", choices=["NHD", "HND"])
    ap.add_argument("--impl", default="kvr", choices=["kvr", "reference"])
    ap.add_argument("--latency", action="store_true",
                    help="also report launch-to-launch latency and CUDA-graph replay time per call, rotating over 8 "
                         "buffer sets (SURVEY.md 8(d); always on for --config 0)")
    ap.add_argument("--op", default="splice", choices=["splice", "inplace", "span", "attend"],
                    help="splice = kvr_reposition_splice (the BASELINE.json metric); inplace = kvr_reposition_inplace "
                         "(SURVEY.md 8(f) NEXT-1: re-float resident chunks, 2*B1 bytes per token; device-timed only); "
                         "span = kvr_write_span over the same rows (Delta = 0: byte copies with the same access pattern "
                         "= this library's own copy ceiling, SURVEY.md H1); attend = kvr_rotate_on_read_attention over a "
                         "rotate-on-read workload (--workload attend-serving | attend-32k-x8 | attend-compose4; SURVEY.md "
                         "8(f) rank 4, first alternative; device-timed only)")
    ap.add_argument("--sweep", dest="sweep", action="store_true", default=None, help="force the per_config sweep")
    ap.add_argument("--no-sweep", dest="sweep", action="store_false")
    ap.add_argument("--min-device-s", type=float, default=0.25, help="device time per (config, layout) of the sweep")
    ap.add_argument("--e2e-steps", type=int, default=None)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-next", action="store_true", help="skip the short NEXT-row cases of the default run")
    ap.add_argument("--layers", type=int, default=None,
                    help="profiling aid: keep only the first N layers of the configuration (same kernel, tiles and "
                         "per-layer access pattern, less memory for ncu to save and restore); never a bench number")
    ap.add_argument("--tune", default="", help="kvr_tuning overrides, e.g. ctas_per_sm=1,stages=12")
    return ap.parse_args(argv)


def measured_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except (OSError, KeyError, ValueError):
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def algorithmic_bytes(w):
    """Bytes one step must move: read K, read V, write K, write V of every spliced token."""
    return (4 if w.has_v else 2) * w.layers * w.kv_heads * w.head_dim * w.elt_bytes * w.tokens


def config_block(w, op, config_index, layout, world):
    """The `config` object of the JSON line: identical keys and values in the kvr arm and the reference arm."""
    b = algorithmic_bytes(w)
    return {"workload": w.name, "op": op, "config_index": config_index, "layout": layout,
            "cache_dtype": CACHE_DTYPE[w.dtype], "tokens": w.tokens, "segments": len(w.segments),
            "bytes_per_step": b, "parallelism": f"replicas x{world}",
            "sources": ("precompiled skills: every segment carries KVR_SEG_SRC_STABLE (kvr.h), so a launch may start reading its "
                        "sources while the previous launch on the stream drains") if all(getattr(s_, "src_stable", False) for s_ in w.segments)
                       else "no ordering promise (no early source loads)",
            "l2": (f"inputs larger than L2 ({b // 2} B of sources + as many pool bytes per step vs 126 MB L2); no flush")
                  if b // 2 > 2 * L2_BYTES else
                  (f"working set ({b} B per step) does NOT exceed the 126 MB L2 and is not flushed: a latency-bound "
                   "case, not a bandwidth figure; see 'latency' (8 rotating buffer sets)")}


def bits_to_numpy(t):
    """Bit-pattern tensor (int16 for bf16, uint8 for fp8) -> contiguous numpy array (uint16 / uint8) on the host."""
    import numpy as np
    a = t.detach().cpu().contiguous().numpy()
    return a.view(np.uint16) if a.dtype == np.int16 else a


# --------------------------------------------------------------------------------------- clocks
class ClockSampler:
    """Samples SM clock and throttle reasons through NVML while a timed region runs."""
    BAD = {"hw_slowdown": 0x8, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20}
    NOTE = {"sw_power_cap": 0x4}

    def __init__(self, torch_device):
        self.samples, self.reasons, self.max_mhz, self._stop, self._h = [], 0, None, threading.Event(), None
        try:
            import pynvml
            import torch
            pynvml.nvmlInit()
            self._nv = pynvml
            uuid = str(torch.cuda.get_device_properties(torch_device).uuid)
            try:
                self._h = pynvml.nvmlDeviceGetHandleByUUID(("GPU-" + uuid) if not uuid.startswith("GPU-") else uuid)
            except Exception:
                self._h = pynvml.nvmlDeviceGetHandleByIndex(torch.device(torch_device).index or 0)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM))
        except Exception as e:      # noqa: BLE001 -- no NVML: the clocks object says so
            self.error = repr(e)

    def reset(self):
        self.samples, self.reasons, self._stop = [], 0, threading.Event()

    def sample(self):
        if self._h is None:
            return
        try:
            self.samples.append(int(self._nv.nvmlDeviceGetClockInfo(self._h, self._nv.NVML_CLOCK_SM)))
            self.reasons |= int(self._nv.nvmlDeviceGetCurrentClocksEventReasons(self._h))
        except Exception:           # noqa: BLE001
            pass

    def _run(self):
        while not self._stop.is_set():
            self.sample()
            time.sleep(0.003)

    def __enter__(self):
        self._t = threading.Thread(target=self._run, daemon=True)
        self._t.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        self._t.join()

    def bad(self):
        return any(self.reasons & bit for bit in self.BAD.values())

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["unavailable: " + getattr(self, "error", "no samples")]}
        s = sorted(self.samples)
        names = [n for n, bit in {**self.BAD, **self.NOTE}.items() if self.reasons & bit]
        return {"sm_mhz": s[len(s) // 2], "sm_min_mhz": s[0], "sm_max_mhz": self.max_mhz, "reasons": names, "samples": len(s)}


# --------------------------------------------------------------------------------------- oracle timing
def _oracle_sample(c, layout, k_steps_total, get_sources, cpu_work_target_s=15.0, wall_cap_s=120.0):
    """Times the oracle, as it stands, on a bounded sample of config c: the first `ls` layers of every segment
    (every head, token and element of them).  Returns (ls, layers, threads, run_step, full workload) where run_step()
    performs one sample pass.  The sample is sized from one calibration layer so that a step is ~cpu_work_target_s
    of CPU work and k_steps_total steps stay under wall_cap_s."""
    import numpy as np
    from oracle import kvr_oracle as orc
    from workloads import SENTINEL_BF16, SENTINEL_FP8, config
    threads = orc.host_threads()
    full = config(c, layout)

    def make(ls):
        w = config(c, layout, layers=ls)
        srcs = get_sources(w, ls)
        edt = np.uint16 if w.dtype == "bf16" else np.uint8
        kc = np.full(w.pool_elems(), SENTINEL_BF16 if w.dtype == "bf16" else SENTINEL_FP8, dtype=edt)
        vc = kc.copy()
        return w, srcs, kc, vc

    w1, s1, kc, vc = make(1)
    orc.splice_workload(w1, s1, kc, vc, n_threads=threads)        # untimed: page in the pool, start the thread team
    t0 = time.perf_counter()
    orc.splice_workload(w1, s1, kc, vc, n_threads=threads)
    per_layer = time.perf_counter() - t0
    # the canonical single-thread oracle on the same one-layer sample, if it ends within ~20 s
    single = None
    if per_layer * threads < 20.0:
        t0 = time.perf_counter()
        orc.splice_workload(w1, s1, kc, vc, n_threads=1)
        single = full.tokens / ((time.perf_counter() - t0) * full.layers)
    _oracle_sample.single_thread_value = single
    per_step_target = min(cpu_work_target_s / threads, wall_cap_s / max(1, k_steps_total))
    ls = int(max(1, min(full.layers, per_step_target / max(per_layer, 1e-9))))
    ls = max(ls, min(full.layers, -(-threads // full.kv_heads)))     # enough (layer, head) units for every thread
    threads = min(threads, ls * full.kv_heads)                       # the OpenMP loop runs over (layer, head)
    w, srcs, kc, vc = (w1, s1, kc, vc) if ls == 1 else make(ls)

    def run_step():
        t = time.perf_counter()
        orc.splice_workload(w, srcs, kc, vc, n_threads=threads)
        return time.perf_counter() - t

    return ls, full.layers, threads, run_step, full


def cpu_sources_from_device(dw):
    def get(w, ls):
        return [(bits_to_numpy(k[:ls]), bits_to_numpy(v[:ls])) for k, v in dw.sources]
    return get


def cpu_sources_fresh():
    def get(w, ls):
        from workloads import make_sources
        return [(bits_to_numpy(k), bits_to_numpy(v)) for k, v in make_sources(w, "cpu")]
    return get


def time_oracle(c, layout, steps, warmup, get_sources):
    ls, layers, threads, run_step, full = _oracle_sample(c, layout, steps + warmup, get_sources)
    for _ in range(warmup):
        run_step()
    ts = [run_step() for _ in range(steps)]
    per_step = sum(ts) / len(ts)
    # a KV token spans all layers: the sample covers ls of `layers`, cost is linear in layers (O(L))
    tokens_per_s = full.tokens / (per_step * layers / ls)
    sample = (f"layers 0..{ls - 1} of {layers} (all heads, all {full.tokens} tokens, every element) per step, "
              f"{steps} step(s) after {warmup} warm-up, scaled linearly to {layers} layers")
    return tokens_per_s, per_step, threads, sample, full


def run_reference(args):
    """The oracle arm: imports oracle/ and workloads/ only -- nothing under paper_2606_17107_b200/."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    steps = args.steps if args.steps is not None else 5
    warmup = args.warmup if args.warmup is not None else 1
    c = args.config if args.config is not None else HEADLINE_CONFIG
    value, per_step, threads, sample, full = time_oracle(c, args.layout, steps, warmup, cpu_sources_fresh())
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
        "warmup": warmup, "ms_per_step": per_step * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": config_block(full, "splice", c, args.layout, max(1, args.gpus)),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


def latency_probe(w, device, ctx, stream, sets=8, reps=64):
    """Per-call latency of kvr_reposition_splice on `w` (meant for configs[0], 262 KB: launch-bound), rotating over
    `sets` independent source/pool sets so no call finds its lines in L2 from the call before:
    launch_to_launch_us = stream of back-to-back calls (CUDA events); graph_replay_us = the same calls captured once
    in a CUDA graph and replayed."""
    import torch
    from paper_2606_17107_b200.harness import DeviceWorkload
    dws = [DeviceWorkload(w, device) for _ in range(sets)]
    for d in dws:
        d.run(ctx, stream=stream)
    torch.cuda.synchronize(device)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

    def burst():
        for i in range(sets * reps):
            dws[i % sets].run(ctx, stream=stream)
    burst()
    torch.cuda.synchronize(device)
    ev0.record(stream); burst(); ev1.record(stream)
    torch.cuda.synchronize(device)
    l2l = ev0.elapsed_time(ev1) * 1e3 / (sets * reps)
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.stream(stream):
        with torch.cuda.graph(graph, stream=stream):
            burst()
        graph.replay()
        torch.cuda.synchronize(device)
        ev0.record(stream)
        for _ in range(5):
            graph.replay()
        ev1.record(stream)
    torch.cuda.synchronize(device)
    rep_us = ev0.elapsed_time(ev1) * 1e3 / (5 * sets * reps)
    assert ctx.last_device_status()[0] == 0
    return {"launch_to_launch_us": l2l, "graph_replay_us": rep_us, "buffer_sets": sets, "calls_per_graph": sets * reps,
            "bytes_per_call": int(dws[0].bytes_moved())}


# --------------------------------------------------------------------------------------- the kvr arm
def _median(xs):
    s = sorted(xs)
    n = len(s)
    return s[n // 2] if n % 2 else 0.5 * (s[n // 2 - 1] + s[n // 2])


class Timer:
    """Device timing of one (workload, layout, op) on one stream.  All numbers come from CUDA events recorded on
    the launching stream; nothing is timed under a profiler."""

    def __init__(self, device, stream, rep, sampler):
        self.device, self.stream, self.rep, self.sampler = device, stream, rep, sampler

    def warm(self, run_step, warmup):
        """`warmup` untimed steps, then keep warming until the GPU has been busy for >= 0.3 s: an idle B200 sits at
        ~120 MHz SM clock and needs tens of ms of load to reach its running clocks.  Returns (ramp steps, s/step)."""
        import torch
        for _ in range(warmup):
            run_step()
        torch.cuda.synchronize(self.device)
        ramp, t_ramp = 0, time.perf_counter()
        while time.perf_counter() - t_ramp < 0.3 and ramp < 100000:
            for _ in range(8):
                run_step()
            ramp += 8
            torch.cuda.synchronize(self.device)
        return ramp, (time.perf_counter() - t_ramp) / max(1, ramp)

    def exact_block(self, run_step, steps):
        """EXACTLY `steps` steps bracketed by barrier + synchronize on both sides.  Returns seconds."""
        import torch
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize(self.device)
        self.rep.barrier()
        ev0.record(self.stream)
        for _ in range(steps):
            run_step()
        ev1.record(self.stream)
        self.sampler.sample()                  # the queue is still draining: a sample under load even for short runs
        torch.cuda.synchronize(self.device)
        self.rep.barrier()
        return ev0.elapsed_time(ev1) * 1e-3

    def single_calls(self, run_step, n=15):
        """`n` ISOLATED steps: the device is idle when each one starts (synchronize on both sides), so nothing of the
        previous call's tail overlaps its ramp (no programmatic dependent launch, no early source loads).  This is the
        figure for the paper's use -- one transplant per request on the TTFT path, one re-float per turn
        (PAPER.md:528).  CUDA events around one launch add a few microseconds.  Returns the per-call seconds."""
        import torch
        out = []
        for _ in range(n):
            ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize(self.device)
            ev0.record(self.stream)
            run_step()
            ev1.record(self.stream)
            torch.cuda.synchronize(self.device)
            out.append(ev0.elapsed_time(ev1) * 1e-3)
        return out

    def blocks(self, run_step, steps, est_step_s, min_device_s, max_blocks=2000):
        """Blocks of `steps` steps back to back (one event between blocks, no host sync inside) until the device has
        been timed for >= min_device_s.  Returns the per-block seconds."""
        import torch
        block_s = max(steps * est_step_s, 1e-9)
        n = int(min(max_blocks, max(3 if 3 * block_s < 2.0 else 1, -(-min_device_s // block_s))))
        evs = [torch.cuda.Event(enable_timing=True) for _ in range(n + 1)]
        torch.cuda.synchronize(self.device)
        evs[0].record(self.stream)
        for b in range(n):
            for _ in range(steps):
                run_step()
            evs[b + 1].record(self.stream)
        self.sampler.sample()
        torch.cuda.synchronize(self.device)
        return [evs[b].elapsed_time(evs[b + 1]) * 1e-3 for b in range(n)]


def measure_case(kvr, timer, ctx_of, w, dw, op, steps, warmup, min_device_s, peak, headline):
    """Times one (workload, layout, op).  Returns the per_config entry; with `headline` also the bracketed block."""
    ctx = ctx_of(dw)
    stream = timer.stream
    bytes_per_step = dw.bytes_moved()
    assert op != "splice" or bytes_per_step == algorithmic_bytes(w), (bytes_per_step, algorithmic_bytes(w))
    run_step = lambda: dw.run(ctx, stream=stream)
    if op == "inplace":
        dw.run(ctx, stream=stream)                       # the chunks must be resident first (finite keys in the slots)
        spans = dw.inplace_spans([161 + 7 * i for i in range(len(w.segments))])
        bytes_per_step = kvr.kvr_inplace_bytes_moved(dw.model, spans)
        run_step = lambda: dw.run_inplace(ctx, spans, stream=stream)
    elif op == "span":
        spans_w = dw.write_spans()
        run_step = lambda: ctx.write_span(dw.dst, spans_w, stream=stream)

    out = {}
    for attempt in range(2):                   # a region that saw a thermal / hw slowdown is re-measured once
        ramp, est = timer.warm(run_step, warmup)
        st = ctx.last_device_status()
        assert st[0] == kvr.KVR_OK, st
        timer.sampler.reset()
        launches0 = ctx.launch_count()
        with timer.sampler:
            exact_s = timer.exact_block(run_step, steps) if headline else None
            launches_exact = ctx.launch_count() - launches0
            blk = timer.blocks(run_step, steps, est, min_device_s)
            single = timer.single_calls(run_step)
        out["remeasured"] = attempt > 0
        if not timer.sampler.bad():
            break
    st = ctx.last_device_status()
    assert st[0] == kvr.KVR_OK, st
    info = ctx.last_launch_info()
    per_step = [b / steps for b in blk]
    med, best, worst = _median(per_step), min(per_step), max(per_step)
    gbs = lambda s: bytes_per_step / s / 1e9
    out.update({
        "workload": w.name, "layout": w.layout, "op": op, "cache_dtype": CACHE_DTYPE[w.dtype], "tokens": w.tokens,
        "segments": len(w.segments), "bytes_per_step": int(bytes_per_step),
        "ms_per_step": med * 1e3, "best_ms_per_step": best * 1e3, "worst_ms_per_step": worst * 1e3,
        "spread": (worst - best) / med, "blocks": len(blk), "steps_per_block": steps, "device_s": sum(blk),
        "tokens_per_s": w.tokens / med,
        "achieved": gbs(med), "best_achieved": gbs(best), "unit": "GB/s", "frac": gbs(med) / peak,
        "best_frac": gbs(best) / peak, "gb_s_of_nominal_8000": gbs(med) / 8000.0,
        "single_call_us": _median(single) * 1e6, "single_call_achieved": gbs(_median(single)),
        "single_call_best_us": min(single) * 1e6, "single_call_calls": len(single),
        "clocks": timer.sampler.summary(), "traffic": traffic_of(w.name, w.layout, op),
        "kernel": {1: "kvr_generic_kernel", 2: "kvr_ring_kernel", 4: "kvr_window_inplace_kernel", 5: "kvr_generic_vec_kernel"}.get(info["path"], "?"),
        "grid": info["grid"], "block": info["block"], "smem": info["smem"],
        "warmup": warmup, "warmup_ramp_steps": ramp,
    })
    return out, exact_s, launches_exact, ctx


def measure_attend(kvr, timer, w, device, peak, steps, warmup, min_device_s, tune=None):
    """Times kvr_rotate_on_read_attention on `w` (one layer per step; source sets rotated so no call finds its keys in
    L2).  Returns (entry, exact seconds of `steps` steps, launches in them, the device workloads)."""
    from paper_2606_17107_b200.harness import DeviceReadWorkload
    sets = max(1, min(8, int(-(-3 * L2_BYTES // max(1, w.bytes_read())))))
    dws = [DeviceReadWorkload(w, device) for _ in range(sets)]
    ctx = kvr.Context(dws[0].model, device=device.index)
    if tune:
        ctx.set_tuning(**tune)
    state = {"i": 0}

    def run_step():
        dws[state["i"] % sets].run(ctx, stream=timer.stream)
        state["i"] += 1
    ramp, est = timer.warm(run_step, warmup)
    timer.sampler.reset()
    l0 = ctx.launch_count()
    with timer.sampler:
        exact_s = timer.exact_block(run_step, steps)
        launches = ctx.launch_count() - l0
        blk = timer.blocks(run_step, steps, est, min_device_s)
        single = timer.single_calls(run_step)
    per = [b / steps for b in blk]
    med, best, worst = _median(per), min(per), max(per)
    info = ctx.last_launch_info()
    b = dws[0].bytes_read()
    ctx.close()
    entry = {"workload": w.name, "op": "attend", "bytes_per_step": int(b), "ms_per_step": med * 1e3,
             "achieved": b / med / 1e9, "best_achieved": b / best / 1e9, "unit": "GB/s", "frac": b / med / 1e9 / peak,
             "spread": (worst - best) / med, "blocks": len(blk), "steps_per_block": steps,
             "single_call_us": _median(single) * 1e6, "single_call_achieved": b / _median(single) / 1e9,
             "tokens_per_s": w.tokens / med, "clocks": timer.sampler.summary(), "source_sets": sets,
             "kernel": "kvr_attend_kernel", "grid": info["grid"], "block": info["block"], "smem": info["smem"],
             "warmup": warmup, "warmup_ramp_steps": ramp}
    return entry, exact_s, launches, dws


NEXT_ROWS = [("inplace", "config", 2), ("span", "config", 1), ("splice", "adapter", "mla-dsv2-lite"),
             ("splice", "adapter", "compose-qwen3-8b"), ("attend", "read", "attend-serving")]


def next_rows(kvr, timer, ctx_of, peak, device, min_device_s=0.1):
    """One short timed case per SURVEY.md 8(f) row (in place, span overwrite, the MLA adapter, the compose workload,
    rotate-on-read attention) so that the default run's line carries them: median GB/s of back-to-back calls, fraction of
    the measured peak, GB/s of an isolated call, clocks.  No oracle leg here (parity is the tests' business)."""
    import torch
    from paper_2606_17107_b200.harness import DeviceWorkload
    from workloads import adapter_config, attention_config, config
    keep = ("workload", "layout", "op", "bytes_per_step", "ms_per_step", "achieved", "best_achieved", "frac", "unit",
            "single_call_us", "single_call_achieved", "kernel", "grid", "clocks", "blocks", "steps_per_block")
    rows = []
    for op, kind, which in NEXT_ROWS:
        if kind == "read":
            entry, _, _, dws = measure_attend(kvr, timer, attention_config(which), device, peak, 20, 3, min_device_s)
            del dws
        else:
            w = config(which, "NHD") if kind == "config" else adapter_config(which, "NHD")
            dw = DeviceWorkload(w, device)
            entry, _, _, ctx = measure_case(kvr, timer, ctx_of, w, dw, op, 20, 3, min_device_s, peak, headline=False)
            ctx.close()
            del dw
        rows.append({k: entry[k] for k in keep if k in entry})
        torch.cuda.empty_cache()
    return rows


def run_kvr(args):
    import torch
    from paper_2606_17107_b200 import build as _kbuild
    _kbuild.build()        # no-op when the in-tree library is newer than its sources; never a CPU fallback
    from paper_2606_17107_b200 import kvr
    from paper_2606_17107_b200.harness import DeviceWorkload
    from paper_2606_17107_b200.replicas import Replicas, aggregate_throughput
    from workloads import config

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the kvr path has no CPU fallback")
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    device = torch.device("cuda", local_rank)
    torch.cuda.set_device(device)
    rep = Replicas(backend="nccl", device=device)
    single = args.config is not None or bool(args.workload) or args.op != "splice"
    steps = args.steps if args.steps is not None else (1000 if single else 20)
    warmup = max(3, args.warmup if args.warmup is not None else (50 if single else 5))
    sweep = args.sweep if args.sweep is not None else (not single and rep.world == 1)
    head_c = args.config if args.config is not None else HEADLINE_CONFIG
    peak, peak_src = measured_peak()
    stream = torch.cuda.Stream(device=device)
    timer = Timer(device, stream, rep, ClockSampler(device))     # NVML init happens here, before any warm-up
    tune = {k: int(v) for k, v in (kv.split("=") for kv in args.tune.split(","))} if args.tune else {}

    ctxs = []

    def ctx_of(dw):
        ctx = kvr.Context(dw.model, device=local_rank)
        if tune:
            ctx.set_tuning(**tune)
        ctxs.append(ctx)
        return ctx

    # ---- sweep: configs[1..4] x {NHD, HND}; the headline case is measured last and keeps its buffers ----
    per_config, head = [], None
    cases = []
    if sweep:
        for c in SWEEP_CONFIGS:
            for lay in SWEEP_LAYOUTS:
                if not (c == head_c and lay == args.layout):
                    cases.append((c, lay))
    cases.append((head_c, args.layout))
    sources, sources_c = None, None
    for c, lay in cases:
        is_head = (c, lay) == (head_c, args.layout)
        if args.workload and is_head:
            from workloads import adapter_config
            w = adapter_config(args.workload, lay)
            args.no_cpu_baseline = True
        else:
            w = config(c, lay, layers=args.layers)
        if sources_c != c:
            sources, sources_c = None, c                 # frees the previous configuration's sources
        dw = DeviceWorkload(w, device, sources=sources)   # the two layouts of a configuration share its sources
        sources = dw.sources
        entry, exact_s, launches, ctx = measure_case(kvr, timer, ctx_of, w, dw, args.op if is_head else "splice",
                                                     steps, warmup, args.min_device_s, peak, headline=is_head)
        entry["config_index"] = None if (args.workload and is_head) else c
        per_config.append(entry)
        if is_head:
            head = (w, dw, ctx, entry, exact_s, launches)
        else:
            ctx.close()
            del dw
            torch.cuda.empty_cache()
    per_config.sort(key=lambda e: (e["config_index"] if e["config_index"] is not None else -1, e["layout"]))

    w, dw, ctx, entry, seconds, launches = head
    if args.op != "splice":
        args.no_e2e = args.no_cpu_baseline = True
    tokens, bytes_per_step = w.tokens, entry["bytes_per_step"]
    agg = aggregate_throughput(rep, tokens * steps, seconds)
    achieved = bytes_per_step / (seconds / steps) / 1e9      # this rank's kernel: one launch per step

    latency = None
    if (args.latency or (not args.workload and head_c == 0)) and args.op == "splice" and rep.world == 1:
        latency = latency_probe(w, device, ctx, stream)

    # ---- end to end: sources in pinned host memory, through kvr_reposition_splice_host ----
    e2e = None
    if not args.no_e2e:
        dw.make_host_sources()
        e2e_steps = args.e2e_steps if args.e2e_steps is not None else max(3, min(20, steps))
        for _ in range(2):
            dw.run_host(ctx, stream=stream)
            assert ctx.last_device_status()[0] == kvr.KVR_OK
        h2d = ctx.last_h2d_bytes() + len(dw.host_segs) * 96 * max(1, (w.layers + 3) // 4)
        torch.cuda.synchronize(device)
        rep.barrier()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            dw.run_host(ctx, stream=stream)
            st = ctx.last_device_status()      # device -> host read of the step's result (status word), syncs
            assert st[0] == kvr.KVR_OK, st
        torch.cuda.synchronize(device)
        e2e_seconds = time.perf_counter() - t0
        rep.barrier()
        e_agg = aggregate_throughput(rep, tokens * e2e_steps, e2e_seconds)
        # the ceiling of this leg: a plain pinned-host -> device cudaMemcpyAsync of one source tensor, timed alone
        hk = max((k for k, _ in dw.host_sources), key=lambda t: t.numel())
        scratch = torch.empty(hk.shape, dtype=hk.dtype, device=device)
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        with torch.cuda.stream(stream):
            scratch.copy_(hk, non_blocking=True)
            ev0.record(stream)
            for _ in range(3):
                scratch.copy_(hk, non_blocking=True)
            ev1.record(stream)
        torch.cuda.synchronize(device)
        h2d_peak = 3 * hk.numel() * hk.element_size() / (ev0.elapsed_time(ev1) * 1e-3) / 1e9
        del scratch
        e2e_ms = e_agg["seconds"] / e2e_steps * 1e3
        e2e = {"value": e_agg["per_second"], "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": 16,
               "steps": e2e_steps, "ms_per_step": e2e_ms,
               "h2d_gbs": h2d / (e2e_ms * 1e-3) / 1e9, "h2d_peak_gbs": h2d_peak,
               "h2d_frac": h2d / (e2e_ms * 1e-3) / 1e9 / h2d_peak,
               "h2d_peak_source": f"pinned cudaMemcpyAsync of one {hk.numel() * hk.element_size()} B source tensor, 3 copies, CUDA events",
               "api": "kvr_reposition_splice_host (pinned host K/V sources -> staged H2D overlapped with the kernel) "
                      "+ kvr_last_device_status"}
        dw.host_sources = dw.host_segs = None

    # ---- oracle on the host cores (rank 0, N = 1 only): 1 warm-up + 3 timed passes over a bounded sample ----
    cpu = None
    if rep.world == 1 and not args.no_cpu_baseline:
        v, per_step, threads, sample, _ = time_oracle(head_c, args.layout, 3, 1, cpu_sources_from_device(dw))
        cpu = {"value": v, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample,
               "single_thread_value": getattr(_oracle_sample, "single_thread_value", None),
               "single_thread_sample": "layer 0 of every segment, one thread, scaled linearly to all layers"}

    nxt = None
    if sweep and rep.world == 1 and args.op == "splice" and not args.workload and not args.no_next:
        nxt = next_rows(kvr, timer, ctx_of, peak, device)

    for c_ in ctxs:
        c_.close()
    if rep.rank == 0:
        cfg = config_block(w, args.op, None if args.workload else head_c, args.layout, rep.world)
        cfg["bytes_per_step"] = int(bytes_per_step)
        if args.layers is not None:
            cfg["layers_override"] = args.layers           # a profiling run, not a bench number
        line = {
            "metric": {"splice": METRIC, "inplace": "KV tokens repositioned in place/sec",
                       "span": "KV tokens overwritten (Delta = 0 copy)/sec"}[args.op],
            "value": agg["per_second"], "unit": UNIT, "n_gpus": rep.world, "steps": steps,
            "warmup": warmup, "warmup_ramp_steps": entry["warmup_ramp_steps"],
            "ms_per_step": agg["seconds"] / steps * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": w.dtype if w.dtype == "bf16" else "fp8-e4m3",
            "arithmetic": "fp32 registers (bf16: compensated rotate) on an fp64 sincos table; one rounding to the cache dtype",
            "data": "synthetic", "config": cfg,
            "launch": {"kernel": entry["kernel"], "grid": entry["grid"], "block": entry["block"], "smem": entry["smem"]},
            "gpu_launches": launches,
            "clocks": entry["clocks"],
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                         "traffic": entry["traffic"], "peak_source": peak_src,
                         "gb_s_of_nominal_8000": achieved / 8000.0,
                         "median_achieved": entry["achieved"], "best_achieved": entry["best_achieved"],
                         "spread": entry["spread"], "blocks": entry["blocks"]},
            "e2e": e2e,
            "cpu_baseline": cpu,
        }
        if sweep or len(per_config) > 1:
            line["per_config"] = per_config
        else:
            line["timing"] = {k: entry[k] for k in ("ms_per_step", "best_ms_per_step", "worst_ms_per_step", "spread",
                                                     "blocks", "steps_per_block", "device_s", "remeasured")}
        if latency is not None:
            line["latency"] = latency
        if nxt is not None:
            line["next"] = nxt
        # LAST key, short on purpose: whoever keeps only the tail of this line still sees every case
        line["per_config_summary"] = summary_of(per_config, nxt)
        print(json.dumps(line), flush=True)
    rep.close()
    return 0


def summary_of(per_config, nxt):
    """Short on purpose (about 600 bytes) and ordered so that configs[1..4] come last: per case
    [GB/s back to back, fraction of the measured peak, GB/s of an isolated call, median SM MHz, bad clocks]."""
    def row(e):
        return [round(e["achieved"]), round(e["frac"], 3), round(e["single_call_achieved"]),
                round(e["clocks"].get("sm_mhz") or 0), int(any(r in ClockSampler.BAD for r in e["clocks"].get("reasons", [])))]
    out = {"_": "GB/s,frac,isolated GB/s,MHz,badclk"}
    for e in nxt or []:
        name = e["workload"].split("-")[0] if e["workload"].startswith("cfg") else e["workload"]
        out[name if e["op"] in ("splice", "attend") else f'{e["op"]}:{name}'] = row(e)
    for e in per_config:
        name = f'cfg{e["config_index"]}' if e.get("config_index") is not None else e["workload"]
        out[f'{name}:{e["layout"]}' + ("" if e["op"] == "splice" else ":" + e["op"])] = row(e)
    return out


def run_attend(args):
    """--op attend: one step = one kvr_rotate_on_read_attention call (one layer) over a rotate-on-read workload.
    HBM roofline: K and V of the layer are read once (2 * kv_heads * head_dim * 2 bytes per token); the contraction
    flops (2 * 2 * q_heads * head_dim per token, on the tensor cores) are reported beside it."""
    import torch
    from paper_2606_17107_b200 import build as _kbuild
    _kbuild.build()
    from paper_2606_17107_b200 import kvr
    from paper_2606_17107_b200.harness import DeviceReadWorkload
    from paper_2606_17107_b200.replicas import Replicas
    from workloads import attention_config
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the kvr path has no CPU fallback")
    device = torch.device("cuda", int(os.environ.get("LOCAL_RANK", "0")))
    torch.cuda.set_device(device)
    rep = Replicas(backend="nccl", device=device)
    steps = args.steps if args.steps is not None else 200
    warmup = max(3, args.warmup if args.warmup is not None else 20)
    peak, peak_src = measured_peak()
    stream = torch.cuda.Stream(device=device)
    timer = Timer(device, stream, rep, ClockSampler(device))
    w = attention_config(args.workload or "attend-serving")
    # sets of sources rotated step by step so that no call finds its keys in the 126 MB L2 from the call before
    sets = max(1, min(8, int(-(-3 * L2_BYTES // max(1, w.bytes_read())))))
    dws = [DeviceReadWorkload(w, device) for _ in range(sets)]
    ctx = kvr.Context(dws[0].model, device=device.index)
    if args.tune:
        ctx.set_tuning(**{k: int(v) for k, v in (kv.split("=") for kv in args.tune.split(","))})
    state = {"i": 0}

    def run_step():
        dws[state["i"] % sets].run(ctx, stream=stream)
        state["i"] += 1
    ramp, est = timer.warm(run_step, warmup)
    timer.sampler.reset()
    l0 = ctx.launch_count()
    with timer.sampler:
        exact_s = timer.exact_block(run_step, steps)
        launches = ctx.launch_count() - l0
        blk = timer.blocks(run_step, steps, est, args.min_device_s)
    per = [b / steps for b in blk]
    med, best, worst = _median(per), min(per), max(per)
    info = ctx.last_launch_info()
    b = dws[0].bytes_read()
    flops = 4.0 * w.q_heads * w.head_dim * w.tokens
    achieved = b / (exact_s / steps) / 1e9
    ctx.close()
    # the oracle (as it stands) on the host cores, over request 0 of the workload, scaled by tokens
    cpu = None
    if rep.world == 1 and not args.no_cpu_baseline:
        from oracle import kvr_oracle as orc
        seg0 = [(i, s_) for i, s_ in enumerate(w.segments) if s_.request == 0]
        srcs0 = [(bits_to_numpy(dws[0].sources[i][0][w.layer]), bits_to_numpy(dws[0].sources[i][1][w.layer]), s_.delta) for i, s_ in seg0]
        q0 = bits_to_numpy(dws[0].q[0])
        threads = min(orc.host_threads(), w.q_heads)
        kw = dict(q=q0, kv_heads=w.kv_heads, rotary_dim=w.rotary_dim, pairing={"neox": 0, "gptj": 1}[w.pairing],
                  inv_freq=w.inv_freq, scale=w.scale, segments=srcs0, n_threads=threads)
        orc.rotate_on_read_attention(**kw)
        t0 = time.perf_counter()
        for _ in range(3):
            orc.rotate_on_read_attention(**kw)
        tok0 = sum(s_.len for _, s_ in seg0)
        cpu = {"value": tok0 / ((time.perf_counter() - t0) / 3), "unit": UNIT, "cores": threads, "kind": "oracle",
               "sample": f"request 0 of {w.n_req} ({tok0} of {w.tokens} tokens, every query head), 3 passes after 1 warm-up"}
    if rep.rank == 0:
        line = {
            "metric": "KV tokens attended by rotate-on-read/sec (one layer)", "value": w.tokens * rep.world / (exact_s / steps),
            "unit": UNIT, "n_gpus": rep.world, "steps": steps, "warmup": warmup, "warmup_ramp_steps": ramp,
            "ms_per_step": exact_s / steps * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "bf16", "arithmetic": "bf16 tensor-core contractions (tcgen05, fp32 accumulation in TMEM), fp32 softmax, "
                     "fp64 counter-rotation of the query",
            "data": "synthetic",
            "config": {"workload": w.name, "op": "attend", "requests": w.n_req, "segments": len(w.segments), "tokens": w.tokens,
                       "q_heads": w.q_heads, "kv_heads": w.kv_heads, "head_dim": w.head_dim, "bytes_per_step": int(b),
                       "parallelism": f"replicas x{rep.world}",
                       "l2": f"{sets} independent source sets rotated step by step ({sets * b} B > 126 MB L2)"},
            "launch": {"kernel": "kvr_attend_kernel", "grid": info["grid"], "block": info["block"], "smem": info["smem"]},
            "gpu_launches": launches, "clocks": timer.sampler.summary(),
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                         "traffic": traffic_of(w.name, "src", "attend"), "peak_source": peak_src,
                         "median_achieved": b / med / 1e9, "best_achieved": b / best / 1e9, "spread": (worst - best) / med,
                         "blocks": len(blk), "tensor_tflops": flops / (exact_s / steps) / 1e12},
            "e2e": None, "cpu_baseline": cpu,
        }
        print(json.dumps(line), flush=True)
    rep.close()
    return 0


def main():
    args = parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.op == "attend":
        return run_attend(args)
    return run_kvr(args)


if __name__ == "__main__":
    sys.exit(main())
