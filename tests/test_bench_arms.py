"""bench.py's two arms (no GPU needed): the oracle arm maps nothing of the product package into its process, both
arms print the same `config` object, and the sweep covers the configurations the north_star's target names."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

_PROBE = r"""
import json, sys
sys.argv = ["bench.py", "--impl", "reference", "--config", "0", "--steps", "1", "--warmup", "0"]
import bench
rc = bench.main()
mods = sorted(m for m in sys.modules if m.split(".")[0] == "paper_2606_17107_b200")
maps = sorted({l.split()[-1] for l in open("/proc/self/maps") if l.rstrip().endswith(".so") and "/repo/" in l})
print("PROBE " + json.dumps({"rc": rc, "mods": mods, "maps": maps}))
"""


def test_reference_arm_imports_nothing_of_the_product_package():
    out = subprocess.run([sys.executable, "-c", _PROBE], cwd=ROOT, capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = out.stdout.strip().splitlines()
    line = json.loads(next(l for l in lines if l.startswith("{")))
    probe = json.loads(next(l for l in lines if l.startswith("PROBE "))[6:])
    assert probe["rc"] == 0 and probe["mods"] == [], probe
    assert not any("libkvr.so" in m for m in probe["maps"]), probe["maps"]
    assert any(m.endswith("oracle/libkvr_oracle.so") for m in probe["maps"]), probe["maps"]
    assert line["impl"] == "reference" and line["gpu_launches"] == 0 and line["config"]["workload"] == "cfg0-tiny"
    assert line["e2e"] == {"value": line["value"], "unit": line["unit"], "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["value"] == line["value"]


def test_both_arms_describe_the_workload_with_the_same_config_object():
    sys.path.insert(0, ROOT)
    import bench
    from workloads import config
    for c in (1, 4):
        w = config(c, "NHD", layers=1)
        a = bench.config_block(w, "splice", c, "NHD", 1)
        assert set(a) == {"workload", "op", "config_index", "layout", "cache_dtype", "tokens", "segments",
                          "bytes_per_step", "parallelism", "sources", "l2"}
        assert a["bytes_per_step"] == 4 * w.layers * w.kv_heads * w.head_dim * w.elt_bytes * w.tokens
    args = bench.parse_args([])
    assert args.config is None and bench.HEADLINE_CONFIG == 4          # the headline is the largest bf16 configuration
    assert bench.SWEEP_CONFIGS == (1, 2, 3, 4) and bench.SWEEP_LAYOUTS == ("NHD", "HND")


def test_traffic_table_is_keyed_by_workload_and_layout():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.NCU_TRAFFIC_BYTES, "profiles/traffic.txt is missing or empty"
    for key in bench.NCU_TRAFFIC_BYTES:
        parts = key.split(":")
        assert len(parts) in (2, 3) and parts[1] in ("NHD", "HND", "src"), key   # "src": rotate-on-read attention reads the sources in place (no pool layout)
    assert bench.traffic_of("cfg1-qwen3-8b", "NHD", "splice") is not None
    assert bench.traffic_of("no-such-workload", "NHD", "splice") is None
