"""The reference arm of bench.py (the CPU oracle on a bounded sample) runs without a GPU and prints the
contract's JSON line."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_reference_arm_prints_one_contract_line():
    res = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1",
                          "--warmup", "0"], capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [l for l in res.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["metric"] == "prefill_tokens_per_s_per_layer_at_20pct_density"
    assert d["unit"] == "tokens/s" and d["higher_is_better"] is True and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"]["value"] == d["value"] and d["e2e"]["h2d_bytes_per_step"] == 0
    assert d["config"]["workload"].startswith("cfg2")
    # the same config keys as the GPU arm prints (bench_parts.prefill_bench uses the same gen.workload_config)
    assert {"layers", "seq_len", "h_q", "h_kv", "head_dim", "block", "blocks", "tau", "density",
            "tile_pairs_per_layer"} <= set(d["config"])
    assert d["config"]["tau"] == 103 and d["config"]["blocks"] == 512 and d["config"]["tile_pairs_per_layer"] == 47483


def test_reference_arm_never_maps_the_cuda_library():
    """The reference arm is the oracle alone: importing what it imports must not pull in the product package
    (whose import loads libsw.so).  bench.py asserts the same at run time."""
    code = ("import sys, bench; from oracle import sw_oracle; from synth import gen; "
            "assert 'paper_2602_07397_b200' not in sys.modules; "
            "maps = open('/proc/self/maps').read(); assert 'libsw.so' not in maps; print('clean')")
    res = subprocess.run([sys.executable, "-c", code], capture_output=True, text=True, timeout=300, cwd=ROOT)
    assert res.returncode == 0 and "clean" in res.stdout, res.stderr[-2000:]
