"""Host-side plumbing of bench.py that needs no GPU: the algorithmic byte / flop counts of SURVEY.md 8(d), the roofline
object, and the lookup of the committed ncu capture that `roofline.traffic` is read from."""
import importlib.util
import json
import os

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
_spec = importlib.util.spec_from_file_location("bench", os.path.join(ROOT, "bench.py"))
bench = importlib.util.module_from_spec(_spec)
_spec.loader.exec_module(bench)


def test_algorithmic_counts_match_the_scope_table():
    params, in_bytes, flops = bench.layer_counts("layer", 512)
    assert params == 218103808                                   # parameters per layer
    assert flops == 2 * params * 512 == 223338299392             # 223.3 GF per layer at T = 512
    # each distinct X once (q/k/v share one, gate/up share one) + every dY: 71.3 MB
    xs = 4096 + 4096 + 4096 + 14336
    dys = 4096 + 1024 + 1024 + 4096 + 14336 + 14336 + 4096
    assert in_bytes == 2 * 512 * (xs + dys)
    p, b, f = bench.layer_counts("gate", 8192)
    assert p == 14336 * 4096 and b == 2 * 8192 * (4096 + 14336) and f == 2 * p * 8192
    assert abs(bench.MOMENT_BYTES["int8"] - 8.0625) < 1e-12 and bench.MOMENT_BYTES["fp32"] == 20.0


def test_roofline_object_picks_the_binding_term():
    clocks = {"sm_mhz": 1965, "sm_max_mhz": 1965, "reasons": []}
    hbm, tf_burst, tf_sus, _ = bench.measured_peaks()
    p, b, f = bench.layer_counts("layer", 512)
    r, t_sus = bench.roofline_obj(p, b, f, 20.0, 730.0, clocks)
    assert r["bound"] == "hbm" and abs(r["frac"] - (p * 20.0 + b) / 730.0 / 1e3 / hbm) < 1e-9 and r["unit"] == "GB/s"
    assert r["hbm_term_us"] > r["tensor_term_us"] and abs(t_sus - f / tf_sus / 1e6) < 1e-9
    p, b, f = bench.layer_counts("gate", 8192)
    r, _ = bench.roofline_obj(p, b, f, 20.0, 750.0, clocks)
    assert r["bound"] == "tensor" and r["peak"] == tf_burst and r["peak_kind"] == "burst"
    capped = {"sm_mhz": 1500, "sm_max_mhz": 1965, "reasons": ["sw_power_cap"]}
    r, _ = bench.roofline_obj(p, b, f, 20.0, 900.0, capped)
    assert r["peak"] == tf_sus and r["peak_kind"] == "sustained"


def test_traffic_comes_from_the_newest_matching_committed_capture():
    sig = "forge_fused_kernel<0, 0, 32, 4, 2, 2, 64, 128, 128, 2, 2, 2>"
    nbytes, src = bench.ncu_traffic(sig, "fp32")
    assert src["file"].startswith("profiles/r02_fused_fp32_full") and sig in src["kernel"].replace("forge::", "")
    assert 4.2e9 < nbytes < 4.5e9                                # 0.99 x the 4.433 GB algorithmic bytes
    # a capture of another instantiation must not be used
    nbytes, src = bench.ncu_traffic("forge_fused_kernel<0, 0, 99, 4, 2, 2, 64, 128, 128, 2, 2, 2>", "fp32")
    assert nbytes is None and "reason" in src
    nbytes, src = bench.ncu_traffic(sig, "no_such_workload")
    assert nbytes is None


def test_committed_bench_line_has_the_contract_keys():
    line = json.loads(open(os.path.join(ROOT, "profiles", "r02_bench_default.json.txt")).read().strip().splitlines()[-1])
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "config", "roofline", "cpu_baseline", "e2e", "gpu_launches", "clocks", "configs"):
        assert k in line, k
    assert {"bound", "achieved", "peak", "unit", "frac", "traffic"} <= set(line["roofline"])
    assert {"value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step"} <= set(line["e2e"])
    assert {"value", "unit", "cores", "kind", "sample"} <= set(line["cpu_baseline"])
    assert len(line["configs"]) == 7 and line["higher_is_better"] is False and line["vs_baseline"] is None
