#!/usr/bin/env python
"""bench.py -- measures BASELINE.json's metric: fused wgrad+AdamW microseconds per Llama-3.1-8B layer
(7 projections as one grouped launch, T=512, bf16 W, fp32 m/v; BASELINE.json configs[1]) and its
fraction of the HBM roofline on one B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--moments fp32|bf16|int8|fp8] [--impl reference]
                  [--workload layer|q|..|down|model] [--tokens T] [--shard rows] [--backward]

A "step" is one pass of the whole hot path over one synthetic layer:
one forge_wgrad_adamw_grouped call.  Inputs are resident in HBM before the timed region; the
working set (4.4 GB of state per layer) is far larger than the 126 MB L2, so no flush is needed.

The default run prints ONE JSON line: the headline (configs[1]) with `roofline`, `e2e`, `cpu_baseline`,
`sustained`, the same-GPU unfused arms, `layer_backward` (dgrad + fused step in one call), and under `configs` the
other BASELINE.json configurations -- configs[2] (bf16, int8 moments), configs[3] (gate_proj at T = 512 / 2048 / 8192)
and configs[4] (the 75 GB stack) -- each timed with its own clock record against this box's MEASURED_PEAKS.json.

N > 1: `--gpus N` without WORLD_SIZE in the environment spawns N ranks itself (torchrun works too).  Default mode is
replicas (every rank its own layer, weak scaling, no collective on the data path: the tiles are independent,
PAPER.md:273-279, 302); `--shard rows` splits ONE layer's weight rows over the ranks (shard.py, Prop. 2(i): strong
scaling, still no collective).  `--impl reference` times the CPU oracle (the only "reference implementation" this
build has), a whole layer per step.
"""
from __future__ import annotations

import argparse
import glob
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "fused wgrad+AdamW us/layer (Llama-3.1-8B layer, 7 projections, BT=512, 1xB200)"
UNIT = "us/layer"
MOMENT_BYTES = {"fp32": 20.0, "bf16": 12.0, "int8": 8.0 + 2 * 2 * 4 / 256, "fp8": 8.0}   # SURVEY.md 8(d), B/element
MOMENT_ENUM = {"fp32": 0, "bf16": 1, "int8": 2, "fp8": 3}
T_TOKENS = 512
SEED = 20260622 + 1


def measured_peaks():
    """(HBM GB/s, bf16 TF/s burst, bf16 TF/s sustained, source)."""
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            d = json.load(f)
        return (float(d["hbm_gbs"]), float(d["bf16_tflops"]), float(d.get("bf16_tflops_sustained", d["bf16_tflops"])),
                "measured (MEASURED_PEAKS.json)")
    return 6650.0, 1590.0, 1400.0, "fallback (B200_PROFILING.md)"


def workload_shapes(workload: str):
    """configs[1]/[2]: the whole layer (default, the headline); configs[3]: gate_proj alone."""
    from paper_2606_22932_b200 import synth
    if workload == "layer":
        return synth.LLAMA8B_LAYER
    return tuple(s for s in synth.LLAMA8B_LAYER if s[0] == workload)


def layer_counts(workload: str = "layer", tokens: int = T_TOKENS):
    """(weight elements, operand bytes with each distinct X counted once, flops) of one launch."""
    from paper_2606_22932_b200 import synth
    shapes = workload_shapes(workload)
    params = sum(o * i for _, o, i in shapes)
    xs = {}
    for name, o, i in shapes:
        xs[(synth.X_GROUP[name], i)] = i
    in_bytes = 2 * tokens * (sum(xs.values()) + sum(o for _, o, _ in shapes))
    flops = 2 * params * tokens
    return params, in_bytes, flops


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons with NVML during the timed region."""

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.stop_flag, self.sm, self.reasons, self.max_mhz = index, False, [], set(), None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {nv.nvmlClocksThrottleReasonHwSlowdown: "hw_slowdown",
                 nv.nvmlClocksThrottleReasonHwThermalSlowdown: "hw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonSwThermalSlowdown: "sw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonSwPowerCap: "sw_power_cap"}
        while not self.stop_flag:
            try:
                self.sm.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, n in names.items():
                    if r & bit:
                        self.reasons.add(n)
            except Exception:
                pass
            time.sleep(0.002)

    def result(self):
        sm = sorted(self.sm)
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons)}


# ------------------------------------------------------------------------------------------------
# workload construction (synthetic, seeded; shapes of BASELINE.json configs[1] / [2] / [3])
# ------------------------------------------------------------------------------------------------
def make_device_layer(moments: str, seed: int, device, workload: str = "layer", tokens: int = T_TOKENS):
    """One Llama-3.1-8B layer's 7 problems (or one projection of it) on `device` (inputs resident in HBM).  The int8 /
    fp8 state is drawn directly as codes and scales (synth.random_*_state): no quantiser runs outside the library."""
    import torch
    from paper_2606_22932_b200 import synth
    probs = synth.make_layer(tokens, seed, shapes=workload_shapes(workload), device=device)
    out = []
    for k, p in enumerate(probs):
        d = dict(X=p.X, dY=p.dY, W=p.W)
        if moments == "fp32":
            d["m"], d["v"] = p.m, p.v
        elif moments == "bf16":
            d["m"], d["v"] = p.m.to(torch.bfloat16), p.v.to(torch.bfloat16)
        elif moments == "fp8":
            d["m"], d["v"], d["m_scale"], d["v_scale"] = synth.random_fp8_state(p.out, p.inn, seed * 100 + k, device)
        else:
            d["m"], d["v"], d["m_scale"], d["v_scale"] = synth.random_int8_state(p.out, p.inn, seed * 100 + k, device)
        out.append(d)
    return out


def make_host_layer(moments: str, seed: int):
    """The same layer in pinned host memory for the end-to-end (host buffer) measurement."""
    layer = make_device_layer(moments, seed, "cpu")
    return [{k: v.contiguous().pin_memory() for k, v in d.items()} for d in layer]


# ------------------------------------------------------------------------------------------------
# ncu evidence: DRAM traffic of the dispatched instantiation from the committed captures under profiles/
# ------------------------------------------------------------------------------------------------
def ncu_traffic(signature: str, tag: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch from the newest `profiles/r*_fused_<tag>_full.csv`
    (tag = the workload: fp32 | bf16 | int8 | fp8 for the layer, gate_<T> for configs[3]) whose `Kernel Name` is the
    instantiation this run dispatched (forge_last_kernel); (None, reason) if no capture matches."""
    best = None
    for path in sorted(glob.glob(os.path.join(ROOT, "profiles", f"r*_fused_{tag}_full.csv")), reverse=True):
        name, rd, wr = None, None, None
        scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
        try:
            with open(path) as f:
                for line in f:
                    parts = line.rstrip("\n").split(",")
                    if parts[0] == "Kernel Name":
                        name = line.split(",", 2)[2].strip().strip('"')
                    elif parts[0] == "dram__bytes_read.sum":
                        rd = float(parts[2]) * scale.get(parts[1], 1.0)
                    elif parts[0] == "dram__bytes_write.sum":
                        wr = float(parts[2]) * scale.get(parts[1], 1.0)
        except Exception:
            continue
        if name and rd is not None and wr is not None and signature and signature in name.replace("forge::", ""):
            best = {"bytes": rd + wr, "file": os.path.relpath(path, ROOT), "kernel": name}
            break
    if best:
        return best["bytes"], best
    return None, {"bytes": None, "reason": f"no ncu --set full capture of {signature!r} for workload {tag!r} under profiles/"}


# ------------------------------------------------------------------------------------------------
# CPU oracle timing (cpu_baseline leg and --impl reference)
# ------------------------------------------------------------------------------------------------
_CPU_LAYER = {}


def oracle_time_sample(frac_den: int, seed: int):
    """Times the oracle, as it stands, on rows [0, out/frac_den) of every projection of one layer (frac_den = 1: the
    whole layer).  Returns (seconds, description, threads)."""
    from oracle import forge_oracle as fo
    from paper_2606_22932_b200 import synth
    hp = synth.HP_DEFAULT
    if seed not in _CPU_LAYER:
        _CPU_LAYER[seed] = synth.make_layer(T_TOKENS, seed)
    layer = _CPU_LAYER[seed]
    work = []
    for p in layer:
        r = max(1, p.out // frac_den)
        work.append((synth.bf16_bits(p.dY), synth.bf16_bits(p.X), synth.bf16_bits(p.W)[:r].copy(),
                     p.m.numpy()[:r].copy(), p.v.numpy()[:r].copy(), r))
    fo.lib()
    t0 = time.perf_counter()
    for dY, X, W, m, v, r in work:
        G = fo.wgrad(dY, X, rows=(0, r))
        fo.adamw_fp32(W, m, v, G, 10, hp["lr"], hp["beta1"], hp["beta2"], hp["eps"], hp["wd"])
    dt = time.perf_counter() - t0
    what = "the whole layer" if frac_den == 1 else f"first 1/{frac_den} of the rows of each projection"
    return dt, f"{what}: 7 projections, T=512, fp32 moments", fo.num_threads()


def cpu_baseline(seed: int):
    """The oracle on the host cores over a WHOLE layer when that takes under ~40 s (it does: ~12 s on the GPU box's 16
    threads); otherwise over the largest 1/4 or 1/16 row sample that does, scaled to the metric's unit, and `sample`
    says which."""
    dt, desc, threads = oracle_time_sample(16, seed)
    den = 1 if dt * 16 < 40.0 else (4 if dt * 4 < 40.0 else 16)
    if den != 16:
        dt, desc, threads = oracle_time_sample(den, seed)
    return {"value": dt * den * 1e6, "unit": UNIT, "cores": threads, "kind": "oracle",
            "sample": desc + ("" if den == 1 else f", scaled x{den}"), "sample_seconds": round(dt, 3)}


def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores; rank 0 only.  Every timed step is ONE WHOLE
    LAYER (about 12 s on the GPU box's 16 threads): `steps` is the number that actually ran inside a ~100 s budget,
    never an extrapolation.  The warm-up is one 1/16-layer pass (loads the library, touches the inputs)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    budget_s = 100.0
    oracle_time_sample(16, SEED)
    times, desc, threads = [], "", 0
    t_begin = time.perf_counter()
    for _ in range(max(1, args.steps)):
        dt, desc, threads = oracle_time_sample(1, SEED)
        times.append(dt)
        if time.perf_counter() - t_begin + dt > budget_s:
            break
    us = sum(times) / len(times) * 1e6
    line = {"impl": "reference", "metric": METRIC, "value": us, "unit": UNIT, "n_gpus": args.gpus,
            "steps": len(times), "warmup": 1, "ms_per_step": us / 1e3, "higher_is_better": False,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "configs[1]: Llama-3.1-8B layer, 7 projections in one grouped launch, T=512",
                       "moments": "fp32", "params_per_layer": layer_counts()[0], "tokens": T_TOKENS},
            "cpu_baseline": {"value": us, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": desc},
            "e2e": {"value": us, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0,
            "note": f"requested steps={args.steps} warmup={args.warmup}; ran {len(times)} whole-layer steps (budget {budget_s:.0f} s) after one 1/16-layer warm-up"}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------
# timing and roofline helpers of the CUDA arm
# ------------------------------------------------------------------------------------------------
def time_steps(step, steps: int, warmup: int, stream, local: int, barrier=None):
    """W untimed warm-up calls, then exactly K calls bracketed by CUDA events on the launching stream (barrier +
    synchronize on both sides), NVML clock samples taken while they execute.  step(t) enqueues one step."""
    import torch
    for i in range(warmup):
        step(1 + i)
    if barrier:
        barrier()
    torch.cuda.synchronize()
    sampler = ClockSampler(local)
    sampler.start()
    evs = [torch.cuda.Event(enable_timing=True) for _ in range(steps + 1)]
    evs[0].record(stream)
    for i in range(steps):
        step(1 + warmup + i)
        evs[i + 1].record(stream)
    time.sleep(0.004)                              # the launches are asynchronous: let the sampler see the GPU under load
    if barrier:
        barrier()
    torch.cuda.synchronize()
    sampler.stop_flag = True
    per = sorted(evs[i].elapsed_time(evs[i + 1]) for i in range(steps))
    return {"total_ms": evs[0].elapsed_time(evs[-1]), "median_ms": per[len(per) // 2], "clocks": sampler.result()}


def roofline_obj(params, in_bytes, flops, bytes_per_elem, launch_us, clocks):
    """Per-shape roofline max(flops / P_bf16, bytes / B_HBM) (north_star) against the MEASURED peaks.  The tensor term
    takes the cuBLAS figure of the power state the timed region ran in (B200_PROFILING.md): K launches that stay at
    the boost clock are a burst measurement, a region that reached the power cap is compared with the sustained one."""
    hbm_peak, tf_burst, tf_sus, peak_src = measured_peaks()
    alg_bytes = params * bytes_per_elem + in_bytes
    gbs, tfs = alg_bytes / launch_us / 1e3, flops / launch_us / 1e6
    capped = "sw_power_cap" in clocks["reasons"] or bool(clocks["sm_mhz"] and clocks["sm_max_mhz"] and clocks["sm_mhz"] < 0.95 * clocks["sm_max_mhz"])
    tf_peak, tf_kind = (tf_sus, "sustained") if capped else (tf_burst, "burst")
    t_hbm, t_tc = alg_bytes / hbm_peak / 1e3, flops / tf_peak / 1e6
    if t_hbm >= t_tc:
        r = {"bound": "hbm", "achieved": gbs, "peak": hbm_peak, "unit": "GB/s", "frac": gbs / hbm_peak}
    else:
        r = {"bound": "tensor", "achieved": tfs, "peak": tf_peak, "unit": "TFLOP/s", "frac": tfs / tf_peak,
             "peak_kind": tf_kind, "burst_peak": tf_burst, "sustained_peak": tf_sus}
    r.update({"traffic": None, "peak_source": peak_src, "algorithmic_bytes_per_launch": alg_bytes, "flops_per_launch": flops,
              "roofline_us": max(t_hbm, t_tc), "hbm_term_us": t_hbm, "tensor_term_us": t_tc,
              "frac_of_max_term": max(t_hbm, t_tc) / launch_us, "launch_us_avg": launch_us, "gbs": gbs, "tflops": tfs,
              "frac_of_datasheet_8TBs": gbs / 8000.0, "frac_of_datasheet_2250TF": tfs / 2250.0})
    return r, flops / tf_sus / 1e6


def time_unfused_baselines(layer, hp, steps):
    """Context arms on the same GPU: cuBLAS dW then a separate optimizer pass.
    B3: fp32 dW (cuBLAS via torch.mm) + this library's elementwise kernel over the materialised G
        (byte-matched control, 28 B/element + the GEMM);
    B1: all-bf16 cuBLAS dW + torch._fused_adamw_ on bf16 W/m/v (the paper's "fused AdamW" arm)."""
    import torch
    from paper_2606_22932_b200 import binding as fb
    res = {}
    Gs = [torch.empty(d["W"].shape, dtype=torch.float32, device=d["W"].device) for d in layer]
    has_out_dtype = True
    try:
        torch.mm(layer[1]["dY"].t(), layer[1]["X"], out_dtype=torch.float32)
    except Exception:
        has_out_dtype = False

    def run_b3():
        for d, G in zip(layer, Gs):
            if has_out_dtype:
                torch.mm(d["dY"].t(), d["X"], out_dtype=torch.float32, out=G)
            else:   # bf16 cuBLAS output widened afterwards (torch build without out_dtype)
                G.copy_(torch.mm(d["dY"].t(), d["X"]))
            fb.forge_adamw_from_g(G, d["W"], d["m"], d["v"], 10, hp["lr"], hp["beta1"], hp["beta2"], hp["eps"], hp["wd"])

    def timeit(fn, n):
        for _ in range(2):
            fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(n):
            fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / n * 1e3

    if layer[0]["m"].dtype == torch.float32:
        res["cublas_dw_fp32_plus_elementwise_adamw_us"] = timeit(run_b3, steps)
        res["cublas_dw_out_dtype_fp32"] = has_out_dtype
    try:
        Wb = [d["W"].clone() for d in layer]
        mb = [torch.zeros_like(w) for w in Wb]
        vb = [torch.zeros_like(w) for w in Wb]
        st = [torch.tensor(9.0, device=w.device) for w in Wb]

        def run_b1():
            grads = [torch.mm(d["dY"].t(), d["X"]) for d in layer]
            torch._fused_adamw_(Wb, grads, mb, vb, [], st, lr=hp["lr"], beta1=hp["beta1"], beta2=hp["beta2"],
                                weight_decay=hp["wd"], eps=hp["eps"], amsgrad=False, maximize=False)
        res["cublas_dw_bf16_plus_torch_fused_adamw_bf16_us"] = timeit(run_b1, steps)
    except Exception as ex:  # pragma: no cover
        res["cublas_dw_bf16_plus_torch_fused_adamw_bf16_us"] = None
        res["b1_error"] = str(ex)[:200]
    return res


def backward_leg(layer, hpt, mdt, steps, stream, local):
    """forge_layer_backward_grouped (the hand-written tcgen05 dgrad of all 7 projections in one
    launch, then the fused launch) next to cuBLAS dgrad (torch.mm, 7 GEMMs) + the same fused call, on this box."""
    import torch
    from paper_2606_22932_b200 import binding as fb
    dXs = [torch.empty((d["X"].shape[0], d["W"].shape[1]), dtype=torch.bfloat16, device=d["W"].device) for d in layer]
    arr = fb.make_problem_array(layer)
    flops = sum(2.0 * d["X"].shape[0] * d["W"].shape[0] * d["W"].shape[1] for d in layer)

    def ours(t):
        fb.forge_layer_backward_grouped(layer, dXs, t, *hpt, mdt, stream=stream)

    def cublas(t):
        for d, dX in zip(layer, dXs):
            torch.mm(d["dY"], d["W"], out=dX)
        fb.forge_wgrad_adamw_grouped(layer, t, *hpt, mdt, stream=stream, _arr=arr)

    def cublas_dgrad_only(t):
        for d, dX in zip(layer, dXs):
            torch.mm(d["dY"], d["W"], out=dX)

    a = time_steps(ours, steps, 3, stream, local)
    sig = fb.lib().forge_last_kernel().decode()
    b = time_steps(cublas, steps, 3, stream, local)
    c = time_steps(cublas_dgrad_only, steps, 3, stream, local)
    f = time_steps(lambda t: fb.forge_wgrad_adamw_grouped(layer, t, *hpt, mdt, stream=stream, _arr=arr), steps, 3, stream, local)
    ours_us, fused_us = a["total_ms"] / steps * 1e3, f["total_ms"] / steps * 1e3
    dgrad_us = max(ours_us - fused_us, 1e-3)
    _, tf_burst, tf_sus, _ = measured_peaks()
    return {"value": ours_us, "unit": UNIT, "api": "forge_layer_backward_grouped: 1 dgrad launch (tcgen05, all 7 projections) + 1 fused launch",
            "fused_step_alone_us": fused_us, "dgrad_us_by_difference": dgrad_us, "dgrad_tflops": flops / dgrad_us / 1e6,
            "dgrad_frac_of_bf16_burst_peak": flops / dgrad_us / 1e6 / tf_burst, "dgrad_flops": flops,
            "cublas_dgrad_plus_fused_us": b["total_ms"] / steps * 1e3, "cublas_dgrad_alone_us": c["total_ms"] / steps * 1e3,
            "cublas_dgrad_tflops": flops / (c["total_ms"] / steps * 1e3) / 1e6, "last_kernel": sig, "clocks": a["clocks"]}


def model_leg(dev, tokens: int, steps: int, with_pool: bool):
    """BASELINE.json configs[4]: 32 layers + lm_head resident (75 GB of state), one optimizer step layer by
    layer in reverse order; total step time and peak device memory with and without a materialised dW pool."""
    import torch
    from paper_2606_22932_b200 import binding as fb
    from paper_2606_22932_b200 import stack, synth
    hp = synth.HP_DEFAULT
    free0, total = torch.cuda.mem_get_info()
    need = 7_504_658_432 * 10 + (3 << 30)
    if free0 < need:
        return {"skipped": f"configs[4] needs {need / 1e9:.1f} GB of free device memory, {free0 / 1e9:.1f} GB available"}
    st = stack.build_stack(dev, tokens=tokens)
    torch.cuda.synchronize()
    stream = torch.cuda.current_stream()
    local = dev.index or 0

    def timed(fn, n, warm):
        torch.cuda.reset_peak_memory_stats()
        r = time_steps(fn, n, warm, stream, local)
        return r["total_ms"] / n, torch.cuda.max_memory_allocated(), r["clocks"]

    n = max(1, min(steps, 5))
    launches0 = fb.forge_launch_count()
    fused_ms, fused_peak, clocks = timed(lambda t: stack.step_fused(st, t, hp, stream), n, 1)
    launches = (fb.forge_launch_count() - launches0) // (n + 1)
    alg_bytes = st.params * 20.0 + st.input_bytes
    hbm_peak, _, _, peak_src = measured_peaks()
    gbs = alg_bytes / (fused_ms * 1e-3) / 1e9
    out = {"value": fused_ms, "unit": "ms/step", "steps": n, "warmup": 1,
           "workload": "configs[4]: 32 x 7 projections + lm_head[128256,4096], bf16 W + fp32 m/v resident, reverse layer order",
           "params": st.params, "state_bytes": st.state_bytes, "input_bytes": st.input_bytes, "tokens": tokens,
           "roofline": {"bound": "hbm", "achieved": gbs, "peak": hbm_peak, "unit": "GB/s", "frac": gbs / hbm_peak, "traffic": None,
                        "peak_source": peak_src, "algorithmic_bytes_per_step": alg_bytes, "roofline_ms": alg_bytes / hbm_peak / 1e6},
           "gpu_launches_per_step": int(launches), "clocks": clocks,
           "peak_device_memory": {"fused_bytes": int(fused_peak), "dw_bytes_allocated_by_fused_path": 0,
                                  "device_total_bytes": int(total)}}
    if with_pool:
        pool = stack.alloc_dw_pool(st, dev)
        pool_bytes = sum(g.numel() * 4 for layer in pool for g in layer)
        pool_ms, pool_peak, _ = timed(lambda t: stack.step_dw_pool(st, pool, t, hp), max(1, n // 2), 1)
        out["peak_device_memory"].update({"dw_pool_arm_bytes": int(pool_peak), "dw_pool_bytes": int(pool_bytes)})
        out["dw_pool_arm"] = {"ms_per_step": pool_ms, "what": "cuBLAS fp32 dW for all layers into a 30 GB pool, then elementwise AdamW over the pool"}
        out["speedup_vs_dw_pool_arm"] = pool_ms / fused_ms
        del pool
    del st
    torch.cuda.empty_cache()
    return out


def run_model(args):
    import torch
    dev = torch.device("cuda", int(os.environ.get("LOCAL_RANK", "0")))
    torch.cuda.set_device(dev)
    r = model_leg(dev, args.tokens, args.steps, with_pool=True)
    if "skipped" in r:
        raise SystemExit(r["skipped"])
    line = {"metric": "full Llama-3.1-8B linear stack optimizer step, ms (32 layers + lm_head, BT=%d, 1xB200)" % args.tokens,
            "value": r["value"], "unit": "ms/step", "n_gpus": 1, "steps": r["steps"], "warmup": 1, "ms_per_step": r["value"],
            "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": r["workload"], "params": r["params"], "state_bytes": r["state_bytes"],
                       "input_bytes": r["input_bytes"], "tokens": args.tokens, "l2": "75 GB working set >> 126 MB L2"},
            "roofline": r["roofline"], "gpu_launches": r["gpu_launches_per_step"] * r["steps"], "clocks": r["clocks"],
            "peak_device_memory": r["peak_device_memory"], "dw_pool_arm": r.get("dw_pool_arm"),
            "speedup_vs_dw_pool_arm": r.get("speedup_vs_dw_pool_arm")}
    print(json.dumps(line), flush=True)


def config_leg(name, moments, workload, tokens, dev, steps, hpt, stream, local, tag):
    """One extra BASELINE.json configuration inside the default run: build, time K launches, free."""
    import torch
    from paper_2606_22932_b200 import binding as fb
    layer = make_device_layer(moments, SEED, dev, workload, tokens)
    arr = fb.make_problem_array(layer)
    mdt = MOMENT_ENUM[moments]
    r = time_steps(lambda t: fb.forge_wgrad_adamw_grouped(layer, t, *hpt, mdt, stream=stream, _arr=arr), steps, 3, stream, local)
    sig = fb.lib().forge_last_kernel().decode()
    us = r["total_ms"] / steps * 1e3
    params, in_bytes, flops = layer_counts(workload, tokens)
    roof, _ = roofline_obj(params, in_bytes, flops, MOMENT_BYTES[moments], us, r["clocks"])
    roof["traffic"], roof["traffic_source"] = ncu_traffic(sig, tag)
    del layer, arr
    torch.cuda.empty_cache()
    return {"config": name, "us": us, "launch_us_median": r["median_ms"] * 1e3, "steps": steps, "moments": moments,
            "workload": workload, "tokens": tokens, "kernel": sig, "roofline": roof, "clocks": r["clocks"]}


def run_cuda(args):
    if args.workload == "model":
        return run_model(args)
    import torch
    import torch.distributed as dist
    from paper_2606_22932_b200 import binding as fb
    from paper_2606_22932_b200 import shard, synth

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; there is no CPU fallback for the product path")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    fb.lib()                                       # fails loudly if the CUDA library is missing
    hp = synth.HP_DEFAULT
    mdt = MOMENT_ENUM[args.moments]
    sharded = args.shard == "rows" and world > 1
    # replicas: every rank its own layer (own seed); --shard rows: ONE layer (same seed everywhere), each rank keeps
    # its 128-aligned row range of every W / m / v and the matching column slice of dY (shard.py; Prop. 2(i))
    layer = make_device_layer(args.moments, SEED + (0 if sharded else rank), dev, args.workload, args.tokens)
    if sharded:
        if args.moments == "fp8":
            raise SystemExit("--shard rows: fp8 moments keep one scale per TENSOR; shard fp32 / bf16 / int8 state")
        full = layer
        layer = [s for s in (shard.shard_problem(d, world, rank) for d in full) if s is not None]
        layer = [{k: v for k, v in d.items() if k != "rows"} for d in layer]
    nst = fb.FAMILY_STATES.get(args.optimizer, 0)
    if args.optimizer == "storeg":
        if args.workload in ("layer", "model"):
            raise SystemExit("--optimizer storeg is the single-projection control: use --workload q|k|v|o|gate|up|down")
    elif args.optimizer != "adamw":                  # keep only the states the family has
        if args.moments in ("int8", "fp8"):
            raise SystemExit("int8 / fp8 state is implemented for AdamW only")
        for d in layer:
            v_like = d["v"]                        # non-negative: the single state of rmsprop / adagrad
            d["v"] = d["v"] if nst >= 2 else None
            d["m"] = (d["m"] if nst == 2 or args.optimizer in ("momentum", "lion") else v_like) if nst >= 1 else None
    arr = fb.make_problem_array(layer)
    hpt = (hp["lr"], hp["beta1"], hp["beta2"], hp["eps"], hp["wd"])
    stream = torch.cuda.current_stream()
    # --distinct-layers N: the timed loop rotates over N resident layers (distinct W, m, v, X, dY) instead of
    # re-stepping one, the footprint a real model presents (profiles/r01_summary.md, "Footprint")
    rot = [(layer, arr)]
    if args.distinct_layers > 1:
        if args.optimizer != "adamw" or sharded:
            raise SystemExit("--distinct-layers is implemented for --optimizer adamw, unsharded")
        for k in range(1, args.distinct_layers):
            lk = make_device_layer(args.moments, SEED + 1000 * k + rank, dev, args.workload, args.tokens)
            rot.append((lk, fb.make_problem_array(lk)))

    G_ctl = torch.empty(layer[0]["W"].shape, dtype=torch.float32, device=dev) if args.optimizer == "storeg" else None
    dp_plan = dp_pool = None
    if args.schedule == "bucket":                    # the data-parallel bucket-transient schedule
        if args.optimizer != "adamw" or args.moments == "fp8" or args.distinct_layers > 1 or sharded:
            raise SystemExit("--schedule bucket: AdamW with fp32 / bf16 / int8 moments, unsharded")
        from paper_2606_22932_b200 import dp
        dp_plan = dp.BucketPlan([tuple(d["W"].shape) for d in layer], args.bucket_mb << 20, slots=2)
        dp_pool = [torch.empty(dp_plan.slot_elems, dtype=torch.float32, device=dev) for _ in range(dp_plan.slots)]

    def step(t):
        if args.optimizer == "storeg":             # the paper's store-G control: same mainloop, G stored
            fb.forge_wgrad_store_g(layer[0]["X"], layer[0]["dY"], G_ctl, stream=stream)
        elif dp_plan is not None:                      # store-G into the rotating bucket, (all-reduce,) update from it
            dp.bucket_step_adamw(layer, t, hpt, dp_plan, dp_pool, group=dist.group.WORLD if world > 1 else None)
        elif args.optimizer == "adamw":
            lk, ak = rot[t % len(rot)]
            fb.forge_wgrad_adamw_grouped(lk, t, *hpt, mdt, stream=stream, _arr=ak)
        else:
            fb.forge_wgrad_step_grouped(layer, args.optimizer, t, hp["lr"], hp["beta1"], hp["beta2"], hp["eps"], hp["wd"],
                                        momentum=0.9, state_dtype=mdt, stream=stream, _arr=arr)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    launches0 = fb.forge_launch_count()
    r = time_steps(step, args.steps, args.warmup, stream, local, barrier)
    launches = fb.forge_launch_count() - launches0 - 0
    launches = launches * args.steps // (args.steps + args.warmup)
    signature = fb.lib().forge_last_kernel().decode()
    total_ms = shard.max_over_ranks(r["total_ms"], device=dev)
    ms_per_step = total_ms / args.steps
    layers_per_step = 1 if sharded else world          # shards: all ranks together step ONE layer
    us_per_layer = ms_per_step * 1e3 / layers_per_step

    params, in_bytes, flops = layer_counts(args.workload, args.tokens)
    if sharded:                                        # this rank's share of the launch (its rows; X whole, dY its columns)
        params = sum(d["W"].numel() for d in layer)
        flops = 2 * params * args.tokens
        xs = {d["X"].data_ptr(): d["X"].numel() for d in layer}
        in_bytes = 2 * (sum(xs.values()) + sum(d["dY"].shape[0] * d["dY"].shape[1] for d in layer))
    state_b = {"fp32": 8.0, "bf16": 4.0}.get(args.moments, 0.0)
    bpe = (MOMENT_BYTES[args.moments] if args.optimizer == "adamw" else
           (4.0 if args.optimizer == "storeg" else 4.0 + nst * state_b))          # store-G: 4 B/element of G out
    kernel_us = r["total_ms"] / args.steps * 1e3          # this rank's average launch duration
    clk = r["clocks"]
    roofline, t_tensor_sus_us = roofline_obj(params, in_bytes, flops, bpe, kernel_us, clk)
    roofline["launch_us_median"] = r["median_ms"] * 1e3
    is_headline = (args.workload == "layer" and args.tokens == T_TOKENS and args.optimizer == "adamw" and dp_plan is None
                   and not sharded)
    tag = args.moments if args.workload == "layer" else f"{args.workload}_{args.tokens}"
    if args.optimizer == "adamw" and dp_plan is None and not sharded and (args.workload == "layer" or args.moments == "fp32"):
        roofline["traffic"], roofline["traffic_source"] = ncu_traffic(signature, tag)
    roofline["kernel"] = signature

    line = {"metric": METRIC, "value": us_per_layer, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": False,
            "scaling": "strong" if sharded else "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": (("configs[1]: Llama-3.1-8B layer, 7 projections in one grouped launch, T=512"
                                     if args.moments == "fp32" else f"configs[2]: same layer, {args.moments} moments")
                                    if (is_headline or sharded) else f"configs[3]-style: {args.workload} of a Llama-3.1-8B layer, T={args.tokens}, "
                                    f"{args.optimizer} with {nst} {args.moments} state tensor(s)"),
                       "moments": args.moments, "params_per_layer": layer_counts(args.workload, args.tokens)[0], "tokens": args.tokens,
                       "distinct_layers": len(rot),
                       "schedule": ("fused" if dp_plan is None else
                                    f"dp bucket-transient: {len(dp_plan.buckets)} buckets, {dp_plan.transient_bytes >> 20} MiB of fp32 "
                                    f"gradient in flight, all-reduce over {world} rank(s)"),
                       "l2": "working set 4.4 GB/layer >> 126 MB L2, no flush needed",
                       "parallelism": (f"one layer row-sharded over {world} ranks (shard.py), no collective" if sharded
                                       else f"replicated layers x{world}, no collective")},
            "roofline": roofline, "gpu_launches": int(launches), "clocks": clk,
            "dw_bytes_allocated": 0 if dp_plan is None else dp_plan.transient_bytes,
            "library_workspace_bytes": fb.forge_workspace_bytes()}

    if rank == 0 and ((not args.no_extras and is_headline) or args.sustained):
        # ---- the same launch under SUSTAINED load: about 1.2 s of back-to-back launches, the last third timed.
        # The timed region above (K launches, tens of ms) runs at the boost clock; a training loop does not: after
        # ~0.1 s of continuous load the board reaches its power cap and the SM clock falls (profiles/r01_summary.md,
        # "Power state").  `value` stays the K-step figure the contract asks for; this is the long-run companion.
        def sustained_leg():
            n_sus = int(1.2e3 / max(ms_per_step, 1e-3)) + 1
            n_tail = n_sus // 3
            s_evs = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
            for i in range(n_sus - n_tail):
                step(1 + i)
            s_evs[0].record(stream)
            for i in range(n_tail):
                step(1 + i)
            s_evs[1].record(stream)
            while not s_evs[0].query():                # start sampling when the timed tail starts executing
                time.sleep(0.002)
            sus_sampler = ClockSampler(local)
            sus_sampler.start()
            torch.cuda.synchronize()
            sus_sampler.stop_flag = True
            sus_us = s_evs[0].elapsed_time(s_evs[1]) / n_tail * 1e3
            time.sleep(1.0)                            # let the power state recover before the next leg
            return {"value": sus_us, "unit": UNIT, "launches": n_sus, "timed": f"last {n_tail} launches",
                    "frac": max(roofline["hbm_term_us"], t_tensor_sus_us) / sus_us, "tensor_peak_kind": "sustained",
                    "ratio_to_boost": sus_us / kernel_us, "clocks": sus_sampler.result(),
                    "tuning": "sustained_clock" if fb.forge_get_tuning() == fb.TUNE_SUSTAINED_CLOCK else "boost_clock"}

        line["sustained"] = sustained_leg()
        if fb.forge_get_tuning() == fb.TUNE_BOOST_CLOCK and args.moments in ("fp32", "bf16") and args.optimizer == "adamw":
            # the same loop after forge_set_tuning(FORGE_TUNE_SUSTAINED_CLOCK): the instantiation meant for a board at
            # its power cap (bit-identical results; include/forge.h).  The headline `value` is the default tuning.
            fb.forge_set_tuning(fb.TUNE_SUSTAINED_CLOCK)
            try:
                for i in range(3):
                    step(1 + i)
                torch.cuda.synchronize()
                line["sustained_with_sustained_clock_tuning"] = sustained_leg()
                r2 = time_steps(step, args.steps, 3, stream, local)
                line["sustained_with_sustained_clock_tuning"]["boost_us"] = r2["total_ms"] / args.steps * 1e3
                line["sustained_with_sustained_clock_tuning"]["kernel"] = fb.lib().forge_last_kernel().decode()
            finally:
                fb.forge_set_tuning(fb.TUNE_BOOST_CLOCK)
    if rank == 0 and world == 1 and args.backward:
        line["layer_backward"] = backward_leg(layer, hpt, mdt, max(5, min(args.steps, 20)), stream, local)
    if rank == 0 and not args.no_extras and is_headline:
        # ---- end to end through the C ABI with HOST buffers (H2D + kernel + D2H inside the call)
        host = make_host_layer(args.moments, SEED)
        h2d = sum(sum(v.numel() * v.element_size() for v in d.values()) for d in host)
        d2h = sum(sum(d[k].numel() * d[k].element_size() for k in d if k not in ("X", "dY")) for d in host)
        host_arr = fb.make_problem_array(host)

        def e2e_step(tt):
            fb.forge_wgrad_adamw_grouped_host(host, tt, *hpt, mdt, _arr=host_arr)
        e2e_step(1)
        n_e2e = max(1, min(3, args.steps))
        t0 = time.perf_counter()
        for i in range(n_e2e):
            e2e_step(2 + i)
        torch.cuda.synchronize()
        e2e_us = (time.perf_counter() - t0) / n_e2e * 1e6
        line["e2e"] = {"value": e2e_us, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                       "steps": n_e2e, "api": "forge_wgrad_adamw_grouped_host, 7 problems pipelined over 3 streams (pinned host buffers)"}
        del host
        if world == 1:
            if not args.backward:
                line["layer_backward"] = backward_leg(layer, hpt, mdt, 10, stream, local)
            line["baselines_same_gpu"] = time_unfused_baselines(layer, hp, max(3, min(10, args.steps)))
            # ---- the other BASELINE.json configurations, timed on this box in this run
            del layer, arr, rot
            torch.cuda.empty_cache()
            k = max(10, min(args.steps, 20))
            cfgs = []
            for name, mom, wl, tok, tag2 in (("configs[2] bf16 moments", "bf16", "layer", 512, "bf16"),
                                             ("configs[2] int8 moments", "int8", "layer", 512, "int8"),
                                             ("fp8 moments (8(f) rank 1)", "fp8", "layer", 512, "fp8"),
                                             ("configs[3] gate T=512", "fp32", "gate", 512, "gate_512"),
                                             ("configs[3] gate T=2048", "fp32", "gate", 2048, "gate_2048"),
                                             ("configs[3] gate T=8192", "fp32", "gate", 8192, "gate_8192")):
                cfgs.append(config_leg(name, mom, wl, tok, dev, k, hpt, stream, local, tag2))
                time.sleep(0.3)
            m4 = model_leg(dev, T_TOKENS, 3, with_pool=False)
            m4["config"] = "configs[4] full stack"
            cfgs.append(m4)
            line["configs"] = cfgs
            line["cpu_baseline"] = cpu_baseline(SEED)
    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def _spawn_entry(rank: int, world: int, port: int, argv):
    os.environ.update({"RANK": str(rank), "LOCAL_RANK": str(rank), "WORLD_SIZE": str(world),
                       "MASTER_ADDR": "127.0.0.1", "MASTER_PORT": str(port)})
    sys.argv = argv
    main()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=30)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--moments", choices=["fp32", "bf16", "int8", "fp8"], default="fp32")
    ap.add_argument("--impl", choices=["cuda", "reference"], default="cuda")
    ap.add_argument("--workload", choices=["layer", "q", "k", "v", "o", "gate", "up", "down", "model"], default="layer",
                    help="layer = BASELINE.json configs[1] (the metric); a projection name = that problem alone (configs[3]); model = configs[4]")
    ap.add_argument("--optimizer", default="adamw", choices=["adamw", "sgd", "momentum", "lion", "rmsprop", "adagrad", "adamax", "nadam", "radam", "storeg"],
                    help="SURVEY.md 8(f) rank 1: the other coordinate-wise families on the same fused mainloop")
    ap.add_argument("--tokens", type=int, default=T_TOKENS, help="T (configs[3] sweeps 512/2048/8192 on gate)")
    ap.add_argument("--distinct-layers", type=int, default=1,
                    help="rotate the timed loop over N resident layers (default 1: the same layer re-stepped)")
    ap.add_argument("--schedule", choices=["fused", "bucket"], default="fused",
                    help="bucket = the data-parallel schedule of dp.py (gradient through a rotating fp32 bucket)")
    ap.add_argument("--bucket-mb", type=int, default=256)
    ap.add_argument("--shard", choices=["none", "rows"], default="none",
                    help="rows = N > 1 ranks split ONE layer's weight rows (strong scaling); none = one layer per rank (weak)")
    ap.add_argument("--backward", action="store_true", help="add the layer-backward leg (dgrad + fused step) with --no-extras / other modes")
    ap.add_argument("--sustained", action="store_true", help="add the sustained-load leg even with --no-extras / other workloads")
    ap.add_argument("--no-extras", action="store_true", help="skip e2e, same-GPU baselines, the extra configs and the CPU oracle leg")
    ap.add_argument("--tuning", choices=["boost", "sustained"], default="boost",
                    help="forge_set_tuning: which clock the launches are tuned for (bit-identical results; default boost)")
    ap.add_argument("--profiling-lib", action="store_true",
                    help="load libforge_b200_prof.so (the -DFORGE_PROFILING build: FORGE_CFG / FORGE_GRID / FORGE_ABLATE); profiles/ commands only")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3)
    if args.impl == "reference":
        return run_reference(args)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # no launcher: spawn the ranks here, one per GPU, NCCL's communicator lines (NCCL_DEBUG=INFO) to stderr
        import socket
        import torch
        if torch.cuda.device_count() < args.gpus:
            raise SystemExit(f"bench.py --gpus {args.gpus}: only {torch.cuda.device_count()} CUDA device(s) visible")
        os.environ.setdefault("NCCL_DEBUG", "INFO")
        os.environ.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
        os.environ.setdefault("NCCL_DEBUG_FILE", "/dev/stderr")
        with socket.socket() as s:
            s.bind(("127.0.0.1", 0))
            port = s.getsockname()[1]
        import torch.multiprocessing as mp
        mp.spawn(_spawn_entry, args=(args.gpus, port, list(sys.argv)), nprocs=args.gpus, join=True)
        return
    from paper_2606_22932_b200 import binding as fb
    if args.profiling_lib:
        fb.use_profiling_library(True)
    if args.tuning == "sustained":
        fb.forge_set_tuning(fb.TUNE_SUSTAINED_CLOCK)
    run_cuda(args)


if __name__ == "__main__":
    main()
