#!/usr/bin/env python
"""bench.py — throughput of the B200 hot path on BASELINE.json's workloads.

One "step" = one best_step_* call advancing ALL chains by `inner` sampler steps (ONE persistent kernel launch
on the bf16 path).  `value` = whole-job chain-steps/s with the state resident in HBM; `e2e` = the same metric
through the C-ABI with HOST buffers (best_state_set from pinned host memory, best_step_*, best_state_get to host
memory inside the timed region).

Default line = BASELINE configs[2]: HMC, 16 384 chains x L = 16 on 27->512^4->1, bf16 -- the largest single-GPU
configuration of the 512-wide net and the one north_star states its target on (">= 16k chains").  `extra`
carries the other configs (each with its own roofline fraction), trace-on throughput, best_logp_grad timed
directly, the configs[4] batch sweep with covariance adaptation (min / median over repeats, with the
non-adaptive time beside it) and the small-batch L2 figures.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload hmc|lcdm_mala|aies|...]
                  [--precision bf16|fp32] [--impl ours|reference]
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

# dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from the committed
# `ncu --set full` captures of THIS round's code (default line: profiles/r2c_ncu_full.md; the other three:
# profiles/r2d_ncu_full.md); None where no capture exists.
NCU_TRAFFIC_BYTES = {("hmc", "bf16"): 11.073280e6 + 126.469120e6,          # best_tc_kernel<2,256>, 8 trajectories per launch
                     ("lcdm_mala_16k", "bf16"): 17.137920e6 + 1362.267e6,    # best_tc_kernel<1,256>, 100 steps per launch
                     ("lcdm_mh_16k", "bf16"): 5.554176e6 + 0.0,              # best_tc_kernel<0,256>, 100 steps per launch
                     ("lcdm_mala", "bf16"): 5.254912e6 + 0.310272e6}         # best_tc_kernel<1,233>, 100 steps per launch
NCU_TRAFFIC_SOURCE = "profiles/r2c_ncu_full.md"

# PAPER.md Table 1 (L211-219), best published figure per sampler: sampler steps/s at 20 (1000) chains on a Tesla
# V100 with XLA JIT -- another machine, an emulator of unstated size: context, not a target
PAPER_TABLE1_GPU_JIT = {"mh": (8688, 2932), "mala": (3534, 1028), "hmc": (1856, 294), "aies": (8238, 2901)}

WORKLOADS = {
    # name: maker kwargs, method, sampler kwargs, inner = sampler steps per bench step, cfg = BASELINE configs index
    "hmc": dict(cfg=2, make="lcdm", n_chains=16384, mlp_scale=3.0, method="hmc", eps=0.1, n_leapfrog=16, inner=8),
    "lcdm_mala": dict(cfg=1, make="lcdm", n_chains=4096, mlp_scale=1.0, method="mala", eps=0.3, inner=100),
    "lcdm_mala_16k": dict(cfg=1, make="lcdm", n_chains=16384, mlp_scale=1.0, method="mala", eps=0.3, inner=100),
    "lcdm_mh_16k": dict(cfg=1, make="lcdm", n_chains=16384, mlp_scale=1.0, method="mh", eps=0.3, inner=100),
    "aies": dict(cfg=3, make="sterile", n_chains=32768, mlp_scale=1.0, method="aies", a=2.0, inner=10),
    "sterile_mala_16k": dict(cfg=4, make="sterile", n_chains=16384, mlp_scale=1.0, method="mala", eps=0.01, inner=20),
    "sterile_mh_16k": dict(cfg=4, make="sterile", n_chains=16384, mlp_scale=1.0, method="mh", eps=0.3, inner=20),
    "sterile_hmc_16k": dict(cfg=4, make="sterile", n_chains=16384, mlp_scale=1.0, method="hmc", eps=0.03, n_leapfrog=8, inner=4),
    "sterile_hmc_65k": dict(cfg=4, make="sterile", n_chains=65536, mlp_scale=1.0, method="hmc", eps=0.03, n_leapfrog=8, inner=4),
    "lcdm256_hmc": dict(cfg=2, make="lcdm", hidden=256, n_chains=16384, mlp_scale=3.0, method="hmc", eps=0.1, n_leapfrog=16, inner=8),
    # small-batch (latency / L2-bound) points of configs[4], for the ncu captures in profiles/
    "sterile_mala_1k": dict(cfg=4, make="sterile", n_chains=1024, mlp_scale=1.0, method="mala", eps=0.01, inner=100),
    "sterile_mala_64": dict(cfg=4, make="sterile", n_chains=64, mlp_scale=1.0, method="mala", eps=0.01, inner=100),
    "tiny_mala": dict(cfg=0, make="tiny", n_chains=64, mlp_scale=0.1, method="mala", eps=0.3, inner=100),
}
DEFAULT_WORKLOAD = "hmc"


def make_workload(spec, n_chains=None):
    from paper_2606_04895_b200 import workloads as WL
    n = n_chains or spec["n_chains"]
    if spec["make"] == "lcdm":
        return WL.lcdm(n_chains=n, mlp_scale=spec["mlp_scale"], hidden=spec.get("hidden", 512))
    if spec["make"] == "tiny":
        return WL.tiny(n_chains=n)
    if spec["make"] == "sterile":
        return WL.sterile(n_chains=n)
    raise KeyError(spec["make"])


def shard_workload(spec, rank, world):
    """Weak scaling: chains are independent, so every rank advances its OWN
    spec['n_chains'] chains of the same target with NO data-path collective.  Rank r's chains are the GLOBAL
    chains r*B .. r*B + B - 1: their θ₀ comes from seed 1000 + r and their Philox streams from chain offset r*B
    (best_state_set_chain_offset), so no two ranks share a stream.  Returns (workload, chain0)."""
    w = make_workload(spec)
    if world > 1:
        w = w.with_chains(spec["n_chains"], seed=1000 + rank)
    return w, rank * spec["n_chains"]


def max_over_ranks(value, world, device="cuda"):
    """device-timed milliseconds -> max over ranks (the slowest rank defines the step)"""
    if world <= 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def evals_per_chain_step(spec):
    return spec.get("n_leapfrog", 1) if spec["method"] == "hmc" else 1


def flops_per_chain_step(w, spec):
    per_eval = (4 if spec["method"] in ("mala", "hmc") else 2) * w.macs   # fwd 2·MACs, +bwd 2·MACs
    return per_eval * evals_per_chain_step(spec)


def run_steps(st, spec, n, seed, stream=0, trace=None, thin=0):
    m = spec["method"]
    if m == "mala":
        st.step_mala(n, seed, spec["eps"], trace=trace, thin=thin, stream=stream)
    elif m == "mh":
        st.step_mh(n, seed, spec["eps"], trace=trace, thin=thin, stream=stream)
    elif m == "hmc":
        st.step_hmc(n, seed, spec["eps"], spec["n_leapfrog"], trace=trace, thin=thin, stream=stream)
    elif m == "aies_de":
        st.step_aies_de(n, seed, spec.get("sigma_gamma", 0.1), trace=trace, thin=thin, stream=stream)
    else:
        st.step_aies(n, seed, spec.get("a", 2.0), trace=trace, thin=thin, stream=stream)


class ClockSampler(threading.Thread):
    """SM clocks / throttle reasons while the timed region runs (B200_PROFILING.md): NVML, else nvidia-smi."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.rows, self._stop_evt = index, [], threading.Event()

    def _nvml(self):
        """NVML handle for fast sampling (a query takes < 1 ms; an nvidia-smi process ~100 ms, longer than
        the whole timed region of a short run).  None when pynvml is not usable: nvidia-smi is then polled."""
        try:
            import pynvml
            pynvml.nvmlInit()
            return pynvml, pynvml.nvmlDeviceGetHandleByIndex(self.index)
        except Exception:
            return None

    def run(self):
        nv = self._nvml()
        while not self._stop_evt.is_set():
            try:
                if nv is not None:
                    nvml, h = nv
                    try:
                        rs = nvml.nvmlDeviceGetCurrentClocksEventReasons(h)
                    except Exception:
                        rs = nvml.nvmlDeviceGetCurrentClocksThrottleReasons(h)
                    bits = (nvml.nvmlClocksThrottleReasonHwSlowdown, nvml.nvmlClocksThrottleReasonHwThermalSlowdown,
                            nvml.nvmlClocksThrottleReasonSwThermalSlowdown, nvml.nvmlClocksThrottleReasonSwPowerCap)
                    self.rows.append([str(nvml.nvmlDeviceGetClockInfo(h, nvml.NVML_CLOCK_SM)),
                                      str(nvml.nvmlDeviceGetMaxClockInfo(h, nvml.NVML_CLOCK_SM))]
                                     + ["Active" if rs & b else "Not Active" for b in bits])
                    self._stop_evt.wait(0.005)
                    continue
                out = subprocess.run(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                      "-i", str(self.index)], capture_output=True, text=True, timeout=5).stdout
                self.rows.append([x.strip() for x in out.strip().split(",")])
            except Exception:
                nv = None
            self._stop_evt.wait(0.1)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=6)
        sm = [float(r[0]) for r in self.rows if len(r) >= 6 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) >= 6 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({names[i] for r in self.rows if len(r) >= 6 for i in range(4) if r[2 + i] == "Active"})
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm)}


def oracle_steps(ost, spec, n):
    m = spec["method"]
    eps = float(np.float32(spec.get("eps", 0.0)))
    if m == "mala":
        ost.step_mala(n, 1, eps)
    elif m == "mh":
        ost.step_mh(n, 1, eps)
    elif m == "hmc":
        ost.step_hmc(n, 1, eps, spec["n_leapfrog"])
    else:
        ost.step_aies(n, 1, spec.get("a", 2.0))


def cpu_baseline(spec, budget_s=12.0, n_sample=None):
    """The oracle as it stands (fp64 scalar loops, OpenMP over chains: a correctness checker, never tuned),
    timed on the host cores on a bounded sample of the same workload."""
    from oracle import oracle as O
    if n_sample is None:
        n_sample = 256 if spec["make"] != "tiny" else 64
    w = make_workload(spec, n_sample)
    ost = O.Oracle(w).new_state(w.theta0)
    steps_done, t0 = 0, time.perf_counter()
    chunk = 1 if spec["method"] == "hmc" else 2
    while True:
        oracle_steps(ost, spec, chunk)
        steps_done += chunk
        el = time.perf_counter() - t0
        if el > budget_s:
            break
    return {"value": n_sample * steps_done / el, "unit": "chain-steps/s", "cores": O.num_threads(),
            "kind": "oracle", "sample": f"{n_sample} chains x {steps_done} {spec['method']} steps "
                                        f"({el:.1f} s, OpenMP over chains, fp64 scalar loops; a checker, not a tuned CPU code)"}


def reference_arm(args, spec):
    """--impl reference: the oracle on the host cores; each step = a bounded sample of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import oracle as O
    n_sample = 64
    inner = 1
    w = make_workload(spec, n_sample)
    ost = O.Oracle(w).new_state(w.theta0)
    for _ in range(args.warmup):
        oracle_steps(ost, spec, inner)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle_steps(ost, spec, inner)
    el = time.perf_counter() - t0
    val = n_sample * inner * args.steps / el
    sample = f"{n_sample} chains x {inner} {spec['method']} step per bench step (oracle, fp64, {O.num_threads()} threads)"
    line = {"impl": "reference", "metric": "chain-steps/s", "value": val, "unit": "chain-steps/s",
            "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * el / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": args.workload, "sample": sample},
            "cpu_baseline": {"value": val, "unit": "chain-steps/s", "cores": O.num_threads(), "kind": "oracle",
                             "sample": sample},
            "e2e": {"value": val, "unit": "chain-steps/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default=DEFAULT_WORKLOAD, choices=sorted(WORKLOADS))
    ap.add_argument("--precision", default="bf16", choices=["bf16", "fp32", "fp32tc"])
    ap.add_argument("--inner", type=int, default=0, help="sampler steps per bench step (0 = workload default)")
    ap.add_argument("--chains", type=int, default=0, help="override the number of chains per GPU")
    ap.add_argument("--trace", action="store_true", help="write the trace (thin = 1) inside the timed region")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extra", action="store_true")
    args = ap.parse_args()
    spec = dict(WORKLOADS[args.workload])
    if args.inner:
        spec["inner"] = args.inner
    if args.chains:
        spec["n_chains"] = args.chains
    if args.impl == "reference":
        reference_arm(args, spec)
        return

    import torch
    import __graft_entry__ as entry
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if rank == 0:
        entry.build()
    torch.cuda.set_device(local_rank)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
        dist.barrier()
    from paper_2606_04895_b200 import binding as B
    B.lib()
    prec = {"bf16": B.PREC_BF16, "fp32": B.PREC_FP32, "fp32tc": B.PREC_FP32_TC}[args.precision]

    def barrier():
        if world > 1:
            torch.distributed.barrier()
        torch.cuda.synchronize()

    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda")   # > 126 MB L2

    def measure(spec, steps, warmup, with_e2e=False, prec=prec, adapt_every=0, trace=False, clocks=False, exchange=None):
        """Times `steps` bench steps (CUDA events on the launching stream, L2 flushed before each, max over ranks).
        Returns dict(ms_total, ms_list (this rank), launches, clocks, accept_rate, e2e...)."""
        w, chain0 = shard_workload(spec, rank, world)
        ctx = B.Context(w, prec)
        st = ctx.new_state(w.theta0)
        st.set_chain_offset(chain0)
        if adapt_every:
            st.set_adaptation(adapt_every, 1e-6)
        if exchange:                                   # (kind, all-gather callback): SURVEY 8(e) exchange at world size 1
            if exchange[0] == "adapt":
                st.set_adaptation_exchange(exchange[1], 1)
            else:
                st.set_aies_exchange(exchange[1], 0, 1)
        stream = torch.cuda.current_stream().cuda_stream
        inner = spec["inner"]
        tr = torch.empty(inner, w.n_chains, w.d, device="cuda") if trace else None
        thin = 1 if trace else 0
        for i in range(warmup):
            run_steps(st, spec, inner, 7, stream, tr, thin)
        barrier()
        ck = None
        if clocks:
            ck = ClockSampler(local_rank)
            ck.start()
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        l0 = B.launch_count()
        for i in range(steps):
            flush.fill_(i & 0xFF)                      # L2 flush between timed iterations (untimed)
            ev[i][0].record()
            run_steps(st, spec, inner, 7, stream, tr, thin)
            ev[i][1].record()
        barrier()
        launches = B.launch_count() - l0
        ckr = ck.stop() if ck is not None else None
        ms_list = [a.elapsed_time(b) for a, b in ev]
        dev_ms = max_over_ranks(sum(ms_list), world)
        acc = st.get(want_grad=False)
        res = dict(w=w, ms_total=dev_ms, ms_list=ms_list, launches=int(launches), clocks=ckr,
                   accept_rate=float(acc["n_accept"].mean() / max(acc["step"], 1)))
        if with_e2e:
            host_theta = torch.from_numpy(w.theta0).pin_memory()
            out_theta = np.zeros_like(w.theta0)
            out_logp = np.zeros(w.n_chains, np.float32)
            lib = B.lib()
            n_e2e = max(10, steps)

            def e2e_once():
                st.set(host_theta, step=0)                       # H2D of θ (+ logp/grad refresh on device)
                run_steps(st, spec, inner, 7, stream)
                rc = lib.best_state_get(st._h, out_theta.ctypes.data, out_logp.ctypes.data, None, None, None,
                                        None, None)              # D2H of θ, logp (synchronises)
                assert rc == 0
            e2e_once()
            barrier()
            t0 = time.perf_counter()
            for _ in range(n_e2e):
                e2e_once()
            barrier()
            el = time.perf_counter() - t0
            res["e2e_s_per_step"] = max_over_ranks(el, world) / n_e2e
            res["h2d"] = int(w.theta0.nbytes)
            res["d2h"] = int(out_theta.nbytes + out_logp.nbytes)
        st.close()
        ctx.close()
        return res

    peaks = {}
    pk_path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(pk_path):
        peaks = json.load(open(pk_path))
    peak_tf = peaks.get("bf16_tflops", 1590.0)
    peak_src = "MEASURED_PEAKS.json bf16_tflops (burst), of measured" if peaks else "1590 TF fallback, of fallback"
    fp32_peak_tf = 148 * 128 * 2 * 1.965e9 / 1e12

    def summarize(sp, rr, n):
        """throughput figures of a measure() result over n bench steps"""
        ms = rr["ms_total"] / n
        v = sp["n_chains"] * world * sp["inner"] / (ms * 1e-3)
        tf = flops_per_chain_step(rr["w"], sp) * v / 1e12
        return {"chain_steps_per_s": v, "grad_evals_per_s": v * evals_per_chain_step(sp), "tflops": tf,
                "frac_of_peak": tf / peak_tf, "ms_per_step": ms, "ms_min": min(rr["ms_list"]),
                "ms_median": float(np.median(rr["ms_list"])), "accept_rate": rr["accept_rate"], "inner": sp["inner"],
                "gpu_launches": rr["launches"], "n_chains": sp["n_chains"]}

    r = measure(spec, args.steps, args.warmup, with_e2e=True, trace=args.trace, clocks=True)
    w = r["w"]
    Btot = spec["n_chains"] * world
    inner = spec["inner"]
    ms_per_step = r["ms_total"] / args.steps
    value = Btot * inner / (ms_per_step * 1e-3)
    flops_per_launch = flops_per_chain_step(w, spec) * spec["n_chains"] * inner
    launches_per_step = max(1, r["launches"] // max(args.steps, 1))
    achieved_tf = flops_per_launch / (ms_per_step * 1e-3) / 1e12
    this_peak, this_src = (peak_tf, peak_src) if args.precision == "bf16" else \
        (fp32_peak_tf, "FP32 FFMA peak 148 SM x 128 lanes x 2 x 1.965 GHz (derived)")
    is_default_size = spec["n_chains"] == WORKLOADS[args.workload]["n_chains"] and inner == WORKLOADS[args.workload]["inner"]
    line = {
        "metric": "chain-steps/s", "value": value, "unit": "chain-steps/s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": args.precision, "data": "synthetic",
        "config": {"workload": f"{args.workload} (BASELINE configs[{spec['cfg']}]): d={w.d}, MLP "
                               + "x".join(map(str, w.widths)) + f", {spec['n_chains']} chains/GPU, {spec['method']}",
                   "sampler_steps_per_step": inner, "method": spec["method"],
                   "n_leapfrog": spec.get("n_leapfrog"), "eps": spec.get("eps"), "trace": bool(args.trace),
                   "l2": "flushed (256 MB write) between timed iterations", "precision": args.precision,
                   "unit_note": "HMC: one chain-step = one trajectory of n_leapfrog gradient evaluations"},
        "grad_evals_per_s": value * evals_per_chain_step(spec),
        "accept_rate": r["accept_rate"],
        "clocks": r["clocks"],
        "gpu_launches": r["launches"],
        "e2e": {"value": Btot * inner / r["e2e_s_per_step"], "unit": "chain-steps/s",
                "h2d_bytes_per_step": r["h2d"], "d2h_bytes_per_step": r["d2h"]},
        "roofline": {"bound": "tensor" if args.precision == "bf16" else "alu", "achieved": achieved_tf,
                     "peak": this_peak, "unit": "TFLOP/s", "frac": achieved_tf / this_peak,
                     "traffic": NCU_TRAFFIC_BYTES.get((args.workload, args.precision)) if is_default_size else None,
                     "traffic_unit": "bytes per launch (ncu dram read+write, %s)" % (NCU_TRAFFIC_SOURCE if args.workload == DEFAULT_WORKLOAD else "profiles/r2d_ncu_full.md"),
                     "peak_source": this_src,
                     "frac_of_sustained": (achieved_tf / peaks["bf16_tflops_sustained"]) if peaks and args.precision == "bf16" else None,
                     "kernel": "best_tc_kernel<%s>" % spec["method"], "flops_per_launch": flops_per_launch,
                     "kernel_launches_per_step": launches_per_step, "ms_min": min(r["ms_list"]),
                     "ms_median": float(np.median(r["ms_list"]))},
        "paper_context": {"table1_gpu_jit_steps_per_s_at_20_and_1000_chains": PAPER_TABLE1_GPU_JIT.get(spec["method"]),
                          "hardware": "Tesla V100, XLA JIT, emulator size and precision not stated (PAPER.md L211-219)"},
    }
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(spec)
        line["cpu_baseline"]["note"] = "GPU/CPU ratio is against the scalar fp64 oracle, a correctness checker"
    if world == 1 and not args.no_extra and args.workload == DEFAULT_WORKLOAD:
        extra = {}
        n_x = max(5, args.steps // 4)
        # the other configs, each with its own fraction of the measured peak
        for name in ("lcdm_mala", "lcdm_mala_16k", "lcdm_mh_16k", "aies", "sterile_mala_16k", "sterile_hmc_65k", "hmc_fp32",
                     "hmc_fp32tc"):
            sp = dict(WORKLOADS[name.replace("_fp32tc", "").replace("_fp32", "")])
            if name.endswith("_fp32"):      # exact path: one trajectory per bench step
                sp["inner"] = 1
                rr = measure(sp, n_x, 3, prec=B.PREC_FP32)
                extra[name] = summarize(sp, rr, n_x)
                extra[name]["frac_of_peak"] = extra[name]["tflops"] / fp32_peak_tf
                extra[name]["peak"] = "FP32 FFMA 74.5 TFLOP/s (derived)"
            elif name.endswith("_fp32tc"):  # exact path with split-operand tensor-core GEMMs (3 fp16 MMAs per product)
                sp["inner"] = 1
                rr = measure(sp, n_x, 3, prec=B.PREC_FP32_TC)
                extra[name] = summarize(sp, rr, n_x)
                extra[name]["frac_of_peak"] = extra[name]["tflops"] / (peak_tf / 3.0)
                extra[name]["peak"] = "measured bf16 peak / 3 (three fp16 MMAs per product; fp16 and bf16 share the pipe rate)"
            else:
                rr = measure(sp, n_x, 3)
                extra[name] = summarize(sp, rr, n_x)
        # trace on (thin = 1: every post-accept state written by the kernel) next to trace off
        tr_on = {}
        for name in ("hmc", "lcdm_mala_16k", "lcdm_mh_16k"):
            sp = dict(WORKLOADS[name])
            off = summarize(sp, measure(sp, n_x, 3), n_x) if name != "hmc" else None
            on = summarize(sp, measure(sp, n_x, 3, trace=True), n_x)
            base = off["chain_steps_per_s"] if off else value
            tr_on[name] = {"trace_on_chain_steps_per_s": on["chain_steps_per_s"], "trace_off_chain_steps_per_s": base,
                           "ratio": on["chain_steps_per_s"] / base,
                           "trace_bytes_per_chain_step": 4 * make_workload(sp, 8).d}
        extra["trace_on"] = tr_on
        # best_logp_grad timed directly (BASELINE metric "emulator logp+grad evals/s"): device buffers in and out
        lg = {}
        for make, net in (("lcdm", "27x512^4x1"), ("sterile", "29x1024^4x1")):
            for npts in (16384, 65536, 262144):   # one wave of CTAs walks all tiles (Run::n_tiles): 1 / 3.5 / 14 passes
                sp = dict(make=make, mlp_scale=1.0, n_chains=npts)
                ww = make_workload(sp)
                ctx = B.Context(ww, B.PREC_BF16)
                th = torch.from_numpy(ww.theta0).cuda()
                lp = torch.empty(npts, device="cuda")
                g = torch.empty(npts, ww.d, device="cuda")
                stream = torch.cuda.current_stream().cuda_stream
                for want_grad in (False, True):
                    ms = []
                    for i in range(3 + 7):
                        flush.fill_(i)
                        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                        e0.record()
                        ctx.logp_grad(th, npts, lp, g if want_grad else None, stream=stream)
                        e1.record()
                        torch.cuda.synchronize()
                        if i >= 3:
                            ms.append(e0.elapsed_time(e1))
                    med = float(np.median(ms))
                    fl = (4 if want_grad else 2) * ww.macs * npts
                    lg[f"{make}_{npts}_{'fwd_grad' if want_grad else 'fwd'}"] = {
                        "net": net, "evals_per_s": npts / (med * 1e-3), "ms_median": med, "ms_min": min(ms),
                        "tflops": fl / (med * 1e-3) / 1e12, "frac_of_peak": fl / (med * 1e-3) / 1e12 / peak_tf}
                ctx.close()
        extra["logp_grad"] = lg
        # BASELINE configs[4]: chain-steps/s vs batch size on the 29->1024^4->1 banana target with the running
        # covariance -> Cholesky update every 500 steps on device; 5 timed repeats per point (min / median), the
        # same point without adaptation beside it
        sweep = {}
        for meth, kw in (("mh", dict(eps=0.3)), ("mala", dict(eps=0.01)), ("hmc", dict(eps=0.03, n_leapfrog=8))):
            for nb in (1, 64, 1024, 16384, 65536):
                n_steps = 500 if not (meth == "hmc" and nb > 16384) else 100
                sp = dict(cfg=4, make="sterile", n_chains=nb, mlp_scale=1.0, method=meth, inner=n_steps, **kw)
                ra = measure(sp, 5, 1, adapt_every=500)
                rn = measure(sp, 3, 1)
                med = float(np.median(ra["ms_list"]))
                v = nb * n_steps / (med * 1e-3)
                sweep[f"{meth}_{nb}"] = {"chain_steps_per_s": v, "ms_per_sampler_step": med / n_steps,
                                         "ms_per_sampler_step_min": min(ra["ms_list"]) / n_steps,
                                         "ms_per_sampler_step_no_adapt": float(np.median(rn["ms_list"])) / n_steps,
                                         "adapt_overhead": med / float(np.median(rn["ms_list"])) - 1.0,
                                         "tflops": flops_per_chain_step(ra["w"], sp) * v / 1e12,
                                         "accept_rate": ra["accept_rate"], "sampler_steps": n_steps, "repeats": 5,
                                         "gpu_launches_per_call": ra["launches"] // 5}
        # the oracle beside the curve (north_star: "a chain-steps/s vs batch-size curve reported against the
        # oracle"): B = 1 and 64 chains in full for ~1.5 s each, and 256 chains for MH / MALA -- OpenMP over
        # chains saturates the host cores well before that, so the 256-chain figure also stands for 1k..65k
        if not args.no_cpu_baseline:
            orc = {}
            for meth, kw, nbs in (("mh", dict(eps=0.3), (1, 64, 256)), ("mala", dict(eps=0.01), (1, 64, 256)),
                                  ("hmc", dict(eps=0.03, n_leapfrog=8), (1, 64))):
                for nb in nbs:
                    sp = dict(cfg=4, make="sterile", n_chains=nb, mlp_scale=1.0, method=meth, **kw)
                    cb = cpu_baseline(sp, budget_s=1.5, n_sample=nb)
                    orc[f"{meth}_{nb}"] = {"chain_steps_per_s": cb["value"], "sample": cb["sample"]}
            orc["cores"] = cb["cores"]
            sweep["oracle"] = orc
        extra["sweep_adapt500"] = sweep
        # Small-batch path: every tile streams the forward and the backward weight pack from L2
        # once per evaluation: algorithmic bytes = tiles x 2|W| per MALA step, |W| = 2 B x MACs (bf16, unpadded).
        # Denominator: best_probe_l2_read (148 CTAs re-reading a 32 MiB buffer that stays in the 126 MB L2).
        l2_gbs = max(B.probe_l2_read(32 << 20, 20) for _ in range(3))
        small = {"l2_resident_read_GB_per_s": l2_gbs, "hbm_copy_GB_per_s": peaks.get("hbm_gbs")}
        macs = make_workload(dict(make="sterile", mlp_scale=1.0, n_chains=8)).macs
        for nb in (1, 64, 1024):
            k = sweep[f"mala_{nb}"]
            per_tile = 64 if nb <= 4736 else 128      # geometry 232 (32 chains per CTA of a pair) while it fits one wave
            tiles = (nb + per_tile - 1) // per_tile
            by = tiles * 2 * 2 * macs
            gbs = by / (k["ms_per_sampler_step_no_adapt"] * 1e-3) / 1e9
            small[f"mala_{nb}"] = {"tiles": tiles, "weight_bytes_per_step": by,
                                   "ms_per_sampler_step": k["ms_per_sampler_step_no_adapt"],
                                   "achieved_l2_GB_per_s": gbs, "frac_of_l2_read": gbs / l2_gbs}
        extra["small_batch"] = small
        # SURVEY 8(e) exchanges (best_set_adaptation_exchange, best_set_aies_exchange) with the all-gather of
        # distributed.py over a real NCCL group of ONE rank (all one GPU allows): what pack + NCCL call + combine /
        # unpack add to a covariance window and to an ensemble half-step -- latency, there is nothing to transfer
        try:
            import socket
            import torch.distributed as dist
            from paper_2606_04895_b200 import distributed as D
            with socket.socket() as sk:
                sk.bind(("127.0.0.1", 0))
                port = sk.getsockname()[1]
            dist.init_process_group("nccl", init_method=f"tcp://127.0.0.1:{port}", rank=0, world_size=1,
                                    device_id=torch.device("cuda", local_rank))
            try:
                fn = D.allgather_exchange()
                xo = {}
                sp = dict(cfg=4, make="sterile", n_chains=16384, mlp_scale=1.0, method="mh", inner=500, eps=0.3)
                a = float(np.median(measure(sp, 3, 1, adapt_every=500)["ms_list"]))
                b = float(np.median(measure(sp, 3, 1, adapt_every=500, exchange=("adapt", fn))["ms_list"]))
                xo["adapt_window_mh_16k"] = {"ms_per_500_step_window": a, "ms_with_exchange": b,
                                             "added_us_per_window": 1e3 * (b - a)}
                sp = dict(WORKLOADS["aies"])
                a = float(np.median(measure(sp, n_x, 3)["ms_list"])) / sp["inner"]
                b = float(np.median(measure(sp, n_x, 3, exchange=("aies", fn))["ms_list"])) / sp["inner"]
                xo["aies_32k"] = {"ms_per_sampler_step": a, "ms_with_exchange": b,
                                  "added_us_per_half_step": 1e3 * (b - a) / 2,
                                  "bytes_gathered_per_half_step": 8 * (make_workload(sp, 8).d + 1) * sp["n_chains"] // 2}
                extra["exchange_world1"] = xo
            finally:
                dist.destroy_process_group()
        except Exception as e:                          # noqa: BLE001  (NCCL not usable on this box: say so, go on)
            extra["exchange_world1"] = {"error": str(e)[:200]}
        # DE move on the AIES config, the burn-in loop on configs[1], R - 1 of a trace
        sp = dict(WORKLOADS["aies"], method="aies_de", sigma_gamma=0.1)
        extra["aies_de"] = summarize(sp, measure(sp, n_x, 3), n_x)
        sp1 = WORKLOADS["lcdm_mala"]
        w1 = make_workload(sp1)
        w1.L = np.diag(np.sqrt(np.diag(w1.Sigma)))
        ctx = B.Context(w1, prec)
        st = ctx.new_state(w1.theta0)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        eps, _, _, hist = st.burn_in("mala", 3, 600, 200, 10, 7, 0.05, 0.574)
        torch.cuda.synchronize()
        el = time.perf_counter() - t0
        tr = torch.zeros(500, w1.n_chains, w1.d, device="cuda")
        a0 = st.get(want_grad=False)["n_accept"].sum()
        st.step_mala(500, 7, eps, trace=tr, thin=1)
        torch.cuda.synchronize()
        acc = float((st.get(want_grad=False)["n_accept"].sum() - a0) / (500 * w1.n_chains))
        B.rminus1(tr)
        t_r = 1e9
        for _ in range(5):                       # best of 5 (host timer around a synchronising call)
            t0 = time.perf_counter()
            r1 = B.rminus1(tr)
            t_r = min(t_r, time.perf_counter() - t0)
        extra["burn_in"] = {"config": "configs[1] from a diagonal whitening: 3 iterations x 600 MALA steps, "
                                      "200 of them adapting the step in blocks of 10, target acceptance 0.574",
                            "wall_s": el, "chain_steps_per_s": 3 * 600 * w1.n_chains / el, "eps": eps,
                            "adaptation_blocks": int(len(hist)), "accept_rate_after": acc}
        extra["rminus1"] = {"trace": [500, int(w1.n_chains), int(w1.d)], "value": r1, "ms": 1e3 * t_r,
                            "GB_per_s": tr.numel() * 4 / t_r / 1e9}
        st.close()
        ctx.close()
        line["extra"] = extra
    if rank == 0:
        print(json.dumps(line))
    if world > 1:
        torch.distributed.destroy_process_group()


if __name__ == "__main__":
    main()
