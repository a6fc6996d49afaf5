#!/usr/bin/env python
"""bench.py — measures BASELINE.json's metric on the SLP MoE layer.

A "step" is one pass of the whole hot path (router, permute, quantise, expert-weight streaming
overlapped with the grouped FP8 GEMMs, shared expert, combine) over one batch of synthetic tokens.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload NAME] [--impl ours|reference]
                  [--parallelism token|smallep]

Workloads (BASELINE.json configs): cfg1_streamed (default: the configuration the metric is quoted on,
T = 4096, DeepSeek-V3 shape, weights streamed from pinned host memory), cfg2_streamed / cfg2_resident
(T = 32768 single pass), cfg3_streamed, cfg4_streamed / cfg4_resident, cfg5_k2_streamed (384 experts),
cfg0_resident.  Prints ONE JSON line (rank 0).  The default run also carries, under their own keys, the
rest of BASELINE's metric: the resident 32K-token call (mean, min and a sustained soak, against the
nominal, the measured-bf16-derived and the on-box measured FP8 peaks), the streamed 32K single pass and
the 8 x 4096 chunked pass.

Multi-GPU: `--gpus N` without a torchrun environment starts N ranks itself (torch.distributed.run on
127.0.0.1), one per GPU, each bound to the CPUs of its GPU's NUMA node.
  --parallelism token    every rank runs its own T tokens through its own replica, no data-path
                         collective ("scaling": "weak"); SURVEY.md 8(e) option 1.
  --parallelism smallep  the paper's SmallEP: all-gather the hidden states, every
                         rank routes all tokens and streams / runs only its E / N experts, reduce-scatter
                         of the fp32 partial sums ("scaling": "strong": T tokens in total).
`--dry-run` replaces the GPU work by fixed per-rank numbers and uses gloo, so the rank plumbing (launch,
rendezvous, max-over-ranks reduction, rank-0 JSON) is covered by a CPU test.
"""

import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

WORKLOADS = {
    "cfg0_resident": (0, "resident"),
    "cfg1_streamed": (1, "streamed"),
    "cfg1_resident": (1, "resident"),
    "cfg2_streamed": (2, "streamed"),
    "cfg2_resident": (2, "resident"),
    "cfg3_streamed": (3, "streamed"),
    "cfg4_streamed": (4, "streamed"),
    "cfg4_resident": (4, "resident"),
    "cfg5_k2_streamed": (5, "streamed"),
    "cfg5_k2_resident": (5, "resident"),
}
METRIC = "prefill tok/s per MoE layer (host-streamed FP8); resident FP8 TFLOP/s vs peak"
# dram__bytes_read.sum + dram__bytes_write.sum of ONE gemm_tc_kernel<0> launch from the committed
# `ncu --set full` captures (profiles/r2_layer_ncu.md: the whole resident 32K layer in one launch;
# profiles/r2_streamed_gemm_ncu.md: one 64-expert group of the streamed T = 4096 layer); None = not captured.
NCU_TRAFFIC_BYTES = {"cfg2_resident": 10.55e9, "cfg1_streamed": 2.136e9}
FP8_NOMINAL_TFLOPS = 4500.0


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        p = json.load(open(path))
        return dict(hbm_gbs=p["hbm_gbs"], bf16_tflops=p["bf16_tflops"],
                    bf16_tflops_sustained=p.get("bf16_tflops_sustained", p["bf16_tflops"]), source="measured")
    return dict(hbm_gbs=6650.0, bf16_tflops=1590.0, bf16_tflops_sustained=1400.0, source="fallback")


class ClockSampler:
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, device):
        self.device = device
        self.tmp = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.device), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"], stdout=self.tmp,
                                         stderr=subprocess.DEVNULL)
        except OSError:
            self.proc = None

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        self.tmp.flush()
        rows = [r.strip().split(", ") for r in open(self.tmp.name) if r.strip()]
        os.unlink(self.tmp.name)
        sm, mx, reasons = [], [], set()
        for r in rows:
            try:
                sm.append(float(r[1]))
                mx.append(float(r[2]))
            except (ValueError, IndexError):
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[5:9]):
                if v.strip().lower() == "active":
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


# --------------------------------------------------------------------------------------------------
# multi-GPU launch: one process per GPU, NUMA-local host memory
# --------------------------------------------------------------------------------------------------
def relaunch_under_torchrun(args, argv):
    """`python bench.py --gpus N` outside a torchrun environment: start N ranks on this node."""
    port = 29500 + (os.getpid() % 2000)
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + argv
    env = dict(os.environ)
    env.setdefault("NCCL_DEBUG", "WARN")   # keep the communicator log on (ranks / transport visible to the driver)
    return subprocess.call(cmd, env=env)


def bind_to_gpu_numa_node(local_rank, dry_run=False):
    """Pin this rank's CPU affinity (and with it the first-touch placement of its pinned weight copy) to the
    NUMA node of its GPU.  Best effort: returns a description for the JSON line."""
    try:
        if dry_run:
            return "dry-run: not bound"
        import torch
        bus = torch.cuda.get_device_properties(local_rank).pci_bus_id if hasattr(torch.cuda.get_device_properties(local_rank), "pci_bus_id") else None
        if bus is None:
            out = subprocess.run(["nvidia-smi", "-i", str(local_rank), "--query-gpu=pci.bus_id", "--format=csv,noheader"],
                                 capture_output=True, text=True, timeout=10).stdout.strip()
            bus = out[-12:].lower() if out else None     # 00000000:1B:00.0 -> 0000:1b:00.0
        node_path = f"/sys/bus/pci/devices/{bus}/numa_node" if bus else None
        node = int(open(node_path).read()) if node_path and os.path.exists(node_path) else -1
        if node < 0:
            return "numa node unknown: not bound"
        cpus = []
        for part in open(f"/sys/devices/system/node/node{node}/cpulist").read().strip().split(","):
            lo, _, hi = part.partition("-")
            cpus.extend(range(int(lo), int(hi or lo) + 1))
        allowed = sorted(set(cpus) & os.sched_getaffinity(0))
        if allowed:
            os.sched_setaffinity(0, allowed)
            return f"gpu {local_rank} -> numa node {node} ({len(allowed)} cpus)"
        return f"numa node {node} has no allowed cpu: not bound"
    except Exception as ex:  # never fail the bench over placement
        return f"not bound ({type(ex).__name__})"


# --------------------------------------------------------------------------------------------------
# CPU baseline = the oracle as it stands, on a bounded sample
# --------------------------------------------------------------------------------------------------
def cpu_oracle_sample(cfg, W_np, hidden_bits, n_experts_sample, n_shared_tokens):
    """Times the oracle, as it stands, on a bounded sample of the workload and EXTRAPOLATES to the whole
    layer: full routing + quantisation for all T tokens (timed as is), the expert FFNs of the first
    `n_experts_sample` routed experts over ALL their rows (scaled by E / sample), and the shared expert
    over `n_shared_tokens` rows (scaled by T / n)."""
    import numpy as np
    from oracle import router, quantize_rows_1x128, expert_ffn
    t0 = time.perf_counter()
    route = router(hidden_bits, W_np["router_w"], W_np.get("router_bias"), top_k=cfg.k, n_group=cfg.G,
                   topk_group=cfg.Gk, scoring=cfg.scoring, norm_topk=cfg.norm_topk, routed_scale=cfg.routed_scale)
    x32 = (hidden_bits.astype(np.uint32) << 16).view(np.float32)
    xq, xs = quantize_rows_1x128(x32)
    t_route = time.perf_counter() - t0
    t0 = time.perf_counter()
    rows_done = 0
    for e in range(n_experts_sample):
        rows = np.nonzero((route["idx"] == e).any(axis=1))[0]
        if len(rows) == 0:
            continue
        expert_ffn(xq[rows], xs[rows], W_np["gate_q"][e], W_np["gate_s"][e], W_np["up_q"][e], W_np["up_s"][e],
                   W_np["down_q"][e], W_np["down_s"][e])
        rows_done += len(rows)
    t_exp = time.perf_counter() - t0
    t_sh = 0.0
    if cfg.n_shared:
        t0 = time.perf_counter()
        expert_ffn(xq[:n_shared_tokens], xs[:n_shared_tokens], W_np["shared_gate_q"], W_np["shared_gate_s"],
                   W_np["shared_up_q"], W_np["shared_up_s"], W_np["shared_down_q"], W_np["shared_down_s"])
        t_sh = time.perf_counter() - t0
    T = hidden_bits.shape[0]
    est = t_route + t_exp * (cfg.E / n_experts_sample) + t_sh * (T / max(1, n_shared_tokens))
    sample = (f"ESTIMATED by extrapolation from a bounded sample of the float64 numpy oracle: router+quantise all {T} tokens "
              f"({t_route:.2f}s), FFN of routed experts 0..{n_experts_sample - 1} of {cfg.E} over all their {rows_done} rows "
              f"({t_exp:.2f}s, scaled x{cfg.E / n_experts_sample:.0f}), shared expert on {n_shared_tokens} rows ({t_sh:.2f}s, "
              f"scaled x{T / max(1, n_shared_tokens):.0f})")
    return T / est, sample, t_route + t_exp + t_sh, rows_done + (n_shared_tokens if cfg.n_shared else 0)


def cpu_oracle_full(cfg, W_np, hidden_bits):
    """One timed pass of oracle.moe_layer, as it stands, over ALL T tokens and all experts of the workload
    ("the timed number comes from a full-T run").  Returns tokens/s and the seconds it took."""
    from oracle import moe_layer
    t0 = time.perf_counter()
    moe_layer(hidden_bits, W_np, top_k=cfg.k, n_group=cfg.G, topk_group=cfg.Gk, scoring=cfg.scoring,
              norm_topk=cfg.norm_topk, routed_scale=cfg.routed_scale)
    dt = time.perf_counter() - t0
    return hidden_bits.shape[0] / dt, dt


def torch_h2d_gbs(dev, nbytes=1 << 30, repeats=10):
    """Pinned host -> device copy rate measured WITHOUT the library: one torch pinned tensor, Tensor.copy_ on the
    current stream, CUDA events, best of `repeats`.  An independent check of slp_measure_h2d's figure."""
    import torch
    try:
        src = torch.empty(nbytes, dtype=torch.uint8).pin_memory()
        src.fill_(1)
        dst = torch.empty(nbytes, dtype=torch.uint8, device=dev)
        best = 0.0
        for i in range(repeats + 1):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            dst.copy_(src, non_blocking=True)
            e1.record()
            torch.cuda.synchronize()
            if i > 0:
                best = max(best, nbytes / (e0.elapsed_time(e1) * 1e-3) / 1e9)
        return best
    except Exception as ex:  # report, never hide
        return {"error": repr(ex)}


def measure_fp8_dense_peak(dev, sustained_seconds=3.0):
    """On-box FP8 dense GEMM yardstick (cuBLASLt through torch._scaled_mm, 8192^3, e4m3 x e4m3 -> bf16, per-tensor
    scales): best of 10 (burst) and back to back for `sustained_seconds`.  A yardstick for the resident
    fractions only; it is not on the hot path."""
    import torch
    n = 8192
    try:
        a = (torch.randn(n, n, device=dev) * 0.5).to(torch.float8_e4m3fn)
        b = (torch.randn(n, n, device=dev) * 0.5).to(torch.float8_e4m3fn).t()     # column-major second operand
        one = torch.ones((), device=dev, dtype=torch.float32)
        f = lambda: torch._scaled_mm(a, b, scale_a=one, scale_b=one, out_dtype=torch.bfloat16)
        for _ in range(3):
            f()
        torch.cuda.synchronize()
        best = 0.0
        for _ in range(10):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            f()
            e1.record()
            torch.cuda.synchronize()
            best = max(best, 2.0 * n ** 3 / (e0.elapsed_time(e1) * 1e-3) / 1e12)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        reps, t0 = 0, time.perf_counter()
        e0.record()
        while time.perf_counter() - t0 < sustained_seconds:
            for _ in range(50):
                f()
            reps += 50
            torch.cuda.synchronize()
        e1.record()
        torch.cuda.synchronize()
        sustained = 2.0 * n ** 3 * reps / (e0.elapsed_time(e1) * 1e-3) / 1e12
        return {"burst_tflops": best, "sustained_tflops": sustained, "how": f"torch._scaled_mm {n}^3 e4m3 x e4m3 -> bf16, best of 10 / {reps} back to back"}
    except Exception as ex:  # report, never hide
        return {"error": repr(ex)}


def stack_main(args, local_rank):
    """--workload cfg1_stack / cfg2_stack: a multi-layer stack of DeepSeek-V3-shaped layers on one GPU, streamed through ONE
    ring of expert slots shared by the layers (Fig. 5; slp_moe_stack_*).  A step = one layer call;
    K steps walk the layers round-robin back to back on one stream, so every call finds the loader already running
    ahead with its experts.  Reports steady-state ms per layer against the host link, what was prefetched, and the
    implied whole-model figure (context only)."""
    import dataclasses
    import torch
    import __graft_entry__ as entry
    entry.build()
    from paper_2606_10493_b200 import SlpMoeLayer, inputs, measure_h2d_gbs
    n_layers = args.stack_layers
    cfg = inputs.CONFIGS[1 if args.workload == "cfg1_stack" else 2]
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    numa = bind_to_gpu_numa_node(local_rank)
    t0 = time.perf_counter()
    Ws = [inputs.make_weights(dataclasses.replace(cfg, seed=cfg.seed + 100 * l), device=dev, pin=True) for l in range(n_layers)]
    hidden = inputs.make_hidden(cfg, device=dev)
    t_gen = time.perf_counter() - t0
    h2d_peak = max(measure_h2d_gbs(local_rank, cfg.I * cfg.H, 1 << 30, 5), measure_h2d_gbs(local_rank, 256 << 20, 1 << 30, 5))
    stack = SlpMoeLayer(cfg, Ws, device=local_rank, staging_slots=args.staging_slots, experts_per_launch=args.experts_per_launch)
    out = torch.empty_like(hidden)
    per_layer_bytes = cfg.E * 3 * cfg.I * cfg.H
    try:
        for i in range(max(args.warmup, n_layers)):          # at least one full walk, so the steady state is reached
            stack.prefill(hidden, out, layer=i % n_layers)
        torch.cuda.synchronize()
        first = max(args.warmup, n_layers)
        sampler = ClockSampler(local_rank)
        sampler.start()
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
        stats = []
        ev[0].record()
        for i in range(args.steps):
            stack.prefill(hidden, out, layer=(first + i) % n_layers)
            ev[i + 1].record()                                # no stats() here: it waits for the call and would serialise the walk
        # The window opens with one layer already loaded (the warm-up's last call prefetched it) and every call enqueues the
        # next layer's copies, so it has to close when the LAST call's prefetch has landed too: then exactly K weight
        # passes crossed the link inside it.  Closing at the last call's compute would count K - 1 passes as K.
        torch.cuda.synchronize()                              # all streams of the device, the library's copy stream included
        ev_end = torch.cuda.Event(enable_timing=True)
        ev_end.record()
        torch.cuda.synchronize()
        stats.append(stack.stats())                           # the last call of the back-to-back walk
        clocks = sampler.stop()
        per_call = [ev[i].elapsed_time(ev[i + 1]) for i in range(args.steps)]
        ms = ev[0].elapsed_time(ev_end) / args.steps
        iso = []                                              # same walk with a device synchronise between calls
        for i in range(n_layers):
            stack.prefill(hidden, out, layer=(first + args.steps + i) % n_layers)
            torch.cuda.synchronize()
            iso.append(stack.stats())
    finally:
        stack.close()
    gbs = per_layer_bytes / (ms * 1e-3) / 1e9
    line = {"metric": METRIC, "value": cfg.T / (ms * 1e-3), "unit": "tokens/s", "n_gpus": 1, "steps": args.steps, "warmup": max(args.warmup, n_layers),
            "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "e4m3 x e4m3 -> f32",
            "data": "synthetic", "clocks": clocks, "e2e": None,
            "gpu_launches": int(statistics.mean(s["kernel_launches"] for s in stats + iso)),
            "config": {"workload": args.workload, "config": cfg.name, "T": cfg.T, "layers": n_layers, "mode": "streamed, one ring shared by the layers",
                       "pinned_host_gb": n_layers * per_layer_bytes / 1e9, "numa": numa, "l2": "inputs_exceed_l2",
                       "step": "one layer call; layers walked round-robin back to back on one stream"},
            "link_roofline": {"bound": "host_link", "bytes_per_step": per_layer_bytes, "peak": h2d_peak, "unit": "GB/s",
                              "achieved_whole_step": gbs, "frac": gbs / h2d_peak},
            "per_call_ms": {"first": per_call[0], "steady_mean": statistics.mean(per_call[1:]) if len(per_call) > 1 else None,
                            "steady_min": min(per_call[1:]) if len(per_call) > 1 else None, "steady_max": max(per_call[1:]) if len(per_call) > 1 else None,
                            "note": "call-to-call CUDA events on the caller's stream; the first timed call finds its layer loaded by the warm-up, "
                                    "every later one waits for the pass its predecessor started"},
            "prefetch": {"experts_from_prefetch_per_call": statistics.mean(s["experts_from_prefetch"] for s in stats + iso),
                         "experts_copied_by_the_call_itself": statistics.mean(s["experts_copied"] for s in stats + iso),
                         "bytes_prefetched_per_call": statistics.mean(s["bytes_prefetched"] for s in stats + iso),
                         "note": "counters of the last back-to-back call and of the isolated walk"},
            "isolated_call": {"ms_total": [s["ms_total"] for s in iso], "ms_route": [s["ms_route"] for s in iso],
                              "ms_experts": [s["ms_experts"] for s in iso], "ms_combine": [s["ms_combine"] for s in iso],
                              "note": "device synchronise between calls: the next layer's copies have been running since the previous call was "
                                      "enqueued, so an isolated call is SHORTER than a weight pass"},
            "whole_model_context": {"layers": 58, "tokens_per_s": cfg.T / (58 * ms * 1e-3),
                                    "note": "58 MoE layers at this per-layer time, MoE layers only (no attention); the paper reports "
                                            "1,200 tok/s for the whole model on its own hardware (context, not a comparison)"},
            "gen_seconds": t_gen}
    print(json.dumps(line))
    return 0


def dry_run_main(args, rank, world):
    """CPU-only rank plumbing: gloo rendezvous, the same reductions, rank-0 JSON (no GPU work, fixed numbers)."""
    import torch.distributed as dist
    from paper_2606_10493_b200 import inputs, sharding
    cfg = inputs.CONFIGS[WORKLOADS[args.workload][0]]
    if world > 1:
        dist.init_process_group("gloo")
    ms_rank = 100.0 + 10.0 * rank                       # the slowest rank decides
    tokens_rank = cfg.T if args.parallelism == "token" else sharding.token_range(cfg.T, rank, world)[1] - sharding.token_range(cfg.T, rank, world)[0]
    value, ms = sharding.whole_job_tokens_per_s(tokens_rank, ms_rank, device="cpu")
    if rank == 0:
        print(json.dumps({"metric": METRIC, "value": value, "unit": "tokens/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                          "ms_per_step": ms, "higher_is_better": True, "scaling": "weak" if args.parallelism == "token" else "strong",
                          "vs_baseline": None, "dtype": "none (dry run)", "data": "none (dry run)", "dry_run": True,
                          "config": {"workload": args.workload, "parallelism": f"{args.parallelism} x{world}"}}))
    if world > 1 or par == "smallep":
        dist.destroy_process_group()
    return 0


def main(argv=None):
    argv = sys.argv[1:] if argv is None else argv
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="cfg1_streamed", choices=sorted(WORKLOADS) + ["cfg1_stack", "cfg2_stack"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--parallelism", default="token", choices=["token", "smallep"])
    ap.add_argument("--dry-run", action="store_true", help="CPU-only rank plumbing check (gloo), no GPU work")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extras", action="store_true", help="skip the resident / 32K / soak / fp8-peak extras of the default run")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer leg (profiling runs)")
    ap.add_argument("--cpu-baseline-sample", action="store_true", help="cpu_baseline from the bounded, extrapolated sample only (skips the timed full oracle pass)")
    ap.add_argument("--triage", default=None, help="triage spec (slp_moe_debug_set_triage) for A/B runs (e.g. gemm=pair); not a product option")
    ap.add_argument("--stack-layers", type=int, default=3, help="layers of the cfg1_stack / cfg2_stack workloads")
    ap.add_argument("--staging-slots", type=int, default=0)
    ap.add_argument("--experts-per-launch", type=int, default=0)
    args = ap.parse_args(argv)

    if args.gpus > 1 and "WORLD_SIZE" not in os.environ and args.impl == "ours":
        return relaunch_under_torchrun(args, argv)

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.dry_run:
        return dry_run_main(args, rank, world)
    if args.workload in ("cfg1_stack", "cfg2_stack"):
        if world != 1 or args.impl != "ours":
            print(json.dumps({"error": "the stack workloads run on one GPU, our arm only"}))
            return 2
        return stack_main(args, local_rank)

    import numpy as np
    import torch
    from paper_2606_10493_b200 import inputs

    cfg_id, mode = WORKLOADS[args.workload]
    cfg = inputs.CONFIGS[cfg_id]
    ncores = len(os.sched_getaffinity(0))
    par = args.parallelism   # smallep with one GPU: a one-rank NCCL group, so the collective calls run (as copies) and are timed
    config = {"workload": args.workload, "config": cfg.name, "T": cfg.T, "hidden": cfg.H, "n_experts": cfg.E,
              "top_k": cfg.k, "n_group": cfg.G, "topk_group": cfg.Gk, "moe_intermediate": cfg.I,
              "n_shared": cfg.n_shared, "mode": mode,
              "parallelism": (f"token-sharded x{world} (no collective)" if par == "token" else
                              f"smallep x{world} (all-gather hidden, expert-sharded streaming, reduce-scatter fp32 partials)"),
              "l2": "inputs_exceed_l2" if cfg_id >= 1 else "tiny (launch-latency regime)",
              "aggregate": "mean over the timed steps (min reported separately where given)"}

    # ------------------------------------------------------------------ reference arm = oracle
    if args.impl == "reference":
        if rank != 0:
            return 0
        torch.set_num_threads(ncores)
        n_exp = 2 if cfg.E >= 64 else cfg.E
        dev = "cuda" if torch.cuda.is_available() else "cpu"
        affinity0 = os.sched_getaffinity(0)
        numa = bind_to_gpu_numa_node(local_rank) if dev == "cuda" else "no gpu: not bound"   # the same key our arm's config carries
        os.sched_setaffinity(0, affinity0)
        W = inputs.make_weights(cfg, device=dev, experts=range(n_exp))
        W_np = inputs.weights_as_numpy(W)
        hb = inputs.hidden_as_bits(inputs.make_hidden(cfg, device=dev))
        # Each step is a BOUNDED SAMPLE of the workload (a full float64 pass takes over a minute, K of them would not end
        # within minutes): the FFNs of the first n_exp routed experts over all their rows, the shared expert over 128 rows,
        # and the router + hidden quantisation of as many tokens as those FFN rows amount to (rows / (k + n_shared)), so
        # every stage is sampled at the same fraction of the layer.  Which rows the sampled experts own comes from one
        # untimed routing of the whole prompt (set-up).  Reported as measured: ms_per_step is the wall time of one step,
        # `value` the step's token-equivalents per second.  Nothing is extrapolated to a time that was not spent.
        import numpy as np
        from oracle import router, quantize_rows_1x128, expert_ffn
        rkw = dict(top_k=cfg.k, n_group=cfg.G, topk_group=cfg.Gk, scoring=cfg.scoring, norm_topk=cfg.norm_topk, routed_scale=cfg.routed_scale)
        route = router(hb, W_np["router_w"], W_np.get("router_bias"), **rkw)
        xq, xs = quantize_rows_1x128((hb.astype(np.uint32) << 16).view(np.float32))
        rows_of = [np.nonzero((route["idx"] == e).any(axis=1))[0] for e in range(n_exp)]
        n_sh = min(cfg.T, 128) if cfg.n_shared else 0
        rows = sum(len(r) for r in rows_of) + n_sh
        n_tok = max(1, round(rows / (cfg.k + cfg.n_shared)))
        secs, toks = [], []
        for i in range(args.warmup + args.steps):
            t0 = time.perf_counter()
            router(hb[:n_tok], W_np["router_w"], W_np.get("router_bias"), **rkw)
            quantize_rows_1x128((hb[:n_tok].astype(np.uint32) << 16).view(np.float32))
            for e, r in enumerate(rows_of):
                if len(r):
                    expert_ffn(xq[r], xs[r], W_np["gate_q"][e], W_np["gate_s"][e], W_np["up_q"][e], W_np["up_s"][e], W_np["down_q"][e], W_np["down_s"][e])
            if n_sh:
                expert_ffn(xq[:n_sh], xs[:n_sh], W_np["shared_gate_q"], W_np["shared_gate_s"], W_np["shared_up_q"], W_np["shared_up_s"],
                           W_np["shared_down_q"], W_np["shared_down_s"])
            dt = time.perf_counter() - t0
            if i >= args.warmup:
                secs.append(dt)
                toks.append(rows / (cfg.k + cfg.n_shared))
        ms_step = 1e3 * statistics.mean(secs)
        tok_step = statistics.mean(toks)
        v = tok_step / (ms_step * 1e-3)
        sample = (f"measured, not extrapolated: each step = FFN of routed experts 0..{n_exp - 1} of {cfg.E} over all their rows + shared expert on "
                  f"{n_sh} rows ({rows} FFN rows = {tok_step:.1f} token-equivalents at k + n_shared = {cfg.k + cfg.n_shared} rows per token) + router and "
                  f"hidden quantisation of {n_tok} tokens, in {ms_step:.0f} ms")
        config["numa"] = numa
        print(json.dumps({"metric": METRIC, "value": v, "unit": "tokens/s", "n_gpus": args.gpus, "steps": args.steps,
                          "warmup": args.warmup, "ms_per_step": ms_step, "tokens_per_step": tok_step, "higher_is_better": True,
                          "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic", "impl": "reference",
                          "config": config,
                          "cpu_baseline": {"value": v, "unit": "tokens/s", "cores": ncores, "kind": "oracle", "estimated": False, "sample": sample},
                          "e2e": {"value": v, "unit": "tokens/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))
        return 0

    # ------------------------------------------------------------------ our arm
    import __graft_entry__ as entry
    entry.build()
    from paper_2606_10493_b200 import SlpMoeLayer, measure_h2d_gbs, sharding, query_plan

    assert torch.cuda.is_available(), "bench.py needs a CUDA device (there is no CPU path)"
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    # Bind to the GPU's NUMA node BEFORE any pinned allocation (first touch decides where the weight copy lives); a single
    # rank first measures the pinned-copy rate unbound, so the line can show both.  The affinity is widened again for the
    # CPU baseline at the end (the oracle uses every core the process started with).
    affinity0 = os.sched_getaffinity(0)
    h2d_peak_unbound = measure_h2d_gbs(local_rank, 256 << 20, 1 << 30, 5) if (world == 1 and mode == "streamed") else None
    config["numa"] = bind_to_gpu_numa_node(local_rank)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
    elif par == "smallep":
        import socket
        import torch.distributed as dist
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
        dist.init_process_group("nccl", init_method=f"tcp://127.0.0.1:{port}", rank=0, world_size=1, device_id=dev)
    peaks = load_peaks()
    stream = torch.cuda.current_stream()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    # ---- inputs and the layer (token mode: a full replica per rank; smallep: this rank's expert range only) ----
    t_gen = time.perf_counter()
    if par == "smallep":
        from paper_2606_10493_b200 import smallep
        e0, e1 = smallep.expert_range(cfg.E, rank, world)
        W = inputs.make_weights(cfg, device=dev, pin=True, experts=range(e0, e1))
        t0, t1 = sharding.token_range(cfg.T, rank, world)
        hidden = inputs.make_hidden(cfg, device=dev)[t0:t1].contiguous()        # this rank's token shard of the SAME prompt
        layer = SlpMoeLayer(cfg, W, device=local_rank, staging_slots=args.staging_slots, experts_per_launch=args.experts_per_launch,
                            expert_range=(e0, e1), triage=args.triage)
        runner = smallep.SmallEpLayer(layer, cfg, rank, world, always_collective=True)
        tokens_this_rank = t1 - t0
    else:
        W = inputs.make_weights(cfg, device=dev, pin=True)
        hidden = inputs.make_hidden(cfg, device=dev, first_chunk=sharding.weak_scaling_first_chunk(cfg.T, rank))  # each rank its own tokens
        layer = SlpMoeLayer(cfg, W, device=local_rank, staging_slots=args.staging_slots,
                            experts_per_launch=args.experts_per_launch, triage=args.triage)
        runner = None
        tokens_this_rank = cfg.T
    t_gen = time.perf_counter() - t_gen
    layer.set_residency(mode)
    out = torch.empty_like(hidden)

    def step(lyr=None, h=None, o=None):
        if runner is not None and lyr is None:
            runner.prefill(hidden, out)
        else:
            (lyr or layer).prefill(hidden if h is None else h, out if o is None else o)

    def timed_steps(n_steps, sampler=None, **kw):
        """W warm-up steps, then exactly n_steps back to back on one stream (no host sync inside the timed
        region), bracketed by barrier + synchronize; returns mean ms per step on this rank."""
        for _ in range(args.warmup):
            step(**kw)
        barrier()
        if sampler:
            sampler.start()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record(stream)
        for _ in range(n_steps):
            step(**kw)
        ev1.record(stream)
        barrier()
        clocks = sampler.stop() if sampler else None
        return ev0.elapsed_time(ev1) / n_steps, clocks

    def isolated_calls(n, lyr=None, **kw):
        """n calls with a device synchronise between them: per-call latency without cross-call copy prefetch;
        returns the list of the library's per-call stats."""
        stats = []
        for _ in range(n):
            step(lyr=lyr, **kw)
            torch.cuda.synchronize()
            stats.append((lyr or layer).stats())
        return stats

    # host-link peak of this box: the better of per-matrix chunks and 256 MiB chunks (the engine merges
    # consecutive experts into one copy when the host layout allows, profiles/r1_h2d_chunks.md)
    h2d_peak = max(measure_h2d_gbs(local_rank, cfg.I * cfg.H, 1 << 30, 5),
                   measure_h2d_gbs(local_rank, 256 << 20, 1 << 30, 5)) if mode == "streamed" else None
    h2d_peak_torch = torch_h2d_gbs(dev) if (mode == "streamed" and rank == 0) else None
    ms_rank, clocks = timed_steps(args.steps, ClockSampler(local_rank))
    value, ms = sharding.whole_job_tokens_per_s(tokens_this_rank, ms_rank, device=dev)   # all ranks' tokens / slowest rank's device time
    iso = isolated_calls(max(3, min(10, args.steps)))
    mean = lambda key, ss=None: statistics.mean(s[key] for s in (ss or iso))

    # ---- kernel-level numbers from the library's own CUDA events on the launching stream ----
    st = iso[-1]
    n_pairs = max(1, st["timed_gemm_pairs"])
    idx, _, counts = layer.debug_routing(hidden.shape[0] if par == "token" else cfg.T)
    own = slice(*(layer.expert_range or (0, cfg.E)))
    rows_routed = int(counts[own].sum())
    rows_total = rows_routed + (tokens_this_rank if cfg.n_shared else 0)
    n_exp_run = int((counts[own] > 0).sum()) + cfg.n_shared
    flops_call = inputs.fp8_flops_per_token(cfg) * cfg.T
    # gate/up kernel: algorithmic bytes = weights (2*I*H per expert run) + A rows + hq written + scales
    gu_bytes = n_exp_run * 2 * cfg.I * cfg.H + rows_total * (cfg.H + cfg.I) + rows_total * 4 * (cfg.H // 128 + cfg.I // 128)
    gu_flops = 2.0 * 2 * cfg.I * cfg.H * rows_total
    gu_time = mean("ms_gateup_sum") * 1e-3
    # Streamed mode launches the (resident) shared expert apart from the routed groups: T rows against ONE expert is a
    # tensor-bound launch however HBM-bound the routed groups are, so the roofline of the dominant kernel is taken over
    # the routed launches and the shared-expert launch is reported beside it.
    shared_launch = None
    sh_time = mean("ms_gateup_shared") * 1e-3
    if sh_time > 0 and cfg.n_shared and rows_routed > 0:
        sh_rows = rows_total - rows_routed
        sh_bytes = 2 * cfg.I * cfg.H + sh_rows * (cfg.H + cfg.I) + sh_rows * 4 * (cfg.H // 128 + cfg.I // 128)
        sh_flops = 2.0 * 2 * cfg.I * cfg.H * sh_rows
        shared_launch = {"kernel": "gemm_tc_kernel<0>, the shared expert's own launch", "rows": sh_rows, "ms": sh_time * 1e3,
                         "tflops": sh_flops / sh_time / 1e12, "gbs": sh_bytes / sh_time / 1e9}
        gu_bytes -= sh_bytes
        gu_flops -= sh_flops
        gu_time -= sh_time
        rows_total, n_exp_run, n_pairs = rows_routed, n_exp_run - 1, max(1, n_pairs - 1)
    fp8_peak = 2.0 * (peaks["bf16_tflops"] if mode == "resident" else peaks["bf16_tflops_sustained"])
    ridge_rows = fp8_peak * 1e12 / (peaks["hbm_gbs"] * 1e9) / 2.0   # rows/expert where 2*M flop/B crosses the ridge
    tensor_bound = (rows_total / max(1, n_exp_run)) >= ridge_rows
    if tensor_bound:
        roofline = {"kernel": "gemm_tc_kernel<0> (gate/up + SwiGLU + requant)", "bound": "tensor",
                    "achieved": gu_flops / gu_time / 1e12, "peak": fp8_peak, "unit": "TFLOP/s",
                    "peak_source": f"2 x bf16 {peaks['source']} ({'burst' if mode == 'resident' else 'sustained'}), fp8:bf16 nominal ratio"}
    else:
        roofline = {"kernel": "gemm_tc_kernel<0> (gate/up + SwiGLU + requant)", "bound": "hbm",
                    "achieved": gu_bytes / gu_time / 1e9, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                    "peak_source": f"hbm copy {peaks['source']}"}
    roofline["frac"] = roofline["achieved"] / roofline["peak"]
    roofline["traffic"] = NCU_TRAFFIC_BYTES.get(args.workload)
    roofline["traffic_source"] = "constant from the committed ncu --set full capture of one launch (profiles/), not measured in this run"
    # the ncu capture is of ONE launch: the whole layer in resident mode, one group of experts_per_launch
    # routed experts in streamed mode; the algorithmic bytes of that same launch, for comparison
    epl = query_plan(cfg, staging_slots=args.staging_slots, experts_per_launch=args.experts_per_launch)["experts_per_launch"]
    roofline["traffic_launch_algorithmic_bytes"] = gu_bytes if mode == "resident" else gu_bytes * min(epl, cfg.E) / max(1, n_exp_run)
    roofline["algorithmic_bytes_per_launch"] = gu_bytes / n_pairs
    roofline["algorithmic_flops_per_launch"] = gu_flops / n_pairs
    roofline["ms_per_launch"] = gu_time * 1e3 / n_pairs
    roofline["launches_per_step"] = n_pairs
    roofline["down_ms_per_launch"] = (mean("ms_down_sum") - (mean("ms_down_shared") if shared_launch else 0.0)) / n_pairs
    roofline["sm_mhz_during_kernel"] = mean("sm_mhz_gateup")
    roofline["down_sm_mhz_during_kernel"] = mean("sm_mhz_down")
    roofline["aggregate"] = f"mean over {len(iso)} isolated calls"
    if shared_launch:
        roofline["launches"] = "routed-expert launches only (the shared expert's own, tensor-bound launch is under shared_expert_launch)"
        roofline["shared_expert_launch"] = shared_launch

    stage_keys = ("ms_total", "ms_route", "ms_experts", "ms_combine", "ms_copy_span", "ms_gateup_sum", "ms_down_sum")
    extra = {"tflops_per_call": flops_call * (world if par == "token" else 1) / (ms * 1e-3) / 1e12,
             "fp8_peak_nominal_tflops": FP8_NOMINAL_TFLOPS,
             "frac_of_nominal_fp8": flops_call * (world if par == "token" else 1) / (ms * 1e-3) / (FP8_NOMINAL_TFLOPS * 1e12) / world,
             "stage_ms": {k: mean(k) for k in stage_keys},
             "isolated_call": {"ms_mean": mean("ms_total"), "ms_min": min(s["ms_total"] for s in iso), "calls": len(iso),
                               "note": "device synchronise between calls: no cross-call copy prefetch (include/slp_moe.h, slp_moe_prefill)"},
             "gen_seconds": t_gen}
    if mode == "streamed":
        link_gbs = statistics.mean(s["bytes_copied"] / (s["ms_copy_span"] * 1e-3) / 1e9 for s in iso if s["ms_copy_span"] > 0)
        step_gbs = st["bytes_copied"] / (ms_rank * 1e-3) / 1e9
        extra["link_roofline"] = {"bound": "host_link", "bytes_per_step": st["bytes_copied"], "peak": h2d_peak, "unit": "GB/s",
                                  "achieved_copy_span": link_gbs, "achieved_whole_step": step_gbs,
                                  "frac": step_gbs / h2d_peak, "frac_isolated_call": st["bytes_copied"] / (mean("ms_total") * 1e-3) / 1e9 / h2d_peak,
                                  "peak_source": "slp_measure_h2d, pinned, best of per-matrix and 256 MiB chunks, best of 5 each (the same cudaMemcpyAsync path the engine uses; "
                                                 "profiles/r1_h2d_chunks.md has an SM zero-copy cross-check)",
                                  "h2d_copies_per_step": st["h2d_copies"],
                                  "peak_unbound": h2d_peak_unbound, "peak_torch_crosscheck": h2d_peak_torch,
                                  "peak_note": "peak = measured after binding to the GPU's NUMA node (config.numa); peak_unbound = 256 MiB chunks "
                                               "before binding; peak_torch_crosscheck = 1 GiB torch pinned -> device copy_, best of 10, "
                                               "not through libslpmoe.so"}

    # ---- end to end through the host entry point: hidden from pinned host memory, result read back ----
    e2e = None
    if not args.no_e2e and par == "token":
        hin = hidden.cpu().pin_memory()
        hout = torch.empty_like(hin).pin_memory()
        for _ in range(max(1, args.warmup // 2)):
            layer.prefill_host(hin, hout)
        barrier()
        t0 = time.perf_counter()
        n_e2e = max(2, args.steps // 2)
        for _ in range(n_e2e):
            layer.prefill_host(hin, hout)
        e2e_s = (time.perf_counter() - t0) / n_e2e
        e2e_s = sharding.max_over_ranks(e2e_s, device=dev)
        e2e = {"value": world * cfg.T / e2e_s, "unit": "tokens/s",
               "h2d_bytes_per_step": cfg.T * cfg.H * 2 + (st["bytes_copied"] if mode == "streamed" else 0),
               "d2h_bytes_per_step": cfg.T * cfg.H * 2}
    gpu_launches = st["kernel_launches"] * args.steps

    # ---- the rest of BASELINE's metric on the same weights: 32K tokens resident / streamed / chunked ----
    if not args.no_extras and rank == 0 and world == 1 and cfg_id == 1 and mode == "streamed":
        try:
            layer.close()
            cfg2 = inputs.CONFIGS[2]
            big = SlpMoeLayer(cfg2, W, device=local_rank, triage=args.triage)
            h2 = inputs.make_hidden(cfg2, device=dev)
            o2 = torch.empty_like(h2)
            fl2 = inputs.fp8_flops_per_token(cfg2) * cfg2.T
            # streamed: one 32K pass, and 8 chunks of 4096 (one weight pass per chunk)
            for _ in range(2):
                big.prefill(h2, o2)
            torch.cuda.synchronize()
            s32 = isolated_calls(3, lyr=big, h=h2, o=o2)
            ms32 = statistics.mean(s["ms_total"] for s in s32)
            extra["streamed_32k"] = {"workload": "cfg2_streamed (single pass)", "ms_per_call": ms32, "ms_min": min(s["ms_total"] for s in s32),
                                     "tokens_per_s": cfg2.T / (ms32 * 1e-3), "calls": len(s32),
                                     "link_frac": s32[-1]["bytes_copied"] / (ms32 * 1e-3) / 1e9 / h2d_peak, "bytes_per_call": s32[-1]["bytes_copied"]}
            ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            chunks = [(h2[r0:r0 + 4096], o2[r0:r0 + 4096]) for r0 in range(0, cfg2.T, 4096)]
            for hc, oc in chunks[:2]:
                big.prefill(hc, oc)
            torch.cuda.synchronize()
            reps = 2
            ev0.record(stream)
            for _ in range(reps):
                for hc, oc in chunks:
                    big.prefill(hc, oc)
            ev1.record(stream)
            torch.cuda.synchronize()
            msc = ev0.elapsed_time(ev1) / reps
            extra["streamed_32k_chunked"] = {"workload": "cfg2_streamed (8 chunks of 4096, one weight pass per chunk, back to back)", "ms_per_32k": msc,
                                             "tokens_per_s": cfg2.T / (msc * 1e-3), "link_frac": 8 * s32[-1]["bytes_copied"] / (msc * 1e-3) / 1e9 / h2d_peak}
            # resident: isolated calls (mean / min), then a soak of back-to-back calls (sustained clocks)
            big.set_residency("resident")
            for _ in range(3):
                big.prefill(h2, o2)
            torch.cuda.synchronize()
            sres = isolated_calls(10, lyr=big, h=h2, o=o2)
            msr = statistics.mean(s["ms_total"] for s in sres)
            fp8 = measure_fp8_dense_peak(dev)
            soak_n = 150
            sampler = ClockSampler(local_rank)
            sampler.start()
            ev0.record(stream)
            for _ in range(soak_n):
                big.prefill(h2, o2)
            ev1.record(stream)
            torch.cuda.synchronize()
            soak_clocks = sampler.stop()
            ms_soak = ev0.elapsed_time(ev1) / soak_n
            peak8 = 2.0 * peaks["bf16_tflops"]
            tf = lambda m: fl2 / (m * 1e-3) / 1e12
            res = {"workload": "cfg2_resident", "calls": len(sres), "ms_per_call": msr, "ms_min": min(s["ms_total"] for s in sres),
                   "tokens_per_s": cfg2.T / (msr * 1e-3), "tflops_per_call": tf(msr),
                   "frac_of_nominal_fp8": tf(msr) / FP8_NOMINAL_TFLOPS, "frac_of_2x_measured_bf16": tf(msr) / peak8,
                   "sustained": {"calls": soak_n, "ms_per_call": ms_soak, "tflops_per_call": tf(ms_soak), "frac_of_nominal_fp8": tf(ms_soak) / FP8_NOMINAL_TFLOPS,
                                 "frac_of_2x_measured_bf16_sustained": tf(ms_soak) / (2.0 * peaks["bf16_tflops_sustained"]), "clocks": soak_clocks},
                   "fp8_dense_peak_measured": fp8,
                   "stage_ms": {k: statistics.mean(s[k] for s in sres) for k in ("ms_route", "ms_experts", "ms_combine", "ms_gateup_sum", "ms_down_sum")},
                   "aggregate": "mean over isolated calls; ms_min separately"}
            if "burst_tflops" in fp8:
                res["frac_of_measured_fp8_burst"] = tf(msr) / fp8["burst_tflops"]
                res["sustained"]["frac_of_measured_fp8_sustained"] = tf(ms_soak) / fp8["sustained_tflops"]
            gu2 = statistics.mean(s["ms_gateup_sum"] for s in sres)
            rr = {"kernel": "gemm_tc_kernel<0> (gate/up + SwiGLU + requant)", "bound": "tensor",
                  "achieved": 2.0 * 2 * cfg2.I * cfg2.H * (cfg2.T * (cfg2.k + cfg2.n_shared)) / (gu2 * 1e-3) / 1e12,
                  "peak": peak8, "unit": "TFLOP/s", "traffic": NCU_TRAFFIC_BYTES["cfg2_resident"],
                  "peak_source": "2 x bf16 measured (burst), fp8:bf16 nominal ratio", "aggregate": "mean over isolated calls",
                  "sm_mhz_during_kernel": statistics.mean(s["sm_mhz_gateup"] for s in sres)}
            rr["frac"] = rr["achieved"] / rr["peak"]
            if "burst_tflops" in fp8:
                rr["frac_of_measured_fp8_burst"] = rr["achieved"] / fp8["burst_tflops"]
            res["roofline"] = rr
            extra["resident_32k"] = res
            big.close()
        except Exception as ex:  # report, never hide
            extra["extras_error"] = repr(ex)
    else:
        layer.close()

    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        os.sched_setaffinity(0, affinity0)   # the NUMA binding was for the pinned weights; the oracle gets every core
        torch.set_num_threads(ncores)
        n_exp = 2 if cfg.E >= 64 else cfg.E
        W_np, hb = inputs.weights_as_numpy(W), inputs.hidden_as_bits(hidden)
        v, sample, _, _ = cpu_oracle_sample(cfg, W_np, hb, n_exp, min(cfg.T, 128))
        cpu_baseline = {"value": v, "unit": "tokens/s", "cores": ncores, "kind": "oracle", "estimated": True, "sample": sample}
        # The headline workload gets ONE timed full pass of the oracle (all T tokens, all experts) when the sample says it
        # ends within about two and a half minutes on this box; otherwise the extrapolated sample above stays, labelled.
        if not args.cpu_baseline_sample and cfg.T / v <= 150.0:
            v_full, dt = cpu_oracle_full(cfg, W_np, hb)
            cpu_baseline = {"value": v_full, "unit": "tokens/s", "cores": ncores, "kind": "oracle", "estimated": False,
                            "sample": f"one timed pass of oracle.moe_layer over all {cfg.T} tokens and all {cfg.E} experts of {cfg.name}: {dt:.1f} s "
                                      f"(the bounded sample had predicted {cfg.T / v:.1f} s)"}

    if rank == 0:
        print(json.dumps({"metric": METRIC, "value": value, "unit": "tokens/s", "n_gpus": world, "steps": args.steps,
                          "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
                          "scaling": "weak" if par == "token" else "strong",
                          "vs_baseline": None, "dtype": "e4m3 x e4m3 -> f32", "data": "synthetic", "config": config,
                          "clocks": clocks, "e2e": e2e, "gpu_launches": gpu_launches, "roofline": roofline,
                          "cpu_baseline": cpu_baseline, **extra}))
    if world > 1 or par == "smallep":
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
