#!/usr/bin/env python
"""bench.py — measures BASELINE.json's metric on the SLP MoE layer.

A "step" is one pass of the whole hot path (router, permute, quantise, expert-weight streaming
overlapped with the grouped FP8 GEMMs, shared expert, combine) over one batch of synthetic tokens.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload NAME] [--impl ours|reference]

Workloads (BASELINE.json configs): cfg1_streamed (default; T=4096, DeepSeek-V3 shape, weights
streamed from pinned host memory), cfg2_streamed / cfg2_resident (T=32768 single pass),
cfg4_streamed / cfg4_resident, cfg0_resident.  Prints ONE JSON line (rank 0).
Multi-GPU (torchrun): the path shards by tokens with no data-path collective — every rank runs its
own T tokens through its own layer replica ("scaling": "weak").
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
}
METRIC = "prefill tok/s per MoE layer (host-streamed FP8); resident FP8 TFLOP/s vs peak"
# dram__bytes_read.sum + dram__bytes_write.sum of one gemm_tc_kernel<0> launch, from the committed ncu
# --set full captures (profiles/r1_layer_ncu.md, profiles/r1_streamed_gemm_ncu.md); None = not captured.
NCU_TRAFFIC_BYTES = {"cfg2_resident": 10.65e9, "cfg1_streamed": 2.143e9}


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


def cpu_oracle_sample(cfg, W_np, hidden_bits, n_experts_sample, n_shared_tokens):
    """Times the oracle, as it stands, on a bounded sample of the workload and scales it to the
    whole layer: full routing + quantisation for all T tokens (timed as is), the expert FFNs of
    the first `n_experts_sample` routed experts over ALL their rows (scaled by E / sample), and
    the shared expert over `n_shared_tokens` rows (scaled by T / n)."""
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
    sample = (f"router+quantise all {T} tokens ({t_route:.2f}s), FFN of routed experts 0..{n_experts_sample - 1} of {cfg.E} "
              f"over all their {rows_done} rows ({t_exp:.2f}s, scaled x{cfg.E / n_experts_sample:.0f}), shared expert on "
              f"{n_shared_tokens} rows ({t_sh:.2f}s, scaled x{T / max(1, n_shared_tokens):.0f})")
    return T / est, sample, t_route + t_exp + t_sh


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="cfg1_streamed", choices=sorted(WORKLOADS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-resident-extra", action="store_true")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer leg (profiling runs)")
    ap.add_argument("--triage", default=None, help="SLP_TRIAGE value for A/B runs (e.g. gemm=pair); not a product option")
    ap.add_argument("--staging-slots", type=int, default=0)
    ap.add_argument("--experts-per-launch", type=int, default=0)
    args = ap.parse_args()

    import numpy as np
    import torch
    from paper_2606_10493_b200 import inputs

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    cfg_id, mode = WORKLOADS[args.workload]
    cfg = inputs.CONFIGS[cfg_id]
    ncores = len(os.sched_getaffinity(0))
    config = {"workload": args.workload, "config": cfg.name, "T": cfg.T, "hidden": cfg.H, "n_experts": cfg.E,
              "top_k": cfg.k, "n_group": cfg.G, "topk_group": cfg.Gk, "moe_intermediate": cfg.I,
              "n_shared": cfg.n_shared, "mode": mode, "parallelism": f"token-sharded x{world} (no collective)",
              "l2": "inputs_exceed_l2" if cfg_id >= 1 else "tiny (launch-latency regime)"}

    # ------------------------------------------------------------------ reference arm = oracle
    if args.impl == "reference":
        if rank != 0:
            return 0
        torch.set_num_threads(ncores)
        n_exp = 2 if cfg.E >= 64 else cfg.E
        dev = "cuda" if torch.cuda.is_available() else "cpu"
        W = inputs.make_weights(cfg, device=dev, experts=range(n_exp))
        W_np = inputs.weights_as_numpy(W)
        hb = inputs.hidden_as_bits(inputs.make_hidden(cfg, device=dev))
        vals, secs = [], []
        for i in range(args.warmup + args.steps):
            v, sample, s = cpu_oracle_sample(cfg, W_np, hb, n_exp, min(cfg.T, 128))
            if i >= args.warmup:
                vals.append(v)
                secs.append(s)
        v = statistics.median(vals)
        print(json.dumps({"metric": METRIC, "value": v, "unit": "tokens/s", "n_gpus": args.gpus, "steps": args.steps,
                          "warmup": args.warmup, "ms_per_step": 1e3 * cfg.T / v, "higher_is_better": True,
                          "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic", "impl": "reference",
                          "config": config, "cpu_baseline": {"value": v, "unit": "tokens/s", "cores": ncores, "kind": "oracle", "sample": sample},
                          "e2e": {"value": v, "unit": "tokens/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))
        return 0

    # ------------------------------------------------------------------ our arm
    import __graft_entry__ as entry
    entry.build()
    from paper_2606_10493_b200 import SlpMoeLayer, measure_h2d_gbs, sharding

    assert torch.cuda.is_available(), "bench.py needs a CUDA device (there is no CPU path)"
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
    peaks = load_peaks()

    t_gen = time.perf_counter()
    W = inputs.make_weights(cfg, device=dev, pin=True)
    hidden = inputs.make_hidden(cfg, device=dev, first_chunk=sharding.weak_scaling_first_chunk(cfg.T, rank))  # each rank its own tokens
    t_gen = time.perf_counter() - t_gen
    layer = SlpMoeLayer(cfg, W, device=local_rank, staging_slots=args.staging_slots,
                        experts_per_launch=args.experts_per_launch, triage=args.triage)
    layer.set_residency(mode)
    out = torch.empty_like(hidden)
    stream = torch.cuda.current_stream()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    def timed_steps(n_steps, sampler=None):
        for _ in range(args.warmup):
            layer.prefill(hidden, out)
        barrier()
        if sampler:
            sampler.start()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(n_steps):          # back-to-back on one stream, no host sync inside the timed region
            layer.prefill(hidden, out)
        e1.record(stream)
        barrier()
        clocks = sampler.stop() if sampler else None
        per_call = [layer.stats()]        # CUDA-event stage/kernel times of the last timed call
        return e0.elapsed_time(e1) / n_steps, per_call, clocks

    # host-link peak of this box: the better of per-matrix chunks and 256 MiB chunks (the engine merges
    # consecutive experts into one copy when the host layout allows, profiles/r1_h2d_chunks.md)
    h2d_peak = max(measure_h2d_gbs(local_rank, cfg.I * cfg.H, 1 << 30, 5),
                   measure_h2d_gbs(local_rank, 256 << 20, 1 << 30, 5)) if mode == "streamed" else None
    ms, per_call, clocks = timed_steps(args.steps, ClockSampler(local_rank))
    value, ms = sharding.whole_job_tokens_per_s(cfg.T, ms, device=dev)   # all ranks' tokens / slowest rank's device time

    # kernel-level numbers from the library's own CUDA events on the launching stream
    st = per_call[-1]
    n_pairs = max(1, st["timed_gemm_pairs"])
    gu_ms = statistics.mean(s["ms_gateup_sum"] for s in per_call) / n_pairs
    dn_ms = statistics.mean(s["ms_down_sum"] for s in per_call) / n_pairs
    idx, _, counts = layer.debug_routing(cfg.T)
    rows_total = int(counts.sum()) + (cfg.T if cfg.n_shared else 0)
    n_exp_run = int((counts > 0).sum()) + cfg.n_shared
    flops_call = inputs.fp8_flops_per_token(cfg) * cfg.T
    # gate/up kernel: algorithmic bytes = weights (2*I*H per expert run) + A rows + hq written + scales
    gu_bytes = n_exp_run * 2 * cfg.I * cfg.H + rows_total * (cfg.H + cfg.I) + rows_total * 4 * (cfg.H // 128 + cfg.I // 128)
    gu_flops = 2.0 * 2 * cfg.I * cfg.H * rows_total
    gu_time = statistics.mean(s["ms_gateup_sum"] for s in per_call) * 1e-3
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
    # the ncu capture is of ONE launch: the whole layer in resident mode, one group of experts_per_launch
    # routed experts in streamed mode; the algorithmic bytes of that same launch, for comparison
    from paper_2606_10493_b200 import query_plan
    epl = query_plan(cfg, staging_slots=args.staging_slots, experts_per_launch=args.experts_per_launch)["experts_per_launch"]
    roofline["traffic_launch_algorithmic_bytes"] = gu_bytes if mode == "resident" else gu_bytes * min(epl, cfg.E) / max(1, n_exp_run)
    roofline["algorithmic_bytes_per_launch"] = gu_bytes / max(1, st["timed_gemm_pairs"])
    roofline["algorithmic_flops_per_launch"] = gu_flops / max(1, st["timed_gemm_pairs"])
    roofline["ms_per_launch"] = gu_ms
    roofline["launches_per_step"] = st["timed_gemm_pairs"]
    roofline["down_ms_per_launch"] = dn_ms
    roofline["sm_mhz_during_kernel"] = st["sm_mhz_gateup"]
    roofline["down_sm_mhz_during_kernel"] = st["sm_mhz_down"]

    extra = {"tflops_per_call": flops_call / (ms * 1e-3) / 1e12,
             "fp8_peak_nominal_tflops": 4500.0, "frac_of_nominal_fp8": flops_call / (ms * 1e-3) / 4.5e15,
             "stage_ms": {k: statistics.mean(s[k] for s in per_call) for k in ("ms_total", "ms_route", "ms_experts", "ms_combine", "ms_copy_span")},
             "gen_seconds": t_gen}
    if mode == "streamed":
        link_gbs = statistics.mean(s["bytes_copied"] / (s["ms_copy_span"] * 1e-3) / 1e9 for s in per_call if s["ms_copy_span"] > 0)
        step_gbs = st["bytes_copied"] / (ms * 1e-3) / 1e9
        extra["link_roofline"] = {"bound": "host_link", "bytes_per_step": st["bytes_copied"], "peak": h2d_peak, "unit": "GB/s",
                                  "achieved_copy_span": link_gbs, "achieved_whole_step": step_gbs,
                                  "frac": step_gbs / h2d_peak, "peak_source": "slp_measure_h2d, pinned, best of per-matrix and 256 MiB chunks, best of 5 each",
                                  "h2d_copies_per_step": st["h2d_copies"]}

    # end-to-end through the host entry point: hidden from pinned host memory, result read back
    e2e = None
    if not args.no_e2e:
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

    # resident-mode 32K number on the same weights (the second half of BASELINE's metric)
    if not args.no_resident_extra and rank == 0 and cfg_id == 1 and mode == "streamed":
        try:
            layer.close()
            cfg2 = inputs.CONFIGS[2]
            big = SlpMoeLayer(cfg2, W, device=local_rank, triage=args.triage)
            big.set_residency("resident")
            h2 = inputs.make_hidden(cfg2, device=dev)
            o2 = torch.empty_like(h2)
            for _ in range(3):
                big.prefill(h2, o2)
            torch.cuda.synchronize()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            reps = 5
            stats2 = []
            a.record(stream)
            for _ in range(reps):
                big.prefill(h2, o2)
                torch.cuda.synchronize()
                stats2.append(big.stats())
            b.record(stream)
            torch.cuda.synchronize()
            ms2 = min(s["ms_total"] for s in stats2)
            fl2 = inputs.fp8_flops_per_token(cfg2) * cfg2.T
            peak8 = 2.0 * peaks["bf16_tflops"]
            extra["resident_32k"] = {"workload": "cfg2_resident", "ms_per_call": ms2, "tokens_per_s": cfg2.T / (ms2 * 1e-3),
                                     "tflops_per_call": fl2 / (ms2 * 1e-3) / 1e12,
                                     "frac_of_nominal_fp8": fl2 / (ms2 * 1e-3) / 4.5e15,
                                     "frac_of_measured_fp8": fl2 / (ms2 * 1e-3) / (peak8 * 1e12),
                                     "roofline": {"kernel": "gemm_tc_kernel<0> (gate/up + SwiGLU + requant)", "bound": "tensor",
                                                  "achieved": 2.0 * 2 * cfg2.I * cfg2.H * (cfg2.T * (cfg2.k + cfg2.n_shared)) / (min(s["ms_gateup_sum"] for s in stats2) * 1e-3) / 1e12,
                                                  "peak": peak8, "unit": "TFLOP/s", "traffic": NCU_TRAFFIC_BYTES["cfg2_resident"],
                                                  "peak_source": "2 x bf16 measured (burst), fp8:bf16 nominal ratio",
                                                  "sm_mhz_during_kernel": statistics.mean(s["sm_mhz_gateup"] for s in stats2)},
                                     "stage_ms": {k: statistics.mean(s[k] for s in stats2) for k in ("ms_route", "ms_experts", "ms_combine", "ms_gateup_sum", "ms_down_sum")}}
            rr = extra["resident_32k"]["roofline"]
            rr["frac"] = rr["achieved"] / rr["peak"]
            big.close()
        except Exception as ex:  # report, never hide
            extra["resident_32k"] = {"error": repr(ex)}
    else:
        layer.close()

    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        torch.set_num_threads(ncores)
        n_exp = 2 if cfg.E >= 64 else cfg.E
        v, sample, _ = cpu_oracle_sample(cfg, inputs.weights_as_numpy(W), inputs.hidden_as_bits(hidden), n_exp, min(cfg.T, 128))
        cpu_baseline = {"value": v, "unit": "tokens/s", "cores": ncores, "kind": "oracle", "sample": sample}

    if rank == 0:
        print(json.dumps({"metric": METRIC, "value": value, "unit": "tokens/s", "n_gpus": world, "steps": args.steps,
                          "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
                          "vs_baseline": None, "dtype": "e4m3 x e4m3 -> f32", "data": "synthetic", "config": config,
                          "clocks": clocks, "e2e": e2e, "gpu_launches": gpu_launches, "roofline": roofline,
                          "cpu_baseline": cpu_baseline, **extra}))
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
