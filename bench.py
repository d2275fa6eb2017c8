#!/usr/bin/env python
"""bench.py -- the RingX hot path on B200: attention TFLOP/s of the chunked forward (and backward), one JSON line.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config C3]

A "step" is one pass of the WHOLE hot path over one batch of synthetic input of
the named BASELINE.json config (default C3: bf16, B=1, H=8, N=262144, d=128, kv_chunk=32768 -- the configuration
the north_star's target "bf16 forward at N >= 262,144" is quoted on): `ringx_attn_fwd` (8 KV-chunk passes of the
tcgen05 kernel + 7 Eq. 5 merges) followed by `ringx_attn_bwd` (D_i preprocess, 8 backward chunk passes, dQ
convert).  `--pass fwd` times the forward alone.  FLOPs: forward 4*B*H*N^2*d, backward
10*B*H*N^2*d; `value` is their sum over the step time, and the line also carries forward-only and backward-only
TFLOP/s from the live per-kernel CUDA-event timing.  Inputs are seeded synthetic (paper_2507_16697_b200/workloads.py), resident in HBM for
`value`; `e2e` times the same metric through the C ABI with HOST buffers (H2D + D2H inside the timed region).
Multi-GPU (--gpus N under torchrun): the path has no exchange step on one node (batch x heads
are independent) -> every rank runs the workload on its own seeded batch, no data-path collective, "weak".
`--impl reference` times the fp64 CPU oracle (oracle/), as it stands, on a bounded sample of the workload.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402
import torch  # noqa: E402

METRIC = ("attention TFLOPS fwd+bwd at 1 B200 (fwd 4*B*H*N^2*d + bwd 10*B*H*N^2*d per step; fwd-only and bwd-only in "
          "`fwd`/`bwd`; fraction of dense bf16 tensor peak in roofline.frac)")
UNIT = "TFLOP/s"
FALLBACK_PEAKS = {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0}


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            d = json.load(open(p))
            return {k: float(d[k]) for k in FALLBACK_PEAKS if k in d} | {"source": "measured"}
        except Exception:
            pass
    return dict(FALLBACK_PEAKS) | {"source": "fallback"}


def load_traffic(key):
    """DRAM bytes per launch of the dominant kernel from the committed ncu --set full capture (or None)."""
    p = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(p):
        try:
            return json.load(open(p)).get(key)
        except Exception:
            return None
    return None


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms DURING the timed region."""
    FIELDS = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")
    NAMES = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")

    def __init__(self, gpu_index: int):
        self.gpu = gpu_index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.gpu}", f"--query-gpu={self.FIELDS}", "--format=csv,noheader,nounits",
                 "-lms", "200"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if self.proc is None:
            return None
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, smax, power, reasons = [], [], [], set()
        for line in self.lines:
            f = [x.strip() for x in line.split(",")]
            if len(f) < 8:
                continue
            try:
                sm.append(float(f[1])); smax.append(float(f[2])); power.append(float(f[3]))
            except ValueError:
                continue
            for name, val in zip(self.NAMES, f[4:8]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return None
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(smax)), "power_w_max": float(max(power)),
                "samples": len(sm), "reasons": sorted(reasons)}


def host_cores() -> int:
    try:
        return len(os.sched_getaffinity(0))
    except Exception:
        return os.cpu_count() or 1


def oracle_sample(cfg, k64, v64, q_rows64, do_rows64=None, block=256):
    """The oracle as it stands on a bounded sample: `attention_fwd` (and `attention_bwd` when dO rows are given) of
    the sampled query rows of one head against ALL keys of that head.  Returns (seconds, flops)."""
    from oracle import attention as orc
    t0 = time.perf_counter()
    for r0 in range(0, q_rows64.shape[0], block):
        orc.attention_fwd(q_rows64[r0:r0 + block], k64, v64, cfg.scale)
        if do_rows64 is not None:
            orc.attention_bwd(q_rows64[r0:r0 + block], k64, v64, do_rows64[r0:r0 + block], cfg.scale)
    dt = time.perf_counter() - t0
    return dt, (4.0 if do_rows64 is None else 14.0) * q_rows64.shape[0] * cfg.N * cfg.d


def run_reference(args, cfg, rank):
    """--impl reference: the fp64 numpy oracle on this box's host cores, each step a bounded sample."""
    from paper_2507_16697_b200 import workloads as wl
    if rank != 0:
        return
    rows_per_step = args.ref_rows
    # one head of the workload, generated on the host by the same counter-based recipe (first rows of head 0)
    head = wl.Config(cfg.name, cfg.dtype, 1, 1, cfg.N, cfg.d, cfg.kv_chunk, cfg.qk_gain, False, cfg.seed)
    bwd = args.passes == "fwd+bwd"
    q, k, v, do = wl.make_qkv(head, with_do=True)
    k64, v64 = wl.to_f64_numpy(k[0, 0]), wl.to_f64_numpy(v[0, 0])
    q64, do64 = wl.to_f64_numpy(q[0, 0]), wl.to_f64_numpy(do[0, 0])
    rng = np.random.default_rng(0)
    for _ in range(args.warmup):
        rows = rng.integers(0, cfg.N, 64)
        oracle_sample(cfg, k64, v64, q64[rows], do64[rows] if bwd else None)
    t_total, f_total = 0.0, 0.0
    for _ in range(args.steps):
        rows = rng.integers(0, cfg.N, rows_per_step)
        dt, fl = oracle_sample(cfg, k64, v64, q64[rows], do64[rows] if bwd else None)
        t_total += dt
        f_total += fl
    value = f_total / t_total / 1e12
    sample = (f"{rows_per_step} query rows of head 0 against all {cfg.N} keys per step "
              f"({rows_per_step * cfg.N:.3g} of the config's {cfg.B * cfg.H * cfg.N * cfg.N:.3g} query-key pairs)")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t_total / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(cfg, args.passes),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": host_cores(), "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def workload_config(cfg, what):
    return {"workload": f"{cfg.name}: {cfg.dtype} {what}, non-causal, B={cfg.B} H={cfg.H} N={cfg.N} d={cfg.d} "
                        f"kv_chunk={cfg.kv_chunk} ({cfg.N // cfg.kv_chunk} ring passes)",
            "B": cfg.B, "H": cfg.H, "N": cfg.N, "d": cfg.d, "kv_chunk": cfg.kv_chunk, "qk_gain": cfg.qk_gain,
            "pass": what, "seed": cfg.seed, "l2": "inputs larger than L2 (no flush needed)"
            if 3 * cfg.B * cfg.H * cfg.N * cfg.d * 2 > 126e6 else "L2 flushed between steps"}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="C3", choices=["C2", "C3", "C4", "C5"])
    ap.add_argument("--pass", dest="passes", default="fwd+bwd", choices=["fwd", "fwd+bwd"])
    ap.add_argument("--ref-rows", type=int, default=256, help="query rows per step of the reference arm")
    ap.add_argument("--cpu-baseline-seconds", type=float, default=15.0)
    ap.add_argument("--no-extra", action="store_true", help="skip the short C2/C4 side measurements")
    ap.add_argument("--schedule", default="replicas", choices=["replicas", "ringx_b", "ringx_a"],
                    help="replicas (default: the single-GPU hot path, one seeded batch per rank) or one of the paper's "
                         "sequence-parallel schedules over the ranks (PAPER.md:137-147): the config's sequence is sharded "
                         "over the W ranks and every step is one RingX forward + backward")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    from paper_2507_16697_b200 import workloads as wl
    cfg = wl.CONFIGS[args.config]
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))

    if args.impl == "reference":
        run_reference(args, cfg, rank)
        return

    from paper_2507_16697_b200 import multirank, ringx
    from paper_2507_16697_b200.build import build_library
    if rank == 0:
        build_library()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --impl ours needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
        dist.barrier()
    ringx.lib()
    if args.schedule != "replicas":
        run_schedule(args, cfg, rank, world, dev, dist)
        return

    def barrier():
        if dist is not None:
            dist.barrier()

    # ---------------------------------------------------------------- inputs (seeded, per-rank batch)
    rcfg = multirank.rank_config(cfg, rank)
    do_bwd = args.passes == "fwd+bwd"
    tensors = wl.make_qkv(rcfg, with_do=do_bwd, device=dev)
    q, k, v = tensors[:3]
    dO = tensors[3] if do_bwd else None
    B, H, N, d = q.shape
    o = torch.empty_like(q)
    lse = torch.empty((B, H, N), dtype=torch.float32, device=dev)
    ws_f = torch.empty(max(256, ringx.ringx_attn_fwd_workspace_bytes(B, H, N, d, cfg.kv_chunk, q.dtype)),
                       dtype=torch.uint8, device=dev)
    ws_b = None
    if do_bwd:
        ws_b = torch.empty(max(256, ringx.ringx_attn_bwd_workspace_bytes(B, H, N, d, cfg.kv_chunk, q.dtype)),
                           dtype=torch.uint8, device=dev)
    flops_step = cfg.fwd_flops + (cfg.bwd_flops if do_bwd else 0.0)
    launches = [0]

    def step():
        ringx.ringx_attn_fwd(q, k, v, cfg.kv_chunk, cfg.scale, o=o, lse=lse, workspace=ws_f)
        n = ringx.ringx_last_launch_count()
        if do_bwd:
            ringx.ringx_attn_bwd(q, k, v, o, lse, dO, cfg.kv_chunk, cfg.scale, workspace=ws_b)
            n += ringx.ringx_last_launch_count()
        launches[0] += n

    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize()

    # ---------------------------------------------------------------- timed region
    sampler = ClockSampler(local_rank) if rank == 0 else None
    launches[0] = 0
    ringx.ringx_profile_enable(True)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    torch.cuda.synchronize()
    if sampler:
        sampler.start()
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    torch.cuda.synchronize()
    barrier()
    clocks = sampler.stop() if sampler else None
    prof = ringx.ringx_profile_read()
    ringx.ringx_profile_enable(False)
    ms_total = multirank.max_over_ranks(e0.elapsed_time(e1), dist, dev)
    ms_step = ms_total / args.steps
    value = multirank.aggregate_tflops(world, flops_step, ms_step)
    gpu_launches = launches[0]

    # ---------------------------------------------------------------- roofline of the dominant kernel(s)
    peaks = load_peaks()

    def roofline_of(kind):
        ms, n = prof[kind]
        if not n:
            return None
        per_launch = (10.0 if kind == "attn_bwd" else 4.0) * B * H * N * cfg.kv_chunk * d
        ach = per_launch / (ms / n * 1e-3) / 1e12
        return {
            "bound": "tensor", "kernel": "attn_chunk_fwd_kernel" if kind == "attn_fwd" else "attn_chunk_bwd_kernel",
            "achieved": ach, "peak": peaks["bf16_tflops_sustained"], "unit": "TFLOP/s",
            "frac": ach / peaks["bf16_tflops_sustained"],
            "peak_kind": f"bf16 dense, sustained (kernel timed inside a long step), {peaks['source']}",
            "peak_burst": peaks["bf16_tflops"], "frac_of_burst": ach / peaks["bf16_tflops"],
            "frac_of_nominal_2250": ach / 2250.0, "flops_per_launch": per_launch, "launches_timed": n,
            "avg_launch_ms": ms / n, "share_of_step": ms / ms_total if world == 1 else None,
            "traffic": load_traffic(f"{cfg.name}_{kind}"),
        }

    dom = "attn_bwd" if prof["attn_bwd"][0] > prof["attn_fwd"][0] else "attn_fwd"
    roofline = roofline_of(dom)
    roofline_other = roofline_of("attn_fwd" if dom == "attn_bwd" else "attn_bwd")
    fwd_ms = (prof["attn_fwd"][0] + prof["merge"][0]) / args.steps
    bwd_ms = (prof["attn_bwd"][0] + prof["bwd_aux"][0]) / args.steps
    fwd_info = {"ms_per_step": fwd_ms, "tflops": cfg.fwd_flops / fwd_ms / 1e9,
                "frac_of_sustained_peak": cfg.fwd_flops / fwd_ms / 1e9 / peaks["bf16_tflops_sustained"],
                "frac_of_burst_peak": cfg.fwd_flops / fwd_ms / 1e9 / peaks["bf16_tflops"]} if fwd_ms > 0 else None
    bwd_info = {"ms_per_step": bwd_ms, "tflops": cfg.bwd_flops / bwd_ms / 1e9,
                "frac_of_sustained_peak": cfg.bwd_flops / bwd_ms / 1e9 / peaks["bf16_tflops_sustained"],
                "frac_of_burst_peak": cfg.bwd_flops / bwd_ms / 1e9 / peaks["bf16_tflops"]} if bwd_ms > 0 else None
    # the Eq. 5 merge kernel (north_star subsystem 3): the bf16 forward folds Eq. 5 in the chunk kernel's epilogue, so
    # ringx_lse_merge -- the entry RingX_a/b and the fp32 path use -- is timed on its own on this workload's [R,d] partials
    merge_info = None
    if rank == 0:
        R = B * H * N
        pa, pb = torch.randn(R, d, device=dev), torch.randn(R, d, device=dev)
        la, lb = torch.randn(R, device=dev), torch.randn(R, device=dev)
        for _ in range(3):
            ringx.ringx_lse_merge(pa, la, pb, lb, inplace=True)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        n_merge = 10
        e0.record()
        for _ in range(n_merge):
            ringx.ringx_lse_merge(pa, la, pb, lb, inplace=True)
        e1.record()
        torch.cuda.synchronize()
        mms = e0.elapsed_time(e1) / n_merge
        mbytes = 3.0 * R * (d * 4 + 4)
        merge_info = {"bound": "hbm", "kernel": "lse_merge_kernel<float,float>", "avg_launch_ms": mms,
                      "launches_timed": n_merge, "achieved": mbytes / (mms * 1e-3) / 1e9, "peak": peaks["hbm_gbs"],
                      "unit": "GB/s", "frac": mbytes / (mms * 1e-3) / 1e9 / peaks["hbm_gbs"],
                      "note": "timed alone, back to back, in place on operand a (fp32 partials of the workload's shape)"}
        del pa, pb, la, lb

    # ---------------------------------------------------------------- e2e: HOST buffers through the C ABI
    n_e2e = max(1, min(args.steps, 3))
    tb = q.numel() * q.element_size()
    if do_bwd:
        host_in = [t.cpu().pin_memory() for t in (q, k, v, dO)]
        outs = (torch.empty_like(host_in[0]).pin_memory(), torch.empty((B, H, N), dtype=torch.float32).pin_memory(),
                torch.empty_like(host_in[0]).pin_memory(), torch.empty_like(host_in[0]).pin_memory(),
                torch.empty_like(host_in[0]).pin_memory())
        ws_h = torch.empty(ringx.ringx_attn_fwd_bwd_host_workspace_bytes(B, H, N, d, cfg.kv_chunk, q.dtype),
                           dtype=torch.uint8, device=dev)
        call = lambda: ringx.ringx_attn_fwd_bwd_host(*host_in, cfg.kv_chunk, cfg.scale, outs=outs, workspace=ws_h)
        h2d, d2h = 4 * tb, 4 * tb + lse.numel() * 4
        entry = "ringx_attn_fwd_bwd_host (pinned host q,k,v,dO -> device, fwd+bwd, o,lse,dq,dk,dv -> host, synchronised)"
    else:
        host_in = [t.cpu().pin_memory() for t in (q, k, v)]
        oh = torch.empty_like(host_in[0]).pin_memory()
        lh = torch.empty((B, H, N), dtype=torch.float32).pin_memory()
        ws_h = torch.empty(ringx.ringx_attn_fwd_host_workspace_bytes(B, H, N, d, cfg.kv_chunk, q.dtype),
                           dtype=torch.uint8, device=dev)
        call = lambda: ringx.ringx_attn_fwd_host(*host_in, cfg.kv_chunk, cfg.scale, o_host=oh, lse_host=lh,
                                                 workspace=ws_h)
        h2d, d2h = 3 * tb, tb + lse.numel() * 4
        entry = "ringx_attn_fwd_host (pinned host q,k,v -> device, forward, o+lse -> host, synchronised)"
    call()
    barrier()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(n_e2e):
        call()
    torch.cuda.synchronize()
    dt = multirank.max_over_ranks((time.perf_counter() - t0) / n_e2e, dist, dev)
    e2e = {"value": multirank.aggregate_tflops(world, flops_step, dt * 1e3), "unit": UNIT, "ms_per_step": dt * 1e3, "steps": n_e2e,
           "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "entry": entry}
    del ws_h, host_in

    # ---------------------------------------------------------------- short side measurements (not the metric)
    extra = {}
    if rank == 0 and not args.no_extra:
        extra["C1"] = c1_measure(ringx, wl, dev)
        for name in ("C2", "C4", "C5"):
            if name == cfg.name:
                continue
            extra[name] = side_measure(ringx, wl, wl.CONFIGS[name], dev, oracle_seconds=args.cpu_baseline_seconds / 5.0)
        extra["next_rows"] = next_rows_measure(ringx, wl, dev)
        if do_bwd:
            # the workload's backward with ringx_set_deterministic (int32 fixed-point dQ accumulator): context, not the metric
            ringx.ringx_set_deterministic(True)
            try:
                det_ms = timed_loop(lambda: ringx.ringx_attn_bwd(q, k, v, o, lse, dO, cfg.kv_chunk, cfg.scale,
                                                                 workspace=ws_b), min_seconds=2.0, min_reps=3)
            finally:
                ringx.ringx_set_deterministic(False)
            extra["deterministic_bwd"] = summarise(det_ms, cfg.bwd_flops)

    # ---------------------------------------------------------------- CPU baseline: the oracle, bounded sample
    cpu_baseline = None
    if rank == 0 and world == 1:
        k64, v64 = wl.to_f64_numpy(k[0, 0]), wl.to_f64_numpy(v[0, 0])
        q64 = wl.to_f64_numpy(q[0, 0, :8192])
        do64 = wl.to_f64_numpy(dO[0, 0, :8192]) if do_bwd else None
        dt0, _ = oracle_sample(cfg, k64, v64, q64[:128], do64[:128] if do_bwd else None)
        n_rows = int(min(q64.shape[0], max(128, args.cpu_baseline_seconds / (dt0 / 128.0) // 128 * 128)))
        dt, fl = oracle_sample(cfg, k64, v64, q64[:n_rows], do64[:n_rows] if do_bwd else None)
        cpu_baseline = {"value": fl / dt / 1e12, "unit": UNIT, "cores": host_cores(), "kind": "oracle",
                        "seconds": dt,
                        "sample": f"first {n_rows} query rows of head (0,0) against all {N} keys "
                                  f"(oracle.attention_fwd" + (" + attention_bwd" if do_bwd else "") +
                                  ", fp64 numpy, blocks of 256 rows)",
                        "full_config_seconds_extrapolated": flops_step / (fl / dt),
                        "extrapolation": "linear in query rows x heads",
                        # the other BASELINE.json configs: measured sample + labelled extrapolation each
                        "per_config": {name: extra[name]["cpu_baseline"] for name in extra
                                       if isinstance(extra[name], dict) and "cpu_baseline" in extra[name]}}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
            "config": workload_config(cfg, args.passes),
            "clocks": clocks, "e2e": e2e, "gpu_launches": gpu_launches,
            "roofline": roofline, "roofline_other_kernel": roofline_other, "merge_kernel": merge_info,
            "fwd": fwd_info, "bwd": bwd_info, "cpu_baseline": cpu_baseline, "extra": extra,
            "frac_of_bf16_peak": {"sustained": value / world / peaks["bf16_tflops_sustained"],
                                  "burst": value / world / peaks["bf16_tflops"], "nominal_2250": value / world / 2250.0,
                                  "source": peaks["source"]},
        }
        # LAST key, < 1 KB: the side figures in one place, so that a reader who keeps only the tail of the line still has the
        # d = 64 configs, the merge kernel, the MLA widths and the deterministic backward (TFLOP/s unless named _gbs)
        def _get(*path):
            node = extra
            for key in path:
                if not isinstance(node, dict) or key not in node:
                    return None
                node = node[key]
            return round(float(node), 1)
        line["summary"] = {
            "fwd_tflops": round(fwd_info["tflops"], 1) if fwd_info else None,
            "bwd_tflops": round(bwd_info["tflops"], 1) if bwd_info else None,
            "C2_fwd": _get("C2", "fwd_tflops"), "C4_fwd": _get("C4", "fwd_tflops"), "C4_bwd": _get("C4", "bwd_tflops"),
            "C5_fwd": _get("C5", "fwd_tflops"),
            "merge_gbs": round(merge_info["achieved"], 1) if merge_info else None,
            "mla_fwd": _get("next_rows", "mla_dqk192_dv128_H8_N65536", "fwd_tflops"),
            "mla_bwd": _get("next_rows", "mla_dqk192_dv128_H8_N65536", "bwd_tflops"),
            "gqa_fwd": _get("next_rows", "gqa_16q4kv_N32768_d128", "fwd_tflops"),
            "gqa_bwd": _get("next_rows", "gqa_16q4kv_N32768_d128", "bwd_tflops"),
            "split_kv": _get("next_rows", "split_kv_Nq2048_Nk65536_H8_d128", "split_tflops"),
            "bwd_partial": _get("next_rows", "bwd_partial_Nq16384_Nk16384_d128", "tflops"),
            "det_bwd": _get("deterministic_bwd", "tflops_median"),
            "tokeniser_gbs": _get("next_rows", "fidelity_tokens_512cube", "k4_f32", "gbs"),
            "qkv_proj": _get("next_rows", "projections_S262144_h1024", "qkv_tflops"),
            "block_fwd_bwd": _get("next_rows", "block_fwd_bwd_S262144_h1024", "tflops"),
        }
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


def run_schedule(args, cfg, rank, world, dev, dist):
    """--schedule ringx_b | ringx_a: the paper's schedules (paper_2507_16697_b200/ringx_dist.py) over the W ranks of the
    launch.  Every rank holds N/W tokens of every head; a step is one forward + one backward of the WHOLE sequence
    (strong scaling: the work per step is fixed, `value` = its FLOPs over the slowest rank's time).  No multi-GPU box
    has been available to this project: at W = 1 this is the single-device path behind the same interface."""
    from paper_2507_16697_b200 import multirank, ringx, ringx_dist, workloads as wl
    if dist is None:
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29531")
        dist.init_process_group("nccl", rank=0, world_size=1, device_id=dev)
    B, H, N, d = cfg.B, cfg.H, cfg.N, cfg.d
    Nl = N // world
    if N % world or Nl % 256:
        raise SystemExit(f"--schedule needs N / W to be a multiple of 256 (N = {N}, W = {world})")
    fwd, bwd = ((ringx_dist.ringx_b_forward, ringx_dist.ringx_b_backward) if args.schedule == "ringx_b" else
                (ringx_dist.ringx_a_forward, ringx_dist.ringx_a_backward))

    def local(which):          # this rank's sequence chunk of the config's seeded tensor (same bits as the single-GPU run)
        full = wl.make_tensor(cfg, which, device=dev)
        return full[:, :, rank * Nl:(rank + 1) * Nl].contiguous()

    q, k, v, dO = local("q"), local("k"), local("v"), local("do")
    comm = ringx_dist.TorchComm()

    def step():
        o, lse, ctx = fwd(q, k, v, cfg.scale, comm=comm)
        return (o, lse) + tuple(bwd(ctx, dO, comm=comm))

    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize()
    sampler = ClockSampler(dev.index or 0) if rank == 0 else None
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    dist.barrier()
    torch.cuda.synchronize()
    if sampler:
        sampler.start()
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    torch.cuda.synchronize()
    dist.barrier()
    clocks = sampler.stop() if sampler else None
    ms_step = multirank.max_over_ranks(e0.elapsed_time(e1), dist if world > 1 else None, dev) / args.steps
    flops = cfg.fwd_flops + cfg.bwd_flops
    # end to end: pinned host chunks up, the schedule step, the local results down
    host = [t.cpu().pin_memory() for t in (q, k, v, dO)]
    t0 = time.perf_counter()
    dq_, dk_, dv_, do_ = (h.to(dev, non_blocking=True) for h in host)
    o, lse, ctx = fwd(dq_, dk_, dv_, cfg.scale, comm=comm)
    outs = [t.cpu() for t in (o, lse) + tuple(bwd(ctx, do_, comm=comm))]
    torch.cuda.synchronize()
    dt = multirank.max_over_ranks(time.perf_counter() - t0, dist if world > 1 else None, dev)
    tb = q.numel() * q.element_size()
    if rank == 0:
        peaks = load_peaks()
        value = flops / ms_step / 1e9
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": ms_step, "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "bf16",
                "data": "synthetic", "config": dict(workload_config(cfg, "fwd+bwd"), schedule=args.schedule,
                                                    tokens_per_rank=Nl),
                "clocks": clocks,
                "e2e": {"value": flops / dt / 1e12, "unit": UNIT, "ms_per_step": dt * 1e3, "steps": 1,
                        "h2d_bytes_per_step": 4 * tb * world, "d2h_bytes_per_step": (4 * tb + lse.numel() * 4) * world,
                        "entry": f"ringx_dist {args.schedule} forward + backward on pinned host chunks"},
                "gpu_launches": None, "roofline": None, "cpu_baseline": None,
                "frac_of_bf16_peak": {"sustained": value / world / peaks["bf16_tflops_sustained"], "source": peaks["source"]}}
        print(json.dumps(line), flush=True)
    dist.barrier()
    dist.destroy_process_group()


def timed_loop(fn, min_seconds=0.5, min_reps=5, max_reps=400):
    """Per-call CUDA-event timings of `fn` after a warm loop of >= min_seconds (so that clocks and power have settled
    where they will sit under this kernel), collected for >= min_seconds and >= min_reps calls.  Returns the list of ms."""
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    n_warm = 0
    while n_warm < 3 or time.perf_counter() - t0 < min_seconds:
        fn()
        torch.cuda.synchronize()
        n_warm += 1
    per_call = max((time.perf_counter() - t0) / n_warm, 1e-5)
    reps = int(min(max_reps, max(min_reps if per_call < 0.5 else 3, math.ceil(min_seconds / per_call))))
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(reps)]
    for a, b in evs:
        a.record()
        fn()
        b.record()
    torch.cuda.synchronize()
    return [a.elapsed_time(b) for a, b in evs]


def summarise(ms_list, flops):
    med, best = float(np.median(ms_list)), float(min(ms_list))
    return {"ms_median": med, "ms_best": best, "reps": len(ms_list), "tflops_median": flops / med / 1e9,
            "tflops_best": flops / best / 1e9}


def oracle_extrapolated(cfg, q, k, v, do, seconds):
    """cpu_baseline of a config: the oracle as it stands on a sample of query rows of head (0,0) against all keys, sized
    for ~`seconds` of CPU work; the time for the whole config is a LINEAR EXTRAPOLATION (rows are independent), labelled so."""
    from paper_2507_16697_b200 import workloads as wl
    k64, v64 = wl.to_f64_numpy(k[0, 0]), wl.to_f64_numpy(v[0, 0])
    cap = min(cfg.N, 4096)
    q64 = wl.to_f64_numpy(q[0, 0, :cap])
    do64 = wl.to_f64_numpy(do[0, 0, :cap]) if do is not None else None
    n0 = min(32, cap)
    dt0, _ = oracle_sample(cfg, k64, v64, q64[:n0], do64[:n0] if do64 is not None else None, block=64)
    n_rows = int(min(cap, max(n0, seconds / (dt0 / n0) // 32 * 32)))
    dt, fl = oracle_sample(cfg, k64, v64, q64[:n_rows], do64[:n_rows] if do64 is not None else None, block=64)
    full = cfg.fwd_flops + (cfg.bwd_flops if do is not None else 0.0)
    return {"value": fl / dt / 1e12, "unit": UNIT, "cores": host_cores(), "kind": "oracle", "seconds": dt,
            "sample": f"first {n_rows} query rows of head (0,0) against all {cfg.N} keys (oracle.attention_fwd"
                      + (" + attention_bwd" if do is not None else "") + ", fp64 numpy)",
            "full_config_seconds_extrapolated": full / (fl / dt), "extrapolation": "linear in query rows x heads"}


def side_measure(ringx, wl, cfg, dev, oracle_seconds=0.0):
    """Forward (and backward) timing of another BASELINE.json config; context, not the metric.  Each call is timed on its
    own with CUDA events for >= 0.5 s after a >= 0.5 s warm loop; median and best are both reported."""
    tensors = wl.make_qkv(cfg, with_do=cfg.backward, device=dev)
    q, k, v = tensors[:3]
    B, H, N, d = q.shape
    o = torch.empty_like(q)
    lse = torch.empty((B, H, N), dtype=torch.float32, device=dev)
    ws = torch.empty(max(256, ringx.ringx_attn_fwd_workspace_bytes(B, H, N, d, cfg.kv_chunk, q.dtype)),
                     dtype=torch.uint8, device=dev)
    out = {}
    r = summarise(timed_loop(lambda: ringx.ringx_attn_fwd(q, k, v, cfg.kv_chunk, cfg.scale, o=o, lse=lse, workspace=ws)),
                  cfg.fwd_flops)
    out["fwd"] = r
    out["fwd_ms"], out["fwd_tflops"] = r["ms_median"], r["tflops_median"]
    if cfg.backward:
        wsb = torch.empty(max(256, ringx.ringx_attn_bwd_workspace_bytes(B, H, N, d, cfg.kv_chunk, q.dtype)),
                          dtype=torch.uint8, device=dev)
        dq, dk, dv = torch.empty_like(q), torch.empty_like(q), torch.empty_like(q)
        r = summarise(timed_loop(lambda: ringx.ringx_attn_bwd(q, k, v, o, lse, tensors[3], cfg.kv_chunk, cfg.scale,
                                                              workspace=wsb, dq=dq, dk=dk, dv=dv)), cfg.bwd_flops)
        out["bwd"] = r
        out["bwd_ms"], out["bwd_tflops"] = r["ms_median"], r["tflops_median"]
    if oracle_seconds > 0:
        out["cpu_baseline"] = oracle_extrapolated(cfg, q, k, v, tensors[3] if cfg.backward else None, oracle_seconds)
    return out


def c1_measure(ringx, wl, dev):
    """BASELINE.json configs[0] (fp32, N = 1024, 4 chunks): the fp32 (3-term bf16 split, tensor-core) path's time and the oracle's, both on the whole config."""
    from oracle import attention as orc
    cfg = wl.CONFIGS["C1"]
    q, k, v = wl.make_qkv(cfg, device=dev)
    r = summarise(timed_loop(lambda: ringx.ringx_attn_fwd(q, k, v, cfg.kv_chunk, cfg.scale), min_seconds=0.2), cfg.fwd_flops)
    q64, k64, v64 = (wl.to_f64_numpy(t[0, 0]) for t in (q, k, v))
    t0 = time.perf_counter()
    orc.attention_fwd_chunked(q64, k64, v64, cfg.scale, list(range(0, cfg.N + 1, cfg.kv_chunk)))
    dt = time.perf_counter() - t0
    return {"fwd": r, "cpu_baseline": {"value": cfg.fwd_flops / dt / 1e12, "unit": UNIT, "cores": host_cores(),
                                       "kind": "oracle", "seconds": dt,
                                       "sample": "the whole config (oracle.attention_fwd_chunked, 4 chunks of 256)"}}


def next_rows_measure(ringx, wl, dev, reps=5):
    """Short timings of the SURVEY.md §8(f) rows built so far (context, not the metric): grouped-query attention,
    the per-device RingX backward step, and the N-operand Eq. 5 kernels of RingX_a."""
    out = {}

    def timeit(fn):
        # the same loop as side_measure: >= 0.5 s warm, then >= 0.5 s and >= `reps` calls timed one by one; the median, so that
        # every figure of the line is a sustained one and reads the same way in every run
        return float(np.median(timed_loop(fn, min_seconds=0.5, min_reps=reps)))

    # GQA: 16 query heads on 4 kv heads, N = 32768, d = 128, 4 passes of 8192 keys
    B, Hq, Hkv, N, d, chunk = 1, 16, 4, 32768, 128, 8192
    scale = d ** -0.5
    q = wl.make_tensor((B, Hq, N, d), "q", seed=77, dtype="bf16", device=dev)
    do = wl.make_tensor((B, Hq, N, d), "do", seed=77, dtype="bf16", device=dev)
    k = wl.make_tensor((B, Hkv, N, d), "k", seed=77, dtype="bf16", device=dev)
    v = wl.make_tensor((B, Hkv, N, d), "v", seed=77, dtype="bf16", device=dev)
    o, lse = ringx.ringx_attn_fwd_gqa(q, k, v, chunk, scale)
    fl = 4.0 * B * Hq * N * N * d
    ms = timeit(lambda: ringx.ringx_attn_fwd_gqa(q, k, v, chunk, scale, o=o, lse=lse))
    out["gqa_16q4kv_N32768_d128"] = {"fwd_tflops": fl / ms / 1e9}
    ms = timeit(lambda: ringx.ringx_attn_bwd_gqa(q, k, v, o, lse, do, chunk, scale))
    out["gqa_16q4kv_N32768_d128"]["bwd_tflops"] = 2.5 * fl / ms / 1e9
    # MLA shapes (d_qk = 192, d_v = 128): 8 heads, N = 65536, 4 passes of 16384 keys; FLOPs 2 N^2 (192 + 128) forward,
    # 2 N^2 (192 + 128 + 128 + 192 + 192) backward per head
    Hm, Nm, cm = 8, 65536, 16384
    qm, km = (wl.make_tensor((1, Hm, Nm, 192), w, seed=78, dtype="bf16", device=dev) for w in "qk")
    vm, dom = (wl.make_tensor((1, Hm, Nm, 128), w, seed=78, dtype="bf16", device=dev) for w in ("v", "do"))
    om, lm_ = ringx.ringx_attn_fwd_mla(qm, km, vm, cm, 192 ** -0.5)
    ms = timeit(lambda: ringx.ringx_attn_fwd_mla(qm, km, vm, cm, 192 ** -0.5, o=om, lse=lm_))
    out["mla_dqk192_dv128_H8_N65536"] = {"fwd_tflops": 2.0 * Hm * Nm * Nm * 320 / ms / 1e9}
    ms = timeit(lambda: ringx.ringx_attn_bwd_mla(qm, km, vm, om, lm_, dom, cm, 192 ** -0.5))
    out["mla_dqk192_dv128_H8_N65536"]["bwd_tflops"] = 2.0 * Hm * Nm * Nm * 832 / ms / 1e9
    del qm, km, vm, dom, om, lm_
    # RingX backward step: 16384 local query rows against one 16384-key chunk of another rank (global lse)
    ql, ol, dol = (t[:, :4, :16384].contiguous() for t in (q, o, do))
    lsel = lse[:, :4, :16384].contiguous()
    kc, vc = k[:, :, 16384:].contiguous(), v[:, :, 16384:].contiguous()
    acc = torch.zeros(ql.shape, dtype=torch.float32, device=dev)
    ms = timeit(lambda: ringx.ringx_attn_bwd_partial(ql, kc, vc, ol, lsel, dol, scale, dq_acc=acc))
    out["bwd_partial_Nq16384_Nk16384_d128"] = {"tflops": 10.0 * B * 4 * 16384 * 16384 * d / ms / 1e9}
    # split-KV: the paper's per-device regime: 2048 local query tokens x 8 heads = 64 CTAs against a
    # 65536-key gathered chunk; the library splits the keys over CTA groups and merges by Eq. 5 inside the pass
    qs = q[:, :8, :2048].contiguous()
    ks, vs = torch.cat([k, k], dim=2)[:, :, :65536].contiguous(), torch.cat([v, v], dim=2)[:, :, :65536].contiguous()
    ks = ks.repeat(1, 2, 1, 1).contiguous()
    vs = vs.repeat(1, 2, 1, 1).contiguous()
    fls = 4.0 * 8 * 2048 * 65536 * d
    ms0 = timeit(lambda: ringx.ringx_attn_chunk_fwd(qs, ks, vs, scale))
    ms1 = timeit(lambda: ringx.ringx_attn_chunk_fwd_ex(qs, ks, vs, scale))
    out["split_kv_Nq2048_Nk65536_H8_d128"] = {"unsplit_tflops": fls / ms0 / 1e9, "split_tflops": fls / ms1 / 1e9}
    del qs, ks, vs
    # Eq. 5 with N operands: bytes per row = d*4 read + d*4 written (+ 12 / + 12)
    rows = 1 << 21
    lo = torch.randn(rows, d, device=dev)
    ll = torch.randn(rows, device=dev)
    lm = ll + 1.0
    ms = timeit(lambda: ringx.ringx_eq5_scale(lo, ll, lm, inplace=True))
    out["eq5_scale_gbs"] = rows * (2 * d * 4 + 12) / ms / 1e6
    den = torch.ones(rows, device=dev)
    ms = timeit(lambda: ringx.ringx_eq5_finalize(lo, den, lm, out_dtype=torch.float32))
    out["eq5_finalize_gbs"] = rows * (2 * d * 4 + 12) / ms / 1e6
    del lo, ll, lm, den, q, k, v, o, do, acc
    # NEXT-4, the Turbulence-Transformer tokeniser: 512^3 x 4 fp32 state (2.1 GB, larger than L2),
    # Gaussian filter k^3 with stride k.  Algorithmic bytes = 16 per input voxel + 16 (8 for bf16) per token.
    G = 512
    y = wl.make_field(1, G, G, G, seed=20250722, device=dev)
    tok = {}
    for kk, odt in ((4, torch.float32), (2, torch.bfloat16), (8, torch.float32), (1, torch.float32)):
        size = (G, G, G) if kk > 1 else (G // 2, G, G)      # k = 1: a half-domain crop (pure copy)
        t = ringx.ringx_fidelity_tokens(y, (0, 0, 0), size, kk, out_dtype=odt)
        ms = timeit(lambda: ringx.ringx_fidelity_tokens(y, (0, 0, 0), size, kk, tokens=t))
        nvox = size[0] * size[1] * size[2]
        byt = nvox * 16 + (nvox // kk ** 3) * 4 * t.element_size()
        tok[f"k{kk}_{'bf16' if odt == torch.bfloat16 else 'f32'}"] = {"ms": ms, "gbs": byt / ms / 1e6,
                                                                   "tokens": nvox // kk ** 3}
    peaks = load_peaks()
    tok["roofline"] = {"bound": "hbm", "kernel": "fidelity_tokens_kernel (k=4, f32 tokens)", "achieved": tok["k4_f32"]["gbs"],
                       "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": tok["k4_f32"]["gbs"] / peaks["hbm_gbs"]}
    out["fidelity_tokens_512cube"] = tok
    del y, t
    # NEXT-4, Table II's projection GEMMs around the attention kernel at C3's block shape
    # (B=1, S=262144, h=1024): 6*b*S*h^2 and 2*b*S*h^2 FLOPs; the head split / merge is fused into the TMA coordinates.
    B, S, H, d = 1, 262144, 8, 128
    h = H * d
    x, wq, wo = wl.make_block_inputs(B, S, H, d, device=dev)
    q, k, v = ringx.ringx_qkv_proj(x, wq, H)
    ms_q = timeit(lambda: ringx.ringx_qkv_proj(x, wq, H, q=q, k=k, v=v))
    yb = ringx.ringx_out_proj(q, wo)
    ms_o = timeit(lambda: ringx.ringx_out_proj(q, wo, y=yb))
    tq, to = 6.0 * B * S * h * h / ms_q / 1e9, 2.0 * B * S * h * h / ms_o / 1e9
    dyb = wl.make_tensor((B, S, h), "do", seed=5, device=dev)
    ms_ob = timeit(lambda: ringx.ringx_out_proj_bwd(dyb, q, wo))          # data + weight gradient: 2 x 2*b*S*h^2
    ms_qb = timeit(lambda: ringx.ringx_qkv_proj_bwd(q, k, v, x, wq))      # 2 x 6*b*S*h^2
    # the whole block of Table II as a training step: projections + attention, forward and backward
    ws_f = torch.empty(ringx.ringx_attn_block_fwd_workspace_bytes(B, S, H, d, 32768), dtype=torch.uint8, device=dev)
    ws_b = torch.empty(ringx.ringx_attn_block_bwd_workspace_bytes(B, S, H, d, 32768), dtype=torch.uint8, device=dev)

    def block_step():
        ringx.ringx_attn_block_fwd(x, wq, wo, H, 32768, d ** -0.5, y=yb, workspace=ws_f)
        ringx.ringx_attn_block_bwd(x, wq, wo, dyb, ws_f, H, 32768, d ** -0.5, workspace=ws_b)

    block_step()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    block_step()
    e1.record()
    torch.cuda.synchronize()
    ms_blk = e0.elapsed_time(e1)
    fl_blk = 14.0 * B * H * S * S * d + 3.0 * 8.0 * B * S * h * h        # attention fwd+bwd + projections fwd+bwd
    out["block_fwd_bwd_S262144_h1024"] = {"ms": ms_blk, "tflops": fl_blk / ms_blk / 1e9}
    del ws_f, ws_b
    out["projections_S262144_h1024"] = {
        "qkv_ms": ms_q, "qkv_tflops": tq, "out_ms": ms_o, "out_tflops": to,
        "out_bwd_ms": ms_ob, "out_bwd_tflops": 4.0 * B * S * h * h / ms_ob / 1e9,
        "qkv_bwd_ms": ms_qb, "qkv_bwd_tflops": 12.0 * B * S * h * h / ms_qb / 1e9,
        "roofline": {"bound": "tensor", "kernel": "proj_gemm_kernel<QKV>", "achieved": tq, "peak": peaks["bf16_tflops"],
                     "unit": "TFLOP/s", "frac": tq / peaks["bf16_tflops"],
                     "peak_kind": "bf16 dense, burst (kernel timed alone), measured"}}
    return out


if __name__ == "__main__":
    main()
