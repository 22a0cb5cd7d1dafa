#!/usr/bin/env python
"""bench.py — TTT update+apply throughput of the B200-native hot path.

Metric (BASELINE.json:metric): "TTT update+apply tokens/s on 1 B200; % of dense-BF16 tensor peak".
A step = one `ttt_chunk_step` (update Eq. 8 then apply Eq. 4, all heads) over one chunk of the
workload. Default workload = BASELINE.json:configs[1] ("cfg2": VGGT-Large-shaped single chunk,
8 frames x 1374 tokens, 16 heads x 64, SwiGLU hidden 128, bf16 activations / fp32 fast weights,
L2-normalised K, lr 0.01). Every step is a NEW single-chunk sequence: the fast weights are reset
with `ttt_init` between steps (outside the per-step CUDA events, inside the outer bracket).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg2|cfg3|...] [--impl reference]

N > 1 (torchrun): every rank runs its own independent sequences (weak scaling, no collective on
the data path — heads/sequences are independent units).
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import torch

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import ttt_inputs as ti  # noqa: E402

L2_BYTES = 126 * 2 ** 20


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return {"bf16_tflops": d["bf16_tflops"], "bf16_tflops_sustained": d.get("bf16_tflops_sustained"),
                "hbm_gbs": d["hbm_gbs"], "source": "measured (MEASURED_PEAKS.json)"}
    return {"bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "hbm_gbs": 6650.0,
            "source": "fallback (B200_PROFILING.md)"}


class ClockSampler:
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self._nv = pynvml
            self._h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self._nv = None

    def _run(self):
        nv = self._nv
        names = {"hw_slowdown": getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8),
                 "hw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40),
                 "sw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20),
                 "sw_power_cap": getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4)}
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self._h, nv.NVML_CLOCK_SM))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self._h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self._h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                break
            time.sleep(0.0005)

    def __enter__(self):
        if self._nv is not None:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._thr is not None:
            self._thr.join()

    def summary(self):
        s = sorted(self.samples)
        return {"sm_mhz": (s[len(s) // 2] if s else None), "sm_max_mhz": self.max_mhz,
                "samples": len(s), "reasons": sorted(self.reasons)}


def flops_per_chunk(w: ti.TTTWorkload, M: int, part: str = "step") -> float:
    """Algorithmic tensor flops: update 12 M d H, apply 6 M d H,
    plus Newton-Schulz n (4 r^2 c + 2 r^3) per matrix, r = hd, c = H."""
    base = {"update": 12, "apply": 6, "step": 18}[part] * M * w.d * w.hidden
    if part != "apply" and w.ns_iters:
        base += w.ns_iters * (4 * w.hd ** 2 * w.hidden + 2 * w.hd ** 3) * 3 * w.nh
    return float(base)


def bytes_per_chunk(w: ti.TTTWorkload, M: int) -> float:
    """Algorithmic HBM bytes: read Q, K, V, write O (bf16) + lr (fp32 per head and token)."""
    return float(4 * M * w.d * 2 + 4 * M * w.nh)


# --------------------------------------------------------------------------------------------
# reference arm: the float64 oracle on the host cores
# --------------------------------------------------------------------------------------------
def run_reference(args, w, rank, world):
    if rank != 0:
        return
    from oracle import ttt_oracle as orc
    heads = sorted({0, w.nh - 1})
    ws = ti.scaled(w, nh=len(heads))
    W1, W2, W3 = ti.fast_weights(w)
    Q, K, V, lr = ti.TokenStream(w).next_chunk()
    M = Q.shape[0]
    cols = torch.cat([torch.arange(h * w.hd, (h + 1) * w.hd) for h in heads])
    Qs, Ks, Vs = (X[:, cols].contiguous() for X in (Q, K, V))
    lrs = lr[heads].contiguous()
    Ws = [X[heads].contiguous() for X in (W1, W2, W3)]

    def step():
        o = orc.OracleTTT(*Ws, ns_iters=w.ns_iters, renorm=w.renorm)
        o.chunk_step(Qs, Ks, Vs, lrs)

    for _ in range(min(args.warmup, 1)):
        step()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        step()
    dt = time.perf_counter() - t0
    ms = dt / args.steps * 1e3
    # heads are independent: tokens/s for all nh heads = tokens * (heads run / nh) / time
    value = M * len(heads) / w.nh / (ms * 1e-3)
    sample = f"heads {heads} of {w.nh}, all {M} tokens of one chunk per step (exact: heads are independent)"
    line = {"impl": "reference", "metric": "ttt_update_apply_tokens_per_s", "value": value,
            "unit": "tokens/s", "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "tokens_per_step": M, "nh": w.nh, "hd": w.hd,
                       "hidden": w.hidden, "ns_iters": w.ns_iters, "renorm": w.renorm},
            "cpu_baseline": {"value": value, "unit": "tokens/s", "cores": orc.num_threads(),
                             "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": "tokens/s", "h2d_bytes_per_step": 0,
                    "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def cpu_baseline(w, budget_s=12.0):
    from oracle import ttt_oracle as orc
    heads = list(range(w.nh))
    W1, W2, W3 = ti.fast_weights(w)
    Q, K, V, lr = ti.TokenStream(w).next_chunk()
    M = Q.shape[0]
    reps, t0 = 0, time.perf_counter()
    while True:
        o = orc.OracleTTT(W1, W2, W3, ns_iters=w.ns_iters, renorm=w.renorm)
        o.chunk_step(Q, K, V, lr)
        reps += 1
        if time.perf_counter() - t0 > budget_s or reps >= 64:
            break
    dt = time.perf_counter() - t0
    return {"value": reps * M / dt, "unit": "tokens/s", "cores": orc.num_threads(), "kind": "oracle",
            "sample": f"{reps} x one full chunk ({M} tokens, all {len(heads)} heads) of {w.name}, {dt:.1f} s"}


# --------------------------------------------------------------------------------------------
# our arm
# --------------------------------------------------------------------------------------------
def run_ours(args, w, rank, local_rank, world):
    from paper_2604_08542_b200 import TTT, TTT_BF16, TTT_F32
    dev = torch.device("cuda", local_rank)
    torch.cuda.set_device(dev)
    peaks = _peaks()
    M = w.chunk_tokens
    n_sets = max(4, min(8, -(-2 * L2_BYTES // int(bytes_per_chunk(w, M)))))  # working set > 2x L2
    W1, W2, W3 = (x.to(dev) for x in ti.fast_weights(w))
    sets = []
    for r in range(n_sets):
        stream = ti.TokenStream(ti.scaled(w, seed=w.seed + 1000 * rank + r))
        Q, K, V, lr = stream.next_chunk()
        sets.append([Q, K, V, lr])
    host = [[x.pin_memory() for x in s] for s in sets[:2]]
    dsets = [[x.to(dev) for x in s] + [torch.empty(M, w.d, dtype=w.torch_dtype, device=dev)] for s in sets]
    ttt = TTT(w.nh, w.hd, w.hidden, TTT_BF16 if w.act_dtype == "bf16" else TTT_F32,
              ns_iters=w.ns_iters, renorm=w.renorm, max_tokens=M, device=local_rank)

    def barrier():
        torch.cuda.synchronize(dev)
        if world > 1:
            torch.distributed.barrier()
        torch.cuda.synchronize(dev)

    def step(i):
        Q, K, V, lr, O = dsets[i % n_sets]
        ttt.ttt_chunk_step(Q, K, V, lr, O=O)

    for i in range(max(args.warmup, 3)):
        ttt.ttt_init(W1, W2, W3)
        step(i)
    barrier()
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
           for _ in range(args.steps)]
    n0 = ttt.launch_count()
    with ClockSampler(local_rank) as clocks:
        t0 = time.perf_counter()
        for i in range(args.steps):
            ttt.ttt_init(W1, W2, W3)                       # new sequence: reset the memory
            evs[i][0].record()
            step(i)
            evs[i][1].record()
        barrier()
        wall_ms = (time.perf_counter() - t0) * 1e3
    launches = ttt.launch_count() - n0
    step_ms = [a.elapsed_time(b) for a, b in evs]
    total_ms = torch.tensor([sum(step_ms)], dtype=torch.float64, device=dev)
    if world > 1:
        torch.distributed.all_reduce(total_ms, op=torch.distributed.ReduceOp.MAX)
    ms_per_step = float(total_ms.item()) / args.steps
    value = world * M / (ms_per_step * 1e-3)

    # ---- per-kernel pass: same work as update / commit / apply calls with events between ----
    kev = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(args.steps)]
    for i in range(args.steps):
        Q, K, V, lr, O = dsets[i % n_sets]
        ttt.ttt_init(W1, W2, W3)
        kev[i][0].record(); ttt.ttt_accumulate(K, V, lr)
        kev[i][1].record(); ttt.ttt_commit()
        kev[i][2].record(); ttt.ttt_apply(Q, O=O)
        kev[i][3].record()
    torch.cuda.synchronize(dev)
    k_ms = [sum(e[j].elapsed_time(e[j + 1]) for e in kev) / args.steps for j in range(3)]
    upd_tflops = flops_per_chunk(w, M, "update") / (k_ms[0] * 1e-3) / 1e12 if w.ns_iters == 0 else \
        12.0 * M * w.d * w.hidden / (k_ms[0] * 1e-3) / 1e12
    app_tflops = flops_per_chunk(w, M, "apply") / (k_ms[2] * 1e-3) / 1e12
    step_tflops = flops_per_chunk(w, M, "step") / (ms_per_step * 1e-3) / 1e12
    # dram__bytes_read.sum + dram__bytes_write.sum of bf16_update_kernel, one launch, from the
    # `ncu --set full` captures summarised in profiles/r01e_cfg2_startup_commit.md (cfg2), r01d_cfg2_cfg4_update.md
    # (cfg4) and r01c_cfg5.md (None = not captured)
    traffic = {"cfg2": 48135424 + 533760, "cfg4": 187718912 + 4704512,
               "cfg5": 186227456 + 9412352}.get(w.name)
    # (the per-kernel pass calls ttt_accumulate / ttt_commit / ttt_apply separately; inside
    #  ttt_chunk_step the plain commit is fused into the update kernel's tail)
    upd_kernel = ("bf16_update_wide_kernel" if w.hd == 128 else "bf16_update_kernel") \
        if w.act_dtype == "bf16" else "f32 path"
    roofline = {"kernel": upd_kernel,
                "bound": "tensor", "achieved": upd_tflops, "peak": peaks["bf16_tflops"],
                "unit": "TFLOP/s", "frac": upd_tflops / peaks["bf16_tflops"], "traffic": traffic,
                "peak_source": peaks["source"] + ", burst figure (step is tens of microseconds)",
                "flops_per_launch": 12.0 * M * w.d * w.hidden,
                "kernel_ms": {"update(accumulate)": k_ms[0], "commit": k_ms[1], "apply": k_ms[2]},
                "apply_tflops": app_tflops, "apply_frac": app_tflops / peaks["bf16_tflops"],
                "step_tflops": step_tflops, "step_frac": step_tflops / peaks["bf16_tflops"],
                "step_frac_of_sustained": (step_tflops / peaks["bf16_tflops_sustained"]
                                           if peaks["bf16_tflops_sustained"] else None),
                "hbm_gbs_algorithmic": bytes_per_chunk(w, M) / (ms_per_step * 1e-3) / 1e9,
                "hbm_frac": bytes_per_chunk(w, M) / (ms_per_step * 1e-3) / 1e9 / peaks["hbm_gbs"]}

    # ---- end to end: pinned host buffers in, O back to the host, through the same C-ABI call ----
    e2e = None
    if not args.no_e2e:
        n_e2e = min(args.steps, 20)
        streams = [torch.cuda.Stream(dev) for _ in range(2)]
        hO = [torch.empty(M, w.d, dtype=w.torch_dtype).pin_memory() for _ in range(2)]
        ctxs = [ttt, TTT(w.nh, w.hd, w.hidden, TTT_BF16 if w.act_dtype == "bf16" else TTT_F32,
                         ns_iters=w.ns_iters, renorm=w.renorm, max_tokens=M, device=local_rank)]

        def e2e_step(i):
            b = i & 1
            with torch.cuda.stream(streams[b]):
                Q, K, V, lr, O = dsets[b]
                for dst, src in zip((Q, K, V, lr), host[b]):
                    dst.copy_(src, non_blocking=True)
                ctxs[b].ttt_init(W1, W2, W3)
                ctxs[b].ttt_chunk_step(Q, K, V, lr, O=O)
                hO[b].copy_(O, non_blocking=True)

        for i in range(2):
            e2e_step(i)
        barrier()
        t0 = time.perf_counter()
        for i in range(n_e2e):
            streams[i & 1].synchronize()          # buffer b is free again (its O reached the host)
            e2e_step(i)
        barrier()
        dt = torch.tensor([time.perf_counter() - t0], dtype=torch.float64, device=dev)
        if world > 1:
            torch.distributed.all_reduce(dt, op=torch.distributed.ReduceOp.MAX)
        esz = 2 if w.act_dtype == "bf16" else 4
        e2e = {"value": world * n_e2e * M / float(dt.item()), "unit": "tokens/s",
               "h2d_bytes_per_step": 3 * M * w.d * esz + 4 * w.nh * M,
               "d2h_bytes_per_step": M * w.d * esz, "steps": n_e2e,
               "how": "pinned host Q,K,V,lr -> device, ttt_init + ttt_chunk_step, O -> pinned host; "
                      "two streams double-buffered; wall clock, max over ranks"}
        ctxs[1].close()

    if rank != 0:
        ttt.close()
        return
    line = {"metric": "ttt_update_apply_tokens_per_s", "value": value, "unit": "tokens/s",
            "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": w.act_dtype, "data": "synthetic",
            "config": {"workload": w.name, "tokens_per_step": M, "nh": w.nh, "hd": w.hd,
                       "hidden": w.hidden, "ns_iters": w.ns_iters, "renorm": w.renorm,
                       "l2_k": w.l2_k, "lr": w.lr, "parallelism": f"replicas x{world}",
                       "l2_policy": f"{n_sets} distinct resident input/output sets rotated "
                                    f"({n_sets * bytes_per_chunk(w, M) / 2**20:.0f} MiB > 2x L2)",
                       "reset": "ttt_init between steps, outside the per-step CUDA events",
                       "timing": "sum of per-step CUDA-event durations on the launch stream, max over ranks"},
            "pct_of_bf16_peak": 100.0 * step_tflops / peaks["bf16_tflops"],
            "wall_ms_per_step_incl_reset": wall_ms / args.steps,
            "clocks": clocks.summary(), "e2e": e2e, "gpu_launches": int(launches),
            "roofline": roofline}
    if world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(w)
    print(json.dumps(line), flush=True)
    ttt.close()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg2", choices=sorted(ti.CONFIGS))
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    w = ti.CONFIGS[args.workload]
    if args.impl == "reference":
        run_reference(args, w, rank, world)
        return
    if world > 1:
        torch.distributed.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    try:
        run_ours(args, w, rank, local_rank, world)
    finally:
        if world > 1:
            torch.distributed.destroy_process_group()


if __name__ == "__main__":
    main()
