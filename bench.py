#!/usr/bin/env python
"""bench.py — TTT update+apply throughput of the B200-native hot path.

Metric (BASELINE.json:metric): "TTT update+apply tokens/s on 1 B200; % of dense-BF16 tensor peak".
A step = one `ttt_chunk_step` (update Eq. 8 then apply Eq. 4, all heads) over one chunk of the
workload. The metric names no config, so the default run times ALL FOUR performance configs of
BASELINE.json (cfg2 .. cfg5) in one process, plus the paper's own shape (paper_k4: one head of 1024,
hidden 4096, 82 440-token chunks): the top-level `value` / `ms_per_step` /
`config.workload` are those of cfg5, the largest single-GPU configuration of BASELINE.json, and
`workloads` carries the same numbers (with their own `roofline`) for every workload. Every step is a new chunk of a
sequence: the fast weights are reset with `ttt_init` between steps (outside the per-step CUDA
events, inside the outer bracket), inputs rotate over distinct resident sets larger than 2x L2.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg2|cfg3|cfg4|cfg5|all]
                  [--impl reference]          (also --workload paper_k4 | paper_k1)

N > 1: launched by torchrun (RANK / LOCAL_RANK / WORLD_SIZE in the environment) every rank runs its
own independent sequences (weak scaling, no collective on the data path — heads and sequences are
independent units); launched WITHOUT torchrun, `--gpus N` starts the N ranks
itself (torchrun --standalone) and fails loudly if the box has fewer than N GPUs.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import torch

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import ttt_inputs as ti  # noqa: E402

L2_BYTES = 126 * 2 ** 20
PERF_WORKLOADS = ("cfg2", "cfg3", "cfg4", "cfg5", "paper_k4")   # BASELINE.json's four + the paper's own shape
HEADLINE = "cfg5"

# dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the workload's dominant kernel, from the
# `ncu --set full` captures summarised under profiles/ (file and commit named per entry)
_CAP = "profiles/r02_ncu_full.md (commits 5afd7f3 / 3d966e7), capture "
TRAFFIC = {
    "cfg2": {"bytes": 48692992, "capture": _CAP + "r02_cfg2_update"},
    # cfg3's dominant kernel is cfg4's (same grid, 86 instead of 344 tiles per CTA): bytes scaled from the
    # cfg4 capture by the token count (K + V + lr are the kernel's only DRAM traffic, 1.05x algorithmic)
    "cfg3": {"bytes": int(191860736 * 10992 / 43968), "capture": _CAP + "r02_cfg4_update, scaled by tokens"},
    "cfg4": {"bytes": 191860736, "capture": _CAP + "r02_cfg4_update"},
    "cfg5": {"bytes": 196604672, "capture": _CAP + "r02_cfg5_update"},
    "paper_k4": {"bytes": 2872674800 + 4316396344,
                 "capture": _CAP + "r02_k4_forward (update) + r02_k4_mn (gradient): the two launches of ttt_accumulate"},
}


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return {"bf16_tflops": d["bf16_tflops"], "bf16_tflops_sustained": d.get("bf16_tflops_sustained"),
                "hbm_gbs": d["hbm_gbs"], "source": "measured (MEASURED_PEAKS.json)"}
    return {"bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "hbm_gbs": 6650.0,
            "source": "fallback (B200_PROFILING.md)"}


class ClockSampler:
    """Samples SM clock and throttle reasons through NVML for the whole run; only samples taken while
    a GPU-busy phase is open (`with sampler.busy():` — timed loops, per-kernel pass, e2e pass) count."""

    def __init__(self, index: int):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._busy = 0
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
            if self._busy:
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

    class _Busy:
        def __init__(self, s):
            self.s = s

        def __enter__(self):
            self.s._busy += 1

        def __exit__(self, *a):
            self.s._busy -= 1

    def busy(self):
        return ClockSampler._Busy(self)

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


def n_input_sets(w: ti.TTTWorkload) -> int:
    return max(4, min(8, -(-2 * L2_BYTES // int(bytes_per_chunk(w, w.chunk_tokens)))))


def config_of(w: ti.TTTWorkload, world: int) -> dict:
    """The `config` object: identical in the GPU arm and the reference arm (workload description only)."""
    n_sets = n_input_sets(w)
    return {"workload": w.name, "tokens_per_step": w.chunk_tokens, "nh": w.nh, "hd": w.hd,
            "hidden": w.hidden, "ns_iters": w.ns_iters, "renorm": w.renorm, "l2_k": w.l2_k, "lr": w.lr,
            "rho": w.rho, "parallelism": f"replicas x{world}",
            "l2_policy": f"{n_sets} distinct resident input/output sets rotated "
                         f"({n_sets * bytes_per_chunk(w, w.chunk_tokens) / 2**20:.0f} MiB > 2x L2)",
            "reset": "ttt_init between steps, outside the per-step CUDA events",
            "timing": "sum of per-step CUDA-event durations on the launch stream, max over ranks"}


# --------------------------------------------------------------------------------------------
# the float64 oracle on the host cores: cpu_baseline leg and the reference arm
# --------------------------------------------------------------------------------------------
# tokens of one chunk an oracle step works on (all heads, OpenMP over heads): sized so that a step
# takes a few seconds on the box's cores; cfg5's full chunk would take ~13 s
REF_TOKENS = {"cfg2": 10992, "cfg3": 10992, "cfg4": 16384, "cfg5": 8192, "paper_k4": 384, "paper_k1": 1024}


def _oracle_sample(w: ti.TTTWorkload):
    ws = ti.scaled(w, n_frames=w.frames_per_chunk)            # the first chunk only
    W1, W2, W3 = ti.fast_weights(w)
    Q, K, V, lr = ti.TokenStream(ws).next_chunk()
    m = min(REF_TOKENS.get(w.name, w.chunk_tokens), Q.shape[0])
    return (W1, W2, W3), (Q[:m].contiguous(), K[:m].contiguous(), V[:m].contiguous(), lr[:, :m].contiguous()), m


def run_reference(args, w, rank, world):
    """--impl reference: the oracle as it stands, on the host cores, same metric / config / unit.
    Rank 0 alone works; the other ranks exit at once."""
    if rank != 0:
        return
    from oracle import ttt_oracle as orc
    Ws, toks, m = _oracle_sample(w)

    def step():
        o = orc.OracleTTT(*Ws, ns_iters=w.ns_iters, renorm=w.renorm)
        o.chunk_step(*toks)

    for _ in range(min(args.warmup, 1)):
        step()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        step()
    dt = time.perf_counter() - t0
    ms = dt / args.steps * 1e3
    value = m / (ms * 1e-3)
    sample = (f"per step: update + apply of the first {m} tokens of one {w.name} chunk "
              f"({w.chunk_tokens} tokens), all {w.nh} heads, float64; cost is linear in tokens")
    cores = min(orc.num_threads(), w.nh)
    line = {"impl": "reference", "metric": "ttt_update_apply_tokens_per_s", "value": value,
            "unit": "tokens/s", "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "config": config_of(w, args.gpus),
            "cpu_baseline": {"value": value, "unit": "tokens/s", "cores": cores, "kind": "oracle",
                             "sample": sample},
            "e2e": {"value": value, "unit": "tokens/s", "h2d_bytes_per_step": 0,
                    "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def cpu_baseline(w, budget_s=12.0):
    from oracle import ttt_oracle as orc
    Ws, toks, m = _oracle_sample(w)
    reps, t0 = 0, time.perf_counter()
    while True:
        o = orc.OracleTTT(*Ws, ns_iters=w.ns_iters, renorm=w.renorm)
        o.chunk_step(*toks)
        reps += 1
        if time.perf_counter() - t0 > budget_s or reps >= 64:
            break
    dt = time.perf_counter() - t0
    return {"value": reps * m / dt, "unit": "tokens/s", "cores": min(orc.num_threads(), w.nh),
            "kind": "oracle",
            "sample": f"{reps} x update + apply of the first {m} tokens of one {w.name} chunk, all "
                      f"{w.nh} heads (OpenMP over heads), {dt:.1f} s"}


# --------------------------------------------------------------------------------------------
# our arm
# --------------------------------------------------------------------------------------------
def measure(args, w, rank, local_rank, world, clocks, peaks, want_e2e):
    """Times one workload; returns (result dict, launches in the timed region)."""
    from paper_2604_08542_b200 import TTT, TTT_BF16, TTT_F32
    dev = torch.device("cuda", local_rank)
    M = w.chunk_tokens
    n_sets = n_input_sets(w)
    W1, W2, W3 = (x.to(dev) for x in ti.fast_weights(w))
    dsets, host = [], []
    for r in range(n_sets):
        stream = ti.TokenStream(ti.scaled(w, seed=w.seed + 1000 * rank + r, n_frames=w.frames_per_chunk))
        s = list(stream.next_chunk())
        if want_e2e and r < 2:
            host.append([x.pin_memory() for x in s])
        dsets.append([x.to(dev) for x in s] + [torch.empty(M, w.d, dtype=w.torch_dtype, device=dev)])
        del s
    dt_code = TTT_BF16 if w.act_dtype == "bf16" else TTT_F32
    ttt = TTT(w.nh, w.hd, w.hidden, dt_code, ns_iters=w.ns_iters, renorm=w.renorm, max_tokens=M,
              device=local_rank)

    def barrier():
        torch.cuda.synchronize(dev)
        if world > 1:
            torch.distributed.barrier()
        torch.cuda.synchronize(dev)

    def step(i):
        Q, K, V, lr, O = dsets[i % n_sets]
        ttt.ttt_chunk_step(Q, K, V, lr, O=O)

    warm = max(args.warmup, 3)
    for i in range(warm):
        ttt.ttt_init(W1, W2, W3)
        step(i)
    barrier()
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
           for _ in range(args.steps)]
    n0 = ttt.launch_count()
    with clocks.busy():
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

    # ---- per-call pass: the same work as three separate C-ABI calls with events between them ----
    # (inside ttt_chunk_step the plain commit is fused into the update kernel's tail and the apply
    #  overlaps its prologue with the commit through programmatic dependent launch, so these legs,
    #  each including its own launch gap, sum to MORE than a step)
    kev = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(args.steps)]
    with clocks.busy():
        for i in range(args.steps):
            Q, K, V, lr, O = dsets[i % n_sets]
            ttt.ttt_init(W1, W2, W3)
            kev[i][0].record(); ttt.ttt_accumulate(K, V, lr)
            kev[i][1].record(); ttt.ttt_commit()
            kev[i][2].record(); ttt.ttt_apply(Q, O=O)
            kev[i][3].record()
        torch.cuda.synchronize(dev)
    k_ms = [sum(e[j].elapsed_time(e[j + 1]) for e in kev) / args.steps for j in range(3)]
    upd_flops = 12.0 * M * w.d * w.hidden
    upd_tflops = upd_flops / (k_ms[0] * 1e-3) / 1e12
    app_tflops = flops_per_chunk(w, M, "apply") / (k_ms[2] * 1e-3) / 1e12
    step_tflops = flops_per_chunk(w, M, "step") / (ms_per_step * 1e-3) / 1e12
    upd_kernel = ("ld_forward_kernel + ld_mn_gemm_kernel (gradient)" if w.hd > 128 else
                  "bf16_update_wide_kernel" if w.hd == 128 else "bf16_update_kernel") \
        if w.act_dtype == "bf16" else "f32 path"
    tr = TRAFFIC.get(w.name)
    roofline = {"kernel": upd_kernel, "bound": "tensor", "achieved": upd_tflops,
                "peak": peaks["bf16_tflops"], "unit": "TFLOP/s", "frac": upd_tflops / peaks["bf16_tflops"],
                "traffic": tr["bytes"] if tr else None, "traffic_capture": tr["capture"] if tr else None,
                "peak_source": peaks["source"] + ", burst figure (a launch lasts tens to hundreds of "
                               "microseconds); achieved = 12 M d H flops / CUDA-event duration of a "
                               "standalone ttt_accumulate call (one launch of the kernel, launch gap included)",
                "flops_per_launch": upd_flops,
                "standalone_call_ms_incl_launch": {"ttt_accumulate (update kernel)": k_ms[0],
                                                   "ttt_commit (un-fused commit / Newton-Schulz)": k_ms[1],
                                                   "ttt_apply": k_ms[2]},
                "apply_tflops": app_tflops, "apply_frac": app_tflops / peaks["bf16_tflops"],
                "step_tflops": step_tflops, "step_frac": step_tflops / peaks["bf16_tflops"],
                "step_frac_of_sustained": (step_tflops / peaks["bf16_tflops_sustained"]
                                           if peaks["bf16_tflops_sustained"] else None),
                "hbm_gbs_algorithmic": bytes_per_chunk(w, M) / (ms_per_step * 1e-3) / 1e9,
                "hbm_frac": bytes_per_chunk(w, M) / (ms_per_step * 1e-3) / 1e9 / peaks["hbm_gbs"]}

    # ---- end to end: pinned host buffers in, O back to the host, through the same C-ABI call ----
    e2e = None
    if want_e2e:
        n_e2e = min(args.steps, 20)
        streams = [torch.cuda.Stream(dev) for _ in range(2)]
        hO = [torch.empty(M, w.d, dtype=w.torch_dtype).pin_memory() for _ in range(2)]
        ctxs = [ttt, TTT(w.nh, w.hd, w.hidden, dt_code, ns_iters=w.ns_iters, renorm=w.renorm,
                         max_tokens=M, device=local_rank)]

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
        with clocks.busy():
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
        del hO
    ttt.close()
    del dsets, host
    torch.cuda.empty_cache()
    s_sorted = sorted(step_ms)
    res = {"value": value, "unit": "tokens/s", "ms_per_step": ms_per_step,
           "ms_per_step_min": s_sorted[0], "ms_per_step_median": statistics.median(s_sorted),
           "tokens_per_s": value, "pct_of_bf16_peak": 100.0 * step_tflops / peaks["bf16_tflops"],
           "step_frac": step_tflops / peaks["bf16_tflops"],
           "wall_ms_per_step_incl_reset": wall_ms / args.steps, "gpu_launches": int(launches),
           "config": config_of(w, world), "roofline": roofline, "e2e": e2e}
    return res


def run_ours(args, names, rank, local_rank, world):
    dev = torch.device("cuda", local_rank)
    torch.cuda.set_device(dev)
    peaks = _peaks()
    head = HEADLINE if HEADLINE in names else names[-1]
    results = {}
    with ClockSampler(local_rank) as clocks:
        for name in names:
            w = ti.CONFIGS[name]
            results[name] = measure(args, w, rank, local_rank, world, clocks, peaks,
                                    want_e2e=(name == head and not args.no_e2e))
    if rank != 0:
        return
    r = results[head]
    w = ti.CONFIGS[head]
    line = {"metric": "ttt_update_apply_tokens_per_s", "value": r["value"], "unit": "tokens/s",
            "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
            "ms_per_step": r["ms_per_step"], "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": w.act_dtype, "data": "synthetic", "config": r["config"],
            "pct_of_bf16_peak": r["pct_of_bf16_peak"],
            "wall_ms_per_step_incl_reset": r["wall_ms_per_step_incl_reset"],
            "clocks": clocks.summary(), "e2e": r["e2e"],
            "gpu_launches": int(sum(x["gpu_launches"] for x in results.values())),
            "roofline": r["roofline"]}
    if len(results) > 1:
        line["workloads"] = {k: {kk: vv for kk, vv in v.items() if kk != "e2e" or vv is not None}
                             for k, v in results.items()}
    if world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(w)
    print(json.dumps(line), flush=True)


def spawn_ranks(args) -> int:
    """`--gpus N` without torchrun: start the N ranks ourselves (one process per GPU)."""
    have = torch.cuda.device_count()
    if have < args.gpus:
        sys.stderr.write(f"bench.py: --gpus {args.gpus} requested but this box has {have} CUDA device(s)\n")
        return 2
    cmd = [sys.executable, "-m", "torch.distributed.run", "--standalone", "--nnodes=1",
           f"--nproc-per-node={args.gpus}", "--local-addr", "127.0.0.1", os.path.abspath(__file__),
           *sys.argv[1:]]
    env = dict(os.environ)
    env.setdefault("NCCL_DEBUG", "INFO")           # the communicator log shows the rank count
    return subprocess.call(cmd, env=env)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="all", choices=["all", *sorted(ti.CONFIGS)])
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    launched = "WORLD_SIZE" in os.environ
    if args.gpus > 1 and not launched:
        if args.impl == "reference":
            pass                       # rank 0 alone runs the oracle: nothing to spawn
        else:
            sys.exit(spawn_ranks(args))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if launched and world != args.gpus:
        sys.stderr.write(f"bench.py: --gpus {args.gpus} but WORLD_SIZE = {world}\n")
        sys.exit(2)
    names = list(PERF_WORKLOADS) if args.workload == "all" else [args.workload]
    if args.impl == "reference":
        head = HEADLINE if HEADLINE in names else names[-1]
        run_reference(args, ti.CONFIGS[head], rank, world)
        return
    if world > 1:
        torch.distributed.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    try:
        run_ours(args, names, rank, local_rank, world)
    finally:
        if world > 1:
            torch.distributed.destroy_process_group()


if __name__ == "__main__":
    main()
