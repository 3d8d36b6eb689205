#!/usr/bin/env python
"""bench.py -- batch-1 decode throughput of the DF-SSM step on B200 (BASELINE.json `metric`).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 2] [--batch 1]

A "step" is one pass of the whole hot path (S0, L x (S1..S7), S8: include/dfssm.h) over one batch of
tokens, i.e. one decoded token per sequence.  The workload is BASELINE.json configs[2] (Mamba-2
1.3B shape, batch 1): seeded synthetic weights, a uniform-random prompt fed
through the step path (the warm-up steps), then greedy decode with the token kept on the device
(the timed steps).  Prints ONE JSON line (rank 0).

Own arm ("ours"): every step runs in libdfssm.so's CUDA kernels through the C ABI.
Reference arm ("--impl reference"): the CPU oracle as it stands (oracle/), timed on the host cores.
N > 1: independent replicas, one per GPU ("replicas only"); no collective in the
data path; value = tokens of all ranks / max-over-ranks device time.
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
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

import dfssm_synth as ds  # noqa: E402

METRIC = "batch-1 decode tokens/s, 1.3B-shape DF-SSM; achieved HBM GB/s vs peak"
UNIT = "tokens/s"
NOMINAL_HBM_GBS = 8000.0          # BASELINE.json north_star: "~8 TB/s peak"
FALLBACK_HBM_GBS = 6650.0         # B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent


def n_cores() -> int:
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1


def measured_peak():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        try:
            return float(json.loads(p.read_text())["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


# ---------------------------------------------------------------------------------------------
# algorithmic bytes: what the method itself must move
# ---------------------------------------------------------------------------------------------
def algorithmic_bytes(s, batch: int, state_esize: int = 4) -> dict:
    dm, di, dip, r, cd, nh = s.d_model, s.d_inner, s.d_in_proj, s.lora_rank, s.conv_dim, s.nheads
    fmt = getattr(s, "fmt", 0)           # weight-format variants (R25): 5 bits per scaffold weight, 4 bits per LoRA value
    scaffold = s.n_layers * (dip * dm + dm * di) // 8 * (5 if fmt & 1 else 1)
    lora = s.n_layers * r * (dm + dip + di + dm) // (2 if fmt & 2 else 1)
    state = s.n_layers * batch * 2 * (nh * s.headdim * s.d_state * state_esize)      # 2 bytes with --state-fp16 (R24)
    lm_head = s.vocab * dm
    per_layer_small = (4 * dm + 2 * dip + 4 * r + 4 * dip + 16 * cd + 4 * cd + 12 * nh + 4 * di
                       + 2 * dm + 4 * r + 4 * dm)
    conv_state = s.n_layers * batch * 2 * cd * 3 * 4
    other = s.n_layers * per_layer_small + conv_state + 4 * s.vocab + 4 * dm + batch * (dm + 4) \
        + batch * 4 * s.vocab
    return dict(scaffold=scaffold, lora=lora, state=state, lm_head=lm_head, other=other,
                bj_formula=scaffold + lora + state, total=scaffold + lora + state + lm_head + other)


def kernel_class_bytes(s, batch: int, state_esize: int = 4) -> dict:
    """Algorithmic bytes ONE launch of each kernel class moves (weights once, state r+w once)."""
    dm, di, dip, r, cd, nh = s.d_model, s.d_inner, s.d_in_proj, s.lora_rank, s.conv_dim, s.nheads
    B = batch
    return {
        "embed": B * (dm + 4 + 4 * dm),
        "normquant": B * (4 * di + 2 * di) + 4 * di,
        "proj_in": dip * dm // 8 * (5 if getattr(s, "fmt", 0) & 1 else 1) + r * dm // (2 if getattr(s, "fmt", 0) & 2 else 1) + B * (2 * dm + 4 * dip + 4 * r),
        "ssm": B * (2 * nh * s.headdim * s.d_state * state_esize + 2 * cd * 4 * 4 + 4 * dip + 4 * di)
        + 2 * dip + dip * r + 4 * dip + 20 * cd + 12 * nh,
        "proj_out": dm * di // 8 * (5 if getattr(s, "fmt", 0) & 1 else 1) + r * di // (2 if getattr(s, "fmt", 0) & 2 else 1) + B * (2 * di + 4 * dm + 4 * r),
        "epi_out": 2 * dm + dm * r + 4 * dm + B * (4 * dm + 8 * dm),
        "lmhead": s.vocab * dm + 4 * s.vocab + B * (dm + 4 * s.vocab),
        "argmax": B * 4 * s.vocab,
        "mega": algorithmic_bytes(s, B, state_esize)["total"],      # the whole step is one kernel
    }


# ---------------------------------------------------------------------------------------------
# clocks: nvidia-smi sampled DURING the timed region
# ---------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.samples = []
        self.proc = None
        self.thread = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._read, daemon=True)
        self.thread.start()

    def _read(self):
        for line in self.proc.stdout:
            self.samples.append(line.strip())

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for ln in self.samples:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 6:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for n, v in zip(names, f[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


# ---------------------------------------------------------------------------------------------
# the oracle, as it stands, on the host cores (cpu_baseline leg and --impl reference)
# ---------------------------------------------------------------------------------------------
def time_oracle(s, blob, cfg_idx: int, batch: int, budget_s: float, max_steps: int, n_prompt: int = 2, threads: int = 0,
                state_fp16: bool = False):
    """Feed `n_prompt` prompt tokens (untimed), then time greedy decode steps until the budget or
    max_steps is reached.  Returns (tokens/s, steps, seconds, threads)."""
    import oracle
    oracle.build()
    oracle.set_threads(threads if threads > 0 else n_cores())
    m = oracle.OracleModel(blob, batch)
    m.set_state_fp16(state_fp16)
    prompt = ds.token_batch(s.vocab, n_prompt, seed=cfg_idx, batch=batch)
    for t in range(n_prompt):
        m.step(prompt[t])
    tok = np.array(m.next_tokens()[:batch], np.int32)
    steps, t0 = 0, time.perf_counter()
    while steps < max_steps:
        m.step(tok)
        tok = np.array(m.next_tokens()[:batch], np.int32)
        steps += 1
        if time.perf_counter() - t0 >= budget_s:
            break
    dt = time.perf_counter() - t0
    return batch * steps / dt, steps, dt, oracle.get_threads()


def run_reference(args, s, blob):
    """--impl reference: the oracle timed on the host cores, same config / metric / unit."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    # warm-up steps and timed steps both run; the timed sample is bounded to ~2 minutes
    import oracle
    oracle.build()
    oracle.set_threads(n_cores())
    m = oracle.OracleModel(blob, args.batch)
    m.set_state_fp16(args.state_fp16)
    toks = ds.token_batch(s.vocab, max(1, min(args.warmup, 8)), seed=args.config, batch=args.batch)
    for t in range(toks.shape[0]):
        m.step(toks[t])
    tok = np.array(m.next_tokens()[:args.batch], np.int32)
    steps, t0 = 0, time.perf_counter()
    while steps < args.steps and time.perf_counter() - t0 < 120.0:
        m.step(tok)
        tok = np.array(m.next_tokens()[:args.batch], np.int32)
        steps += 1
    dt = time.perf_counter() - t0
    val = args.batch * steps / dt
    sample = (f"{steps} greedy decode steps of config {args.config} batch {args.batch} after {toks.shape[0]} prompt steps "
              f"(bounded to 120 s; {args.steps} steps requested)")
    out = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
        "warmup": int(toks.shape[0]), "ms_per_step": 1e3 * dt / steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "int8 x {-1,+1} -> int32; fp32 state", "data": "synthetic",
        "config": {"workload": workload_name(args.config, args.batch, FORMATS[args.format]), "seed": args.config},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": oracle.get_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(out), flush=True)


# ---------------------------------------------------------------------------------------------
# N > 1: independent replicas ("replicas only") -- the host-side logic, also run on CPU/gloo by tests
# ---------------------------------------------------------------------------------------------
def replica_seed(rank: int, cfg_idx: int) -> int:
    """Every rank decodes its own sequences: the token-stream seed of a replica."""
    return 1000 * rank + cfg_idx


def max_over_ranks(values, dist=None, device="cpu"):
    """Element-wise MAX of per-rank durations over all ranks (the job is as slow as its slowest replica)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return [float(v) for v in values]
    import torch
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t.cpu()]


def whole_job_rate(world: int, batch: int, steps: int, seconds: float) -> float:
    """Tokens of ALL replicas divided by the max-over-ranks time."""
    return world * batch * steps / seconds


FORMATS = {"1bit": 0, "17level": 1, "int4": 2, "17level+int4": 3}


def workload_name(cfg_idx: int, batch: int, fmt: int = 0) -> str:
    names = {0: "cfg0 tiny DF-SSM (2 layers, d_model 256)", 1: "cfg1 Mamba-2-130M-shape DF-SSM",
             2: "cfg2 Mamba-2-1.3B-shape DF-SSM (48 layers, d_model 2048, d_state 128, LoRA r32)",
             3: "cfg3 Mamba-2-1.3B-shape DF-SSM batch sweep", 4: "cfg4 Mamba-2-2.7B-shape DF-SSM"}
    fm = {0: "", 1: ", 17-level scaffold", 2: ", int4 LoRA", 3: ", 17-level scaffold + int4 LoRA"}[fmt]
    return f"{names.get(cfg_idx, f'cfg{cfg_idx}')}{fm}, batch {batch}, greedy decode after a uniform-random prompt"


# ---------------------------------------------------------------------------------------------
# own arm: the CUDA path through the C ABI
# ---------------------------------------------------------------------------------------------
def run_ours(args, s, blob):
    import torch

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the DF-SSM step has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    from paper_2606_10932_b200 import build
    build.build()
    import paper_2606_10932_b200 as pk

    B = args.batch
    from paper_2606_10932_b200 import binding
    esz = 2 if args.state_fp16 else 4
    m = pk.Model(pk.Config.from_shape(s, max_batch=B, flags=binding.FLAG_STATE_FP16 if args.state_fp16 else 0), blob, device=f"cuda:{local}")
    # every rank is an independent replica with its own token streams ("replicas only")
    prompt = ds.token_batch(s.vocab, max(args.warmup, 1), seed=replica_seed(rank, args.config), batch=B)
    prompt_dev = [torch.from_numpy(prompt[t]).cuda() for t in range(prompt.shape[0])]
    nxt = m.next_tokens()[:B]

    def barrier():
        m.sync()
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
            torch.cuda.synchronize()

    # ---- device-resident leg: W prompt steps (untimed), then K greedy steps (timed) ----
    for t in range(args.warmup):
        m.step(prompt_dev[t])
    if args.warmup == 0:
        m.step(prompt_dev[0])
    # at least 32 warm-up steps before anything is timed (greedy steps beyond the W prompt steps, untimed)
    extra_warmup = max(0, 32 - max(args.warmup, 1))
    for _ in range(extra_warmup):
        m.step(nxt)
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.15)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    with torch.cuda.stream(m.stream):
        e0.record()
        for _ in range(args.steps):
            m.step(nxt)
        e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    launches = m.launches_per_step(B) * args.steps
    # best and median of 5 repetitions of the same K steps (the first one is the reported value)
    rep_ms = [ms]
    for _ in range(max(0, args.reps - 1)):
        r0, r1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        with torch.cuda.stream(m.stream):
            r0.record()
            for _ in range(args.steps):
                m.step(nxt)
            r1.record()
        barrier()
        rep_ms.append(r0.elapsed_time(r1))

    # ---- end-to-end leg: host buffers through dfssm_step_host, copies inside the timed region ----
    tok_h = np.ascontiguousarray(m.next_tokens()[:B].cpu().numpy(), np.int32)
    nxt_h = np.zeros(B, np.int32)
    e2e_steps = max(8, min(args.steps, 256))
    for _ in range(3):
        m.step_host(tok_h, nxt_h)
        tok_h[:] = nxt_h
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        m.step_host(tok_h, nxt_h)
        tok_h[:] = nxt_h
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    barrier()
    clocks = sampler.stop() if rank == 0 else None

    # ---- per-kernel-class device times (CUDA events on the library's stream, eager chain) ----
    kt = m.time_kernels(nxt, iters=8)
    barrier()

    ms, e2e_s = max_over_ranks([ms, e2e_s], dist, "cuda")
    rep_ms = max_over_ranks(rep_ms, dist, "cuda")

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    ab = algorithmic_bytes(s, B, esz)
    value = whole_job_rate(world, B, args.steps, ms * 1e-3)
    e2e_val = whole_job_rate(world, B, e2e_steps, e2e_s)
    peak, peak_src = measured_peak()
    step_gbs = ab["total"] * (args.steps / (ms * 1e-3)) / 1e9
    kb = kernel_class_bytes(s, B, esz)
    L = s.n_layers
    counts = {"embed": 1, "normquant": 2 * L + 1, "proj_in": L, "ssm": L, "proj_out": L, "epi_out": L,
              "lmhead": 1, "argmax": 1, "mega": 1}
    # dominant kernel class = the one with the largest share of the step's device time
    dom = max(kt, key=lambda k: kt[k])
    per_launch_us = kt[dom] / max(1, counts.get(dom, 1))
    achieved = kb[dom] / (per_launch_us * 1e-6) / 1e9 if per_launch_us > 0 else 0.0
    traffic, traffic_src = ncu_traffic(args.config, B, dom)
    roofline = {
        "bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "GB/s",
        "frac": achieved / peak, "traffic": traffic, "traffic_source": traffic_src, "peak_source": peak_src,
        "bytes_per_launch": kb[dom], "us_per_launch": per_launch_us,
        "whole_step": {"algorithmic_bytes_per_step": ab["total"], "bj_formula_bytes_per_step": ab["bj_formula"],
                       "achieved_GBps": step_gbs, "frac_of_measured": step_gbs / peak,
                       "frac_of_nominal_8TBps": step_gbs / NOMINAL_HBM_GBS,
                       "bj_formula_frac_of_nominal_8TBps": ab["bj_formula"] * (args.steps / (ms * 1e-3)) / 1e9 / NOMINAL_HBM_GBS},
        "kernel_us_per_step": kt,
    }

    cpu_baseline = None
    if world == 1 and not args.no_cpu_baseline:
        v, n, dt, thr = time_oracle(s, blob, args.config, B, budget_s=15.0, max_steps=64, state_fp16=args.state_fp16)
        v1, n1, dt1, _ = time_oracle(s, blob, args.config, B, budget_s=6.0, max_steps=8, threads=1, state_fp16=args.state_fp16)
        cpu_baseline = {"value": v, "unit": UNIT, "cores": thr, "kind": "oracle",
                        "sample": f"{n} greedy decode steps of the same workload after 2 prompt steps ({dt:.1f} s)",
                        "single_thread": {"value": v1, "unit": UNIT, "cores": 1, "sample": f"{n1} steps ({dt1:.1f} s)"}}

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None,       # BASELINE.md holds no published number for this metric on this workload (the paper's are A100, trained, r16)
        "repeats": {"n": len(rep_ms), "steps_each": args.steps, "best_ms_per_step": min(rep_ms) / args.steps,
                    "median_ms_per_step": statistics.median(rep_ms) / args.steps, "extra_warmup_steps": extra_warmup},
        "speedup_vs_cpu_baseline": (value / cpu_baseline["value"]) if cpu_baseline else None,
        "dtype": ("int8 x {-8..8} -> int32; " if FORMATS[args.format] & 1 else "int8 x {-1,+1} -> int32; ") + ("fp16 state (lossy option, DESIGN.md R24)" if args.state_fp16 else "fp32 state"), "data": "synthetic",
        "config": {"workload": workload_name(args.config, B, FORMATS[args.format]), "seed": args.config, "batch_per_gpu": B,
                   "parallelism": "replicas only" if world > 1 else "single GPU",
                   "l2": f"inputs larger than L2: {ab['total'] / 1e6:.0f} MB streamed per step vs ~126 MB L2"},
        "e2e": {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": 4 * B, "d2h_bytes_per_step": 4 * B,
                "steps": e2e_steps, "call": "dfssm_step_host (host token in, host greedy token out)"},
        "gpu_launches": launches,
        "clocks": clocks,
        "roofline": roofline,
        "cpu_baseline": cpu_baseline,
    }
    print(json.dumps(out), flush=True)
    if dist is not None:
        dist.destroy_process_group()


# dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from the committed `ncu --set full`
# captures (profiles/r02_traffic.csv: config,batch,kernel,dram_bytes_per_launch,commit).  NOT measured by this run: the
# value is reported only while no commit after the one it was captured at touches the kernel's sources; on a box without
# the git history (gpurun snapshots) that cannot be checked and the source string says so.
def ncu_traffic(cfg_idx: int, batch: int, kernel: str):
    t = ROOT / "profiles" / "r02_traffic.csv"
    if not t.exists():
        return None, "no capture committed"
    row = None
    for line in t.read_text().splitlines()[1:]:
        f = [x.strip() for x in line.split(",")]
        if len(f) >= 5 and (int(f[0]), int(f[1]), f[2]) == (cfg_idx, batch, kernel):
            row = f
    if row is None:
        return None, "no capture of this workload"
    src = f"profiles/r02_traffic.csv (ncu --set full capture at commit {row[4][:12]}, not this run)"
    try:
        # the files the captured kernel is built from (k_mega: its own two headers and the shared arithmetic)
        srcs = [f"paper_2606_10932_b200/csrc/{f}" for f in ("dfssm_mega.cuh", "dfssm_mega_host.cuh", "dfssm_math.cuh")] if kernel == "mega" \
            else ["paper_2606_10932_b200/csrc"]
        res = subprocess.run(["git", "-C", str(ROOT), "rev-list", f"{row[4]}..HEAD", "--", *srcs],
                             capture_output=True, text=True, timeout=20)
        if res.returncode != 0:
            return int(row[3]), src + "; staleness unchecked (no git history here)"
        if res.stdout.strip():
            return None, src + "; STALE: csrc/ changed since, re-capture"
        return int(row[3]), src
    except Exception:
        return int(row[3]), src + "; staleness unchecked (git unavailable)"


def respawn_under_torchrun(args) -> int:
    """`python bench.py --gpus N` without torchrun: start the N replicas ourselves (one process per GPU)."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), str(Path(__file__).resolve()), *sys.argv[1:]]
    return subprocess.call(cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=512)
    ap.add_argument("--warmup", type=int, default=128)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2)
    ap.add_argument("--batch", type=int, default=1)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--format", default="1bit", choices=sorted(FORMATS),
                    help="weight format of the synthetic blob (SURVEY 8(f) NEXT-3): 17-level scaffold and / or int4 LoRA; kernel chain only")
    ap.add_argument("--state-fp16", action="store_true",
                    help="SSM state stored as binary16 (DFSSM_FLAG_STATE_FP16, SURVEY 8(f) NEXT-2; lossy; kernel chain only)")
    ap.add_argument("--reps", type=int, default=5, help="repetitions of the K timed steps (the first is the reported value)")
    args = ap.parse_args()
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "ours" and args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        raise SystemExit(respawn_under_torchrun(args))
    if args.impl == "ours" and world != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}: launch with torchrun --nproc-per-node {args.gpus}, or without torchrun")
    if args.impl == "reference" and int(os.environ.get("RANK", "0")) != 0:
        return
    s = ds.shape_for_config(args.config).with_(fmt=FORMATS[args.format])
    blob = ds.make_blob(s, args.config)
    if args.impl == "reference":
        run_reference(args, s, blob)
    else:
        run_ours(args, s, blob)


if __name__ == "__main__":
    main()
