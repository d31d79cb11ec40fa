#!/usr/bin/env python
"""bench.py -- scored tokens/s of the RLHF scoring hot path on B200 (BASELINE.json:metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg1|cfg2|cfg3|cfg4|cfg0]
                    [--impl ours|reference] [--no-extras] [--arm fused|nccl] [--dry-run]
                    [--only hbm|attention]

A step is one pass of the hot path over one synthetic micro-batch of the named workload.
BASELINE.json:metric ("scored tokens/sec (fwd and fwd+bwd) on 1 B200") names no configuration, so
the headline workload is the largest single-GPU configuration that has a host-buffer entry point:
configs[4] (hidden 8192, vocab 256000, 8192 tokens, forward + backward, dW in fp32).  The ONE JSON
line on stdout is compact (< 4 KB, asserted): the headline's value, ONE roofline object (the
dominant contraction), e2e (gc_grpo_step_host from pinned host buffers), cpu_baseline, and under
"workloads" a few scalars for each other configuration: configs[1] (the metric's forward half),
configs[2], configs[3] (dynamic-sampling step).  Everything else -- every roofline object of every
workload, the HBM-bound kernels, the cuBLAS/torch library baseline, the attention workload -- goes
to stderr as one JSON object per line ({"detail": name, ...}), never into the stdout line.
Backward-capable workloads run advantages -> loss forward -> loss backward per step.

N > 1: one rank per GPU under torch.distributed.run (bench.py re-executes itself under it when
--gpus N > 1 and WORLD_SIZE is not set).  Whole groups are sharded across ranks -- every rank
scores its own micro-batch, weak scaling.  Scoring (forward) needs no data-path collective; a
training workload (cfg2 / cfg4) at N > 1 exchanges dW every step: `--arm fused` (default) runs
gc_grpo_loss_bwd_reduce_scatter, whose dW contraction reduce-adds its tiles straight into the
owning rank's shard over NVLink; `--arm nccl` runs the plain backward followed by an NCCL
reduce-scatter; the line reports both.
`--impl reference` times the fp64 CPU oracle (oracle/) on a bounded sample of the same workload.
`--dry-run` (CPU, gloo): starts the ranks, runs the timing reductions on fake numbers and prints
the line -- the launch path without a GPU.
"""
from __future__ import annotations

import argparse
import gc
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np
import torch

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2507_22789_b200 import inputs as I  # noqa: E402
from tests.harness import DeviceBatch, detie_old, synth_policy_logp  # noqa: E402,F401

WORKLOADS = {"cfg0": 0, "cfg1": 1, "cfg2": 2, "cfg3": 3, "cfg4": 4}
HEADLINE = "cfg4"        # the largest single-GPU configuration with a host-buffer entry point
MAX_LINE_BYTES = 4096    # the driver parses the stdout line; round 2's 22 KB line was unreadable
KIND_NAMES = {"fwd_stats": "a2+a3 forward H.W^T + online log-softmax epilogue",
              "recompute_ds": "a10 recompute H.W^T + dS epilogue",
              "dh": "a11 dH = dS.W", "dw": "a12 dW += dS^T.H"}
SMI_FIELDS = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm=d["hbm_gbs"], burst=d["bf16_tflops"], sustained=d["bf16_tflops_sustained"],
                    source="measured")
    return dict(hbm=6650.0, burst=1590.0, sustained=1400.0, source="fallback")


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 50 ms during the timed region."""

    def __init__(self, gpu_ids):
        self.rows = []
        self.proc = None
        self.gpu_ids = gpu_ids

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={SMI_FIELDS}", "--format=csv,noheader,nounits",
                 "-lms", "50", "-i", ",".join(str(g) for g in self.gpu_ids)],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if self.proc is None:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"])
        time.sleep(0.15)
        self.proc.terminate()
        self.thread.join(timeout=2)
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[1])); mx.append(float(r[2])); pw.append(float(r[3]))
            except (ValueError, IndexError):
                continue
            for n, v in zip(names, r[4:8]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        if not sm:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["no samples"])
        return dict(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)),
                    power_w_max=float(max(pw)), samples=len(sm), reasons=sorted(reasons))


# --------------------------------------------------------------------------------------------
# synthetic batch on the device (recipe: DESIGN.md sec 4)
# --------------------------------------------------------------------------------------------
def _bwd_chunk_T(B, T, w):
    # rows of the dS buffer the library picks: difference of two workspace queries
    a = B.workspace_bytes(B.GC_OP_LOSS_BWD, T, w.D, w.V, B.GC_BF16, 0)
    c256 = B.workspace_bytes(B.GC_OP_LOSS_BWD, T, w.D, w.V, B.GC_BF16, 256)
    ld = -(-w.V // 64) * 64
    return 256 + (a - c256) // (ld * 2)


def make_step(B, b: DeviceBatch):
    """Returns (step_fn, kernel launches per step).  All work goes through the C ABI."""
    w = b.w
    compact = b.mask is not None
    tc = w.dtype == "bf16"
    # forward: tcgen05 kernel + combine (+ row selection: count, scan, scatter, H gather, target
    # gather, zero-fill of unscored outputs); SIMT: one kernel
    fwd_launches = (2 + (6 if compact else 0)) if tc else 1
    if not w.backward:
        def step():
            B.gc_grpo_advantages(b.rewards, b.go, 1e-6, False, w.drop_constant_groups)
            return B.gc_token_logprobs(b.H, b.W, b.y, b.mask, w.tau, want_lse=False)
        return step, 1 + fwd_launches

    if w.drop_constant_groups:
        return make_step_dynamic_sampling(B, b)

    def step():
        adv, _ = B.gc_grpo_advantages(b.rewards, b.go, 1e-6, False, w.drop_constant_groups)
        f = B.gc_grpo_loss_fwd(b.H, b.W, b.y, b.mask, w.tau, b.cu, adv, b.old, b.ref, w.clip_lo,
                               w.clip_hi, w.beta)
        B.gc_grpo_loss_bwd(b.H, b.W, b.y, b.mask, w.tau, b.cu, adv, b.old, b.ref, f["logp"],
                           f["lse"], w.clip_lo, w.clip_hi, w.beta, dH=b.dH, dW=b.dW,
                           fwd_state=f["state"])
        return f["out5"]
    # launches: advantages 1, fwd, loss 1 (one cooperative launch), bwd: loss 1 + (row selection
    # reused from the forward) 2 small gathers + dH zero-fill + 3 contractions per chunk (SIMT: 2)
    if tc:
        n_chunks = -(-b.T // _bwd_chunk_T(B, b.T, w))
        bwd = 1 + (3 if compact else 0) + 3 * n_chunks
    else:
        bwd = 1 + 2
    return step, 1 + fwd_launches + 1 + bwd


def make_step_dynamic_sampling(B, b):
    """configs[3]: group filter -> repack + workload balancing (gc_balance_plan: kept samples
    sorted by simulated workload L^2, buckets of one group's size, shuffled) -> gathers of H,
    targets, old / ref log-probs -> forward + backward on the kept batch.  Everything runs on the
    device every step; only the kept sizes (fixed by the seeded rewards) are read once at set-up."""
    w = b.w
    adv_all, keep = B.gc_grpo_advantages(b.rewards, b.go, 1e-6, False, True)
    plan = B.gc_balance_plan(b.cu, b.go, keep, 0, 1, w.group_size, 1234, True, n_tokens_max=b.T)
    Tk, Rk = int(plan["n_tokens"].item()), int(plan["n_kept"].item())
    b.n_scored = Tk
    b.T_kept = Tk
    dH = torch.empty(Tk, w.D, dtype=b.H.dtype, device=b.H.device)
    del b.dH

    def step():
        adv_all, keep = B.gc_grpo_advantages(b.rewards, b.go, 1e-6, False, True)
        p = B.gc_balance_plan(b.cu, b.go, keep, 0, 1, w.group_size, 1234, True, n_tokens_max=b.T)
        Hk = B.gc_gather_rows(b.H, p["src_token"], p["n_tokens"], Tk)
        yk = B.gc_gather_1d(b.y, p["src_token"], p["n_tokens"], Tk)
        oldk = B.gc_gather_1d(b.old, p["src_token"], p["n_tokens"], Tk)
        refk = B.gc_gather_1d(b.ref, p["src_token"], p["n_tokens"], Tk)
        advk = B.gc_gather_1d(adv_all, p["order"], p["n_kept"], Rk)
        cuk = p["cu_out"][:Rk + 1]
        f = B.gc_grpo_loss_fwd(Hk, b.W, yk, None, w.tau, cuk, advk, oldk, refk, w.clip_lo, w.clip_hi,
                               w.beta)
        B.gc_grpo_loss_bwd(Hk, b.W, yk, None, w.tau, cuk, advk, oldk, refk, f["logp"], f["lse"],
                           w.clip_lo, w.clip_hi, w.beta, dH=dH, dW=b.dW)
        return f["out5"]
    n_chunks = -(-Tk // _bwd_chunk_T(B, Tk, w))
    # advantages 1 + plan 7 + gathers 5 + fwd 2 + loss 1 + bwd: loss 1 + 3 per chunk
    return step, 1 + 7 + 5 + 2 + 1 + 1 + 3 * n_chunks


def timed_region(step, steps, warmup, dist_on, B=None):
    """warmup untimed steps, then exactly `steps` steps between barriers; per-step CUDA events.
    With B given, the library also brackets each contraction launch with CUDA events on the
    launch stream (gc_kernel_timing_*): -> (total_ms, per_step_ms, {kind: (ms, launches)})."""
    import torch.distributed as dist
    for _ in range(warmup):
        step()
    torch.cuda.synchronize()
    if dist_on:
        dist.barrier()
        torch.cuda.synchronize()
    if B is not None:
        B.gc_kernel_timing_begin()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
          for _ in range(steps)]
    t_all0, t_all1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t_all0.record()
    for i in range(steps):
        ev[i][0].record()
        step()
        ev[i][1].record()
    t_all1.record()
    torch.cuda.synchronize()
    if dist_on:
        dist.barrier()
        torch.cuda.synchronize()
    total_ms = t_all0.elapsed_time(t_all1)
    per = [a.elapsed_time(b) for a, b in ev]
    kinds = B.gc_kernel_timing_end() if B is not None else None
    return total_ms, per, kinds


# --------------------------------------------------------------------------------------------
# the oracle on the host cores (cpu_baseline leg and --impl reference)
# --------------------------------------------------------------------------------------------
def _oracle_sample(w: I.Workload, n_tokens: int, seed=0):
    """A bounded sample of the workload for the oracle: full D and V, n_tokens tokens of one group."""
    import oracle as O
    full = I.make_layout(w, seed).T
    ws = w if n_tokens >= full else I.reduced(w, groups=1, group_size=2, seq_len=max(n_tokens // 2, 1),
                                              prompt_len=0)
    lay = I.make_layout(ws, seed)
    H, W = I.make_hw(lay.T, ws.D, ws.V, ws.dtype, seed, "cpu")
    y = I.sample_targets(H, W, ws.tau, seed).numpy()
    H64 = H.float().numpy().astype(np.float64)
    W64 = W.float().numpy().astype(np.float64)
    rew = I.make_rewards(ws, seed) if n_tokens >= full else np.array([1.0, 0.0], dtype=np.float32)
    old = ref = None
    if w.backward:
        lp = O.token_logprobs(H64, W64, y, None, ws.tau)[0]
        old = I.perturb_logp(lp, ws.old_std, 1)
        ref = I.perturb_logp(lp, ws.ref_std, 2)

    def step():
        adv, _ = O.grpo_advantages(rew, lay.group_offsets, 1e-6)
        if w.backward:
            O.grpo_forward_backward(H64, W64, y, lay.mask if not lay.mask.all() else None, ws.tau,
                                    lay.cu_seqlens, adv, old, ref, ws.clip_lo, ws.clip_hi, ws.beta)
        else:
            O.token_logprobs(H64, W64, y, None, ws.tau)
    return step, lay.T, ws


def _time_oracle(step, tokens, min_seconds, max_reps=64):
    reps = 0
    t0 = time.perf_counter()
    while True:
        step()
        reps += 1
        dt = time.perf_counter() - t0
        if dt >= min_seconds or reps >= max_reps:
            break
    return tokens * reps / dt, reps, dt


def cpu_baseline(w: I.Workload, budget_tokens: int):
    """The oracle, as it stands, on this box's host cores, on a bounded sample of the workload:
    with every core numpy's BLAS uses, with ONE thread, and configs[0] in full (SURVEY.md sec 8(d)
    "Oracle timing").  About 25 s of CPU work in total."""
    from threadpoolctl import threadpool_info, threadpool_limits
    step, T, ws = _oracle_sample(w, budget_tokens)
    kind = "fwd+bwd" if w.backward else "fwd"
    step()                                                 # touch the pages once
    v_all, reps, dt = _time_oracle(step, T, 10.0)
    threads = max([p.get("num_threads", 1) for p in threadpool_info()] + [1])
    with threadpool_limits(limits=1):
        v_one, reps1, dt1 = _time_oracle(step, T, 6.0, max_reps=8)
    step0, T0, _ = _oracle_sample(I.CONFIGS[0], 1 << 30)
    step0()
    v0, reps0, dt0 = _time_oracle(step0, T0, 2.0, max_reps=200)
    return dict(value=v_all, unit="scored tokens/s", cores=int(threads), kind="oracle",
                sample=f"{reps} x {T} tokens of {w.name} (full D={w.D}, V={w.V}), {kind}, "
                       f"{dt:.1f} s, fp64 numpy",
                seconds=dt,
                one_thread=dict(value=v_one, cores=1,
                                sample=f"{reps1} x {T} tokens, {dt1:.1f} s, BLAS limited to 1 thread"),
                config0_full=dict(value=v0, cores=int(threads), unit="scored tokens/s",
                                  sample=f"{reps0} x configs[0] in full (T={T0}, D=256, V=4096, "
                                         f"fp64), fwd+bwd, {dt0:.1f} s"))


def run_reference(args, w):
    """--impl reference: the oracle on host cores, same config/metric/unit."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from threadpoolctl import threadpool_info
    n_tok = 32 if w.D * w.V > 1e9 else 64 if w.D * w.V > 1e8 else 1 << 30
    step, T, ws = _oracle_sample(w, n_tok)
    for _ in range(args.warmup):
        step()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        step()
    dt = time.perf_counter() - t0
    val = T * args.steps / dt
    threads = max([p.get("num_threads", 1) for p in threadpool_info()] + [1])
    unit = "scored tokens/s"
    sample = f"{T} tokens per step of {w.name} (full D={w.D}, V={w.V}), fp64 numpy oracle"
    print(json.dumps({
        "impl": "reference", "metric": metric_name(w), "value": val, "unit": unit,
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(w, T, args.gpus),
        "cpu_baseline": dict(value=val, unit=unit, cores=int(threads), kind="oracle", sample=sample),
        "e2e": dict(value=val, unit=unit, h2d_bytes_per_step=0, d2h_bytes_per_step=0),
    }))


def metric_name(w):
    return "scored tokens/sec (" + ("fwd+bwd" if w.backward else "fwd") + ")"


def workload_config(w, T, n_gpus, exchange="none"):
    return {"workload": w.name, "tokens_per_gpu": T, "hidden": w.D, "vocab": w.V,
            "groups": w.groups, "group_size": w.group_size, "temperature": w.tau,
            "pass": "fwd+bwd" if w.backward else "fwd",
            "parallelism": f"dp{n_gpus} (whole groups per rank, W replicated; data-path "
                           f"collective: {exchange})",
            "l2": "inputs exceed L2 (W alone is larger than 126 MB); no flush needed"}


# --------------------------------------------------------------------------------------------
# rooflines
# --------------------------------------------------------------------------------------------
def load_traffic(workload, kind):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the named kernel kind, from the
    committed `ncu --set full` capture (profiles/roofline_traffic.csv; profiles/*.md say how) --
    not from this run: a run under a profiler is never a bench value."""
    p = os.path.join(ROOT, "profiles", "roofline_traffic.csv")
    if not os.path.exists(p):
        return None
    for line in open(p):
        f = [x.strip() for x in line.split(",")]
        if len(f) >= 3 and f[0] == workload and f[1] == kind:
            return float(f[2])
    return None


def rooflines(w, tokens, steps, kinds, total_ms, peaks):
    """One roofline object per contraction kind: algorithmic flops per launch (2 T_scored D V per
    pass / launches per pass) / the kernel's average launch duration, measured with CUDA events
    that the library records around each contraction launch on the launch stream inside the timed
    region (gc_kernel_timing_*).  Peak: measured cuBLAS bf16 -- burst for a timed region under 1 s,
    sustained otherwise; both fractions and the nominal-2250 fraction are printed."""
    long_run = total_ms > 1000.0
    peak = peaks["sustained"] if long_run else peaks["burst"]
    pass_flops = 2.0 * tokens * w.D * w.V
    out = []
    for k, (ms, n) in (kinds or {}).items():
        if not n:
            continue
        launches_per_step = n / steps
        launch_ms = ms / n
        flops_per_launch = pass_flops / launches_per_step
        achieved = flops_per_launch / (launch_ms * 1e-3) / 1e12
        out.append({
            "workload": w.name, "kind": k, "bound": "tensor",
            "kernel": f"tc::k_tc_gemm [{k}: {KIND_NAMES[k]}]",
            "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
            "peak_kind": ("sustained" if long_run else "burst") + " cuBLAS bf16, " + peaks["source"],
            "frac_of_burst": achieved / peaks["burst"],
            "frac_of_sustained": achieved / peaks["sustained"],
            "frac_of_nominal_2250": achieved / 2250.0,
            "flops_per_launch": flops_per_launch, "launch_ms": launch_ms,
            "launches_per_step": launches_per_step, "ms_per_step": ms / steps,
            "traffic": load_traffic(w.name, k),
            "traffic_source": "committed ncu --set full capture (profiles/), not this run",
        })
    return out


def dominant(roofs, step_ms):
    if not roofs:
        return {"bound": "tensor", "achieved": None, "peak": None, "unit": "TFLOP/s", "frac": None,
                "traffic": None, "note": "fp32 SIMT parity workload: latency bound, no roofline"}
    d = dict(max(roofs, key=lambda r: r["ms_per_step"]))
    d["contraction_share_of_step"] = sum(r["ms_per_step"] for r in roofs) / step_ms
    d["note"] = ("launch duration = CUDA events recorded by the library around each contraction "
                 "launch on the launch stream, inside the timed region")
    return d


ROOFLINE_KEYS = ("workload", "kind", "kernel", "bound", "achieved", "peak", "unit", "frac",
                 "peak_kind", "frac_of_burst", "frac_of_sustained", "flops_per_launch", "launch_ms",
                 "launches_per_step", "traffic", "contraction_share_of_step")


def detail(name, **kw):
    """Everything that is not the headline goes to stderr, one JSON object per line."""
    print(json.dumps(dict({"detail": name}, **kw)), file=sys.stderr, flush=True)


def workload_scalars(m):
    """A measured workload (measure_workload) reduced to the scalars the stdout line carries."""
    roofs = m.get("rooflines") or []
    worst = min(roofs, key=lambda r: r["frac_of_burst"]) if roofs else None
    out = {"ms_per_step": round(m["ms_per_step"], 4), "value": round(m["value"], 1),
           "step_tflops": round(m["step_tflops"], 1),
           "worst_kind": worst["kind"] if worst else None,
           "worst_frac_of_burst": round(worst["frac_of_burst"], 4) if worst else None,
           "e2e_ms": round(m["e2e"]["ms_per_step"], 4) if m.get("e2e") else None}
    if m.get("library_baseline"):
        out["cublas_gemm_only_ms"] = round(m["library_baseline"]["cublas_gemm_only"]["ms_per_step"], 4)
    return out


def assemble_line(w, *, value, ms_per_step, T, world, steps, warmup, exchange, clocks, gpu_launches,
                  roofs, step_ms, e2e, cpu, workloads, extra_config=None, dp_info=None):
    """The ONE stdout line: headline scalars, one roofline object, e2e, cpu_baseline, and scalars per
    other workload.  No lists of objects, nothing twice (tests/test_bench_line.py feeds it fakes)."""
    dom = dominant(roofs, step_ms)
    out = {
        "metric": metric_name(w), "value": value, "unit": "scored tokens/s",
        "n_gpus": world, "steps": steps, "warmup": warmup, "ms_per_step": ms_per_step,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "bf16" if w.dtype == "bf16" else "f32", "data": "synthetic",
        "config": dict(workload_config(w, T, world, exchange), **(extra_config or {})),
        "clocks": clocks, "gpu_launches": gpu_launches,
        "roofline": {k: dom[k] for k in ROOFLINE_KEYS if k in dom} if dom.get("achieved") else dom,
    }
    if e2e:
        out["e2e"] = {k: e2e[k] for k in ("value", "unit", "ms_per_step", "h2d_bytes_per_step",
                                          "d2h_bytes_per_step") if k in e2e}
    if cpu:
        out["cpu_baseline"] = {"value": cpu["value"], "unit": cpu["unit"], "cores": cpu["cores"],
                               "kind": cpu["kind"], "sample": cpu["sample"]}
        if cpu.get("one_thread"):
            out["cpu_baseline"]["one_thread"] = {"value": cpu["one_thread"]["value"], "cores": 1}
    if workloads:
        out["workloads"] = workloads
    if dp_info:
        out["dp_exchange"] = {k: v for k, v in dp_info.items() if not isinstance(v, (dict, list))}
        if isinstance(dp_info.get("other_arm"), dict):
            out["dp_exchange"]["other_arm_ms_per_step"] = dp_info["other_arm"].get("ms_per_step")
    return out


def emit(out) -> str:
    line = json.dumps(out)
    assert len(line) < MAX_LINE_BYTES, f"stdout line is {len(line)} bytes (limit {MAX_LINE_BYTES})"
    return line


def hbm_kernels(B, device, peaks):
    """The HBM-bound kernels of the path (rows a1, a8, a9) on scaled-up stand-ins -- at the configs'
    own sizes they move < 6 MB (loss) / 0.4 GB (gather) and are launch-latency bound (DESIGN.md
    sec 6.3).  Algorithmic bytes / CUDA-event time, against the measured copy bandwidth."""
    def timeit(fn, n=10):
        for _ in range(3):
            fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(n):
            fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / n
    out = {"peak_gbs": peaks["hbm"], "stand_in": True}
    T = 1 << 26
    g = torch.Generator(device=device).manual_seed(0)
    logp = -3.0 * torch.rand(T, device=device, generator=g)
    old = logp + 0.05 * torch.randn(T, device=device, generator=g)
    ref = logp + 0.1 * torch.randn(T, device=device, generator=g)
    y = torch.randint(0, 1000, (T,), device=device, dtype=torch.int32, generator=g)
    # cfg2's layout scaled up: samples of 1024 tokens = 256 prompt (mask 0) + 768 response tokens;
    # and a stress layout of 16-token responses
    mask = ((torch.arange(T, device=device) % 1024) >= 256).to(torch.uint8)
    for seqlen in (1024, 16):
        R = T // seqlen
        cu = torch.arange(0, T + 1, seqlen, device=device, dtype=torch.int32)
        adv = torch.randn(R, device=device, generator=g)
        for agg, agg_name in ((0, "token_mean"), (1, "seq_mean")):
            ms = timeit(lambda: B.gc_grpo_token_loss(logp, old, ref, y, mask, cu, adv, agg=agg))
            # ALGORITHMIC bytes: per token logp, old, ref, target
            # (4 B each) + mask (1 B) read, g (4 B) written = 21 B; per response cu_seqlens +
            # advantage (8 B), and for seq-mean the per-response count written and read (8 B).
            # What the kernel really moves (ncu, profiles/r3_loss.md: 20.9-22.9 B/token since phase 1
            # keeps the scored flags in a bitmap; 25.8 in round 2) is `traffic_bytes_per_token`
            per_tok = 21.0 + (8.0 + (8.0 if agg else 0.0)) / seqlen
            gbs = per_tok * T / ms / 1e6
            out[f"loss_and_grad_{agg_name}_{seqlen}_token_responses"] = {
                "tokens": T, "responses": R, "bytes_per_token": per_tok,
                "traffic_bytes_per_token": {(0, 1024): 20.94, (1, 1024): 20.96, (0, 16): 21.69,
                                            (1, 16): 22.92}[(agg, seqlen)], "ms": ms, "gbs": gbs,
                "frac": gbs / peaks["hbm"], "launches": 1}
    del logp, old, ref, y, mask, cu, adv
    T2, D = 1 << 19, 4096
    H = torch.randn(T2, D, device=device, generator=g).to(torch.bfloat16)
    y2 = torch.zeros(T2, device=device, dtype=torch.int32)
    m2 = (torch.rand(T2, device=device, generator=g) < 0.75).to(torch.uint8)
    n = int(m2.sum())
    ms = timeit(lambda: B.gc_compact_rows(H, y2, m2))
    gbs = (2.0 * n * D * 2 + 9.0 * T2) / ms / 1e6
    out["compact_and_gather_rows"] = {"rows": T2, "scored_rows": n, "hidden": D, "ms": ms,
                                      "gbs": gbs, "frac": gbs / peaks["hbm"]}
    # PPO critic (NEXT-2): value head forward (reads H once) and backward (reads H, writes dH)
    wv = (torch.randn(D, device=device, generator=g) / 64).to(torch.bfloat16)
    gt = torch.randn(T2, device=device, generator=g)
    ms = timeit(lambda: B.gc_value_head_fwd(H, wv))
    gbs = (2.0 * T2 * D + 4.0 * T2) / ms / 1e6
    out["value_head_fwd"] = {"rows": T2, "hidden": D, "ms": ms, "gbs": gbs, "frac": gbs / peaks["hbm"]}
    ms = timeit(lambda: B.gc_value_head_bwd(H, wv, gt))
    gbs = (4.0 * T2 * D + 4.0 * T2) / ms / 1e6
    out["value_head_bwd"] = {"rows": T2, "hidden": D, "ms": ms, "gbs": gbs, "frac": gbs / peaks["hbm"]}
    return out


def library_baseline(b, steps=20):
    """Context only (not the product path, not the oracle): the same forward scoring the way the
    paper's own stack does it (PyTorch / Megatron-Core library calls) -- one cuBLAS
    GEMM that materialises the [T,V] logits in bf16, then fp32 log-softmax, gather and entropy
    in row blocks so the fp32 intermediates fit.  Reported next to the fused kernel."""
    w = b.w
    def gemm():
        return torch.matmul(b.H, b.W.t())
    def full():
        z = torch.matmul(b.H, b.W.t())
        lp = torch.empty(b.T, dtype=torch.float32, device=z.device)
        en = torch.empty(b.T, dtype=torch.float32, device=z.device)
        for r0 in range(0, b.T, 2048):
            zz = z[r0:r0 + 2048].float() / w.tau
            ls = zz - torch.logsumexp(zz, dim=-1, keepdim=True)
            lp[r0:r0 + 2048] = ls.gather(1, b.y[r0:r0 + 2048].long().clamp_min(0)[:, None])[:, 0]
            en[r0:r0 + 2048] = -(ls.exp() * ls).sum(-1)
        return lp, en
    out = {}
    for name, fn in (("cublas_gemm_only", gemm), ("torch_matmul_logsoftmax_gather_entropy", full)):
        for _ in range(2):
            fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(steps):
            fn()
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / steps
        out[name] = {"ms_per_step": ms, "scored_tokens_per_s": b.n_scored / (ms * 1e-3),
                     "tflops": 2.0 * b.T * w.D * w.V / (ms * 1e-3) / 1e12}
    out["logits_bytes_materialised"] = 2 * b.T * w.V
    return out


# --------------------------------------------------------------------------------------------
# end to end from host buffers
# --------------------------------------------------------------------------------------------
def _event_time(step, steps, warmup):
    for _ in range(warmup):
        step()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(steps):
        step()
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / steps


def e2e_forward(B, b: DeviceBatch, steps, warmup):
    """Same metric through the C-ABI call with HOST buffers (gc_token_logprobs_host): per step H2D
    of H / targets / mask from pinned memory (H band by band, overlapped with the contraction), the
    kernels, D2H of logp + entropy, all inside the timed region."""
    w = b.w
    Hh = b.H.cpu().pin_memory()
    yh = b.y.cpu().pin_memory()
    mh = None if b.mask is None else b.mask.cpu().pin_memory()
    lph = torch.empty(b.T, dtype=torch.float32).pin_memory()
    enh = torch.empty(b.T, dtype=torch.float32).pin_memory()
    ms = _event_time(lambda: B.gc_token_logprobs_host(Hh, b.W, yh, mh, w.tau, logp_host=lph,
                                                      entropy_host=enh), steps, warmup)
    h2d = Hh.numel() * Hh.element_size() + yh.numel() * 4 + (0 if mh is None else mh.numel())
    return {"value": b.n_scored / (ms * 1e-3), "unit": "scored tokens/s", "h2d_bytes_per_step": h2d,
            "d2h_bytes_per_step": 2 * b.T * 4, "ms_per_step": ms,
            "pass": "fwd (gc_token_logprobs_host: H copy overlapped band by band)",
            "checksum_logp": float(lph.sum())}


def e2e_train_step(B, b: DeviceBatch, steps, warmup):
    """fwd+bwd end to end (gc_grpo_step_host): per step H, targets, mask, cu_seqlens, rewards,
    group offsets, old / ref log-probs come from pinned host memory; out5 and dH go back to the
    host; dW is model state and stays on the device."""
    w = b.w
    pin = lambda t: None if t is None else t.cpu().pin_memory()
    Hh, yh, mh = pin(b.H), pin(b.y), pin(b.mask)
    cuh, rwh, goh, oldh, refh = pin(b.cu), pin(b.rewards), pin(b.go), pin(b.old), pin(b.ref)
    out5h = torch.empty(5, dtype=torch.float32).pin_memory()
    dHh = torch.empty(b.T, w.D, dtype=b.H.dtype).pin_memory()
    ms = _event_time(lambda: B.gc_grpo_step_host(Hh, b.W, yh, mh, w.tau, cuh, rwh, goh, oldh, refh,
                                                 b.dW, clip_lo=w.clip_lo, clip_hi=w.clip_hi,
                                                 beta=w.beta, out5_host=out5h, dH_host=dHh),
                     steps, warmup)
    h2d = sum(t.numel() * t.element_size() for t in (Hh, yh, mh, cuh, rwh, goh, oldh, refh)
              if t is not None)
    return {"value": b.n_scored / (ms * 1e-3), "unit": "scored tokens/s", "h2d_bytes_per_step": h2d,
            "d2h_bytes_per_step": dHh.numel() * dHh.element_size() + 20, "ms_per_step": ms,
            "pass": "fwd+bwd (gc_grpo_step_host: H copy overlapped with the forward, dH copied back "
                    "under the last dW contraction; dW stays on the device)",
            "loss": float(out5h[0])}


# --------------------------------------------------------------------------------------------
# one workload, measured
# --------------------------------------------------------------------------------------------
def measure_workload(B, w, device, steps, warmup, peaks, with_e2e, with_library=False):
    b = DeviceBatch(w, seed=0, device=device)
    step, launches = make_step(B, b)
    total_ms, per, kinds = timed_region(step, steps, warmup, False, B)
    ms = total_ms / steps
    roofs = rooflines(w, b.n_scored, steps, kinds, total_ms, peaks)
    passes = 4 if w.backward else 1
    out = {"workload": w.name, "metric": metric_name(w), "value": b.n_scored / (ms * 1e-3),
           "unit": "scored tokens/s", "ms_per_step": ms, "steps": steps, "warmup": warmup,
           "scored_tokens": b.n_scored, "tokens": b.T, "gpu_launches_per_step": launches,
           "step_tflops": 2.0 * b.n_scored * w.D * w.V * passes / (ms * 1e-3) / 1e12,
           "rooflines": roofs}
    if hasattr(b, "T_kept"):
        out["tokens_kept_after_group_filter"] = b.T_kept
        out["flow"] = "advantages(drop) -> gc_balance_plan -> gathers -> fwd+bwd"
    if with_e2e and not w.drop_constant_groups:         # as many timed steps as the device figure
        out["e2e"] = e2e_train_step(B, b, steps, 3) if w.backward else e2e_forward(B, b, steps, 3)
    if with_library:
        out["library_baseline"] = library_baseline(b)
    del b, step
    gc.collect()
    torch.cuda.empty_cache()
    return out


def attention_workload(B, device, peaks):
    """NEXT-4: all-gather-KV attention forward, as the last of 8 context-parallel
    ranks sees it (its 16384-query chunk against all 131072 gathered keys, causal, GQA 16/4 heads,
    head_dim 128, two of the four key/value heads gathered at a time on the side stream), and a single-rank
    32768-token causal case.  Algorithmic flops = 4 * allowed (q, k) pairs * head_dim * Hq."""
    out = {}
    for name, S, Hq, Hkv, world, hps in (("cp8_last_rank_131072", 131072, 16, 4, 8, 2),
                                         ("single_rank_32768", 32768, 32, 8, 1, 2)):
        g = torch.Generator(device=device).manual_seed(0)
        K = torch.randn(S, Hkv, 128, device=device, generator=g).to(torch.bfloat16)
        V = torch.randn(S, Hkv, 128, device=device, generator=g).to(torch.bfloat16)
        cuts = [S * r // world for r in range(world + 1)]
        rows = [b - a for a, b in zip(cuts[:-1], cuts[1:])]
        Ks = [K[a:b].contiguous() for a, b in zip(cuts[:-1], cuts[1:])]
        Vs = [V[a:b].contiguous() for a, b in zip(cuts[:-1], cuts[1:])]
        rank = world - 1
        Q = torch.randn(rows[rank], Hq, 128, device=device, generator=g).to(torch.bfloat16)
        kp, vp = [k.data_ptr() for k in Ks], [v.data_ptr() for v in Vs]
        ms = _event_time(lambda: B.gc_attention_allgather_kv(Q, kp, vp, rows, rank, Hkv, None, True, 0,
                                                             None, hps, want_lse=True), 5, 3)
        q0, n = cuts[rank], rows[rank]
        pairs = n * q0 + n * (n + 1) // 2                   # causal: keys 0 .. q
        flops = 4.0 * pairs * 128 * Hq
        tf = flops / (ms * 1e-3) / 1e12
        out[name] = {"tokens_total": S, "queries_local": n, "q_heads": Hq, "kv_heads": Hkv,
                     "head_dim": 128, "world": world, "kv_heads_per_gather_step": hps, "mask": "causal",
                     "ms": ms, "roofline": {"bound": "tensor", "kernel": "attn::k_attn_fwd",
                                            "achieved": tf, "peak": peaks["burst"], "unit": "TFLOP/s",
                                            "frac": tf / peaks["burst"], "flops_per_call": flops,
                                            "gathered_bytes_per_call": 2 * S * Hkv * 128 * 2}}
        del K, V, Ks, Vs, Q
        torch.cuda.empty_cache()
    return out


# --------------------------------------------------------------------------------------------
# N > 1 training arm: the dW exchange
# --------------------------------------------------------------------------------------------
def make_train_step_dp(B, b, arm, world, rank):
    """Data-parallel training step on this rank's micro-batch (W replicated).  Both arms leave, on
    every rank, its shard [shard_rows, D] of the dW summed over ranks, scaled so that it is the
    gradient of the global token-mean objective (dp.global_grad_scale x 1/world)."""
    import torch.distributed as dist
    from paper_2507_22789_b200 import dp
    w = b.w
    sr = dp.shard_rows_for(w.V, world)
    shard = torch.zeros(sr, w.D, dtype=torch.float32, device=b.H.device)
    scale = dp.global_grad_scale(b.n_scored) / world
    if arm == "fused":
        ptrs, keep = dp.exchange_dw_shards(shard)

        def step():
            shard.zero_()
            torch.cuda.current_stream().synchronize()
            dist.barrier()                              # every shard is zero before any add
            adv, _ = B.gc_grpo_advantages(b.rewards, b.go, 1e-6, False, False)
            f = B.gc_grpo_loss_fwd(b.H, b.W, b.y, b.mask, w.tau, b.cu, adv, b.old, b.ref, w.clip_lo,
                                   w.clip_hi, w.beta)
            B.gc_grpo_loss_bwd_reduce_scatter(b.H, b.W, b.y, b.mask, w.tau, b.cu, adv, b.old, b.ref,
                                              f["logp"], f["lse"], ptrs, sr, clip_lo=w.clip_lo,
                                              clip_hi=w.clip_hi, beta=w.beta, grad_loss=scale,
                                              dH=b.dH, fwd_state=f["state"])
            torch.cuda.current_stream().synchronize()
            dist.barrier()                              # every rank's adds have landed
            return f["out5"]
        step.keep = keep
        return step, shard
    full = torch.zeros(sr * world, w.D, dtype=torch.float32, device=b.H.device)

    def step():
        adv, _ = B.gc_grpo_advantages(b.rewards, b.go, 1e-6, False, False)
        f = B.gc_grpo_loss_fwd(b.H, b.W, b.y, b.mask, w.tau, b.cu, adv, b.old, b.ref, w.clip_lo,
                               w.clip_hi, w.beta)
        B.gc_grpo_loss_bwd(b.H, b.W, b.y, b.mask, w.tau, b.cu, adv, b.old, b.ref, f["logp"], f["lse"],
                           w.clip_lo, w.clip_hi, w.beta, grad_loss=scale, dH=b.dH, dW=full[:w.V],
                           fwd_state=f["state"])
        dist.reduce_scatter_tensor(shard, full)
        return f["out5"]
    return step, shard


def maybe_respawn(args):
    """--gpus N > 1 outside torch.distributed.run: start N ranks of this script (one per GPU,
    rendezvous on 127.0.0.1) and return their exit code."""
    if args.gpus <= 1 or "WORLD_SIZE" in os.environ:
        return None
    port = os.environ.get("MASTER_PORT", "29517")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1",
           f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1", "--master-port", port,
           os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def run_dry(args, w):
    """The N-rank launch path on CPU (gloo): rendezvous, barriers, the max-time / summed-token
    reductions, one JSON line from rank 0.  No kernel runs: value is null."""
    import torch.distributed as dist
    from paper_2507_22789_b200 import dp
    rank, world, _ = dp.env_rank_world()
    if world > 1:
        dist.init_process_group("gloo")
    dp.barrier()
    lay = I.make_layout(w, rank)
    fake_ms = 10.0 + rank
    total_ms, tokens_all = dp.reduce_step_stats(fake_ms * args.steps, float(lay.mask.sum()))
    grad_scale = dp.global_grad_scale(float(lay.mask.sum()))
    dp.barrier()
    if rank == 0:
        print(json.dumps({"metric": metric_name(w), "value": None, "unit": "scored tokens/s",
                          "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                          "ms_per_step": total_ms / args.steps, "dry_run": True,
                          "ranks_started": world, "tokens_all_ranks": tokens_all,
                          "grad_scale_rank0": grad_scale,
                          "config": workload_config(w, lay.T, world)}))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--workload", default=HEADLINE, choices=sorted(WORKLOADS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-extras", action="store_true",
                    help="skip the cpu_baseline / e2e / other-workload extras (rank 0, N=1 only)")
    ap.add_argument("--arm", default="fused", choices=["fused", "nccl"],
                    help="N > 1 training workloads: how dW is exchanged (both are reported)")
    ap.add_argument("--dist-backend", default="nccl", choices=["nccl", "gloo"],
                    help="control-plane backend (gloo: ranks may share a GPU; the NCCL arm is skipped)")
    ap.add_argument("--dry-run", action="store_true")
    ap.add_argument("--only", default=None, choices=["hbm", "attention"],
                    help="run only that part of the extras and print it (profiling aid)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    w = I.CONFIGS[WORKLOADS[args.workload]]
    if args.impl == "reference":
        return run_reference(args, w)
    rc = maybe_respawn(args)
    if rc is not None:
        sys.exit(rc)
    if args.dry_run:
        return run_dry(args, w)

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    dist_on = world > 1
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    dev_index = local_rank % torch.cuda.device_count()
    torch.cuda.set_device(dev_index)
    device = torch.device("cuda", dev_index)
    if dist_on:
        import torch.distributed as dist
        if args.dist_backend == "nccl":
            # let NCCL print its INIT lines (ranks, transports, NVLS) so that the driver can count
            # the ranks that really joined; a caller's own setting wins
            os.environ.setdefault("NCCL_DEBUG", "INFO")
            os.environ.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
            dist.init_process_group("nccl", device_id=device)
        else:
            dist.init_process_group("gloo")
    from paper_2507_22789_b200 import binding as B      # raises if libgcore.so is missing
    from paper_2507_22789_b200 import dp
    peaks = load_peaks()
    if args.only:
        part = hbm_kernels(B, device, peaks) if args.only == "hbm" else attention_workload(B, device, peaks)
        print(json.dumps({args.only: part}))
        return

    # every rank: its own tokens (seed = rank), the same W (seed 0)
    b = DeviceBatch(w, seed=rank, device=device, w_seed=0 if dist_on else None)
    exchange = "none"
    dp_info = None
    if dist_on and w.backward and not w.drop_constant_groups and w.dtype == "bf16":
        exchange = ("dW reduce-scatter fused into the dW contraction (TMA reduce-add into peer "
                    "shards over NVLink)" if args.arm == "fused" else "NCCL reduce-scatter of dW")
        step, shard = make_train_step_dp(B, b, args.arm, world, rank)
        n_chunks = -(-b.T // _bwd_chunk_T(B, b.T, w))
        launches = 1 + (8 if b.mask is not None else 2) + 1 + 1 + (3 if b.mask is not None else 0) \
            + 3 * n_chunks + 1
    else:
        step, launches = make_step(B, b)
    sampler = ClockSampler(list(range(min(world, torch.cuda.device_count()))) if rank == 0 else [])
    if rank == 0:
        sampler.start()
    total_ms, per, kinds = timed_region(step, args.steps, args.warmup, dist_on, B)
    clocks = sampler.stop() if rank == 0 else None
    tokens = b.n_scored
    T_rank = b.T
    total_ms_max, tokens_all = dp.reduce_step_stats(total_ms, tokens)   # max time, summed tokens
    ms_per_step = total_ms_max / args.steps
    value = tokens_all / (ms_per_step * 1e-3)

    if exchange != "none":
        # the other arm, same batch, for comparison; bytes a rank puts on the wire per step
        other = "nccl" if args.arm == "fused" else "fused"
        dp_info = {"arm": args.arm, "ms_per_step": ms_per_step,
                   "wire_bytes_per_rank_per_step": (world - 1) / world * w.V * w.D * 4,
                   "shard_rows": dp.shard_rows_for(w.V, world)}
        same_gpu = world > torch.cuda.device_count()
        if other == "nccl" and (args.dist_backend != "nccl" or same_gpu):
            dp_info["other_arm"] = {"arm": other, "skipped": "ranks share a GPU / gloo control plane"}
        else:
            step2, _ = make_train_step_dp(B, b, other, world, rank)
            k2 = max(3, args.steps // 2)
            t2, _, _ = timed_region(step2, k2, 3, True, None)
            t2, _ = dp.reduce_step_stats(t2, 0.0)
            dp_info["other_arm"] = {"arm": other, "ms_per_step": t2 / k2}

    if rank == 0:
        step_ms = float(np.mean(per))
        roofs = rooflines(w, tokens, args.steps, kinds, total_ms, peaks)
        extra_cfg = ({"tokens_kept_after_group_filter": b.T_kept,
                      "flow": "advantages(drop) -> gc_balance_plan -> gathers -> fwd+bwd"}
                     if hasattr(b, "T_kept") else {})
        e2e = cpu = None
        others = {}
        detail("rooflines", workload=w.name, rooflines=roofs)
        if dp_info:
            detail("dp_exchange", **dp_info)
        if world == 1 and not args.no_extras:
            half = max(3, args.steps // 2)
            if w.dtype == "bf16" and not w.drop_constant_groups:
                e2e = e2e_train_step(B, b, half, 3) if w.backward else e2e_forward(B, b, half, 3)
            cpu = cpu_baseline(w, 64 if w.D * w.V > 1e9 else 256 if w.D * w.V > 1e8 else 1 << 30)
            detail("cpu_baseline", **cpu)
            if args.workload == HEADLINE:
                del b, step
                gc.collect()
                torch.cuda.empty_cache()
                # the metric's forward half, the 8B-class step and the dynamic-sampling step
                for name, k, wu in (("cfg1", args.steps, 3), ("cfg2", max(4, args.steps // 4), 3),
                                    ("cfg3", 3, 3)):
                    m = measure_workload(B, I.CONFIGS[WORKLOADS[name]], device, k, wu, peaks,
                                         with_e2e=(name != "cfg3"), with_library=(name == "cfg1"))
                    detail("workload", **m)
                    others[name] = workload_scalars(m)
                detail("hbm_kernels", **hbm_kernels(B, device, peaks))
                torch.cuda.empty_cache()
                detail("attention_allgather_kv", **attention_workload(B, device, peaks))
        out = assemble_line(w, value=value, ms_per_step=ms_per_step, T=T_rank, world=world,
                            steps=args.steps, warmup=args.warmup, exchange=exchange, clocks=clocks,
                            gpu_launches=launches * args.steps, roofs=roofs, step_ms=step_ms, e2e=e2e,
                            cpu=cpu, workloads=others, extra_config=extra_cfg, dp_info=dp_info)
        final_line = emit(out)
    if dist_on:
        import torch.distributed as dist
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        # after the teardown, so that NCCL's own INFO lines (N > 1) never follow the JSON line
        sys.stdout.flush()
        print(final_line, flush=True)


if __name__ == "__main__":
    main()
