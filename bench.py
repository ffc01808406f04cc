#!/usr/bin/env python
"""bench.py — fused context tokens/s per qcf_layer_step at rho = 0.3 (BASELINE.json metric) on a B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c4] [--configs all|none] [--impl qcf|reference]

One "step" = one pass of the whole hot path (a1 reposition -> a2 score -> a3 top-k -> a4 scatter -> a5 recompute
attention) over one batch of seeded synthetic requests.  The headline workload is the largest
single-layer config at rho = 0.3: BASELINE.json configs[3] ("c4": 16 requests x 8 x 1024-token chunks + 128-token
query, 131 072 context tokens per step, one batched launch per stage).  With --configs all (the default at N = 1) the
same line carries a `configs` sub-dict with configs[1] (c2), configs[4] (c5) and the configs[2] pipeline (c3: TTFT and
speed-up over the library's own full prefill), each measured by the same code with fewer steps.
N > 1 (torchrun, one rank per GPU): requests are independent, so every rank runs its own replica of
the headline workload with no data-path collective — weak scaling; `value` = tokens all ranks processed /
max-over-ranks device time.

Timing: W >= 3 warm-up steps, then exactly K steps, each bracketed by CUDA events on the launching stream; an L2
flush (a write of a 256 MiB buffer followed by a read of a second 256 MiB buffer, so that the cache is left full of
CLEAN foreign lines; outside the event pair) precedes every step (c4's 2.7 GB working set exceeds the 126 MB L2 anyway;
c2's does not).  Barrier + synchronize on both sides of the timed region; max over ranks.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "fused context tokens/s per layer step at r=0.3"
UNIT = "tokens/s"
KERNELS_PER_STEP = 6           # reposition, score pass 1, score pass 2, topk, scatter, attn
FALLBACK_PEAKS = {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0}
BASELINE_CONFIG = {"c1": "configs[0]", "c2": "configs[1]", "c3": "configs[2]", "c4": "configs[3]", "c5": "configs[4]"}
# MUFU.EX2 rate used as the denominator of a2's exponential fraction: 16 per clock per SM (4 per SM sub-partition,
# B300_MICROARCH.md pipe table; consistent with ncu's sm__inst_executed_pipe_xu on the a2 kernels)
MUFU_PER_CLK_PER_SM, N_SM = 16, 148



def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--workload", default="c4")
    ap.add_argument("--ratio", type=float, default=None)
    ap.add_argument("--impl", default="qcf", choices=["qcf", "reference"])
    ap.add_argument("--configs", default=None, choices=["all", "none"],
                    help="all: add the c2 / c5 / c3 sub-records to the line (default when the workload is the default c4 at "
                         "N = 1); none: the headline workload only")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--shard", default="requests", choices=["requests", "heads"],
                    help="requests: one replica per rank, no collective (default, weak scaling); heads: ONE request set split "
                         "over the ranks by kv-head groups with an all-reduce of the scores (strong scaling)")
    return ap.parse_args()


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return d, "measured"
    return dict(FALLBACK_PEAKS), "fallback"


def n_cores() -> int:
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1


def profile_traffic(workload: str, kernel_substr: str):
    """dram__bytes_read.sum + dram__bytes_write.sum of one launch of `kernel_substr` on `workload`, from the committed ncu
    --set full summary profiles/r03_<workload>_kernels.csv (else the round-2 file; the .md beside it names the capture
    command).  None if the summary or the kernel's row is absent — never a hard-coded number."""
    for rnd in ("r03", "r02"):
        path = os.path.join(ROOT, "profiles", "%s_%s_kernels.csv" % (rnd, workload))
        if os.path.exists(path):
            break
    else:
        return None, None
    import csv
    with open(path, newline="") as f:
        rows = list(csv.DictReader(f))
    for r in rows:
        if kernel_substr in r.get("kernel", ""):
            try:
                return int(float(r["dram_bytes_read"]) + float(r["dram_bytes_write"])), os.path.relpath(path, ROOT)
            except (KeyError, ValueError):
                return None, None
    return None, None


# ------------------------------------------------------------------------------------------------ oracle legs

def oracle_inputs(wl, b=0):
    from oracle import qcf_oracle as O
    r = wl.requests[b]
    w = O.widen_bf16
    return (r, [w(wl.pool_k[i]) for i in r.chunk_ids], [w(wl.pool_v[i]) for i in r.chunk_ids],
            w(r.q_probe), w(r.q_new), w(r.k_new), w(r.v_new))


def oracle_sample_stride(wl) -> int:
    """a5 row stride of the oracle's bounded step: about 48 sampled rows per request whatever the config (the fp64 a5 of
    ONE c4 row costs ~34 MFLOP x 32 heads; a1-a4 are always run in full)."""
    r = wl.requests[0]
    n_rows = int(wl.cfg.ratio * r.n_ctx) + r.n_query
    return max(1, n_rows // 48)


def oracle_sampled_step(wl, inp, stride: int):
    """The oracle as it stands on one request: a1 + a2 + a3 + a4 in full, a5 on every `stride`-th row of R (rows are
    independent given the fused cache, so each sampled row is exact).  Returns (seconds actually spent, seconds a whole
    step would take with the a5 part scaled by the causal-pair count sum_r (p_r + 1) of all rows / of the sample)."""
    from oracle import qcf_oracle as O
    r, kp, vp, qp, qn, kn, vn = inp
    t0 = time.perf_counter()
    k_ctx, v_ctx = O.reposition(kp, vp, wl.cfg.rope_theta)
    sc = O.score(qp, k_ctx)
    sel = O.select_topk(sc, O.n_select(r.n_ctx, wl.cfg.ratio))
    k_f, v_f = O.fuse(k_ctx, v_ctx, sel, kn, vn)
    t1 = time.perf_counter()
    rows = np.concatenate([sel, np.arange(r.n_ctx, r.n_ctx + r.n_query)])
    sample = rows[::stride]
    O.recompute_attn(qn[sample], sample, k_f, v_f)
    t2 = time.perf_counter()
    scale = float(np.sum(rows + 1)) / max(float(np.sum(sample + 1)), 1.0)
    return t2 - t0, (t1 - t0) + (t2 - t1) * scale


def blas_threads() -> int:
    try:
        from threadpoolctl import threadpool_info
        n = [p.get("num_threads", 0) for p in threadpool_info() if p.get("user_api") == "blas"]
        return max(n) if n else n_cores()
    except Exception:
        return n_cores()


def cpu_baseline_record(wl, cfg) -> dict:
    """the fp64 numpy oracle on the host cores, one request, bounded sample, at the BLAS library's thread
    count and at 1 thread."""
    inp = oracle_inputs(wl)
    stride = oracle_sample_stride(wl)
    n = wl.requests[0].n_ctx
    spent, full = oracle_sampled_step(wl, inp, stride)
    rec = {"value": n / full, "unit": UNIT, "cores": blas_threads(), "kind": "oracle",
           "sample": "oracle (fp64 numpy) on ONE %s request: a1 + a2 + a3 + a4 in full (scores and top-k over all %d positions), "
                     "a5 on every %d-th row of R; %.1f s spent, a5 time scaled by the causal-pair count of all rows / of the "
                     "sample -> %.1f s per whole step; BLAS threads = %d of %d affinity cores" %
                     (cfg.name, n, stride, spent, full, blas_threads(), n_cores())}
    try:
        from threadpoolctl import threadpool_limits
        with threadpool_limits(limits=1):
            spent1, full1 = oracle_sampled_step(wl, inp, stride * 2)
        rec["value_1_thread"] = n / full1
        rec["sample_1_thread"] = "same with every %d-th row, BLAS limited to 1 thread: %.1f s spent -> %.1f s per step" % (stride * 2, spent1, full1)
    except Exception as e:                                   # pragma: no cover
        rec["value_1_thread"] = None
        rec["sample_1_thread"] = "threadpoolctl unavailable: %s" % e
    return rec


def run_reference(args) -> None:
    """--impl reference: the fp64 oracle on the host cores, same metric / config.  Rank 0 only.  A "step" is the bounded
    sample of oracle_sampled_step; `ms_per_step` is what was actually timed, `value` the whole-step extrapolation."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    from paper_2606_05875_b200 import inputs
    wl = inputs.make_workload(args.workload, ratio=args.ratio, batch=1)
    inp = oracle_inputs(wl)
    stride = oracle_sample_stride(wl)
    for _ in range(max(args.warmup, 0)):
        oracle_sampled_step(wl, inp, stride)
    res = [oracle_sampled_step(wl, inp, stride) for _ in range(args.steps)]
    spent = float(np.mean([a for a, _ in res]))
    full = float(np.mean([b for _, b in res]))
    value = wl.requests[0].n_ctx / full
    sample = ("per step: a1+a2+a3+a4 of one %s request in full, a5 on every %d-th row of R (exact per row); ms_per_step is the "
              "time actually spent (%.0f ms); value = N / (a1..a4 time + a5 time x causal pairs of all rows / of the sample) "
              "= N / %.0f ms; BLAS threads = %d" % (wl.cfg.name, stride, spent * 1e3, full * 1e3, blas_threads()))
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": spent * 1e3, "extrapolated_ms_per_whole_step": full * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": config_dict(wl.cfg, args.gpus, l2="flushed before every timed step (256 MiB write then 256 MiB read, outside the event pair)",
                              batch=inputs.CONFIGS[args.workload].batch),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": blas_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def config_dict(cfg, n_gpus: int, l2: str, batch=None) -> dict:
    b = cfg.batch if batch is None else batch
    return {"workload": "%s: %d request(s)/GPU x %d chunks x %d tokens (N=%d) + %d-token query, Hq/Hkv=%d/%d, d=%d, "
                        "bf16, theta=%g, rho=%g" % (cfg.name, b, cfg.n_chunks, cfg.chunk_len, cfg.n_ctx,
                                                    cfg.n_query, cfg.n_q_heads, cfg.n_kv_heads, cfg.head_dim,
                                                    cfg.rope_theta, cfg.ratio),
            "baseline_config": BASELINE_CONFIG.get(cfg.name, cfg.name),
            "ratio": cfg.ratio, "global_batch": b * n_gpus, "parallelism": "replicas x%d" % n_gpus,
            "l2": l2}


def max_over_ranks(values, dist, device) -> list:
    """MAX over ranks of a list of floats (device timings): every rank contributes, every rank gets the result."""
    import torch
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t]


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms (the profiling recipe's interval) while the timed region runs; a query can stall the GPU for ~2 ms (measured: 1 step in 6000), so it is not polled faster."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc = index, None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            out = self.proc.communicate(timeout=5)[0]
        except subprocess.TimeoutExpired:
            self.proc.kill()
            out = self.proc.communicate()[0]
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in out.splitlines():
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}



# ------------------------------------------------------------------------------------------------ qcf arm

def measure_layer_config(name, ratio, steps, warmup, dev, dist, world, want_e2e, want_cpu) -> dict:
    """Everything bench.py reports about one single-layer workload, measured on `dev` (max over ranks where timed)."""
    import torch
    from paper_2606_05875_b200 import binding, device, inputs

    wl = inputs.make_workload(name, ratio=ratio)     # every rank: its own replica (weak scaling)
    cfg = wl.cfg
    ctx = binding.Context(cfg.n_q_heads, cfg.n_kv_heads, cfg.head_dim, cfg.rope_theta, max(cfg.batch, 1),
                          max(cfg.n_ctx, 1024), max(cfg.n_query, 1))
    dw = device.DeviceWorkload(wl, ctx, device=dev)
    largs = dw.layer_args(lse=None)
    tokens_per_step = int(dw.batch.total_ctx)
    flush_w = torch.empty(256 << 20, dtype=torch.uint8, device=dev)    # > 126 MB L2
    flush_r = torch.zeros(64 << 20, dtype=torch.int32, device=dev)     # 256 MiB, read after the write

    def flush_l2(i):
        flush_w.fill_(i & 0xff)        # evicts everything ...
        flush_r.max()                  # ... and the read pass replaces the dirty lines by clean ones

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident leg: K timed steps, each bracketed by CUDA events on the launching stream.  Stage profiling is
    # OFF here: its event records between the kernels would break the programmatic dependent launch chain (PDL).
    for _ in range(max(warmup, 3)):
        flush_l2(1)
        ctx.qcf_layer_step(dw.batch, largs)
    barrier()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    for i in range(steps):
        flush_l2(i)
        ev[i][0].record()
        ctx.qcf_layer_step(dw.batch, largs)
        ev[i][1].record()
    barrier()
    step_ms = np.array([a.elapsed_time(b) for a, b in ev])
    total_ms = float(step_ms.sum())

    # ---- per-stage device time: a second pass with the library's event hooks between the stages (same flush protocol;
    # the stages then run back to back without PDL overlap, so their sum is a little above the step time)
    n_prof = max(3, min(steps, 100))
    ctx.qcf_set_profiling(True)
    for i in range(3 + n_prof):
        flush_l2(i)
        ctx.qcf_layer_step(dw.batch, largs)
        if i == 2:
            torch.cuda.synchronize()
            ctx.qcf_get_stage_ms()                  # forget the warm-up steps
    barrier()
    stage_ms = np.array(ctx.qcf_get_stage_ms())     # mean per-stage device time over n_prof steps
    ctx.qcf_set_profiling(False)

    # ---- comparator: the library's own dense causal attention over all N + Lq rows (Eq. 2), same flush protocol
    out_full = torch.empty_like(dw.out)
    n_full = max(3, min(steps, 20))
    evf = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n_full)]
    for i in range(3 + n_full):
        flush_l2(i)
        if i >= 3:
            evf[i - 3][0].record()
        ctx.qcf_full_prefill_attn(dw.batch, dw.q_new, dw.k_new, dw.v_new, out_full)
        if i >= 3:
            evf[i - 3][1].record()
    barrier()
    full_ms = float(np.mean([a.elapsed_time(b) for a, b in evf]))
    del out_full

    # ---- end-to-end leg: the same step through the C ABI with HOST (pinned) buffers, copies inside the timed region
    e2e = None
    if want_e2e:
        hw = device.DeviceWorkload(wl, ctx, device="cpu", pin=True)
        hargs = hw.layer_args()
        n_e2e = max(3, min(steps, 10))
        for _ in range(2):
            ctx.qcf_layer_step_host(hw.batch, hargs, hw.pool_rows)
        barrier()
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            ctx.qcf_layer_step_host(hw.batch, hargs, hw.pool_rows)     # synchronises the stream before returning
        torch.cuda.synchronize()
        e2e_s = (time.perf_counter() - t0) / n_e2e
        nb = lambda t: t.numel() * t.element_size()
        q_row_b = cfg.n_q_heads * cfg.head_dim * 2
        kv_row_b = cfg.n_kv_heads * cfg.head_dim * 2
        out_rows = sum(binding.qcf_n_select(n, cfg.ratio) + lq for n, lq in zip(hw.batch.n_ctx, hw.batch.n_query))
        # bytes that cross the bus per step: the pool rows some request reads (shared chunks once), the probe, and — the host
        # buffers are pinned, so the a4 / a5 kernels gather them straight from host memory — the |R_b| fresh rows only
        h2d = 2 * int(hw.batch.pool_rows_touched) * kv_row_b + nb(hw.q_probe) + out_rows * (q_row_b + 2 * kv_row_b)
        d2h = out_rows * q_row_b + nb(hw.sel) + nb(hw.n_sel) + nb(hw.scores)      # only the |R_b| written rows of `out` come back
        e2e = (e2e_s, h2d, d2h, n_e2e)
        del hw, hargs

    # ---- max over ranks
    total_ms, e2e_s, full_ms = max_over_ranks([total_ms, e2e[0] if e2e else 0.0, full_ms], dist if world > 1 else None, dev)
    ms_per_step = total_ms / steps
    value = tokens_per_step * world / (ms_per_step * 1e-3)

    # ---- roofline of the dominant kernel (a5 recompute attention: tensor-bound)
    peaks, peak_kind = load_peaks()
    sel = dw.sel.cpu().numpy()
    n_sel = dw.n_sel.cpu().numpy()
    flops = 0.0
    for b, (n, lq) in enumerate(zip(dw.batch.n_ctx, dw.batch.n_query)):
        pos = np.concatenate([sel[b, : n_sel[b]].astype(np.int64), np.arange(n, n + lq)])
        flops += device.attn_flops(cfg, n, pos)
    a5_ms = float(stage_ms[4])
    achieved = flops / (a5_ms * 1e-3) / 1e12
    # The kernel is a few ms inside a step that is timed for well under a second: by MEASURED_PEAKS.json's own definition the
    # burst figure is the denominator (the sustained one is for kernels inside seconds-long steps).  The fraction of the
    # sustained peak is printed beside it: under the power cap the clocks record shows, the truth lies between the two.
    peak = float(peaks["bf16_tflops"])
    sustained = float(peaks.get("bf16_tflops_sustained", peak))
    traffic, traffic_src = profile_traffic(cfg.name, "attn_tc_kernel")
    work = dw.algorithmic_work()
    roofline = {"kernel": "attn_tc_kernel (a5 recompute attention)", "bound": "tensor", "achieved": achieved,
                "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak, "traffic": traffic, "traffic_source": traffic_src,
                "peak_source": "%s bf16_tflops (burst: a ms-scale kernel in a sub-second timed region)" % peak_kind,
                "frac_of_sustained_peak": achieved / sustained, "sustained_peak": sustained,
                "algorithmic_flops_per_launch": flops, "algorithmic_bytes_per_launch": work["a5_bytes"], "ms_per_launch": a5_ms}
    hbm = float(peaks["hbm_gbs"])
    sm_hz = float(peaks.get("sm_max_mhz", 1965.0)) * 1e6
    mufu_peak = MUFU_PER_CLK_PER_SM * N_SM * sm_hz                   # exponentials per second at the max SM clock
    gbps = lambda nbytes, ms: nbytes / (ms * 1e-3) / 1e9
    a2_ms = float(stage_ms[1])
    a2_fr = {"hbm": gbps(work["a2_bytes"], a2_ms) / hbm, "tensor": work["a2_flops"] / (a2_ms * 1e-3) / 1e12 / peak,
             "mufu": work["a2_exps"] / (a2_ms * 1e-3) / mufu_peak}
    stages = {
        "a1_reposition": {"ms": float(stage_ms[0]), "GBps": gbps(work["a1_bytes"], stage_ms[0]),
                          "frac_hbm": gbps(work["a1_bytes"], stage_ms[0]) / hbm},
        "a2_score": {"ms": a2_ms, "TFLOPps": work["a2_flops"] / (a2_ms * 1e-3) / 1e12, "frac_hbm": a2_fr["hbm"],
                     "frac_tensor": a2_fr["tensor"], "frac_mufu": a2_fr["mufu"], "binding": max(a2_fr, key=a2_fr.get),
                     "note": "single-sweep algorithmic work (K once, 2 Lq Hq N d flop, Lq Hq N exp) / time; the kernel sweeps twice"},
        "a3_topk": {"ms": float(stage_ms[2]), "bound": "latency (<= 128 KB per request in one CTA)"},
        "a4_scatter": {"ms": float(stage_ms[3]), "GBps": gbps(work["a4_bytes"], stage_ms[3]),
                       "frac_hbm": gbps(work["a4_bytes"], stage_ms[3]) / hbm},
        "a5_attn": {"ms": a5_ms, "TFLOPps": achieved, "frac_tensor": achieved / peak},
    }
    full_flops = sum(device.attn_flops(cfg, n, np.arange(n + lq)) for n, lq in zip(dw.batch.n_ctx, dw.batch.n_query))
    comparator = {"kernel": "qcf_full_prefill_attn (dense causal GQA over all N+Lq rows, Eq. 2)", "ms": full_ms,
                  "TFLOPps": full_flops / (full_ms * 1e-3) / 1e12, "frac_tensor_peak": full_flops / (full_ms * 1e-3) / 1e12 / peak,
                  "selective_step_over_full_prefill_attn": ms_per_step / full_ms}
    rec = {
        "value": value, "ms_per_step": ms_per_step, "steps": steps, "warmup": max(warmup, 3),
        "config": config_dict(cfg, world, l2="flushed before every timed step (256 MiB write then 256 MiB read, outside the event pair)"),
        "gpu_launches": KERNELS_PER_STEP * steps, "roofline": roofline, "stages": stages, "full_prefill_attn": comparator,
        "step_ms_min_med_max": [float(step_ms.min()), float(np.median(step_ms)), float(step_ms.max())],
    }
    if e2e:
        rec["e2e"] = {"value": tokens_per_step * world / e2e_s, "unit": UNIT, "h2d_bytes_per_step": int(e2e[1]),
                      "d2h_bytes_per_step": int(e2e[2]), "ms_per_step": e2e_s * 1e3, "steps": e2e[3],
                      "api": "qcf_layer_step_host (pinned host buffers: pool rows and probe uploaded, fresh rows gathered zero-copy by the "
                             "a4 / a5 kernels, |R| output rows downloaded; stream-synchronised per step)"}
    if want_cpu:
        wl1 = inputs.make_workload(name, ratio=ratio, batch=1) if cfg.batch != 1 else wl
        rec["cpu_baseline"] = cpu_baseline_record(wl1, cfg)
    del dw, ctx, flush_w, flush_r
    torch.cuda.empty_cache()
    return rec


def run_qcf(args) -> None:
    import torch
    import torch.distributed as dist

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device — the qcf arm has no CPU fallback")
    torch.cuda.set_device(local)
    dev = "cuda:%d" % local
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(dev))
    if args.gpus != world and rank == 0:
        print("bench.py: --gpus %d but WORLD_SIZE %d; using WORLD_SIZE" % (args.gpus, world), file=sys.stderr)
    args.gpus = world
    sub = args.configs if args.configs is not None else ("all" if (args.workload == "c4" and world == 1 and args.ratio is None) else "none")

    t_wall = time.perf_counter()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.4)
    head = measure_layer_config(args.workload, args.ratio, args.steps, args.warmup, dev, dist, world,
                                want_e2e=not args.no_e2e, want_cpu=(not args.no_cpu_baseline) and rank == 0)
    clocks = sampler.stop() if rank == 0 else None
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    line = {
        "metric": METRIC, "value": head["value"], "unit": UNIT, "n_gpus": world, "steps": head["steps"], "warmup": head["warmup"],
        "ms_per_step": head["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "bf16", "data": "synthetic", "config": head["config"], "clocks": clocks,
        "gpu_launches": head["gpu_launches"], "roofline": head["roofline"], "stages": head["stages"],
        "full_prefill_attn": head["full_prefill_attn"], "step_ms_min_med_max": head["step_ms_min_med_max"],
    }
    for k in ("e2e", "cpu_baseline"):
        if k in head:
            line[k] = head[k]
    if sub == "all":
        # the other BASELINE configs, same code, fewer steps: one driver run reproduces every row of DESIGN.md §7
        cfgs = {}
        for key, name, ratio in (("c1", "c1", None), ("c2", "c2", None), ("c5", "c5", None), ("c4_rho0.1", "c4", 0.1), ("c4_rho0.5", "c4", 0.5)):
            s2 = ClockSampler(local); s2.start(); time.sleep(0.2)
            n_steps = max(10, min(args.steps, 50)) if ratio is None else 10        # configs[3] sweeps rho in {0.1, 0.3, 0.5}
            try:
                r = measure_layer_config(name, ratio, n_steps, args.warmup, dev, dist, world, want_e2e=False, want_cpu=False)
            except Exception as e:                           # the headline number must survive a failing sub-record
                r = {"error": "%s: %s" % (type(e).__name__, e)}
            r["clocks"] = s2.stop()
            cfgs[key] = r
        try:
            cfgs["c3"] = c3_record(args, steps=max(3, min(args.steps, 5)), light=True)
        except Exception as e:                               # the headline number must survive a failing sub-record
            cfgs["c3"] = {"error": "%s: %s" % (type(e).__name__, e)}
        line["configs"] = cfgs
    line["wall_s"] = time.perf_counter() - t_wall
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


# ------------------------------------------------------------------------------------------------ kv-head shards

def run_head_sharded(args) -> None:
    """the step of ONE request set split over the ranks by kv-head groups
    (paper_2606_05875_b200/sharded.py).  Strong scaling: total work is fixed, the only exchange is the all-reduce(sum) of
    scores[B][n_stride] between a2 and the replicated a3.  Not the default arm (requests are independent: replicas)."""
    import torch
    import torch.distributed as dist
    from paper_2606_05875_b200 import device, inputs, sharded

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device — the qcf arm has no CPU fallback")
    torch.cuda.set_device(local)
    dev = "cuda:%d" % local
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(dev))
    wl = inputs.make_workload(args.workload, ratio=args.ratio)
    cfg = wl.cfg
    st = sharded.HeadShardedStep(cfg.n_q_heads, cfg.n_kv_heads, cfg.head_dim, cfg.rope_theta, max(cfg.batch, 1),
                                 max(cfg.n_ctx, 1024), max(cfg.n_query, 1), rank=rank, world=world)
    dw = device.DeviceWorkload(inputs.shard_heads(wl, rank, world), st.ctx, device=dev)
    exchange = "none"
    if world > 1:
        # the score exchange fused into a2 over peer memory (include/qcf.h, qcf_set_score_exchange); NCCL is the rendezvous
        slot = dw.batch.batch * dw.batch.n_stride
        mine = sharded.HeadShardedStep.alloc_exchange_buffer(world, slot, device=dev)
        st.enable_fused_exchange(sharded.share_exchange_buffers(mine, rank, world), slot)
        exchange = "fused into a2 (peer stores + flags), %d B per rank and step" % (slot * 4 * (world - 1))
    kw = dict(k_pool=dw.k_pool, v_pool=dw.v_pool, k_fused=dw.k_fused, v_fused=dw.v_fused, q_probe=dw.q_probe,
              scores=dw.scores, sel=dw.sel, n_sel=dw.n_sel, q_new=dw.q_new, k_new=dw.k_new, v_new=dw.v_new, out=dw.out,
              ratio=cfg.ratio)
    flush_w = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    flush_r = torch.zeros(64 << 20, dtype=torch.int32, device=dev)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    for _ in range(max(args.warmup, 3)):
        st.layer_step(dw.batch, **kw)
    barrier()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    for i in range(args.steps):
        flush_w.fill_(i & 0xff)
        flush_r.max()
        ev[i][0].record()
        st.layer_step(dw.batch, **kw)
        ev[i][1].record()
    barrier()
    total_ms = float(sum(a.elapsed_time(b) for a, b in ev))
    clocks = sampler.stop() if rank == 0 else None
    total_ms, = max_over_ranks([total_ms], dist if world > 1 else None, dev)
    if rank == 0:
        ms = total_ms / args.steps
        line = {"metric": METRIC, "value": int(dw.batch.total_ctx) / (ms * 1e-3), "unit": UNIT, "n_gpus": world,
                "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms, "higher_is_better": True,
                "scaling": "strong", "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
                "config": dict(config_dict(wl.cfg, world, l2="flushed before every timed step"),
                               parallelism="kv-head shards x%d, score exchange: %s" % (world, exchange)),
                "clocks": clocks, "gpu_launches": KERNELS_PER_STEP * args.steps}
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


# ------------------------------------------------------------------------------------------------ config 3 (full stack)

C3_METRIC = "fused context tokens/s through the whole stack at r=0.3 (config 3: stage 1 + 36-layer stage 2)"


def c3_record(args, steps: int, light: bool) -> dict:
    """--workload c3 (or a reduced stack name): BASELINE configs[2].  One "step" = one qcf_stack_fuse call: stage 1
    (anchor probe up to the deepest critical layer, scoring, top-k) + stage 2 (every layer: layer-ahead PIC load and
    stitch on a second stream, a4 + a5 + a7 for the rows R).  `value` has the PIC pools resident in HBM; `e2e` reads
    them from pinned host memory inside the timed region (the paper's setting).  The working set (weights 13.9 GB)
    is far larger than L2, so no flush is needed between steps.  Compared with the library's own full prefill."""
    import torch
    from paper_2606_05875_b200 import binding, inputs, stack_device

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device — the qcf arm has no CPU fallback")
    torch.cuda.set_device(0)
    dev = "cuda:0"
    stack_name = args.workload if args.workload in inputs.STACKS else "c3"
    wl = inputs.make_stack_workload(stack_name, ratio=args.ratio if args.workload in inputs.STACKS else None, with_weights=False)
    sp = wl.spec
    ctx = binding.Context(sp.n_q_heads, sp.n_kv_heads, sp.head_dim, sp.rope_theta, 1, max(sp.n_ctx, 1024), sp.n_query)
    layers, embed = stack_device.device_weights(sp, sp.seed, dev)
    run = stack_device.StackRun(wl, ctx, layers, embed, dev)
    t0 = time.perf_counter()
    run.build_phase1(pinned=True)
    host_k, host_v, host_ak, host_av = run.k_pic, run.v_pic, run.k_anchor, run.v_anchor
    dev_pools = [[t.to(dev) for t in lst] for lst in (host_k, host_v, host_ak, host_av)]
    phase1_s = time.perf_counter() - t0
    sampler = ClockSampler(0)
    sampler.start()
    time.sleep(0.3)

    def timed(fn, n, warm):
        for _ in range(warm):
            fn()
        torch.cuda.synchronize()
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n)]
        for a, b in ev:
            a.record(); fn(); b.record()
        torch.cuda.synchronize()
        return np.array([a.elapsed_time(b) for a, b in ev])

    def use(pools):
        run.k_pic, run.v_pic, run.k_anchor, run.v_anchor = pools

    kv_row_b = sp.n_kv_heads * sp.head_dim * 2
    warm = 3 if light else max(args.warmup, 3)
    use(dev_pools)
    fuse_ms = timed(lambda: run.fuse(True), steps, warm)
    serial_ms = timed(lambda: run.fuse(False), max(3, min(steps, 10)), 1)
    use([host_k, host_v, host_ak, host_av])
    n_e2e = max(3, min(steps, 20))
    t1 = time.perf_counter()
    e2e_ms = timed(lambda: (run.fuse(True), run.hidden[-sp.n_query:].cpu(), run.sel.cpu()), n_e2e, 2)
    e2e_serial_ms = timed(lambda: (run.fuse(False), run.hidden[-sp.n_query:].cpu(), run.sel.cpu()), max(3, min(steps, 5)), 1)
    # selector views on the same kernels: stage 1 alone and the whole pipeline, pools in pinned host
    # memory (the paper's setting: selection-time data movement is what the compressed view saves)
    selectors = {}
    for view in ("qcfuse", "fullview", "final"):
        use([host_k, host_v, host_ak, host_av])
        run.use_selector(view)
        s1 = timed(lambda: run.fuse(True, stages=1), 3 if light else 5, 1 if light else 2)
        tot = timed(lambda: run.fuse(True), 3 if light else 5, 1)
        l_pr = max(run.crit) + 1
        selectors[view] = {"stage1_ms": float(s1.mean()), "pipeline_ms": float(tot.mean()), "probe_layers": l_pr,
                           "scored_layers": len(run.crit), "anchor_rows": run.anchor_rows,
                           "stage1_h2d_bytes": int(2 * kv_row_b * (run.anchor_rows * l_pr + sp.n_ctx * len(run.crit)))}
    # bandwidth-constrained loading (Fig. 13): the loader emulates a KV store of the given GB/s
    sweep = {}
    for view in ("qcfuse", "fullview"):
        run.use_selector(view)
        gs = (12.0, 50.0) if light else (3.0, 6.0, 12.0, 25.0, 50.0)       # the 3 GB/s points take a second per call
        sweep[view] = {str(g): float(timed(lambda: run.fuse(True, load_gbps=g), 1 if light else 2, 1).mean()) for g in gs}
    use([host_k, host_v, host_ak, host_av])
    run.use_selector("qcfuse")
    # time to first token: pipeline + final norm + LM head + argmax of the last query row
    gen = torch.Generator(device=dev); gen.manual_seed(sp.seed + 7)
    w_lm = (torch.randn((sp.vocab, sp.hidden), generator=gen, device=dev) * 0.02).to(torch.bfloat16)
    g_fin = torch.ones(sp.hidden, device=dev, dtype=torch.bfloat16)
    logits = torch.zeros(sp.vocab, device=dev)
    tok = torch.zeros(1, dtype=torch.int32, device=dev)
    hid_full = torch.zeros((run.t, sp.hidden), dtype=torch.bfloat16, device=dev)

    def ttft_fuse():
        run.fuse(True)
        run.stack.qcf_stack_first_token(run.hidden, run.n_rows - 1, g_fin, w_lm, logits, tok)
        return int(tok.cpu()[0])                     # the token is read back: the request's TTFT ends here

    ttft_ms = timed(ttft_fuse, max(3, min(steps, 10)), 1)
    kc = [torch.zeros_like(k) for k in run.k_fused]
    vc = [torch.zeros_like(k) for k in run.k_fused]
    full_ms = timed(lambda: run.full_prefill(kc, vc), max(3, min(steps, 10)), 2)

    def ttft_full():
        run.full_prefill(kc, vc, hid_full)
        run.stack.qcf_stack_first_token(hid_full, run.t - 1, g_fin, w_lm, logits, tok)
        return int(tok.cpu()[0])

    ttft_full_ms = timed(ttft_full, max(3, min(steps, 5)), 1)
    # generation over KV^Fuse: n_dec greedy tokens after the first, caches extended in place
    n_dec = 8
    dec_logits = torch.zeros((n_dec, sp.vocab), device=dev)
    dec_toks = torch.zeros(n_dec, dtype=torch.int32, device=dev)
    run.fuse(True)
    run.stack.qcf_stack_first_token(run.hidden, run.n_rows - 1, g_fin, w_lm, logits, tok)
    decode_ms = timed(lambda: run.stack.qcf_stack_decode(tok, run.t, n_dec, run.k_fused, run.v_fused, g_fin, w_lm, dec_logits, dec_toks),
                      3, 1)
    # the decode attention kernel alone: one new token over every layer's cache in turn (1.5 GB of K/V > L2, so each call
    # reads its 42 MB from HBM)
    q1 = torch.randn((sp.n_q_heads, sp.head_dim), device=dev).to(torch.bfloat16)
    o1 = torch.empty_like(q1)
    n_keys = run.t + n_dec
    dattn_ms = timed(lambda: [ctx.qcf_decode_attn(q1, run.k_fused[l], run.v_fused[l], n_keys, o1) for l in range(sp.n_layers)], 3, 1)
    dattn_us = float(dattn_ms.mean()) * 1e3 / sp.n_layers
    dattn_gbps = 2.0 * n_keys * kv_row_b / (dattn_us * 1e-6) / 1e9
    clocks = sampler.stop()

    fl = run.flops()
    peaks, peak_kind = load_peaks()
    peak = float(peaks.get("bf16_tflops_sustained", peaks["bf16_tflops"]))
    t_fuse = float(fuse_ms.mean())
    ach = (fl["gemm_fuse"] + fl["attn_fuse"]) / (t_fuse * 1e-3) / 1e12
    # dominant kernel: the gate/up projection (52 % of the GEMM flops), timed alone
    M, hid, ffn = run.n_rows, sp.hidden, sp.ffn
    a = torch.randn((M, hid), device=dev).to(torch.bfloat16)
    c = torch.empty((M, ffn), device=dev, dtype=torch.bfloat16)
    gu_ms = float(timed(lambda: ctx.qcf_linear(a, layers[0]["w_gate_up"], None, c, M, 2 * ffn, hid, binding.QCF_EPI_SWIGLU), 20, 3).mean())
    gu_tf = 2.0 * M * 2 * ffn * hid / (gu_ms * 1e-3) / 1e12
    kv_row = sp.n_kv_heads * sp.head_dim * 2
    l_probe = max(sp.crit_layers) + 1
    h2d = 2 * kv_row * (sp.n_ctx * sp.n_layers + run.anchor_rows * l_probe)
    line = {
        "metric": C3_METRIC, "value": sp.n_ctx / (t_fuse * 1e-3), "unit": UNIT, "n_gpus": 1, "steps": steps,
        "warmup": warm, "ms_per_step": t_fuse, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "bf16", "data": "synthetic",
        "config": {"workload": "%s: %d layers, hidden %d, FFN %d, Hq/Hkv=%d/%d, d=%d, %d chunks x %d tokens (N=%d) + %d-token "
                               "query, rho=%g, L*=%s (0-based), anchors %d rows, random-init bf16 weights" %
                               (sp.name, sp.n_layers, sp.hidden, sp.ffn, sp.n_q_heads, sp.n_kv_heads, sp.head_dim, sp.n_chunks,
                                sp.chunk_len, sp.n_ctx, sp.n_query, sp.ratio, list(sp.crit_layers), run.anchor_rows),
                   "baseline_config": "configs[2]" if sp.name == "c3" else sp.name, "ratio": sp.ratio, "global_batch": 1,
                   "parallelism": "replicas x1", "l2": "working set (weights) >> L2: no flush"},
        "clocks": clocks, "gpu_launches": int((sp.n_layers + l_probe) * 11 + 4) * steps,
        "roofline": {"kernel": "gemm_tc_kernel (a7 gate/up projection + SwiGLU, M=%d N=%d K=%d)" % (M, 2 * ffn, hid),
                     "bound": "tensor", "achieved": gu_tf, "peak": peak, "unit": "TFLOP/s", "frac": gu_tf / peak,
                     "traffic": None, "peak_source": "%s bf16_tflops_sustained (kernel inside a long step)" % peak_kind,
                     "ms_per_launch": gu_ms},
        "pipeline": {"fuse_ms_min_med_max": [float(fuse_ms.min()), float(np.median(fuse_ms)), float(fuse_ms.max())],
                     "fuse_serial_loader_ms": float(serial_ms.mean()), "full_prefill_ms": float(full_ms.mean()),
                     "speedup_over_full_prefill": float(full_ms.mean()) / t_fuse,
                     "whole_pipeline_TFLOPps": ach, "whole_pipeline_frac_tensor_peak": ach / peak,
                     "full_prefill_TFLOPps": (fl["gemm_full"] + fl["attn_full"]) / (float(full_ms.mean()) * 1e-3) / 1e12,
                     "ttft_ms_pinned_host": float(ttft_ms.mean()), "ttft_full_prefill_ms": float(ttft_full_ms.mean()),
                     "decode_ms_per_token": float(decode_ms.mean()) / n_dec,
                     "decode_attn_us_per_layer": dattn_us, "decode_attn_GBps": dattn_gbps,
                     "decode_attn_frac_hbm": dattn_gbps / float(load_peaks()[0]["hbm_gbs"]),
                     "decode_weight_stream_GBps": (13.9e9 * sp.n_layers / 36.0 + 2.0 * sp.vocab * sp.hidden) / (float(decode_ms.mean()) / n_dec * 1e-3) / 1e9,
                     "phase1_build_s": phase1_s, "selectors_pinned_host": selectors,
                     "pipeline_ms_vs_load_gbps": sweep},
        "e2e": {"value": sp.n_ctx / (float(e2e_ms.mean()) * 1e-3), "unit": UNIT, "h2d_bytes_per_step": int(h2d),
                "d2h_bytes_per_step": int(sp.n_query * sp.hidden * 2 + sp.n_ctx * 4), "ms_per_step": float(e2e_ms.mean()),
                "ms_per_step_serial_loader": float(e2e_serial_ms.mean()),
                "steps": n_e2e, "api": "qcf_stack_fuse with PIC / anchor pools in pinned host memory (layer-ahead H2D on "
                                       "the loader stream), query-row hidden states and P read back"},
    }
    if not args.no_cpu_baseline and not light:
        line["cpu_baseline"] = c3_cpu_baseline(run, layers, sp)
    del run, layers, embed, dev_pools, host_k, host_v, host_ak, host_av, kc, vc, w_lm
    torch.cuda.empty_cache()
    return line


def c3_cpu_baseline(run, layers, sp) -> dict:
    """The stack oracle as it stands on the host cores, on a bounded sample: ONE layer of stage 2 (layer 0: stitch the
    PIC entries, then fuse_layer) for every 16th row of R; scaled to the whole pipeline by 16 x (n_layers + probe
    layers x Lq / |R|)."""
    import torch
    from oracle import qcf_oracle as O
    from oracle import qcf_stack_oracle as S

    def f64(t):
        return O.widen_bf16(t.detach().cpu().contiguous().view(torch.int16).numpy().view(np.uint16))

    hq, hkv, d = sp.n_q_heads, sp.n_kv_heads, sp.head_dim
    lw = layers[0]
    wqkv = f64(lw["w_qkv"])
    gu = f64(lw["w_gate_up"])
    w = S.LayerWeights(wq=wqkv[: hq * d], wk=wqkv[hq * d: (hq + hkv) * d], wv=wqkv[(hq + hkv) * d:], wo=f64(lw["w_o"]),
                       wg=gu[0::2], wu=gu[1::2], wd=f64(lw["w_down"]), g_attn=f64(lw["g_attn"]), g_ffn=f64(lw["g_ffn"]),
                       g_q=f64(lw["g_q"]), g_k=f64(lw["g_k"]))
    cfg = S.StackConfig(1, sp.hidden, sp.ffn, hq, hkv, d, sp.rope_theta, sp.rms_eps)
    n, lq = sp.n_ctx, sp.n_query
    sel = run.sel[: run.k_sel].cpu().numpy().astype(np.int64)
    stride = 16
    sel_s = sel[::stride]
    rows = np.concatenate([sel_s, np.arange(n, n + lq)[::stride]])
    n_q = len(rows) - len(sel_s)
    k_pic = [f64(run.k_pic[0]).reshape(sp.n_chunks, sp.chunk_len, hkv, d)[i] for i in range(sp.n_chunks)]
    v_pic = [f64(run.v_pic[0]).reshape(sp.n_chunks, sp.chunk_len, hkv, d)[i] for i in range(sp.n_chunks)]
    x = np.random.default_rng(0).standard_normal((len(rows), sp.hidden))
    t0 = time.perf_counter()
    k_ctx, v_ctx = O.reposition(k_pic, v_pic, sp.rope_theta)
    # the sampled query rows stand at their own positions; fuse_layer appends them after N, so give it a cache cut to N + n_q
    S.fuse_layer(x, np.concatenate([sel_s, np.arange(n, n + n_q)]), len(sel_s), k_ctx, v_ctx, w, cfg)
    sec = time.perf_counter() - t0
    l_probe = max(sp.crit_layers) + 1
    total = sec * stride * (sp.n_layers + l_probe * lq / max(run.n_rows, 1))
    return {"value": n / total, "unit": UNIT, "cores": n_cores(), "kind": "oracle",
            "sample": "oracle.reposition + qcf_stack_oracle.fuse_layer (fp64 numpy) of layer 0 on every %d-th row of R (%d rows), "
                      "%.1f s; scaled x%d rows x (%d stage-2 layers + %d probe layers of %d rows)" %
                      (stride, len(rows), sec, stride, sp.n_layers, l_probe, lq)}



def main():
    args = parse_args()
    from paper_2606_05875_b200.inputs import STACKS
    if args.workload in STACKS:
        if args.impl == "reference":
            raise SystemExit("bench.py: --impl reference is defined for the layer-step workloads (c1, c2, c4, c5)")
        if int(os.environ.get("RANK", "0")) != 0:
            return                                            # one request: replicas only
        print(json.dumps(c3_record(args, steps=min(args.steps, 20), light=False)), flush=True)
    elif args.impl == "reference":
        run_reference(args)
    elif args.shard == "heads":
        run_head_sharded(args)
    else:
        run_qcf(args)


if __name__ == "__main__":
    main()
