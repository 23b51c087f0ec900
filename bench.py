#!/usr/bin/env python
"""bench.py -- per-denoising-step sparse attention of Prefilling-dLLM on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload NAME]

A "step" is one pass of the whole hot path (chunk-score reduction -> top-K -> index-driven
gather + Split-S partial attention -> LSE combine) over one batch of seeded synthetic input, i.e. one
`pdllm_step` call through the C ABI.  Default workload: BASELINE.json configs[3] ("32K long-context
sparse", the configuration the metric is quoted on; it fits one GPU).

Prints ONE JSON line (rank 0): `value` = device-timed us per step with inputs resident in HBM;
`e2e` = the same through `pdllm_step_host` with pinned HOST per-step tensors (H2D + D2H inside the timed
region); `roofline` for the dominant kernel (per-stage CUDA events recorded inside the timed region by
`pdllm_step_profiled`); `cpu_baseline` = the fp64 oracle timed on this box's host cores on a bounded
sample.  `--impl reference` times the oracle alone (there is no reference code: /root/reference holds a
paper only).

Multi-GPU: replicas only -- the path is fixed to one GPU by BASELINE.json; under
torchrun every rank runs an independent replica of the step, time = max over ranks.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

from paper_2606_10537_b200 import workloads as W  # noqa: E402

METRIC = "us_per_denoising_step_attention"
UNIT = "us"
FALLBACK_PEAKS = {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0}
SPEC_PEAKS = {"hbm_gbs": 8000.0, "bf16_tflops": 2250.0}      # the peaks BASELINE.json's north_star names
# dram__bytes_read.sum + dram__bytes_write.sum per launch, copied from the committed `ncu --set full` capture named in
# NCU_TRAFFIC_SOURCE (NOT measured by the run that prints it: ncu cannot run inside a timed bench); keyed by
# (workload, kernel); None where no capture exists for that pair.
NCU_TRAFFIC_SOURCE = "profiles/r2_ncu_full.md (ncu --set full capture of these kernels; not measured in this run)"
NCU_TRAFFIC_BYTES = {
    ("sparse32k", "score_kernel"): 1081.614e6 + 3.672064e6,
    ("sparse32k", "attn_kernel"): 154.260e6 + 6.714112e6,
}


def load_peaks():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        try:
            d = json.loads(p.read_text())
            return {k: float(d[k]) for k in FALLBACK_PEAKS if k in d} | {"source": "measured"}
        except Exception:
            pass
    return dict(FALLBACK_PEAKS, source="fallback")


# --------------------------------------------------------------------------- clocks during the timed region
class ClockSampler:
    """Samples SM clock and throttle reasons with NVML every few ms while the timed region runs."""
    BAD = {"hw_slowdown": 0x8, "sw_thermal_slowdown": 0x20, "hw_thermal_slowdown": 0x40}
    NOTE = {"sw_power_cap": 0x4, "hw_power_brake": 0x80}

    def __init__(self, index: int, period_s: float = 0.004):
        self.index, self.period = index, period_s
        self.samples, self.reasons = [], 0
        self._stop = threading.Event()
        self._thr = None
        self.max_mhz = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def _reasons(self):
        for fn in ("nvmlDeviceGetCurrentClocksEventReasons", "nvmlDeviceGetCurrentClocksThrottleReasons"):
            f = getattr(self.nv, fn, None)
            if f is not None:
                try:
                    return int(f(self.h))
                except Exception:
                    continue
        return 0

    def _run(self):
        while not self._stop.is_set():
            try:
                self.samples.append(self.nv.nvmlDeviceGetClockInfo(self.h, self.nv.NVML_CLOCK_SM))
                self.reasons |= self._reasons()
            except Exception:
                pass
            self._stop.wait(self.period)

    def __enter__(self):
        if self.nv is not None:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._thr is not None:
            self._thr.join()

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["unavailable"]}
        names = [n for n, bit in {**self.BAD, **self.NOTE}.items() if self.reasons & bit]
        return {"sm_mhz": statistics.median(self.samples), "sm_max_mhz": self.max_mhz, "reasons": names,
                "samples": len(self.samples)}


# --------------------------------------------------------------------------- the oracle leg (CPU baseline / reference arm)
def oracle_sample(w: W.Workload, inp: dict, threads: int):
    """A bounded sample of the workload for the oracle: the first n KV groups of batch element 0 (with their
    G query heads each), one group per host thread.  Returns (slices, scale-up factor to the whole step)."""
    n = max(1, min(w.H_kv, threads // max(1, min(w.G, threads))))
    sl = dict(Q_dec=np.ascontiguousarray(inp["Q_dec"][:1, : n * w.G]), Kcache=np.ascontiguousarray(inp["Kcache"][:1, :n]),
              Vcache=np.ascontiguousarray(inp["Vcache"][:1, :n]), K_dec=np.ascontiguousarray(inp["K_dec"][:1, :n]),
              V_dec=np.ascontiguousarray(inp["V_dec"][:1, :n]),
              keep=None if inp["keep"] is None else np.ascontiguousarray(inp["keep"][:1, :n]))
    return sl, n, (w.B * w.H_kv) / n


def time_oracle_once(w, sl):
    from oracle import oracle
    t0 = time.perf_counter()
    oracle.step(sl["Q_dec"], sl["Kcache"], sl["Vcache"], sl["keep"], sl["K_dec"], sl["V_dec"], w.K, w.L_q)
    return time.perf_counter() - t0


def time_oracle_pieces(w, sl, n_chunks, ids):
    """The oracle's step on the sample with the scoring restricted to the first n_chunks chunks (each chunk's
    score is independent of the others): returns (seconds scoring n_chunks chunks, seconds for the rest =
    top-K + gather indices + concatenation + attention with the selected ids)."""
    from oracle import oracle
    t0 = time.perf_counter()
    sc = oracle.scores(sl["Q_dec"], np.ascontiguousarray(sl["Kcache"][:, :, :n_chunks]), w.L_q)
    t1 = time.perf_counter()
    oracle.topk(sc, min(w.K, n_chunks))
    oracle.gather_idx(ids, sl["keep"], w.N, w.C)
    oracle.attn(sl["Q_dec"], sl["Kcache"], sl["Vcache"], ids, sl["keep"], sl["K_dec"], sl["V_dec"])
    t2 = time.perf_counter()
    return t1 - t0, t2 - t1


def run_reference(args, w):
    """--impl reference: the oracle, as it stands, on the host cores (rank 0 only).  Each step times a bounded
    sample (some (batch, KV-head) groups; the scoring over some of the N chunks) and scales it to the whole
    step; the sample is sized so that steps + warmup end within a few minutes."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    from oracle import oracle
    cores = oracle.num_threads()
    inp = W.make_inputs(W.small_variant(w, B=1))      # the sample only touches batch element 0
    sl, n, factor = oracle_sample(w, inp, cores)
    ids = np.ascontiguousarray(inp["planted"][:1, :n])
    t_s1, t_rest = time_oracle_pieces(w, sl, 1, ids)  # probe: one chunk
    budget = max(0.05, 150.0 / max(1, args.steps + args.warmup))
    n_chunks = int(max(1, min(w.N, (budget - t_rest) / max(t_s1, 1e-6))))
    for _ in range(args.warmup):
        time_oracle_pieces(w, sl, n_chunks, ids)
    tot = 0.0
    for _ in range(args.steps):
        ts, tr = time_oracle_pieces(w, sl, n_chunks, ids)
        tot += ts * (w.N / n_chunks) + tr
    us = 1e6 * factor * tot / max(1, args.steps)
    sample = (f"per step: {n} of {w.B * w.H_kv} (batch, KV-head) groups (b=0, groups 0..{n - 1}, {w.G} query head(s) each); "
              f"scoring over {n_chunks} of {w.N} chunks scaled x{w.N / n_chunks:g}, attention in full; "
              f"whole sample scaled x{factor:g} to the step")
    line = {"impl": "reference", "metric": METRIC, "value": us, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": us / 1e3, "higher_is_better": False, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(w, None),
            "cpu_baseline": {"value": us, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": us, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


L2_BYTES = 126e6


def needs_flush(w) -> bool:
    """Workloads whose K+V cache is not several times larger than L2 get an explicit L2 flush between iterations."""
    return 2 * w.B * w.H_kv * w.N * w.Cp * w.d * 2 < 4 * L2_BYTES


def workload_config(w, n_splits):
    l2 = ("explicit flush: a 256 MB buffer is rewritten between timed iterations (K+V cache is "
          f"{2 * w.B * w.H_kv * w.N * w.Cp * w.d * 2 / 1e6:.0f} MB, not >> L2); per-iteration CUDA events"
          if needs_flush(w) else
          "inputs larger than L2: the step streams the whole K cache "
          f"({w.score_bytes() / 1e6:.0f} MB) every iteration; no explicit flush")
    label = (f"BASELINE.json configs[{list(W.CONFIGS).index(w.name)}] '{w.name}'" if w.name in W.CONFIGS
             else f"extra workload '{w.name}' (paper Fig. 5(b) decode shape; not a BASELINE.json config)")
    return {"workload": label, "B": w.B, "H": w.H,
            "H_kv": w.H_kv, "d": w.d, "N": w.N, "C": w.C, "K": w.K, "keep": w.keep, "Bk": w.Bk, "L_q": w.L_q,
            "L_d": w.L_d, "prefix_tokens": w.N * w.C, "n_splits": n_splits,
            "call": "pdllm_step (score_chunks -> select_topk -> sparse_attn -> lse_combine)",
            "l2": l2}


# --------------------------------------------------------------------------- multi-rank plumbing (replicas only)
def max_over_ranks(value: float, world: int, device="cuda") -> float:
    """MAX all-reduce of a per-rank time; identity for one rank."""
    if world <= 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([value], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def replica_us_per_step(total_ms: float, steps: int, world: int) -> float:
    """`world` independent replicas each ran `steps` steps in total_ms (max over ranks): whole-job us per step."""
    return 1e3 * total_ms / (steps * world)


# --------------------------------------------------------------------------- our arm
def run_ours(args, w):
    import torch
    import torch.distributed as dist
    from paper_2606_10537_b200 import binding as B

    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the pdllm hot path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    B.lib()
    sms = B.num_sms()
    shape = B.Shape.of(w)
    inp = W.make_inputs(w)
    bf = lambda bits: torch.from_numpy(np.ascontiguousarray(bits).view(np.int16)).cuda().view(torch.bfloat16)
    dQ, dKc, dVc, dKd, dVd = (bf(inp[k]) for k in ("Q_dec", "Kcache", "Vcache", "K_dec", "V_dec"))
    dkeep = None if inp["keep"] is None else torch.from_numpy(inp["keep"]).cuda()
    S = args.n_splits if args.n_splits > 0 else B.auto_splits(shape, sms)
    ws = B.alloc_workspace(shape, args.n_splits)
    out = dict(scores=torch.empty((w.B, w.H_kv, w.N), dtype=torch.float32, device="cuda"),
               chunk_ids=torch.empty((w.B, w.H_kv, w.K), dtype=torch.int32, device="cuda"),
               O=torch.empty((w.B, w.H, w.L, w.d), dtype=torch.bfloat16, device="cuda"),
               LSE=torch.empty((w.B, w.H, w.L), dtype=torch.float32, device="cuda"))

    def step(events=None):
        B.step(shape, dQ, dKc, dVc, dkeep, dKd, dVd, n_splits=args.n_splits, workspace=ws, events=events, **out)

    K, Wm = args.steps, args.warmup
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(5)] for _ in range(K)]
    for row in evs:                       # torch creates the cudaEvent_t on first record
        for e in row:
            e.record()
    for _ in range(Wm):
        step()
    torch.cuda.synchronize()
    ok = bool((out["chunk_ids"].cpu().numpy() == inp["planted"]).all())     # sanity: the planted chunks are found

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    t_begin, t_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    flush = needs_flush(w)
    flush_buf = torch.empty((256 << 20,), dtype=torch.uint8, device="cuda") if flush else None

    per_call = []                         # flush mode: the last timed_loop's per-call times (median / min beside the mean)

    def timed_loop(fn):
        """us per call of fn over K calls: one event pair around the loop, or (flush mode) one pair per call with the
        L2 flush between calls outside the timed intervals."""
        if not flush:
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            for _ in range(K):
                fn()
            b.record()
            barrier()
            return 1e3 * a.elapsed_time(b) / K
        pairs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
        for a, b in pairs:
            flush_buf.zero_()
            a.record()
            fn()
            b.record()
        barrier()
        per_call.clear()
        per_call.extend(1e3 * a.elapsed_time(b) for a, b in pairs)
        return sum(per_call) / K

    # ---- the timed regions, clocks sampled meanwhile: K steps through pdllm_step_profiled (per-stage CUDA events recorded
    # on the launching stream inside the loop: the stage split and the kernels' rooflines; the events cost a few us per
    # step and keep the programmatic dependent launches from overlapping, so this loop is not `value`), then K plain
    # pdllm_step calls (what a user runs) = `value`
    barrier()
    with ClockSampler(local) as clk:
        t_begin.record()
        for k in range(K):
            if flush:
                flush_buf.zero_()
            step(evs[k])
        t_end.record()
        barrier()
        us_plain_rank = timed_loop(step)
    plain_calls = sorted(per_call)        # empty without the flush: one event pair spans the whole loop there
    total_ms = max_over_ranks(us_plain_rank * K / 1e3, world)
    us_per_step = replica_us_per_step(total_ms, K, world)     # replicas: world independent steps ran per iteration
    if flush:
        us_profiled = 1e3 * sum(evs[k][0].elapsed_time(evs[k][4]) for k in range(K)) / K
    else:
        us_profiled = 1e3 * t_begin.elapsed_time(t_end) / K

    staged_calls = sorted(1e3 * evs[k][0].elapsed_time(evs[k][4]) for k in range(K))

    def stage(i, j):
        return 1e3 * sum(evs[k][i].elapsed_time(evs[k][j]) for k in range(K)) / K
    t_score, t_topk, t_attn, t_comb = stage(0, 1), stage(1, 2), stage(2, 3), stage(3, 4)
    if S == 1:
        t_comb = 0.0                      # no combine kernel ran: the interval is the gap between two event records

    # ---- the same step as a CUDA-graph replay: one graph launch per step, no per-kernel launch gaps
    us_graph = None
    try:
        g = torch.cuda.CUDAGraph()
        cs = torch.cuda.Stream()
        cs.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(cs):
            step()
            cs.synchronize()
            with torch.cuda.graph(g, stream=cs):
                step()
        torch.cuda.current_stream().wait_stream(cs)
        for _ in range(3):
            g.replay()
        barrier()
        us_graph = timed_loop(g.replay)
    except Exception as e:                # reported, never fatal: the plain loop is the headline
        us_graph = f"unavailable: {type(e).__name__}: {e}"[:200]

    # ---- sustained regime: the same plain loop over >= 200 steps, where the 1 kW power cap has pulled the SM clock
    # down (the driver's 20-step run ends before it bites); reported beside `value`, with its own clock record
    sustained = None
    if not flush:
        K_save = K
        K = max(200, K_save)
        barrier()
        with ClockSampler(local) as clk_s:
            for _ in range(2):            # the first pass heats, the second is kept
                us_sus = timed_loop(step)
        K = K_save
        sustained = {"steps": max(200, K_save), "us_per_step": us_sus, "clocks": clk_s.summary()}

    # ---- hot L2 (reported separately): workloads whose cache fits L2, stepped back to back WITHOUT the
    # flush, so every call after the first finds K / V in L2.  Never `value`.
    us_hot = us_attn_hot = None
    if flush:
        def hot_loop(fn):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            fn()
            a.record()
            for _ in range(K):
                fn()
            b.record()
            barrier()
            return 1e3 * a.elapsed_time(b) / K
        barrier()
        us_hot = hot_loop(step)

    # the paper's static-selection mode: per step only pdllm_sparse_attn
    ids = out["chunk_ids"].clone()
    barrier()
    us_attn_only = timed_loop(lambda: B.sparse_attn(shape, dQ, dKc, dVc, ids, dkeep, dKd, dVd, n_splits=args.n_splits,
                                                    O=out["O"], LSE=out["LSE"], workspace=ws))
    if flush:
        us_attn_hot = hot_loop(lambda: B.sparse_attn(shape, dQ, dKc, dVc, ids, dkeep, dKd, dVd, n_splits=args.n_splits,
                                                     O=out["O"], LSE=out["LSE"], workspace=ws))

    # ---- e2e: HOST per-step tensors through pdllm_step_host, copies inside the timed region
    pin = lambda bits: torch.from_numpy(np.ascontiguousarray(bits).view(np.int16)).view(torch.bfloat16).pin_memory()
    hQ, hK, hV = pin(inp["Q_dec"]), pin(inp["K_dec"]), pin(inp["V_dec"])
    hO = torch.empty((w.B, w.H, w.L, w.d), dtype=torch.bfloat16).pin_memory()
    hL = torch.empty((w.B, w.H, w.L), dtype=torch.float32).pin_memory()
    hI = torch.empty((w.B, w.H_kv, w.K), dtype=torch.int32).pin_memory()
    scratch = torch.empty((B.step_host_scratch_bytes(shape, args.n_splits, sms),), dtype=torch.uint8, device="cuda")
    stream = torch.cuda.current_stream()
    side = B.SideStream()                 # caller-owned: K_dec / V_dec are copied under the scoring kernel

    def host_step():
        B.step_host(shape, hQ, hK, hV, dKc, dVc, dkeep, args.n_splits, hO, hL, hI, scratch, side=side)
        stream.synchronize()              # the caller reads O / LSE / ids after every step

    for _ in range(Wm):
        host_step()
    barrier()
    t0 = time.perf_counter()
    for _ in range(K):
        host_step()
    barrier()
    e2e_s = max_over_ranks(time.perf_counter() - t0, world)
    e2e_us = replica_us_per_step(1e3 * e2e_s, K, world)
    h2d = hQ.numel() * 2 + hK.numel() * 2 + hV.numel() * 2
    d2h = hO.numel() * 2 + hL.numel() * 4 + hI.numel() * 4
    e2e_ok = bool((hI.numpy() == inp["planted"]).all())

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel + the attention kernel (algorithmic work: DESIGN.md "Measurement").
    # Fractions are given against the MEASURED peaks of this pool (MEASURED_PEAKS.json) and, beside them, against
    # the SPEC peaks BASELINE.json's north_star names (8 TB/s, 2.25 PFLOP/s dense bf16).
    peaks = load_peaks()
    score_gbs = w.score_bytes() / (t_score * 1e-6) / 1e9
    attn_t = t_attn + t_comb
    attn_tf = w.attn_flops() / (attn_t * 1e-6) / 1e12
    attn_gbs = w.attn_bytes() / (attn_t * 1e-6) / 1e9
    roof_score = {"kernel": "score_kernel (a1)", "bound": "hbm", "achieved": score_gbs, "peak": peaks["hbm_gbs"],
                  "unit": "GB/s", "frac": score_gbs / peaks["hbm_gbs"], "peak_source": peaks["source"],
                  "frac_of_spec_peak": score_gbs / SPEC_PEAKS["hbm_gbs"],
                  "traffic": NCU_TRAFFIC_BYTES.get((w.name, "score_kernel")), "traffic_source": NCU_TRAFFIC_SOURCE,
                  "us": t_score, "algorithmic_bytes": w.score_bytes()}
    t_tensor = w.attn_flops() / (peaks["bf16_tflops_sustained"] * 1e12)
    t_hbm = w.attn_bytes() / (peaks["hbm_gbs"] * 1e9)
    t_spec = max(w.attn_flops() / (SPEC_PEAKS["bf16_tflops"] * 1e12), w.attn_bytes() / (SPEC_PEAKS["hbm_gbs"] * 1e9))
    attn_bound = "tensor" if t_tensor >= t_hbm else "hbm"
    roof_attn = {"kernel": "attn_kernel (a3+a4)" + (" + combine_kernel (a5)" if S > 1 else ""), "bound": attn_bound,
                 "achieved": attn_tf if attn_bound == "tensor" else attn_gbs,
                 "peak": peaks["bf16_tflops_sustained"] if attn_bound == "tensor" else peaks["hbm_gbs"],
                 "unit": "TFLOP/s" if attn_bound == "tensor" else "GB/s",
                 "frac": max(t_tensor, t_hbm) / (attn_t * 1e-6), "peak_source": peaks["source"] + " (sustained)",
                 "frac_of_spec_peak": t_spec / (attn_t * 1e-6),
                 "traffic": NCU_TRAFFIC_BYTES.get((w.name, "attn_kernel")), "traffic_source": NCU_TRAFFIC_SOURCE,
                 "us": attn_t, "tflops": attn_tf, "gbs": attn_gbs, "roofline_us": 1e6 * max(t_tensor, t_hbm)}
    dominant = roof_score if t_score >= attn_t else roof_attn
    step_flops = w.score_flops() + w.attn_flops()
    step_bytes = w.score_bytes() + w.attn_bytes() + w.topk_bytes()
    roof_step_us = 1e6 * max(step_flops / (peaks["bf16_tflops_sustained"] * 1e12), step_bytes / (peaks["hbm_gbs"] * 1e9))
    roof_step_spec_us = 1e6 * max(step_flops / (SPEC_PEAKS["bf16_tflops"] * 1e12), step_bytes / (SPEC_PEAKS["hbm_gbs"] * 1e9))
    if sustained is not None:
        sustained["step_roofline_frac"] = roof_step_us / sustained["us_per_step"]

    # ---- the oracle on this box's host cores (bounded sample)
    from oracle import oracle
    cores = oracle.num_threads()
    sl, n, factor = oracle_sample(w, inp, cores)
    reps = 3
    t_or = min(time_oracle_once(w, sl) for _ in range(reps))
    cpu = {"value": 1e6 * t_or * factor, "unit": UNIT, "cores": cores, "kind": "oracle",
           "sample": f"{n} of {w.B * w.H_kv} (batch, KV-head) groups (b=0, groups 0..{n - 1}), best of {reps}, "
                     f"time scaled x{factor:g} to the whole step"}

    clocks = clk.summary()
    line = {"metric": METRIC, "value": us_per_step, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
            "ms_per_step": us_per_step / 1e3, "higher_is_better": False,
            "scaling": "weak", "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
            "config": workload_config(w, S),
            "tflops": step_flops / (us_per_step * world * 1e-6) / 1e12,
            "gbs": step_bytes / (us_per_step * world * 1e-6) / 1e9,
            "step_roofline": {"us": roof_step_us, "frac": roof_step_us / (us_per_step * world),
                              "peak_source": peaks["source"], "frac_of_spec_peak": roof_step_spec_us / (us_per_step * world)},
            "value_is": "K plain pdllm_step calls, one CUDA-event pair around the loop (no per-stage events); stages_us and "
                        "the rooflines come from K more steps through pdllm_step_profiled, run just before",
            "stages_us": {"score_chunks": t_score, "select_topk": t_topk, "sparse_attn_partial": t_attn,
                          "lse_combine": t_comb, "step_with_stage_events": us_profiled,
                          "step_with_stage_events_median_min": [statistics.median(staged_calls), staged_calls[0]],
                          "step_median_min": [statistics.median(plain_calls), plain_calls[0]] if plain_calls else None,
                          "step_cuda_graph_replay": us_graph,
                          "step_hot_l2_back_to_back": us_hot, "sparse_attn_only_hot_l2": us_attn_hot,
                          "sparse_attn_only_static_selection": us_attn_only},
            "sustained": sustained,
            "roofline": dominant, "roofline_attn": roof_attn, "roofline_score": roof_score,
            "e2e": {"value": e2e_us, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "call": "pdllm_step_host (pinned host Q_dec/K_dec/V_dec in; O, LSE, chunk ids out; KV cache resident)",
                    "result_ok": e2e_ok},
            "gpu_launches": K * ((2 if w.N <= B.FOLD_MAX_N else 3) + (1 if S > 1 else 0)),   # a2 runs inside a4 up to FOLD_MAX_N chunks
            "cpu_baseline": cpu, "clocks": clocks, "planted_chunks_recovered": ok}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


# --------------------------------------------------------------------------- the rows after the hot path
def _common_setup(args):
    import torch
    from paper_2606_10537_b200 import binding as B
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the pdllm hot path has no CPU fallback")
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    B.lib()
    return torch, B


def _timed(torch, fn, K, flush_buf=None):
    """us per call over K calls on the current stream (per-call events with an L2 flush between calls when asked)."""
    if flush_buf is None:
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(K):
            fn()
        b.record()
        torch.cuda.synchronize()
        return 1e3 * a.elapsed_time(b) / K
    pairs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
    for a, b in pairs:
        flush_buf.zero_()
        a.record()
        fn()
        b.record()
    torch.cuda.synchronize()
    return 1e3 * sum(a.elapsed_time(b) for a, b in pairs) / K


def _timed_graph(torch, fn, K):
    """us per call of fn replayed as a CUDA graph (for stages of a few microseconds, where the host's launch rate and
    not the device would otherwise be what is timed)."""
    g = torch.cuda.CUDAGraph()
    cs = torch.cuda.Stream()
    cs.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(cs):
        fn()
        cs.synchronize()
        with torch.cuda.graph(g, stream=cs):
            fn()
    torch.cuda.current_stream().wait_stream(cs)
    for _ in range(3):
        g.replay()
    return _timed(torch, g.replay, K)


def _attn_roofline(peaks, flops, nbytes, us, kernel):
    t_tensor, t_hbm = flops / (peaks["bf16_tflops_sustained"] * 1e12), nbytes / (peaks["hbm_gbs"] * 1e9)
    t_spec = max(flops / (SPEC_PEAKS["bf16_tflops"] * 1e12), nbytes / (SPEC_PEAKS["hbm_gbs"] * 1e9))
    bound = "tensor" if t_tensor >= t_hbm else "hbm"
    tf, gbs = flops / (us * 1e-6) / 1e12, nbytes / (us * 1e-6) / 1e9
    return {"kernel": kernel, "bound": bound, "achieved": tf if bound == "tensor" else gbs,
            "peak": peaks["bf16_tflops_sustained"] if bound == "tensor" else peaks["hbm_gbs"],
            "unit": "TFLOP/s" if bound == "tensor" else "GB/s", "frac": max(t_tensor, t_hbm) / (us * 1e-6),
            "frac_of_spec_peak": t_spec / (us * 1e-6), "peak_source": peaks["source"], "traffic": None, "us": us,
            "tflops": tf, "gbs": gbs, "roofline_us": 1e6 * max(t_tensor, t_hbm)}


def _line(args, w, value, config, roofline, cpu, e2e, launches, clocks, extra):
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": 1, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": value / 1e3, "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "bf16",
            "data": "synthetic", "config": config, "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e,
            "gpu_launches": launches, "clocks": clocks}
    line.update(extra)
    print(json.dumps(line))


def run_static(args, w):
    """--mode static: the paper's static-selection mode -- per step only the attention, through the gather
    path (pdllm_sparse_attn) and through the compact cache (pdllm_compact_kv once, then pdllm_static_attn: TMA tiles);
    beside it the per-step re-selection cost with the pooled-key scorer (pdllm_score_chunks_pooled + pdllm_select_topk)
    against the full chunk-score kernel."""
    torch, B = _common_setup(args)
    shape = B.Shape.of(w)
    inp = W.make_inputs(w)
    bf = lambda bits: torch.from_numpy(np.ascontiguousarray(bits).view(np.int16)).cuda().view(torch.bfloat16)
    dQ, dQs, dKc, dVc, dKd, dVd = (bf(inp[k]) for k in ("Q_dec", "Q_score", "Kcache", "Vcache", "K_dec", "V_dec"))
    dkeep = None if inp["keep"] is None else torch.from_numpy(inp["keep"]).cuda()
    K, Wm = args.steps, args.warmup
    flush = torch.empty((256 << 20,), dtype=torch.uint8, device="cuda") if needs_flush(w) else None
    sc = B.score_chunks(shape, dQs, dKc)
    ids = B.select_topk(shape, sc)
    kbar = B.pool_keys(shape, dKc)
    sc_p = B.score_chunks_pooled(shape, dQs, kbar)
    ids_p = B.select_topk(shape, sc_p)
    torch.cuda.synchronize()
    recall = float(np.mean([len(set(a) & set(b)) / w.K for a, b in zip(ids_p.cpu().numpy().reshape(-1, w.K), inp["planted"].reshape(-1, w.K))]))
    ids_ok = bool((ids.cpu().numpy() == inp["planted"]).all())
    Kc, Vc = B.compact_kv(shape, dKc, dVc, ids, dkeep)
    ds = B.DenseShape.static_of(shape)
    S = args.n_splits if args.n_splits > 0 else B.auto_splits(shape, B.num_sms())
    Sd = args.n_splits if args.n_splits > 0 else B.dense_auto_splits(ds, B.num_sms())
    ws, wsd = B.alloc_workspace(shape, args.n_splits), B.alloc_dense_workspace(ds, args.n_splits)
    O = torch.empty((w.B, w.H, w.L, w.d), dtype=torch.bfloat16, device="cuda")
    LSE = torch.empty((w.B, w.H, w.L), dtype=torch.float32, device="cuda")
    gather = lambda: B.sparse_attn(shape, dQ, dKc, dVc, ids, dkeep, dKd, dVd, n_splits=args.n_splits, O=O, LSE=LSE, workspace=ws)
    static = lambda: B.static_attn(ds, dQ, Kc, Vc, dKd, dVd, n_splits=args.n_splits, O=O, LSE=LSE, workspace=wsd)
    pooled = lambda: B.select_topk(shape, B.score_chunks_pooled(shape, dQs, kbar, scores=sc_p), chunk_ids=ids_p)
    full = lambda: B.select_topk(shape, B.score_chunks(shape, dQs, dKc, scores=sc), chunk_ids=ids)
    for _ in range(Wm):
        gather(); static(); pooled()
    torch.cuda.synchronize()
    with ClockSampler(0) as clk:
        us_static = _timed(torch, static, K, flush)
        us_gather = _timed(torch, gather, K, flush)
    us_pooled = _timed_graph(torch, pooled, K)
    us_full = _timed_graph(torch, full, max(3, K // 10))
    us_compact = _timed(torch, lambda: B.compact_kv(shape, dKc, dVc, ids, dkeep, Kc, Vc), max(3, K // 10))
    us_pool = _timed(torch, lambda: B.pool_keys(shape, dKc, kbar), max(3, K // 10))
    # e2e: the per-step tensors come from pinned host memory and O goes back, around the C-ABI call
    pin = lambda bits: torch.from_numpy(np.ascontiguousarray(bits).view(np.int16)).view(torch.bfloat16).pin_memory()
    hQ, hK, hV = pin(inp["Q_dec"]), pin(inp["K_dec"]), pin(inp["V_dec"])
    hO = torch.empty(O.shape, dtype=torch.bfloat16).pin_memory()

    def host_step():
        dQ.copy_(hQ, non_blocking=True); dKd.copy_(hK, non_blocking=True); dVd.copy_(hV, non_blocking=True)
        static()
        hO.copy_(O, non_blocking=True)
        torch.cuda.current_stream().synchronize()
    for _ in range(Wm):
        host_step()
    t0 = time.perf_counter()
    for _ in range(K):
        host_step()
    e2e_us = 1e6 * (time.perf_counter() - t0) / K
    peaks = load_peaks()
    roof = _attn_roofline(peaks, w.attn_flops(), w.attn_bytes(), us_static,
                          "attn_kernel, contiguous mode (3-D TMA tiles)" + (" + combine_kernel" if Sd > 1 else ""))
    roof_g = _attn_roofline(peaks, w.attn_flops(), w.attn_bytes(), us_gather,
                            "attn_kernel, gather mode (cp.async)" + (" + combine_kernel" if S > 1 else ""))
    from oracle import oracle
    cores = oracle.num_threads()
    n = max(1, min(w.H_kv, cores // max(1, min(w.G, cores))))
    sl = {k: np.ascontiguousarray(inp[k][:1, : (n * w.G if k == "Q_dec" else n)]) for k in ("Q_dec", "Kcache", "Vcache", "K_dec", "V_dec")}
    kp = None if inp["keep"] is None else np.ascontiguousarray(inp["keep"][:1, :n])
    t0 = time.perf_counter()
    oracle.attn(sl["Q_dec"], sl["Kcache"], sl["Vcache"], np.ascontiguousarray(inp["planted"][:1, :n]), kp, sl["K_dec"], sl["V_dec"])
    t_or = time.perf_counter() - t0
    factor = w.B * w.H_kv / n
    cpu = {"value": 1e6 * t_or * factor, "unit": UNIT, "cores": cores, "kind": "oracle",
           "sample": f"attention of {n} of {w.B * w.H_kv} (batch, KV-head) groups, time scaled x{factor:g}"}
    cfg = workload_config(w, Sd)
    cfg.update(mode="static", call="pdllm_static_attn over the compact cache of pdllm_compact_kv (static selection, P:116)",
               n_splits_gather=S)
    _line(args, w, us_static, cfg, roof, cpu,
          {"value": e2e_us, "unit": UNIT, "h2d_bytes_per_step": hQ.numel() * 2 + hK.numel() * 2 + hV.numel() * 2,
           "d2h_bytes_per_step": hO.numel() * 2, "call": "pinned host Q_dec/K_dec/V_dec in, O out, around pdllm_static_attn"},
          K * (1 + (1 if Sd > 1 else 0)), clk.summary(),
          {"static_mode_us": {"static_attn_tma_tiles": us_static, "sparse_attn_gather": us_gather,
                              "reselect_pooled_scorer_plus_topk": us_pooled, "reselect_full_scorer_plus_topk": us_full,
                              "compact_kv_once": us_compact, "pool_keys_once": us_pool},
           "roofline_gather": roof_g, "pooled_scorer_recall_of_planted_chunks": recall, "full_scorer_ids_ok": ids_ok})


def run_tokens(args, w):
    """--mode tokens: NEXT-1 on the workload's shape with planted tokens: pdllm_score_tokens (two streaming passes over
    the K cache) and pdllm_select_topb; HBM roofline of the pair of passes."""
    torch, B = _common_setup(args)
    if w.keep >= 1.0:
        w = W.small_variant(w, keep=0.5)
    w = W.small_variant(w, token_gamma=4.0) if not w.unit_logits else W.small_variant(w, token_alpha=24.0)
    shape = B.Shape.of(w)
    inp = W.make_inputs(w)
    bf = lambda bits: torch.from_numpy(np.ascontiguousarray(bits).view(np.int16)).cuda().view(torch.bfloat16)
    dQs, dKc = bf(inp["Q_score"]), bf(inp["Kcache"])
    e = torch.empty((w.B, w.H_kv, w.N, w.Cp), dtype=torch.float32, device="cuda")
    keep = torch.empty((w.B, w.H_kv, w.N, w.Bk), dtype=torch.int32, device="cuda")
    ws = torch.empty((B.lib().pdllm_score_tokens_workspace_bytes(__import__("ctypes").byref(shape.c())),), dtype=torch.uint8, device="cuda")
    sc = torch.empty((w.B, w.H_kv, w.N), dtype=torch.float32, device="cuda")
    K, Wm = args.steps, args.warmup
    flush = torch.empty((256 << 20,), dtype=torch.uint8, device="cuda") if needs_flush(w) else None
    tok = lambda: B.score_tokens(shape, dQs, dKc, token_scores=e, workspace=ws)
    for _ in range(Wm):
        tok(); B.select_topb(shape, e, keep)
    torch.cuda.synchronize()
    ok = bool((keep.cpu().numpy() == inp["keep"]).all())
    with ClockSampler(0) as clk:
        us_tok = _timed(torch, tok, K, flush)
    us_pass1 = _timed(torch, lambda: B.score_chunks(shape, dQs, dKc, scores=sc), K, flush)
    us_topb = _timed_graph(torch, lambda: B.select_topb(shape, e, keep), K)
    rows = w.G * w.L_q
    nbytes = 2 * w.B * w.H_kv * w.N * w.Cp * w.d * 2 + 2 * w.B * w.H * w.L_q * w.d * 2 \
        + 2 * 4 * w.B * w.H_kv * w.N * rows + 4 * w.B * w.H_kv * w.N * w.Cp
    peaks = load_peaks()
    flops = 2 * w.score_flops()           # Q K^T once per pass
    roof = _attn_roofline(peaks, flops, nbytes, us_tok, "score_kernel (row log-masses) + token_score_kernel (NEXT-1)")
    roof["algorithmic_bytes"] = nbytes
    roof["token_score_kernel_alone"] = _attn_roofline(peaks, flops / 2, nbytes / 2, max(us_tok - us_pass1, 1e-3), "token_score_kernel")
    from oracle import oracle
    cores = oracle.num_threads()
    n = max(1, min(w.H_kv, cores))
    nch = max(1, min(w.N, 4))
    t0 = time.perf_counter()
    oracle.token_scores(np.ascontiguousarray(inp["Q_score"][:1, : n * w.G]), np.ascontiguousarray(inp["Kcache"][:1, :n, :nch]), w.L_q)
    t_or = time.perf_counter() - t0
    factor = (w.B * w.H_kv / n) * (w.N / nch)
    cpu = {"value": 1e6 * t_or * factor, "unit": UNIT, "cores": cores, "kind": "oracle",
           "sample": f"token scores of {nch} of {w.N} chunks of {n} of {w.B * w.H_kv} groups, time scaled x{factor:g}"}
    hQ = torch.from_numpy(np.ascontiguousarray(inp["Q_score"]).view(np.int16)).view(torch.bfloat16).pin_memory()
    hkeep = torch.empty(keep.shape, dtype=torch.int32).pin_memory()

    def host_step():
        dQs.copy_(hQ, non_blocking=True)
        tok(); B.select_topb(shape, e, keep)
        hkeep.copy_(keep, non_blocking=True)
        torch.cuda.current_stream().synchronize()
    for _ in range(Wm):
        host_step()
    t0 = time.perf_counter()
    for _ in range(K):
        host_step()
    e2e_us = 1e6 * (time.perf_counter() - t0) / K
    cfg = workload_config(w, None)
    cfg.update(mode="tokens", call="pdllm_score_tokens (+ pdllm_select_topb): Eq. 5 query->chunk eviction scores, top-B retention",
               token_planting={"token_alpha": w.token_alpha, "token_gamma": w.token_gamma})
    _line(args, w, us_tok + us_topb, cfg, roof, cpu,
          {"value": e2e_us, "unit": UNIT, "h2d_bytes_per_step": hQ.numel() * 2, "d2h_bytes_per_step": hkeep.numel() * 4,
           "call": "pinned host query window in, token_keep_idx out, around pdllm_score_tokens + pdllm_select_topb"},
          K * (3 + (1 if rows > 128 else 0)), clk.summary(),
          {"tokens_mode_us": {"score_tokens_two_passes": us_tok, "of_which_chunk_score_pass": us_pass1, "select_topb": us_topb},
           "planted_tokens_recovered": ok})


def run_prefill(args, w):
    """--mode prefill: NEXT-2, the attention of the chunk prefill on the workload's prefix: N sequences [BOS; c_i; q; m]
    (|m| = 16 pseudo-labels) per batch element, all heads; tensor roofline."""
    torch, B = _common_setup(args)
    T = w.Cp + w.L_q + 16
    S = w.B * w.N
    r = np.random.Generator(np.random.Philox(key=[(w.seed << 8) + 9, 0]))
    mk = lambda shp: torch.from_numpy(W.f32_to_bf16_bits(r.standard_normal(shp, dtype=np.float32)).view(np.int16)).view(torch.bfloat16)
    hQ, hK, hV = mk((S, w.H, T, w.d)).pin_memory(), mk((S, w.H_kv, T, w.d)).pin_memory(), mk((S, w.H_kv, T, w.d)).pin_memory()
    dQ, dK, dV = hQ.cuda(), hK.cuda(), hV.cuda()
    ds = B.DenseShape(S, w.H, w.H_kv, w.d, T, T, 0)
    Sd = args.n_splits if args.n_splits > 0 else B.dense_auto_splits(ds, B.num_sms())
    ws = B.alloc_dense_workspace(ds, args.n_splits)
    O = torch.empty((S, w.H, T, w.d), dtype=torch.bfloat16, device="cuda")
    LSE = torch.empty((S, w.H, T), dtype=torch.float32, device="cuda")
    K, Wm = args.steps, args.warmup
    fn = lambda: B.prefill_attn(ds, dQ, dK, dV, n_splits=args.n_splits, O=O, LSE=LSE, workspace=ws)
    for _ in range(Wm):
        fn()
    torch.cuda.synchronize()
    kv_bytes = 2 * S * w.H_kv * T * w.d * 2
    flush = torch.empty((256 << 20,), dtype=torch.uint8, device="cuda") if kv_bytes < 4 * L2_BYTES else None
    with ClockSampler(0) as clk:
        us = _timed(torch, fn, K, flush)
    flops = 4.0 * S * w.H * T * T * w.d
    nbytes = kv_bytes + 2 * S * w.H * T * w.d * 2 + 4 * S * w.H * T
    roof = _attn_roofline(load_peaks(), flops, nbytes, us, "attn_kernel, contiguous mode (chunk prefill)" + (" + combine_kernel" if Sd > 1 else ""))
    from oracle import oracle
    cores = oracle.num_threads()
    nh = max(1, min(w.H_kv, cores // max(1, w.G)))
    Tq = min(T, 256)                      # a bounded sample: the first Tq query rows of nh KV heads of one sequence
    q = np.ascontiguousarray(hQ.view(torch.int16).numpy().view(np.uint16)[:1, : nh * w.G])
    k = np.ascontiguousarray(hK.view(torch.int16).numpy().view(np.uint16)[:1, :nh])
    v = np.ascontiguousarray(hV.view(torch.int16).numpy().view(np.uint16)[:1, :nh])
    t0 = time.perf_counter()
    oracle.prefill_attn(q, k, v)
    t_or = time.perf_counter() - t0
    factor = S * w.H_kv / nh
    cpu = {"value": 1e6 * t_or * factor, "unit": UNIT, "cores": cores, "kind": "oracle",
           "sample": f"one sequence, {nh} of {w.H_kv} KV heads (all {T} rows), time scaled x{factor:g}"}
    hO = torch.empty(O.shape, dtype=torch.bfloat16).pin_memory()

    def host_step():
        dQ.copy_(hQ, non_blocking=True); dK.copy_(hK, non_blocking=True); dV.copy_(hV, non_blocking=True)
        fn()
        hO.copy_(O, non_blocking=True)
        torch.cuda.current_stream().synchronize()
    for _ in range(min(Wm, 3)):
        host_step()
    Ke = max(3, K // 10)
    t0 = time.perf_counter()
    for _ in range(Ke):
        host_step()
    e2e_us = 1e6 * (time.perf_counter() - t0) / Ke
    cfg = {"workload": f"chunk prefill of '{w.name}': {S} sequences [BOS; c_i; q; m] of T = {T} rows (C = {w.C}, L_q = {w.L_q}, |m| = 16)",
           "mode": "prefill", "S": S, "H": w.H, "H_kv": w.H_kv, "d": w.d, "T": T, "n_splits": Sd,
           "call": "pdllm_prefill_attn (Eq. 2; SURVEY 8(f) NEXT-2)",
           "l2": "explicit 256 MB flush between iterations" if flush is not None else "K/V larger than L2, no explicit flush"}
    _line(args, w, us, cfg, roof, cpu,
          {"value": e2e_us, "unit": UNIT, "h2d_bytes_per_step": (hQ.numel() + hK.numel() + hV.numel()) * 2,
           "d2h_bytes_per_step": hO.numel() * 2, "call": "pinned host Q/K/V in, O out, around pdllm_prefill_attn"},
          K * (1 + (1 if Sd > 1 else 0)), clk.summary(), {})


# --------------------------------------------------------------------------- BASELINE.json configs[4]: the sweep
def sampled_parity(B, torch, w, shape, t):
    """parity of 4 sampled (b, h) of one layer-step against the fp64 oracle, and the oracle's time on
    them.  Returns dict(ok, score_err, o_err, o_norm, lse_err, oracle_s) -- the R12 gates decide `ok`; chunk ids are
    checked as the oracle's top-K of the GPU's own scores (random data has no planted gap: same-precision decision)."""
    from oracle import oracle
    out = B.step(shape, t["Q"], t["Kc"], t["Vc"], None, t["Kd"], t["Vd"], workspace=t["ws"], **t["out"])
    torch.cuda.synchronize()
    picks = sorted({(0, 0), (w.B - 1, w.H - 1), (w.B // 2, 7 % w.H), (0, 19 % w.H)})
    u16 = lambda x: x.contiguous().view(torch.int16).cpu().numpy().view(np.uint16)
    res = dict(ok=True, score_err=0.0, o_err=0.0, o_norm=0.0, lse_err=0.0, oracle_s=0.0, heads=len(picks))
    for b, h in picks:
        sl = lambda x: u16(x[b:b + 1, h:h + 1])
        Q, Kc, Vc, Kd, Vd = sl(t["Q"]), sl(t["Kc"]), sl(t["Vc"]), sl(t["Kd"]), sl(t["Vd"])
        t0 = time.perf_counter()
        sc = oracle.scores(Q, Kc, w.L_q)
        g_sc = out["scores"][b, h].double().cpu().numpy()
        ids = out["chunk_ids"][b:b + 1, h:h + 1].cpu().numpy()
        O_ref, LSE_ref = oracle.attn(Q, Kc, Vc, ids, None, Kd, Vd)
        res["oracle_s"] += time.perf_counter() - t0
        O = (u16(out["O"][b:b + 1, h:h + 1]).astype(np.uint32) << 16).view(np.float32).astype(np.float64)
        LSE = out["LSE"][b:b + 1, h:h + 1].double().cpu().numpy()
        d_o = np.abs(O - O_ref)
        res["score_err"] = max(res["score_err"], float(np.abs(g_sc - sc[0, 0]).max()))
        res["o_err"] = max(res["o_err"], float(d_o.max()))
        res["o_norm"] = max(res["o_norm"], float(d_o.max() / np.abs(O_ref).max()))
        res["lse_err"] = max(res["lse_err"], float(np.abs(LSE - LSE_ref).max()))
        ids_ok = bool((oracle.topk(g_sc[None, None], w.K) == ids).all())
        res["ok"] = bool(res["ok"] and ids_ok and (d_o <= 2e-2 + 1e-2 * np.abs(O_ref)).all() and res["o_norm"] <= 1e-2
                         and res["lse_err"] <= 1e-3 and res["score_err"] <= 1e-3)
    return res


def run_sweep(args):
    """--mode sweep: paper_2606_10537_b200.sweep's points with the oracle leg per point (parity of 4 sampled (b, h); the
    oracle's time on them scaled to all B*H heads of the layer-step, labelled extrapolated)."""
    torch, B = _common_setup(args)
    from paper_2606_10537_b200 import sweep as SW
    g = torch.Generator(device="cuda").manual_seed(20260615)
    rows = []

    def hook(w, shape, t, row):
        r = sampled_parity(B, torch, w, shape, t)
        row["oracle_us_extrapolated"] = 1e6 * r["oracle_s"] * (w.B * w.H) / r["heads"]
        row["parity"] = ("ok" if r["ok"] else "FAIL") + f" (O {r['o_err']:.1e}/{r['o_norm']:.1e}, LSE {r['lse_err']:.1e}, s {r['score_err']:.1e})"
        row["parity_ok"] = r["ok"]

    for pt in SW.grid_points(args.quick):
        row = SW.run_point(B, torch, g, pt, args.layers, 3, 100.0, hook)
        rows.append(row)
        print(json.dumps(row), flush=True)
    t = SW.table(rows)
    if args.out:
        Path(args.out).write_text(t)
    print(t)
    if not all(r.get("parity_ok", False) for r in rows):
        raise SystemExit("bench.py --mode sweep: a sampled parity check failed")


def run_splitsweep(args, w):
    """--mode splitsweep: SURVEY 8(d): the workload's attention for every split count S = 1 .. min(64, KV tiles), the
    partial-attention kernel and the LSE-combine kernel timed apart (CUDA events between them inside pdllm_step_profiled's
    attention stage are not exposed for pdllm_sparse_attn, so the two are timed as: whole call, and pdllm_lse_combine
    alone on partials of the same size)."""
    torch, B = _common_setup(args)
    shape = B.Shape.of(w)
    inp = W.make_inputs(w)
    bf = lambda bits: torch.from_numpy(np.ascontiguousarray(bits).view(np.int16)).cuda().view(torch.bfloat16)
    dQ, dKc, dVc, dKd, dVd = (bf(inp[k]) for k in ("Q_dec", "Kcache", "Vcache", "K_dec", "V_dec"))
    dkeep = None if inp["keep"] is None else torch.from_numpy(inp["keep"]).cuda()
    ids = torch.from_numpy(inp["planted"]).cuda()
    O = torch.empty((w.B, w.H, w.L, w.d), dtype=torch.bfloat16, device="cuda")
    LSE = torch.empty((w.B, w.H, w.L), dtype=torch.float32, device="cuda")
    flush = torch.empty((256 << 20,), dtype=torch.uint8, device="cuda") if needs_flush(w) else None
    tiles = -(-w.S_kv // 128)
    auto = B.auto_splits(shape, B.num_sms())
    rows_n = w.B * w.H * w.L
    lines = [f"| S | attention call us (cold L2) | of which LSE combine us | partial traffic MB (write + read) | note |", "|---|---|---|---|---|"]
    for S in range(1, min(64, tiles) + 1):
        ws = B.alloc_workspace(shape, S)
        fn = lambda: B.sparse_attn(shape, dQ, dKc, dVc, ids, dkeep, dKd, dVd, n_splits=S, O=O, LSE=LSE, workspace=ws)
        for _ in range(3):
            fn()
        us = _timed(torch, fn, args.steps, flush)
        us_c = 0.0
        if S > 1:
            Op = torch.randn((S, rows_n, w.d), device="cuda"); lp = torch.randn((S, rows_n), device="cuda")
            O2 = torch.empty((rows_n, w.d), dtype=torch.bfloat16, device="cuda"); L2 = torch.empty((rows_n,), dtype=torch.float32, device="cuda")
            us_c = _timed(torch, lambda: B.lse_combine(Op, lp, O2, L2), args.steps, flush)
        mb = 0.0 if S == 1 else 2 * S * rows_n * (w.d + 1) * 4 / 1e6
        lines.append(f"| {S} | {us:.1f} | {us_c:.1f} | {mb:.1f} | {'auto (pdllm_auto_splits)' if S == auto else ''} |")
        print(lines[-1], flush=True)
    t = "\n".join(lines) + "\n"
    if args.out:
        Path(args.out).write_text(t)
    print(t)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--workload", choices=list(W.CONFIGS) + list(W.EXTRA), default="sparse32k")
    ap.add_argument("--n-splits", type=int, default=0, help="0 = pdllm_auto_splits")
    ap.add_argument("--quick", action="store_true", help="--mode sweep: a 13-point subset")
    ap.add_argument("--layers", type=int, default=32, help="--mode sweep: stacked layers per point")
    ap.add_argument("--out", default="", help="--mode sweep / splitsweep: write the markdown table here")
    ap.add_argument("--mode", choices=["step", "static", "tokens", "prefill", "sweep", "splitsweep"], default="step",
                    help="step: pdllm_step (the metric's per-step call, default); static / tokens / prefill: the rows "
                         "after the hot path (SURVEY 8(f)), 1 GPU")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "ours" and args.gpus > 1 and int(os.environ.get("WORLD_SIZE", "1")) != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} needs one rank per GPU: launch with `python -m torch.distributed.run "
                         f"--nnodes=1 --nproc-per-node {args.gpus} --master-addr 127.0.0.1 --master-port P bench.py --gpus "
                         f"{args.gpus} ...` (replicas only, DESIGN.md section 10); refusing to print an n_gpus=1 line")
    w = W.CONFIGS[args.workload] if args.workload in W.CONFIGS else W.EXTRA[args.workload]
    if args.impl == "reference":
        run_reference(args, w)
    elif args.mode == "sweep":
        run_sweep(args)
    elif args.mode == "splitsweep":
        run_splitsweep(args, w)
    elif args.mode == "static":
        run_static(args, w)
    elif args.mode == "tokens":
        run_tokens(args, w)
    elif args.mode == "prefill":
        run_prefill(args, w)
    elif w.strict:
        raise SystemExit(f"bench.py: workload {w.name} has no query rows in Q_dec (strict R8 rows): use --mode static")
    else:
        run_ours(args, w)


if __name__ == "__main__":
    main()
