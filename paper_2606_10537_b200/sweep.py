"""Throughput sweep of the per-step path (BASELINE.json configs[4]): stacked LLaDA-8B-like attention layers.

    python -m paper_2606_10537_b200.sweep [--quick] [--layers 32] [--out sweep.md]

For every point (prefix in {8K,16K,32K}, C in {512,1024}, K in {2,4,8,16} (K <= N), L_d in {64,256,512}, L_q = 64,
B in {1,8}; H = H_kv = 32, d = 128, keep = 100 %) the step `pdllm_step` (scoring -> top-K -> Split-S attention ->
combine) runs over `layers` independent K/V caches in turn (so consecutive calls never find their cache in L2), and,
as the comparator the configs name, the SAME attention kernel runs dense (K = N: every chunk selected) on the same
shapes.  Inputs are seeded device-side Gaussians.  This module only times (the product never touches the oracle);
`python bench.py --mode sweep` runs the same points and adds, per point, the oracle leg SURVEY 8(d) asks for: parity of
4 sampled (b, h) against the fp64 oracle and the oracle's time on those heads extrapolated to the layer-step
(tests/test_gpu_sweep.py checks the shape classes as tests).  Prints one JSON line per point and writes a markdown
table; each point carries the SM clock and throttle reasons read right after its step loop.

Reported per point: us per layer-step, the attention's us / TFLOP/s / GB/s and its fraction of the roofline (the slower
of FLOPs at the measured sustained bf16 peak and algorithmic bytes at the measured HBM peak), the scoring's us and GB/s,
and the dense attention's us.
"""
from __future__ import annotations

import argparse
import itertools
import json
from pathlib import Path

ROOT = Path(__file__).resolve().parent.parent


def peaks():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        d = json.loads(p.read_text())
        return float(d["hbm_gbs"]), float(d["bf16_tflops_sustained"]), "measured"
    return 6650.0, 1400.0, "fallback"


def clock_state():
    """(SM MHz, active throttle-reason names) right now, via NVML; (None, ["unavailable"]) without it."""
    try:
        import pynvml
        pynvml.nvmlInit()
        h = pynvml.nvmlDeviceGetHandleByIndex(0)
        mhz = pynvml.nvmlDeviceGetClockInfo(h, pynvml.NVML_CLOCK_SM)
        f = getattr(pynvml, "nvmlDeviceGetCurrentClocksEventReasons", None) or pynvml.nvmlDeviceGetCurrentClocksThrottleReasons
        r = int(f(h))
        names = [n for n, bit in (("sw_power_cap", 0x4), ("hw_slowdown", 0x8), ("sw_thermal_slowdown", 0x20),
                                  ("hw_thermal_slowdown", 0x40), ("hw_power_brake", 0x80)) if r & bit]
        return mhz, names
    except Exception:
        return None, ["unavailable"]


def grid_points(quick=False):
    """BASELINE.json configs[4]: (prefix, C, K, L_d, B) with K <= N = prefix / C."""
    grid = list(itertools.product((8192, 16384, 32768), (512, 1024), (2, 4, 8, 16), (64, 256, 512), (1, 8)))
    if quick:
        grid = [pt for pt in grid if pt[1] == 512 and pt[2] in (4, 8) and pt[3] == 256] + [(32768, 1024, 4, 256, 1)]
    return [pt for pt in grid if pt[2] <= pt[0] // pt[1]]


def run_point(B, torch, g, pt, layers_max=32, steps=3, mem_gb=100.0, hook=None):
    """Time one sweep point; returns its row.  `hook(w, shape, tensors, row)` (optional) is called before the caches are
    freed -- bench.py --mode sweep uses it for the oracle leg (this module never touches the oracle)."""
    from .workloads import Workload
    hbm, tf, src = peaks()
    H, d, L_q = 32, 128, 64
    prefix, C, K, L_d, Bn = pt
    N = prefix // C
    w = Workload("sweep", B=Bn, H=H, H_kv=H, d=d, N=N, C=C, K=K, keep=1.0, L_q=L_q, L_d=L_d, alpha=0.0,
                 unit_logits=False, seed=0)
    cache_bytes = 2 * Bn * H * N * (C + 1) * d * 2
    layers = max(1, min(layers_max, int(mem_gb * 1e9 // cache_bytes)))
    rnd = lambda *s: torch.randn(*s, generator=g, device="cuda", dtype=torch.float32).to(torch.bfloat16)
    Kc = [rnd(Bn, H, N, C + 1, d) for _ in range(layers)]
    Vc = [rnd(Bn, H, N, C + 1, d) for _ in range(layers)]
    Q, Kd, Vd = rnd(Bn, H, w.L, d), rnd(Bn, H, w.L, d), rnd(Bn, H, w.L, d)
    shape = B.Shape.of(w)
    dense = B.Shape(Bn, H, H, d, N, C, min(N, 64), C + 1, L_q, w.L, w.L)
    ws = B.alloc_workspace(shape, 0)
    ws_dense = B.alloc_workspace(dense, 0)
    out = dict(scores=torch.empty((Bn, H, N), dtype=torch.float32, device="cuda"),
               chunk_ids=torch.empty((Bn, H, K), dtype=torch.int32, device="cuda"),
               O=torch.empty((Bn, H, w.L, d), dtype=torch.bfloat16, device="cuda"),
               LSE=torch.empty((Bn, H, w.L), dtype=torch.float32, device="cuda"))
    all_ids = torch.arange(dense.K, dtype=torch.int32, device="cuda").repeat(Bn, H, 1).contiguous()

    def timed(fn, n):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        fn(0)
        torch.cuda.synchronize()
        a.record()
        for i in range(n):
            fn(i % layers)
        b.record()
        torch.cuda.synchronize()
        return 1e3 * a.elapsed_time(b) / n

    n = steps * layers
    us_step = timed(lambda i: B.step(shape, Q, Kc[i], Vc[i], None, Kd, Vd, workspace=ws, **out), n)
    mhz, reasons = clock_state()                  # right after the heaviest loop of the point
    us_score = timed(lambda i: B.score_chunks(shape, Q, Kc[i], out["scores"]), n)
    ids = out["chunk_ids"].clone()
    us_attn = timed(lambda i: B.sparse_attn(shape, Q, Kc[i], Vc[i], ids, None, Kd, Vd, O=out["O"], LSE=out["LSE"],
                                            workspace=ws), n)
    us_dense = None
    if N <= 64:                                   # K <= 64 is the library's bound on selected chunks
        us_dense = timed(lambda i: B.sparse_attn(dense, Q, Kc[i], Vc[i], all_ids, None, Kd, Vd, O=out["O"],
                                                 LSE=out["LSE"], workspace=ws_dense), max(layers, 4))
    roof_us = 1e6 * max(w.attn_flops() / (tf * 1e12), w.attn_bytes() / (hbm * 1e9))
    row = dict(prefix=prefix, C=C, K=K, L_d=L_d, B=Bn, layers=layers, n_splits=B.auto_splits(shape, B.num_sms()),
               step_us=us_step, score_us=us_score, score_gbs=w.score_bytes() / us_score / 1e3,
               attn_us=us_attn, attn_tflops=w.attn_flops() / us_attn / 1e6, attn_gbs=w.attn_bytes() / us_attn / 1e3,
               attn_roofline_us=roof_us, attn_frac=roof_us / us_attn, dense_attn_us=us_dense, peaks=src,
               sm_mhz=mhz, clock_reasons=reasons)
    if hook is not None:
        hook(w, shape, dict(Q=Q, Kc=Kc[0], Vc=Vc[0], Kd=Kd, Vd=Vd, ws=ws, out=out), row)
    del Kc, Vc
    torch.cuda.empty_cache()
    return row


def table(rows):
    has_or = any("oracle_us_extrapolated" in r for r in rows)
    head = "| prefix | C | K | L_d | B | layers | S | step us | score us (GB/s) | attn us | TFLOP/s | GB/s | of roofline | dense attn us | SM MHz (reasons) |"
    sep = "|---|---|---|---|---|---|---|---|---|---|---|---|---|---|---|"
    if has_or:
        head += " oracle us/layer-step (extrapolated) | parity (4 sampled b,h) |"
        sep += "---|---|"
    lines = [head, sep]
    for r in rows:
        dn = "-" if r["dense_attn_us"] is None else f"{r['dense_attn_us']:.0f}"
        line = (f"| {r['prefix'] // 1024}K | {r['C']} | {r['K']} | {r['L_d']} | {r['B']} | {r['layers']} | {r['n_splits']} | "
                f"{r['step_us']:.1f} | {r['score_us']:.1f} ({r['score_gbs']:.0f}) | {r['attn_us']:.1f} | {r['attn_tflops']:.0f} | "
                f"{r['attn_gbs']:.0f} | {r['attn_frac']:.2f} | {dn} | {r['sm_mhz']} ({','.join(r['clock_reasons']) or 'none'}) |")
        if has_or:
            line += f" {r.get('oracle_us_extrapolated', float('nan')):.3g} | {r.get('parity', '-')} |"
        lines.append(line)
    return "\n".join(lines) + "\n"


def main():
    import torch
    from . import binding as B

    ap = argparse.ArgumentParser()
    ap.add_argument("--quick", action="store_true", help="a 12-point subset")
    ap.add_argument("--layers", type=int, default=32)
    ap.add_argument("--steps", type=int, default=3, help="passes over all layers per point")
    ap.add_argument("--mem-gb", type=float, default=100.0, help="cap on the K/V caches of one point")
    ap.add_argument("--out", default="")
    args = ap.parse_args()
    assert torch.cuda.is_available(), "the sweep needs a CUDA device (no CPU fallback)"
    B.lib()
    g = torch.Generator(device="cuda").manual_seed(20260615)
    rows = []
    for pt in grid_points(args.quick):
        row = run_point(B, torch, g, pt, args.layers, args.steps, args.mem_gb)
        rows.append(row)
        print(json.dumps(row), flush=True)
    t = table(rows)
    if args.out:
        Path(args.out).write_text(t)
    print(t)


if __name__ == "__main__":
    main()
