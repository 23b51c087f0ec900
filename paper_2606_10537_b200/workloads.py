"""Seeded synthetic inputs with the shapes and statistics of the paper's workloads.

This module serves BOTH the CUDA path and the oracle (tests, bench.py, smoke) and
therefore holds none of the method's arithmetic: it only draws random tensors,
rounds them to bf16 and plants a key shift so that top-K has a clear gap
(BASELINE.json configs).  numpy only; no torch, no CUDA.

The paper measures on LongBench MF-en prompts at 8K/16K/32K with
Dream-7B / UltraLLaDA weights; neither dataset nor weights exist here, and the
attention path only sees tensor shapes and value statistics, so seeded Gaussians
with planted relevant chunks stand in for them.
"""
from __future__ import annotations

from concurrent.futures import ThreadPoolExecutor
from dataclasses import dataclass, replace

import numpy as np

BASE_SEED = 20260610

# tensor ids (stream selectors of the counter-based generator)
T_Q, T_KC, T_VC, T_KD, T_VD, T_KEEP, T_PLANT = 1, 2, 3, 4, 5, 6, 7


@dataclass(frozen=True)
class Workload:
    name: str
    B: int
    H: int
    H_kv: int
    d: int
    N: int
    C: int
    K: int
    keep: float          # fraction of the C chunk tokens kept (1.0 -> token_keep_idx is None)
    L_q: int
    L_d: int
    alpha: float         # planted key shift, in units of mean(q) (R20)
    unit_logits: bool    # True: Q,K,V ~ N(0,1)/sqrt(d) (config "tiny"); False: N(0,1)
    seed: int
    # NEXT-1 workloads only -- planted tokens, so that top-B token retention has a clear gap: in every chunk the keys of
    # the slots on the keep list are shifted by token_alpha * mean(q) (works while G*L_q is small enough for the rows to
    # agree with their mean: config "tiny") and / or multiplied by token_gamma (a longer key draws more softmax mass from
    # every row whatever its direction: the N(0,1) configs)
    token_alpha: float = 0.0
    token_gamma: float = 1.0
    # R8's strict reading of P:116 ("only the response tokens are processed", the query KV is cached): Q_dec holds the
    # L_d response rows only while K_dec / V_dec hold the L_q + L_d query + response rows.  False (the BASELINE.json
    # configs): the L_q query rows attend too, L = L_s = L_q + L_d, query rows first.
    strict: bool = False

    @property
    def G(self): return self.H // self.H_kv
    @property
    def Cp(self): return self.C + 1
    @property
    def Bk(self): return self.Cp if self.keep >= 1.0 else 1 + int(round(self.keep * self.C))
    @property
    def L(self): return self.L_d if self.strict else self.L_q + self.L_d
    @property
    def L_s(self): return self.L_q + self.L_d
    @property
    def S_pre(self): return self.K * self.Bk
    @property
    def S_kv(self): return self.S_pre + self.L_s

    # algorithmic work of one step; used by bench.py for TFLOP/s and GB/s
    def attn_flops(self): return 4.0 * self.B * self.H * self.L * self.S_kv * self.d
    def attn_bytes(self):
        return (2 * self.B * self.H_kv * self.S_pre * self.d * 2 + 2 * self.B * self.H_kv * self.L_s * self.d * 2
                + 2 * self.B * self.H * self.L * self.d * 2 + self.B * self.H * self.L * 4
                + 4 * self.B * self.H_kv * self.K * (1 + (self.Bk if self.keep < 1.0 else 0)))
    def score_flops(self): return 2.0 * self.B * self.H * self.L_q * self.N * self.Cp * self.d
    def score_bytes(self):
        return self.B * self.H_kv * self.N * self.Cp * self.d * 2 + self.B * self.H * self.L_q * self.d * 2 + 4 * self.B * self.H_kv * self.N
    def topk_bytes(self): return 4 * self.B * self.H_kv * (self.N + self.K)


# BASELINE.json configs[0..3]; alpha per R20.
CONFIGS = {
    "tiny": Workload("tiny", B=1, H=4, H_kv=4, d=64, N=8, C=64, K=2, keep=0.5, L_q=16, L_d=32,
                     alpha=1.0, unit_logits=True, seed=BASE_SEED + 1),
    "llada8k": Workload("llada8k", B=1, H=32, H_kv=32, d=128, N=16, C=512, K=4, keep=1.0, L_q=64, L_d=256,
                        alpha=0.5, unit_logits=False, seed=BASE_SEED + 2),
    "dream16k": Workload("dream16k", B=1, H=28, H_kv=4, d=128, N=16, C=1024, K=4, keep=0.5, L_q=128, L_d=256,
                         alpha=2.0, unit_logits=False, seed=BASE_SEED + 3),
    "sparse32k": Workload("sparse32k", B=4, H=32, H_kv=32, d=128, N=64, C=512, K=8, keep=0.25, L_q=128, L_d=256,
                          alpha=0.5, unit_logits=False, seed=BASE_SEED + 4),
}

# Not a BASELINE.json config: the paper's own decode-kernel shape (Fig. 5(b): GQA 32/8, d = 128, 32 rows per
# head attending ~4K selected KV: K = 4 chunks of C = 1024), the L << S_kv regime Split-S was made for.
# G*L = 128 packed rows = one query tile per KV group: 8 single items, so everything hangs on the split count.
EXTRA = {
    "fig5b": Workload("fig5b", B=1, H=32, H_kv=8, d=128, N=16, C=1024, K=4, keep=1.0, L_q=16, L_d=16,
                      alpha=2.0, unit_logits=False, seed=BASE_SEED + 6),
}
# SURVEY 8(f) NEXT-4, the Fig. 5(b) shape as the survey wrote it: L = L_d = 32 response rows (strict R8), the cached
# query window L_q = 64 inside K_dec / V_dec, GQA 32/8, d = 128, dense-selected KV of 8K / 16K / 32K tokens
# (K whole chunks of C = 1024 out of a 32K prefix); the paper runs it with S = 4 splits.
for _k, _name in ((8, "fig5b_8k"), (16, "fig5b_16k"), (32, "fig5b_32k")):
    EXTRA[_name] = Workload(_name, B=1, H=32, H_kv=8, d=128, N=32, C=1024, K=_k, keep=1.0, L_q=64, L_d=32,
                            alpha=2.0, unit_logits=False, seed=BASE_SEED + 7 + _k, strict=True)


def small_variant(w: Workload, **kw) -> Workload:
    return replace(w, **kw)


def f32_to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """float32 -> bf16 bit patterns, round-to-nearest-even (inputs are finite)."""
    u = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32)
    r = (u + np.uint32(0x7FFF) + ((u >> np.uint32(16)) & np.uint32(1))) >> np.uint32(16)
    return r.astype(np.uint16)


def bf16_bits_to_f32(b: np.ndarray) -> np.ndarray:
    return (b.astype(np.uint32) << np.uint32(16)).view(np.float32)


def _rng(seed: int, tensor_id: int, slab: int = 0) -> np.random.Generator:
    # Philox is counter-based: (seed, tensor_id, slab) selects an independent stream.
    return np.random.Generator(np.random.Philox(key=[(seed << 8) + tensor_id, slab]))


def _normal(seed, tensor_id, slab, shape, sigma):
    x = _rng(seed, tensor_id, slab).standard_normal(shape, dtype=np.float32)
    if sigma != 1.0:
        x *= np.float32(sigma)
    return x


def make_keep(w: Workload):
    """token_keep_idx int32 [B,H_kv,N,Bk]: slot 0 (BOS) + round(keep*C) distinct sorted slots of 1..C (R7)."""
    if w.keep >= 1.0:
        return None
    m = w.Bk - 1
    rows = w.B * w.H_kv * w.N
    r = _rng(w.seed, T_KEEP).random((rows, w.C), dtype=np.float32)
    sel = np.argpartition(r, m - 1, axis=1)[:, :m] + 1 if m > 0 else np.zeros((rows, 0), np.int64)
    sel = np.sort(sel, axis=1)
    out = np.concatenate([np.zeros((rows, 1), np.int64), sel], axis=1).astype(np.int32)
    return out.reshape(w.B, w.H_kv, w.N, w.Bk)


def make_planted(w: Workload):
    """planted chunk ids int32 [B,H_kv,K], ascending, drawn without replacement per (b,g)."""
    r = _rng(w.seed, T_PLANT).random((w.B * w.H_kv, w.N))
    ids = np.sort(np.argsort(r, axis=1)[:, : w.K], axis=1).astype(np.int32)
    return ids.reshape(w.B, w.H_kv, w.K)


def make_inputs(w: Workload, threads: int = 8) -> dict:
    """All tensors of one step as numpy arrays (bf16 tensors as uint16 bit patterns)."""
    sigma = 1.0 / np.sqrt(w.d) if w.unit_logits else 1.0
    Q = f32_to_bf16_bits(_normal(w.seed, T_Q, 0, (w.B, w.H, w.L_q + w.L_d, w.d), sigma))     # query rows, then response rows
    Kd = f32_to_bf16_bits(_normal(w.seed, T_KD, 0, (w.B, w.H_kv, w.L_s, w.d), sigma))
    Vd = f32_to_bf16_bits(_normal(w.seed, T_VD, 0, (w.B, w.H_kv, w.L_s, w.d), sigma))
    keep = make_keep(w)
    planted = make_planted(w)
    # mean(q) over the G*L_q scoring rows of each KV group, from the bf16-rounded Q
    qf = bf16_bits_to_f32(Q[:, :, : w.L_q, :]).astype(np.float64)
    qbar = qf.reshape(w.B, w.H_kv, w.G * w.L_q, w.d).mean(axis=2).astype(np.float32)   # [B,H_kv,d]

    Kc = np.empty((w.B, w.H_kv, w.N, w.Cp, w.d), np.uint16)
    Vc = np.empty((w.B, w.H_kv, w.N, w.Cp, w.d), np.uint16)

    def slab(bg):
        b, g = divmod(bg, w.H_kv)
        k = _normal(w.seed, T_KC, bg, (w.N, w.Cp, w.d), sigma)
        k[planted[b, g]] += np.float32(w.alpha) * qbar[b, g]        # shift every row of the planted chunks
        if keep is not None and (w.token_alpha > 0.0 or w.token_gamma != 1.0):      # planted tokens: the kept slots
            sel = (np.arange(w.N)[:, None], keep[b, g, :, 1:])
            k[sel] = k[sel] * np.float32(w.token_gamma) + np.float32(w.token_alpha) * qbar[b, g]
        Kc[b, g] = f32_to_bf16_bits(k)
        Vc[b, g] = f32_to_bf16_bits(_normal(w.seed, T_VC, bg, (w.N, w.Cp, w.d), sigma))

    n = w.B * w.H_kv
    if threads > 1 and n > 1:
        with ThreadPoolExecutor(max_workers=threads) as ex:
            list(ex.map(slab, range(n)))
    else:
        for bg in range(n):
            slab(bg)
    Q_score = np.ascontiguousarray(Q[:, :, : w.L_q])                # the scoring rows (the query window)
    Q_dec = np.ascontiguousarray(Q[:, :, w.L_q:]) if w.strict else Q
    return dict(Q_dec=Q_dec, Q_score=Q_score, Kcache=Kc, Vcache=Vc, K_dec=Kd, V_dec=Vd, keep=keep, planted=planted)
