"""GPU-vs-oracle parity of the rows after the hot path through the C ABI: compact static cache + TMA-tile
attention + pooled-key scorer (NEXT-3), chunk-prefill attention (NEXT-2), token scores + top-B (NEXT-1), the paper's
Fig. 5(b) decode shapes (NEXT-4).  Same gates as test_gpu_parity.py (R12); index lists bit-exact."""
import dataclasses

import numpy as np
import pytest
import torch

from oracle import oracle
from paper_2606_10537_b200 import workloads as W

from gpu_util import (LSE_ABS, SCORE_ABS, check_close, check_exact, check_O, dev_bf16, dev_f32, dev_i32,
                      shape_of, to_device)

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    from paper_2606_10537_b200 import binding
    binding.lib()
    return binding


def _inputs(name, **kw):
    w = W.CONFIGS.get(name) or W.EXTRA[name]
    if kw:
        w = W.small_variant(w, **kw)
    return w, W.make_inputs(w)


# --------------------------------------------------------------------------- NEXT-3 compact cache + static attention
@pytest.mark.parametrize("name,kw,splits", [
    ("tiny", {}, [1, 2, 0]),                                                   # S_pre = 66 < one tile, keep list
    ("tiny", dict(C=100, K=3, keep=1.0, L_q=40, L_d=99), [1, 3]),              # ragged prefix tail AND ragged decode tail
    ("tiny", dict(H=8, H_kv=2, d=128, C=200, K=5, keep=0.4, L_q=30, L_d=100), [1, 2, 0]),   # GQA, pair + single items
    ("llada8k", {}, [0, 1]),
    ("dream16k", {}, [0, 4]),
    ("sparse32k", {}, [0]),
])
def test_static_path_compact_then_tma_attention(B, name, kw, splits):
    """pdllm_compact_kv is a bit copy of the oracle's gathered rows; pdllm_static_attn over it gives the oracle's
    attention for the original chunk ids / keep lists (compaction is the identity on O and LSE)."""
    w, inp = _inputs(name, **kw)
    dev = to_device(inp)
    shape = B.Shape.of(w)
    ids = inp["planted"]
    Kc, Vc = B.compact_kv(shape, dev["Kcache"], dev["Vcache"], dev_i32(ids), dev["keep"])
    torch.cuda.synchronize()
    gi = oracle.gather_idx(ids, inp["keep"], w.N, w.C)
    Kc_ref, Vc_ref = oracle.compact_kv(inp["Kcache"], inp["Vcache"], gi)
    assert np.array_equal(Kc.view(torch.int16).cpu().numpy().view(np.uint16), Kc_ref), "Kcompact"
    assert np.array_equal(Vc.view(torch.int16).cpu().numpy().view(np.uint16), Vc_ref), "Vcompact"
    O_ref, LSE_ref = oracle.attn(inp["Q_dec"], inp["Kcache"], inp["Vcache"], ids, inp["keep"], inp["K_dec"], inp["V_dec"])
    ds = B.DenseShape.static_of(shape)
    for S in splits:
        O, LSE = B.static_attn(ds, dev["Q_dec"], Kc, Vc, dev["K_dec"], dev["V_dec"], n_splits=S)
        torch.cuda.synchronize()
        e_o, r_o = check_O(O, O_ref, what=f"static O (S={S})")
        check_close(LSE, LSE_ref, LSE_ABS, what=f"static LSE (S={S})")
        print(f"{name} static S={S}: O max|d| {e_o:.2e} (norm {r_o:.2e})")


def test_static_attn_without_decode_rows(B):
    """L_s = 0: attention over the compact prefix alone (K_dec / V_dec NULL)."""
    w, inp = _inputs("tiny", C=150, K=3, keep=0.7, d=128, H=4, H_kv=2)
    dev = to_device(inp)
    shape = B.Shape.of(w)
    ids = inp["planted"]
    Kc, Vc = B.compact_kv(shape, dev["Kcache"], dev["Vcache"], dev_i32(ids), dev["keep"])
    gi = oracle.gather_idx(ids, inp["keep"], w.N, w.C)
    Kc_ref, Vc_ref = oracle.compact_kv(inp["Kcache"], inp["Vcache"], gi)
    # the oracle's dense definition over those rows: one sequence's prefill attention with separate Q
    q = oracle.bf16_to_f64(inp["Q_dec"]); k = oracle.bf16_to_f64(Kc_ref); v = oracle.bf16_to_f64(Vc_ref)
    z = np.einsum("bhgid,bhjd->bhgij", q.reshape(w.B, w.H_kv, w.G, w.L, w.d), k) / np.sqrt(w.d)
    m = z.max(-1, keepdims=True); p = np.exp(z - m); l = p.sum(-1, keepdims=True)
    O_ref = np.einsum("bhgij,bhjd->bhgid", p / l, v).reshape(w.B, w.H, w.L, w.d)
    LSE_ref = (m + np.log(l))[..., 0].reshape(w.B, w.H, w.L)
    ds = B.DenseShape(w.B, w.H, w.H_kv, w.d, w.S_pre, w.L, 0)
    for S in (1, 2):
        O, LSE = B.static_attn(ds, dev["Q_dec"], Kc, Vc, None, None, n_splits=S)
        torch.cuda.synchronize()
        check_O(O, O_ref); check_close(LSE, LSE_ref, LSE_ABS)


# --------------------------------------------------------------------------- NEXT-3 pooled-key scorer
@pytest.mark.parametrize("name,kw", [("tiny", {}), ("tiny", dict(H=12, H_kv=4, d=128, C=77, N=21, L_q=9, L_d=3)),
                                     ("llada8k", {}), ("dream16k", {}), ("sparse32k", dict(B=1))])
def test_pooled_scorer(B, name, kw):
    w, inp = _inputs(name, **kw)
    shape = B.Shape.of(w)
    dQ, dK = dev_bf16(inp["Q_dec"]), dev_bf16(inp["Kcache"])
    kbar = B.pool_keys(shape, dK)
    torch.cuda.synchronize()
    kbar_ref = oracle.pooled_keys(inp["Kcache"])
    check_close(kbar, kbar_ref, 1e-5, what="pooled keys")
    got = B.score_chunks_pooled(shape, dQ, kbar)
    torch.cuda.synchronize()
    # both sides score the SAME pooled keys (the GPU's fp32 values, widened exactly): what is compared is the scorer
    ref = oracle.pooled_scores(inp["Q_dec"], kbar.double().cpu().numpy(), w.C, w.L_q)
    check_close(got, ref, 1e-4, what="pooled scores")
    ref_full = oracle.pooled_scores(inp["Q_dec"], kbar_ref, w.C, w.L_q)
    check_close(got, ref_full, 1e-3, what="pooled scores vs fp64 pooled keys")
    # recall of the planted chunks under the cheap scorer (reported, asserted only where the shift is a mean shift)
    ids = B.select_topk(shape, got).cpu().numpy()
    recall = np.mean([len(set(ids[b, g]) & set(inp["planted"][b, g])) / w.K for b in range(w.B) for g in range(w.H_kv)])
    print(f"{name} {kw}: pooled-scorer recall of planted chunks = {recall:.3f}")
    assert recall == 1.0          # the planted shift alpha * mean(q) moves the chunk's MEAN key: the pooled scorer sees it


# --------------------------------------------------------------------------- NEXT-2 chunk-prefill attention
@pytest.mark.parametrize("S,H,H_kv,T,d,splits", [
    (3, 4, 4, 81, 64, [1, 0]),                        # [BOS; c; q; m] with C = 64, L_q = 12, |m| = 4: one ragged tile
    (2, 8, 2, 300, 128, [1, 2, 0]),                   # GQA G = 4: 1200 packed rows per KV head, 3 KV tiles
    (5, 2, 2, 128, 128, [1]),                         # exactly one tile
    (8, 32, 8, 1105, 128, [0, 1]),                    # Fig. 5(a)-like: C = 1024 + BOS + L_q = 64 + |m| = 16, GQA 32/8
])
def test_prefill_attn(B, S, H, H_kv, T, d, splits):
    r = np.random.default_rng(S * 1000 + T)
    Q = W.f32_to_bf16_bits(r.standard_normal((S, H, T, d), dtype=np.float32))
    K = W.f32_to_bf16_bits(r.standard_normal((S, H_kv, T, d), dtype=np.float32))
    V = W.f32_to_bf16_bits(r.standard_normal((S, H_kv, T, d), dtype=np.float32))
    O_ref, LSE_ref = oracle.prefill_attn(Q, K, V)
    ds = B.DenseShape(S, H, H_kv, d, T, T, 0)
    dQ, dK, dV = dev_bf16(Q), dev_bf16(K), dev_bf16(V)
    for n_splits in splits:
        O, LSE = B.prefill_attn(ds, dQ, dK, dV, n_splits=n_splits)
        torch.cuda.synchronize()
        e_o, r_o = check_O(O, O_ref, what=f"prefill O (S={n_splits})")
        check_close(LSE, LSE_ref, LSE_ABS, what=f"prefill LSE (S={n_splits})")
        print(f"prefill S={S} H={H}/{H_kv} T={T} d={d} splits={n_splits}: O max|d| {e_o:.2e} (norm {r_o:.2e})")
