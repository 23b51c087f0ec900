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


# --------------------------------------------------------------------------- NEXT-1 token scores + top-B
# |d| <= 1e-4 |ref| + 1e-6 * G*L_q: e is a sum of <= G*L_q fp32 exponentials (relative error ~3e-6 each: ex2.approx /
# the degree-4 polynomial) taken against a row log-mass that is itself good to ~1e-6
def _check_e(got, ref, rows, what):
    g = got.double().cpu().numpy()
    lim = 1e-4 * np.abs(ref) + 1e-6 * rows
    worst = float((np.abs(g - ref) - lim).max())
    assert np.isfinite(g).all() and worst <= 0, f"{what}: gate exceeded by {worst:.3e}"
    np.testing.assert_allclose(g.sum(-1), rows, rtol=2e-5, err_msg=f"{what}: a chunk's slots must sum to G*L_q")


TOKEN_CASES = [
    ("tiny", dict(token_alpha=24.0)),                                           # C1
    ("tiny", dict(C=130, N=5, K=2, keep=0.3, token_alpha=24.0)),                # full tile + 3-row tail
    ("tiny", dict(C=200, H=8, H_kv=2, L_q=40, L_d=8, keep=0.25, token_alpha=40.0)),   # GQA: 160 scoring rows = 2 M tiles
    ("dream16k", dict(token_gamma=3.0)),                                        # C3: 896 scoring rows = 7 M tiles
    ("sparse32k", dict(token_gamma=4.0)),                                       # C4 at full size
]


@pytest.mark.parametrize("name,kw", TOKEN_CASES)
def test_token_scores_and_topb(B, name, kw):
    w, inp = _inputs(name, **kw)
    shape = B.Shape.of(w)
    dQ, dK = dev_bf16(inp["Q_dec"]), dev_bf16(inp["Kcache"])
    e = B.score_tokens(shape, dQ, dK)
    torch.cuda.synchronize()
    e_ref = oracle.token_scores(inp["Q_dec"], inp["Kcache"], w.L_q)
    _check_e(e, e_ref, w.G * w.L_q, f"token scores {name}")
    keep = B.select_topb(shape, e)
    torch.cuda.synchronize()
    # the selection rule itself, decided on the same values on both sides (the GPU's fp32 scores, widened exactly)
    check_exact(keep, oracle.topb(e.double().cpu().numpy(), w.Bk), "top-B of the GPU's scores")
    # the planted tokens leave a clear gap (asserted on the oracle's scores), so the list is also the fp64 oracle's
    keep_ref = oracle.topb(e_ref, w.Bk)
    kept = np.take_along_axis(e_ref, keep_ref[..., 1:].astype(np.int64), -1).min(-1)
    mask = np.ones(e_ref.shape, bool); np.put_along_axis(mask, keep_ref.astype(np.int64), False, -1)
    dropped = np.where(mask, e_ref, -np.inf).max(-1)
    # >= 1e-3 relative: a hundred times the fp32 error of a score (<= 1e-5 relative, see _check_e)
    assert ((kept - dropped) / dropped).min() >= 1e-3, "planted-token gap too small for a bit-exact comparison"
    check_exact(keep, keep_ref, "token_keep_idx vs the oracle")
    check_exact(keep, inp["keep"], "planted tokens (generator sanity)")


@pytest.mark.parametrize("kw", [
    dict(B=5, H=8, H_kv=8, d=64, N=512, C=128, K=4, L_q=16, L_d=8),     # Cp = 129: 69 chunks per CTA, runs cross (b, g) boundaries
    dict(B=1, H=2, H_kv=2, d=128, N=301, C=128, K=3, L_q=128, L_d=8),   # 602 chunks / 296 CTAs: runs of 2-3, groups cut short
    dict(B=1, H=6, H_kv=2, d=64, N=23, C=384, K=3, L_q=60, L_d=4),      # GQA G = 3: 180 rows = 2 M tiles (partials), Cp = 385
    dict(B=1, H=4, H_kv=4, d=128, N=5, C=256, K=2, L_q=40, L_d=8),      # 20 chunks on 20 CTAs: every group a single chunk
    dict(B=1, H=1, H_kv=1, d=128, N=1, C=1024, K=1, L_q=16, L_d=8),     # a single chunk
    dict(B=5, H=8, H_kv=8, d=128, N=64, C=128, K=4, L_q=32, L_d=8),     # runs of 8-9 chunks = groups of 4, 4, (1)
])
def test_token_scores_one_row_tails_in_groups(B, kw):
    """Chunks of 128 t + 1 rows: the token kernel takes the tail slots of up to four consecutive chunks of a CTA's run in
    one tile step, each against its own chunk's row log-masses.  Every slot of every chunk against the oracle."""
    w, inp = _inputs("tiny", **kw)
    shape = B.Shape.of(w)
    e = B.score_tokens(shape, dev_bf16(inp["Q_dec"]), dev_bf16(inp["Kcache"]))
    torch.cuda.synchronize()
    _check_e(e, oracle.token_scores(inp["Q_dec"], inp["Kcache"], w.L_q), w.G * w.L_q, "token scores (grouped tails)")


def test_topb_ties_nan_inf(B):
    C, Bk = 40, 7
    e = np.zeros((1, 1, 7, C + 1), np.float32)
    e[0, 0, 0] = 1.0                                   # all equal: lowest slots win
    e[0, 0, 1, 2::3] = 2.0                             # many ties above a floor
    e[0, 0, 2] = np.nan                                # all NaN == all -inf
    e[0, 0, 3] = -np.inf; e[0, 0, 3, [7, 30]] = 0.5    # fewer finite values than Bk - 1
    e[0, 0, 4] = np.arange(C + 1)[::-1]; e[0, 0, 4, 5] = np.nan; e[0, 0, 4, 40] = np.inf
    e[0, 0, 5] = np.tile([3.0, -0.0, 0.0, 1.0], 11)[: C + 1]                    # -0 ties with +0
    e[0, 0, 6] = np.random.default_rng(0).standard_normal(C + 1); e[0, 0, 6, 0] = 100.0     # BOS kept whatever its score
    for bk in (1, 2, Bk, C, C + 1):
        shape = B.Shape(1, 1, 1, 128, 7, C, 1, bk, 1, 1, 1)
        check_exact(B.select_topb(shape, dev_f32(e)), oracle.topb(e, bk), f"top-B Bk={bk}")


@pytest.mark.parametrize("C,Bk,chunks", [(512, 129, 64), (1024, 513, 16), (2047, 100, 8), (8191, 4000, 3), (5, 3, 200),
                                           # the warp-per-chunk kernel's size classes (C <= 128 / 512 / 1024) and the first size beyond
                                           # (taken from 1024 chunks on)
                                           (128, 64, 1030), (129, 2, 1027), (512, 129, 1100), (513, 513, 1024), (1024, 1025, 1025),
                                           (1024, 257, 1031), (1025, 300, 1024), (31, 32, 2000), (128, 64, 9), (513, 100, 1023)])
def test_topb_random(B, C, Bk, chunks):
    r = np.random.default_rng(C + Bk)
    e = r.standard_normal((1, 1, chunks, C + 1)).astype(np.float32)
    e[0, 0, ::2] = np.round(e[0, 0, ::2] * 4) / 4      # half of the chunks on a coarse grid: many exact ties
    shape = B.Shape(1, 1, 1, 128, chunks, C, 1, Bk, 1, 1, 1)
    check_exact(B.select_topb(shape, dev_f32(e)), oracle.topb(e, Bk), "top-B")


def test_step_with_device_produced_keep_list(B):
    """The list pdllm_select_topb writes is what pdllm_step consumes: score tokens -> top-B -> pdllm_step, against the
    oracle run with the oracle's own list."""
    w, inp = _inputs("tiny", C=150, H=8, H_kv=4, d=128, N=10, K=3, keep=0.4, L_q=24, L_d=40, token_alpha=40.0)
    dev = to_device(inp)
    shape = B.Shape.of(w)
    keep = B.select_topb(shape, B.score_tokens(shape, dev["Q_dec"], dev["Kcache"]))
    out = B.step(shape, dev["Q_dec"], dev["Kcache"], dev["Vcache"], keep, dev["K_dec"], dev["V_dec"], n_splits=2)
    torch.cuda.synchronize()
    keep_ref = oracle.topb(oracle.token_scores(inp["Q_dec"], inp["Kcache"], w.L_q), w.Bk)
    check_exact(keep, keep_ref, "keep list")
    ref = oracle.step(inp["Q_dec"], inp["Kcache"], inp["Vcache"], keep_ref, inp["K_dec"], inp["V_dec"], w.K, w.L_q)
    check_exact(out["chunk_ids"], ref["ids"])
    check_O(out["O"], ref["O"]); check_close(out["LSE"], ref["LSE"], LSE_ABS)


# --------------------------------------------------------------------------- NEXT-4 the paper's Fig. 5(b) decode shapes
@pytest.mark.parametrize("name", ["fig5b_8k", "fig5b_16k", "fig5b_32k"])
def test_fig5b_strict_decode_shapes_full_size(B, name):
    """P:189-193 / Fig. 5(b): L = L_d = 32 response rows per head (R8 strict: the cached query rows sit in K_dec /
    V_dec, L_s = L_q + L_d = 96), GQA 32/8 (one packed 128-row query tile per KV head), dense-selected KV of 8K-32K
    tokens: the static-selection flow -- scores and top-K from the query window, then attention with the paper's
    S = 4 and the automatic split count, through the gather path and through the compact cache (TMA tiles)."""
    w = W.EXTRA[name]
    inp = W.make_inputs(w)
    dev = to_device(inp)
    shape = B.Shape.of(w)
    assert (shape.L, shape.L_s, shape.H // shape.H_kv * shape.L) == (32, 96, 128)
    sc = B.score_chunks(shape, dev_bf16(inp["Q_score"]), dev["Kcache"])
    ids = B.select_topk(shape, sc)
    torch.cuda.synchronize()
    sc_ref = oracle.scores(inp["Q_score"], inp["Kcache"], w.L_q)
    check_close(sc, sc_ref, SCORE_ABS, what="scores")
    ids_ref = oracle.topk(sc_ref, w.K)
    check_exact(ids, ids_ref, "chunk ids")
    O_ref, LSE_ref = oracle.attn(inp["Q_dec"], inp["Kcache"], inp["Vcache"], ids_ref, None, inp["K_dec"], inp["V_dec"])
    for S in (0, 4):
        O, LSE = B.sparse_attn(shape, dev["Q_dec"], dev["Kcache"], dev["Vcache"], ids, None, dev["K_dec"], dev["V_dec"], n_splits=S)
        torch.cuda.synchronize()
        e_o, r_o = check_O(O, O_ref, what=f"O (S={S})")
        check_close(LSE, LSE_ref, LSE_ABS, what=f"LSE (S={S})")
        print(f"{name} gather S={S} (auto={B.auto_splits(shape, B.num_sms())}): O max|d| {e_o:.2e} (norm {r_o:.2e})")
    Kc, Vc = B.compact_kv(shape, dev["Kcache"], dev["Vcache"], ids, None)
    ds = B.DenseShape.static_of(shape)
    for S in (0, 4):
        O, LSE = B.static_attn(ds, dev["Q_dec"], Kc, Vc, dev["K_dec"], dev["V_dec"], n_splits=S)
        torch.cuda.synchronize()
        check_O(O, O_ref, what=f"static O (S={S})")
        check_close(LSE, LSE_ref, LSE_ABS, what=f"static LSE (S={S})")
