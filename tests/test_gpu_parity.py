"""GPU-vs-oracle parity through the C ABI (include/pdllm.h), element by element on the same seeded
inputs.  Bars (SURVEY 8(c) R12 / BASELINE.json north_star): chunk ids and gather indices bit-exact;
O within 2e-2 + 1e-2|ref| per element and max|d|/max|ref| <= 1e-2; LSE and scores within 1e-3.
"""
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
    w = W.CONFIGS[name]
    if kw:
        w = W.small_variant(w, **kw)
    return w, W.make_inputs(w)


# --------------------------------------------------------------------------- a2 top-K
@pytest.mark.parametrize("rows,N,K", [(4, 8, 2), (32, 16, 4), (128, 64, 8), (5, 33, 33), (3, 1, 1), (7, 100, 1),
                                      (9, 513, 16), (2, 4096, 64), (6, 130, 64)])
def test_topk_random(B, rows, N, K):
    r = np.random.default_rng(rows * 1000 + N + K)
    s = r.standard_normal((1, rows, N)).astype(np.float32)
    shape = B.Shape(1, rows, rows, 128, N, 512, K, 513, 1, 1, 1)
    got = B.select_topk(shape, dev_f32(s))
    check_exact(got, oracle.topk(s, K))


def test_topk_ties_nan_inf(B):
    N, K = 40, 6
    s = np.zeros((1, 6, N), np.float32)
    s[0, 0] = 1.0                                   # all equal: lowest indices win
    s[0, 1, ::3] = 2.0                              # many ties above a floor
    s[0, 2] = np.nan                                # all NaN == all -inf
    s[0, 3] = -np.inf; s[0, 3, [7, 30]] = 0.5       # fewer finite values than K
    s[0, 4] = np.arange(N)[::-1]; s[0, 4, 5] = np.nan; s[0, 4, 0] = np.inf
    s[0, 5] = np.tile([3.0, 1.0], N // 2)
    shape = B.Shape(1, 6, 6, 128, N, 512, K, 513, 1, 1, 1)
    check_exact(B.select_topk(shape, dev_f32(s)), oracle.topk(s, K))


# --------------------------------------------------------------------------- a3 gather indices
@pytest.mark.parametrize("name", ["tiny", "sparse32k"])
def test_gather_idx(B, name):
    w = W.CONFIGS[name]
    keep, ids = W.make_keep(w), W.make_planted(w)
    shape = B.Shape.of(w)
    got = B.gather_idx(shape, dev_i32(ids), dev_i32(keep))
    check_exact(got, oracle.gather_idx(ids, keep, w.N, w.C), "gather_idx")


def test_gather_idx_no_keep(B):
    w = W.CONFIGS["llada8k"]
    ids = W.make_planted(w)
    got = B.gather_idx(B.Shape.of(w), dev_i32(ids), None)
    check_exact(got, oracle.gather_idx(ids, None, w.N, w.C), "gather_idx")


# --------------------------------------------------------------------------- a5 combine
@pytest.mark.parametrize("S,rows,d", [(1, 37, 128), (2, 300, 128), (4, 48, 64), (5, 77, 128), (7, 1000, 128), (33, 40, 128),
                                      (64, 129, 64), (65, 33, 128), (100, 50, 64)])
def test_lse_combine(B, S, rows, d):
    r = np.random.default_rng(S * 7 + rows)
    Op = r.standard_normal((S, rows, d)).astype(np.float32)
    lp = (3.0 * r.standard_normal((S, rows))).astype(np.float32)
    if S > 1:
        lp[0, ::5] = -np.inf                         # an empty split for some rows
        lp[:, 3] = -np.inf                           # a row with nothing at all
        Op[:, 3] = 0.0
    O, LSE = B.lse_combine(dev_f32(Op), dev_f32(lp))
    O_ref, LSE_ref = oracle.lse_combine(Op, lp)
    check_O(O, O_ref, what="combine O")
    check_close(LSE, LSE_ref, 1e-5, what="combine LSE")


# --------------------------------------------------------------------------- a1 scores
@pytest.mark.parametrize("name,kw", [
    ("tiny", {}),
    ("tiny", dict(C=127, L_q=16)),                   # Cp = 128: exactly one full tile
    ("tiny", dict(C=130, N=5, K=2)),                 # Cp = 131: full tile + 3-row tail (16-row TMA box)
    ("tiny", dict(C=200, H=8, H_kv=2, L_q=40, L_d=8)),   # GQA G=4, 160 scoring rows -> 2 M tiles (atomic path)
    ("llada8k", {}),
    ("dream16k", {}),
])
def test_scores(B, name, kw):
    w, inp = _inputs(name, **kw)
    shape = B.Shape.of(w)
    got = B.score_chunks(shape, dev_bf16(inp["Q_dec"]), dev_bf16(inp["Kcache"]))
    ref = oracle.scores(inp["Q_dec"], inp["Kcache"], w.L_q)
    err = check_close(got, ref, SCORE_ABS, what="scores")
    ids = B.select_topk(shape, got)
    check_exact(ids, oracle.topk(ref, w.K))
    if not kw:
        check_exact(ids, inp["planted"], "planted chunks")
    print(f"{name} {kw}: scores max|d| = {err:.2e}")


# --------------------------------------------------------------------------- a3+a4+a5 attention
def _attn_case(B, w, inp, splits, ids=None, scale=None):
    dev = to_device(inp)
    ids = inp["planted"] if ids is None else ids
    shape = shape_of(inp, ids.shape[-1], min(w.L_q, inp["Q_dec"].shape[2]))
    if scale is not None:
        shape = dataclasses.replace(shape, scale=scale)
    O_ref, LSE_ref = oracle.attn(inp["Q_dec"], inp["Kcache"], inp["Vcache"], ids, inp["keep"], inp["K_dec"], inp["V_dec"],
                                 scale=scale)
    gi_ref = oracle.gather_idx(ids, inp["keep"], w.N, w.C)
    for S in splits:
        gi = torch.empty(gi_ref.shape, dtype=torch.int32, device="cuda")
        O, LSE = B.sparse_attn(shape, dev["Q_dec"], dev["Kcache"], dev["Vcache"], dev_i32(ids), dev["keep"],
                               dev["K_dec"], dev["V_dec"], n_splits=S, gather_idx_out=gi)
        torch.cuda.synchronize()
        e_o, r_o = check_O(O, O_ref, what=f"O (S={S})")
        e_l = check_close(LSE, LSE_ref, LSE_ABS, what=f"LSE (S={S})")
        check_exact(gi, gi_ref, "gather_idx")
        print(f"{w.name} S={S}: O max|d| {e_o:.2e} (norm {r_o:.2e}), LSE max|d| {e_l:.2e}")


def test_attn_tiny(B):
    w, inp = _inputs("tiny")
    _attn_case(B, w, inp, [1, 2, 4, 0])


@pytest.mark.parametrize("kw", [
    dict(keep=1.0),                                   # no keep list (NULL)
    dict(K=8, keep=1.0),                              # K = N, full mask: dense attention over the whole prefix
    dict(keep=0.0),                                   # only the BOS of each selected chunk survives (Bk = 1)
    dict(L_q=1, L_d=0),                               # a single query row, L_s = 1
    dict(L_q=100, L_d=101, C=100, keep=0.37),         # ragged everything: L = 201, Bk = 38
    dict(H=8, H_kv=2, L_q=20, L_d=30),                # GQA G=4: 200 packed rows, tiles straddle heads
    dict(B=3, H=6, H_kv=3, d=128, C=96, L_q=8, L_d=24),
])
def test_attn_edges(B, kw):
    w, inp = _inputs("tiny", **kw)
    _attn_case(B, w, inp, [1, 3, 64])


def test_attn_llada8k(B):
    w, inp = _inputs("llada8k")
    _attn_case(B, w, inp, [0, 1, 4])


def test_attn_dream16k_split_sweep(B):
    w, inp = _inputs("dream16k")
    _attn_case(B, w, inp, [1, 2, 3, 5, 8, 20, 64, 0])


def test_attn_large_logits(B):
    """A key with logit ~ +50 above the rest (oracle pin iv) and strongly growing maxima across KV tiles:
    exercises the reference-max update and the O rescale."""
    w, inp = _inputs("tiny", C=300, L_q=64, L_d=64, keep=1.0)
    u = np.zeros(w.d, np.float32); u[::2] = 1.0; u /= np.linalg.norm(u)
    Q = W.bf16_bits_to_f32(inp["Q_dec"]) + 4.0 * u                                # logit = (1/8) * 4 * 20 * ramp
    Kc = W.bf16_bits_to_f32(inp["Kcache"]).copy()
    ramp = np.linspace(0.0, 6.0, w.N * w.Cp, dtype=np.float32).reshape(w.N, w.Cp, 1)
    Kc += (20.0 * ramp * u)[None, None]
    inp["Q_dec"], inp["Kcache"] = W.f32_to_bf16_bits(Q), W.f32_to_bf16_bits(Kc)
    _attn_case(B, w, inp, [1, 2])


# --------------------------------------------------------------------------- the per-step call
def test_step_tiny(B):
    w, inp = _inputs("tiny")
    dev = to_device(inp)
    shape = B.Shape.of(w)
    ref = oracle.step(inp["Q_dec"], inp["Kcache"], inp["Vcache"], inp["keep"], inp["K_dec"], inp["V_dec"], w.K, w.L_q)
    for S in (1, 2, 4):
        out = B.step(shape, dev["Q_dec"], dev["Kcache"], dev["Vcache"], dev["keep"], dev["K_dec"], dev["V_dec"], n_splits=S)
        torch.cuda.synchronize()
        check_close(out["scores"], ref["scores"], SCORE_ABS, what="scores")
        check_exact(out["chunk_ids"], ref["ids"])
        check_O(out["O"], ref["O"])
        check_close(out["LSE"], ref["LSE"], LSE_ABS)


def test_step_sparse32k_full_size_all_heads(B):
    """BASELINE configs[3] at full size in bench.py's launch configuration (n_splits = 0): scores, chunk ids,
    gather indices, O and LSE of ALL 128 (b, head) groups against the oracle's own step (ids from
    oracle.topk(oracle.scores), not from the generator's planted list)."""
    w, inp = _inputs("sparse32k")
    dev = to_device(inp)
    shape = B.Shape.of(w)
    gi = torch.empty((w.B, w.H_kv, w.K * w.Bk), dtype=torch.int32, device="cuda")
    out = B.step(shape, dev["Q_dec"], dev["Kcache"], dev["Vcache"], dev["keep"], dev["K_dec"], dev["V_dec"],
                 n_splits=0, gather_idx_out=gi)
    torch.cuda.synchronize()
    ref = oracle.step(inp["Q_dec"], inp["Kcache"], inp["Vcache"], inp["keep"], inp["K_dec"], inp["V_dec"], w.K, w.L_q)
    check_close(out["scores"], ref["scores"], SCORE_ABS, what="scores")
    check_exact(out["chunk_ids"], ref["ids"], "chunk ids vs oracle top-K")
    check_exact(gi, ref["gather_idx"], "gather_idx")
    check_O(out["O"], ref["O"], what="O (all heads)")
    check_close(out["LSE"], ref["LSE"], LSE_ABS, what="LSE (all heads)")
    check_exact(out["chunk_ids"], inp["planted"], "planted chunks (generator sanity)")


def test_step_host_matches_step(B):
    """pdllm_step_host (pinned host buffers, copies on the stream) returns what pdllm_step computes."""
    w, inp = _inputs("tiny")
    dev = to_device(inp)
    shape = B.Shape.of(w)
    pin = lambda bits: torch.from_numpy(bits.view(np.int16)).view(torch.bfloat16).pin_memory()
    hQ, hK, hV = pin(inp["Q_dec"]), pin(inp["K_dec"]), pin(inp["V_dec"])
    hO = torch.empty((w.B, w.H, w.L, w.d), dtype=torch.bfloat16).pin_memory()
    hL = torch.empty((w.B, w.H, w.L), dtype=torch.float32).pin_memory()
    hI = torch.empty((w.B, w.H_kv, w.K), dtype=torch.int32).pin_memory()
    scratch = torch.empty((B.step_host_scratch_bytes(shape, 2, B.num_sms()),), dtype=torch.uint8, device="cuda")
    B.step_host(shape, hQ, hK, hV, dev["Kcache"], dev["Vcache"], dev["keep"], 2, hO, hL, hI, scratch)      # one stream
    torch.cuda.synchronize()
    hO2, hL2, hI2 = torch.empty_like(hO).pin_memory(), torch.empty_like(hL).pin_memory(), torch.empty_like(hI).pin_memory()
    side = B.SideStream()
    for _ in range(3):                               # with the caller's side stream, back to back on one scratch
        B.step_host(shape, hQ, hK, hV, dev["Kcache"], dev["Vcache"], dev["keep"], 2, hO2, hL2, hI2, scratch, side=side)
    torch.cuda.synchronize()
    assert torch.equal(hO.view(torch.int16), hO2.view(torch.int16)) and torch.equal(hL, hL2) and torch.equal(hI, hI2)
    out = B.step(shape, dev["Q_dec"], dev["Kcache"], dev["Vcache"], dev["keep"], dev["K_dec"], dev["V_dec"], n_splits=2)
    torch.cuda.synchronize()
    assert torch.equal(hO.view(torch.int16), out["O"].cpu().view(torch.int16))
    assert torch.equal(hL, out["LSE"].cpu())
    assert torch.equal(hI, out["chunk_ids"].cpu())


def test_errors(B):
    w, inp = _inputs("tiny", C=300, keep=1.0)        # S_kv = 650: several KV tiles, so 2 splits need scratch
    dev = to_device(inp)
    shape = B.Shape.of(w)
    bad = B.Shape(w.B, w.H, 3, w.d, w.N, w.C, w.K, w.Bk, w.L_q, w.L, w.L_s)       # H % H_kv != 0
    with pytest.raises(B.PdllmError):
        B.select_topk(bad, torch.zeros((1, 3, w.N), device="cuda"))
    ws = torch.empty((16,), dtype=torch.uint8, device="cuda")
    with pytest.raises(B.PdllmError):                                             # workspace too small for 2 splits
        B.sparse_attn(shape, dev["Q_dec"], dev["Kcache"], dev["Vcache"], dev_i32(inp["planted"]), dev["keep"],
                      dev["K_dec"], dev["V_dec"], n_splits=2, workspace=ws)


def test_debug_validate_switch(B, monkeypatch):
    """PDLLM_DEBUG_VALIDATE=1 (include/pdllm.h "DEBUG SWITCH"): malformed chunk ids / keep lists are reported as
    PDLLM_ERR_DATA (-7) with nothing enqueued; well-formed lists pass and give the usual result."""
    w, inp = _inputs("tiny")
    dev = to_device(inp)
    shape = B.Shape.of(w)
    ids = dev_i32(inp["planted"])
    monkeypatch.setenv("PDLLM_DEBUG_VALIDATE", "1")
    O_ref, LSE_ref = oracle.attn(inp["Q_dec"], inp["Kcache"], inp["Vcache"], inp["planted"], inp["keep"], inp["K_dec"], inp["V_dec"])
    O, LSE = B.sparse_attn(shape, dev["Q_dec"], dev["Kcache"], dev["Vcache"], ids, dev["keep"], dev["K_dec"], dev["V_dec"], n_splits=1)
    torch.cuda.synchronize()
    check_O(O, O_ref)

    def expect_data_error(fn):
        with pytest.raises(B.PdllmError, match="-7"):
            fn()

    attn = lambda i, k: B.sparse_attn(shape, dev["Q_dec"], dev["Kcache"], dev["Vcache"], i, k, dev["K_dec"], dev["V_dec"], n_splits=1)
    bad_ids = ids.clone(); bad_ids[0, 1, 0] = w.N                      # chunk id == N
    expect_data_error(lambda: attn(bad_ids, dev["keep"]))
    bad_ids = ids.clone(); bad_ids[0, 0, 1] = -1
    expect_data_error(lambda: B.gather_idx(shape, bad_ids, dev["keep"]))
    k = dev["keep"].clone(); k[0, 2, 3, 0] = 1                         # BOS slot not kept first
    expect_data_error(lambda: attn(ids, k))
    k = dev["keep"].clone(); k[0, 1, 5, w.Bk - 1] = w.C + 1            # slot beyond the chunk
    expect_data_error(lambda: attn(ids, k))
    k = dev["keep"].clone(); k[0, 3, 7, 5] = k[0, 3, 7, 4]             # not strictly ascending
    expect_data_error(lambda: attn(ids, k))
    expect_data_error(lambda: B.step(shape, dev["Q_dec"], dev["Kcache"], dev["Vcache"], k, dev["K_dec"], dev["V_dec"], n_splits=1))
    monkeypatch.setenv("PDLLM_DEBUG_VALIDATE", "0")                    # switch off: the well-formed call is untouched
    O2, _ = attn(ids, dev["keep"])
    torch.cuda.synchronize()
    assert torch.equal(O2.view(torch.int16), O.view(torch.int16))


# --------------------------------------------------------------------------- rare paths of the single-pass softmaxes
def _ramp_inputs(C, L_q, L_d, H, H_kv, d, gain):
    """Keys whose logits grow steeply along the cached sequence (each KV tile, and each 32-column block inside a
    tile, outgrows the running reference max by many octaves): exercises the overflow -> rescale paths."""
    w, inp = _inputs("tiny", C=C, L_q=L_q, L_d=L_d, H=H, H_kv=H_kv, d=d, keep=1.0)
    u = np.zeros(w.d, np.float32); u[::2] = 1.0; u /= np.linalg.norm(u)
    Q = W.bf16_bits_to_f32(inp["Q_dec"]) + 4.0 * u
    Kc = W.bf16_bits_to_f32(inp["Kcache"]).copy()
    ramp = np.linspace(0.0, gain, w.N * w.Cp, dtype=np.float32).reshape(w.N, w.Cp, 1)
    Kc += (20.0 * ramp * u)[None, None]
    inp["Q_dec"], inp["Kcache"] = W.f32_to_bf16_bits(Q), W.f32_to_bf16_bits(Kc)
    return w, inp


@pytest.mark.parametrize("H,H_kv,L_q,L_d,d", [(4, 4, 64, 64, 64), (8, 2, 64, 64, 128), (2, 2, 100, 284, 128)])
def test_attn_growing_logits_all_item_kinds(B, H, H_kv, L_q, L_d, d):
    """pair items (two query tiles share K/V), single items (in-CTA Split-S merge) and GQA packing, each with a
    reference max that has to be raised inside tiles."""
    w, inp = _ramp_inputs(C=300, L_q=L_q, L_d=L_d, H=H, H_kv=H_kv, d=d, gain=6.0)
    _attn_case(B, w, inp, [1, 2, 5])


def test_scores_growing_logits(B):
    """chunk scores when the logits inside every chunk outgrow the chunk's first-tile reference max (redo path)."""
    w, inp = _ramp_inputs(C=700, L_q=128, L_d=8, H=4, H_kv=4, d=128, gain=40.0)
    shape = B.Shape.of(w)
    got = B.score_chunks(shape, dev_bf16(inp["Q_dec"]), dev_bf16(inp["Kcache"]))
    ref = oracle.scores(inp["Q_dec"], inp["Kcache"], w.L_q)
    check_close(got, ref, SCORE_ABS * max(1.0, float(np.abs(ref).max()) / 100.0), what="scores (growing logits)")
    check_exact(B.select_topk(shape, got), oracle.topk(ref, w.K))


@pytest.mark.parametrize("kw", [
    dict(H=4, H_kv=4, d=64, C=500, K=3, keep=1.0, L_q=128, L_d=128),     # d = 64: pair items, 13 KV tiles
    dict(H=2, H_kv=2, d=128, C=640, K=8, keep=1.0, L_q=32, L_d=32),      # one query tile per group: single items, 41 tiles
    dict(H=16, H_kv=2, d=128, C=256, K=4, keep=0.3, L_q=48, L_d=80),     # GQA G = 8: 8 query tiles per group
])
def test_attn_item_shapes(B, kw):
    w, inp = _inputs("tiny", **kw)
    _attn_case(B, w, inp, [0, 1, 3, 7])


def test_step_back_to_back_without_sync(B):
    """200 pdllm_step calls enqueued back to back (no host sync in between, the way a denoising loop runs them),
    with and without the combine kernel: every call must reproduce the first, oracle-checked result bit for bit
    (guards the launch-overlap plumbing: programmatic dependent launch, the work-item counter, workspace reuse)."""
    w, inp = _inputs("tiny", C=300, H=8, H_kv=8, d=128, N=12, K=6, keep=1.0, L_q=64, L_d=192)
    dev = to_device(inp)
    shape = B.Shape.of(w)
    ref = oracle.step(inp["Q_dec"], inp["Kcache"], inp["Vcache"], inp["keep"], inp["K_dec"], inp["V_dec"], w.K, w.L_q)
    for S in (1, 2, 3):
        ws = B.alloc_workspace(shape, S)
        first = B.step(shape, dev["Q_dec"], dev["Kcache"], dev["Vcache"], dev["keep"], dev["K_dec"], dev["V_dec"],
                       n_splits=S, workspace=ws)
        torch.cuda.synchronize()
        check_exact(first["chunk_ids"], ref["ids"])
        check_O(first["O"], ref["O"], what=f"O (S={S})")
        check_close(first["LSE"], ref["LSE"], LSE_ABS)
        O0, L0 = first["O"].clone(), first["LSE"].clone()
        out = dict(scores=first["scores"], chunk_ids=first["chunk_ids"], O=first["O"], LSE=first["LSE"])
        for _ in range(200):
            B.step(shape, dev["Q_dec"], dev["Kcache"], dev["Vcache"], dev["keep"], dev["K_dec"], dev["V_dec"],
                   n_splits=S, workspace=ws, **out)
        torch.cuda.synchronize()
        assert torch.equal(out["O"].view(torch.int16), O0.view(torch.int16)), f"O changed across back-to-back steps (S={S})"
        assert torch.equal(out["LSE"], L0), f"LSE changed across back-to-back steps (S={S})"


def test_step_fig5b_decode_shape(B):
    """The paper's decode-kernel shape (Fig. 5(b)): GQA 32/8, 32 rows per head over ~4K selected KV -- one packed
    query tile per KV group, so the whole call is Split-S (auto split count and the paper's S = 4)."""
    w = W.EXTRA["fig5b"]
    inp = W.make_inputs(w)
    dev = to_device(inp)
    shape = B.Shape.of(w)
    ref = oracle.step(inp["Q_dec"], inp["Kcache"], inp["Vcache"], inp["keep"], inp["K_dec"], inp["V_dec"], w.K, w.L_q)
    for S in (0, 4, 1):
        out = B.step(shape, dev["Q_dec"], dev["Kcache"], dev["Vcache"], dev["keep"], dev["K_dec"], dev["V_dec"], n_splits=S)
        torch.cuda.synchronize()
        check_close(out["scores"], ref["scores"], SCORE_ABS, what="scores")
        check_exact(out["chunk_ids"], ref["ids"])
        check_O(out["O"], ref["O"], what=f"O (S={S})")
        check_close(out["LSE"], ref["LSE"], LSE_ABS, what=f"LSE (S={S})")


@pytest.mark.parametrize("half", [0, 1])
@pytest.mark.parametrize("d", [64, 128])
def test_attn_overflow_in_one_column_half(B, half, d):
    """A query row is shared by two softmax threads (columns 0..63 and 64..127 of every 128-key tile).  Here the
    logits outgrow the reference max, tile after tile, ONLY in the columns of one half: the other half sees nothing
    unusual and has to follow the pair's overflow vote (same reference, same rescale) for the row to come out right."""
    w, inp = _inputs("tiny", C=255, K=4, N=4, keep=1.0, L_q=96, L_d=160, H=4, H_kv=2, d=d)      # K = N: virtual row = cache row
    u = np.zeros(w.d, np.float32); u[::2] = 1.0; u /= np.linalg.norm(u)
    Q = W.bf16_bits_to_f32(inp["Q_dec"]) + 4.0 * u
    Kc = W.bf16_bits_to_f32(inp["Kcache"]).copy()                  # [B, H_kv, N, Cp, d]
    v = np.arange(w.N * w.Cp).reshape(w.N, w.Cp)                   # position in the gathered sequence
    boost = np.where((v % 128) // 64 == half, 12.0 * (v // 128), 0.0).astype(np.float32)        # +12*sqrt(d)/8.. per tile
    Kc += (boost[..., None] * u * (np.sqrt(w.d) / 4.0))[None, None]
    inp["Q_dec"], inp["Kcache"] = W.f32_to_bf16_bits(Q), W.f32_to_bf16_bits(Kc)
    _attn_case(B, w, inp, [1, 2])


@pytest.mark.parametrize("tail", [1, 33, 64, 65, 97, 127])
def test_attn_ragged_tail_widths(B, tail):
    """Last KV tile with `tail` valid keys: 1..64 leaves the second column half of the tile empty, 65..127 masks inside
    it; pair items and a single item (L = 300: three query tiles), with and without splits."""
    L = 300
    S_pre = 2 * 101                                                # K = 2 chunks of C + 1 = 101 kept whole
    L_s = next(x for x in range(L, L + 128) if (S_pre + x) % 128 == tail)
    w, inp = _inputs("tiny", C=100, K=2, keep=1.0, L_q=40, L_d=L_s - 40, H=2, H_kv=2, d=128)
    assert (w.K * (w.C + 1) + w.L) % 128 == tail
    _attn_case(B, w, inp, [1, 2])


# --------------------------------------------------------------------------- paths the ABI accepts that round 1 never ran
@pytest.mark.parametrize("kw", [
    dict(N=80, C=20, K=40, keep=0.5, d=64, L_q=16, L_d=48),                     # K in 33..64: chunk ids in the second id register
    dict(N=70, C=12, K=64, keep=1.0, d=128, H=4, H_kv=2, L_q=16, L_d=40),       # K = 64 (the bound), GQA, no keep list
    dict(N=64, C=30, K=33, keep=0.3, d=128, H=2, H_kv=2, L_q=100, L_d=200),     # K = 33, pair + single items
])
def test_attn_many_chunks(B, kw):
    w, inp = _inputs("tiny", **kw)
    _attn_case(B, w, inp, [1, 3, 0])


@pytest.mark.parametrize("L,L_s", [(32, 96), (96, 32), (1, 200), (130, 7)])
def test_attn_rows_differ_from_decode_kv_rows(B, L, L_s):
    """R8's strict shape: only the L = L_d response rows attend while K_dec / V_dec hold the L_s = L_q + L_d
    query + response rows; and the converse (L_s < L)."""
    big = max(L, L_s)
    w, inp = _inputs("tiny", C=150, K=3, keep=0.6, d=128, H=4, H_kv=2, L_q=16, L_d=big - 16)
    inp["Q_dec"] = np.ascontiguousarray(inp["Q_dec"][:, :, :L])
    inp["K_dec"] = np.ascontiguousarray(inp["K_dec"][:, :, :L_s])
    inp["V_dec"] = np.ascontiguousarray(inp["V_dec"][:, :, :L_s])
    _attn_case(B, w, inp, [1, 2, 0])


@pytest.mark.parametrize("scale", [0.05, 0.3])
def test_attn_explicit_scale(B, scale):
    w, inp = _inputs("tiny", C=200, K=3, keep=1.0, d=128, L_q=40, L_d=120)
    _attn_case(B, w, inp, [1, 2], scale=scale)


def test_step_explicit_scale_and_strict_rows(B):
    """pdllm_step with scale = 0.05 (scores, ids and attention all take it)."""
    w, inp = _inputs("tiny", C=200, H=8, H_kv=4, d=128, L_q=24, L_d=40)
    dev = to_device(inp)
    shape = dataclasses.replace(B.Shape.of(w), scale=0.05)
    ref = oracle.step(inp["Q_dec"], inp["Kcache"], inp["Vcache"], inp["keep"], inp["K_dec"], inp["V_dec"], w.K, w.L_q,
                      scale=0.05)
    out = B.step(shape, dev["Q_dec"], dev["Kcache"], dev["Vcache"], dev["keep"], dev["K_dec"], dev["V_dec"], n_splits=2)
    torch.cuda.synchronize()
    check_close(out["scores"], ref["scores"], SCORE_ABS, what="scores")
    check_exact(out["chunk_ids"], ref["ids"])
    check_O(out["O"], ref["O"])
    check_close(out["LSE"], ref["LSE"], LSE_ABS)


@pytest.mark.parametrize("kw", [
    dict(B=5, H=8, H_kv=8, d=64, N=512, C=31, K=4, L_q=16, L_d=8),     # 40 groups x 512 chunks: 69 units per CTA, runs cross
                                                                       # 64-chunk segments and (b, g) boundaries (N = 512)
    dict(B=2, H=64, H_kv=64, d=128, N=256, C=15, K=4, L_q=8, L_d=8),   # 128 groups x 256 chunks, one 16-row tile per chunk
    dict(B=1, H=12, H_kv=4, d=64, N=2000, C=12, K=5, L_q=100, L_d=4),  # GQA G = 3: 300 scoring rows = 3 M tiles, 81 units per CTA
])
def test_scores_long_cta_runs(B, kw):
    _scores_case(B, kw)


@pytest.mark.parametrize("kw", [
    dict(B=5, H=8, H_kv=8, d=64, N=512, C=128, K=4, L_q=16, L_d=8),     # Cp = 129: one main tile + a one-row tail; 69 chunks per CTA:
                                                                        # tail groups of 4 restart at every 64-chunk segment
    dict(B=1, H=4, H_kv=4, d=128, N=5, C=256, K=2, L_q=40, L_d=8),      # 20 chunks on 20 CTAs: every group is a single chunk
    dict(B=1, H=2, H_kv=2, d=128, N=301, C=128, K=3, L_q=128, L_d=8),   # 602 chunks / 296 CTAs: runs of 2-3 chunks, groups cut short
    dict(B=1, H=6, H_kv=2, d=64, N=23, C=384, K=3, L_q=60, L_d=4),      # GQA G = 3: 180 rows = 2 M tiles (partial M tile), Cp = 385
    dict(B=5, H=8, H_kv=8, d=128, N=64, C=128, K=4, L_q=32, L_d=8),     # 2560 chunks / 296 CTAs: runs of 8-9 = groups of 4, 4, (1)
    dict(B=1, H=1, H_kv=1, d=128, N=1, C=1024, K=1, L_q=16, L_d=8),     # a single chunk
])
def test_scores_one_row_tails_in_groups(B, kw):
    """Chunks of 128 t + 1 rows (C = 2^k): the score kernel takes the one-row tails of up to four consecutive chunks of a
    CTA's run in ONE tile step behind the first of them; the later chunks start their running (max, sum) from that
    row.  Runs that start / end inside a group, single-chunk runs, segment restarts, GQA."""
    _scores_case(B, kw)


@pytest.mark.parametrize("gain", [0.0, 1.0, 40.0])
def test_scores_tail_row_dominates_or_vanishes(B, gain):
    """The last cached row of every second chunk scaled by `gain` along the mean query: with 40 its logit sits far above
    the chunk's other 256 (the chunk's running max then starts from the tail row and never rises), with 0 it is an
    average key; both through the grouped-tail path (Cp = 257) and against the oracle."""
    w, inp = _inputs("tiny", B=2, H=4, H_kv=4, d=128, N=11, C=256, K=2, L_q=48, L_d=8)
    Kc = W.bf16_bits_to_f32(inp["Kcache"]).copy()
    qm = W.bf16_bits_to_f32(inp["Q_dec"])[:, :, :w.L_q].mean(axis=2)           # [B, H, d] (H = H_kv here)
    Kc[:, :, ::2, w.C, :] = gain * qm[:, :, None, :]
    inp["Kcache"] = W.f32_to_bf16_bits(Kc)
    shape = B.Shape.of(w)
    got = B.score_chunks(shape, dev_bf16(inp["Q_dec"]), dev_bf16(inp["Kcache"]))
    ref = oracle.scores(inp["Q_dec"], inp["Kcache"], w.L_q)
    check_close(got, ref, SCORE_ABS * max(1.0, float(np.abs(ref).max()) / 100.0), what="scores (tail rows)")


def _scores_case(B, kw):
    w, inp = _inputs("tiny", **kw)
    shape = B.Shape.of(w)
    got = B.score_chunks(shape, dev_bf16(inp["Q_dec"]), dev_bf16(inp["Kcache"]))
    ref = oracle.scores(inp["Q_dec"], inp["Kcache"], w.L_q)
    check_close(got, ref, SCORE_ABS, what="scores (long CTA runs)")
    check_exact(B.select_topk(shape, got), oracle.topk(ref, w.K))


def test_step_gqa_scores_are_bit_reproducible(B):
    """G*L_q > 128: the chunk-score kernel splits the scoring rows into several M tiles.  In pdllm_step their partial
    scores go through the workspace and are summed in M-tile order by the top-K kernel (no float atomics), so repeated
    steps give bit-identical scores; and they match the oracle."""
    w, inp = _inputs("tiny", B=2, H=14, H_kv=2, d=128, N=24, C=200, K=3, keep=0.5, L_q=100, L_d=28)       # G = 7: 700 rows = 6 M tiles
    dev = to_device(inp)
    shape = B.Shape.of(w)
    ref = oracle.step(inp["Q_dec"], inp["Kcache"], inp["Vcache"], inp["keep"], inp["K_dec"], inp["V_dec"], w.K, w.L_q)
    ws = B.alloc_workspace(shape, 2)
    first = B.step(shape, dev["Q_dec"], dev["Kcache"], dev["Vcache"], dev["keep"], dev["K_dec"], dev["V_dec"], n_splits=2, workspace=ws)
    torch.cuda.synchronize()
    check_close(first["scores"], ref["scores"], SCORE_ABS, what="scores")
    check_exact(first["chunk_ids"], ref["ids"])
    check_O(first["O"], ref["O"]); check_close(first["LSE"], ref["LSE"], LSE_ABS)
    s0 = first["scores"].clone()
    for _ in range(50):
        out = B.step(shape, dev["Q_dec"], dev["Kcache"], dev["Vcache"], dev["keep"], dev["K_dec"], dev["V_dec"], n_splits=2, workspace=ws)
        assert torch.equal(out["scores"].view(torch.int32), s0.view(torch.int32)), "scores changed between identical steps"
    torch.cuda.synchronize()


@pytest.mark.parametrize("where", [150, 300, 640])
@pytest.mark.parametrize("L_q,L_d", [(64, 64), (100, 284)])
def test_attn_logit_jump_beyond_the_soft_range(B, where, L_q, L_d):
    """One cached key whose logit sits ~85 nats (> 100 octaves) above everything the row has seen when its tile comes up:
    the single-pass softmax would form P = 2^120; the row sum trips the hard limit and the tile is redone behind an exact
    row max (the careful pass), with l and O rescaled.  Pair and single items, the key in the 2nd / 3rd / 6th KV tile."""
    w, inp = _inputs("tiny", C=400, N=3, K=3, keep=1.0, L_q=L_q, L_d=L_d, H=2, H_kv=2, d=128)       # K = N: virtual row = cache row
    u = np.zeros(w.d, np.float32); u[::2] = 1.0; u /= np.linalg.norm(u)
    Q = W.bf16_bits_to_f32(inp["Q_dec"]) + 4.0 * u
    Kc = W.bf16_bits_to_f32(inp["Kcache"]).copy().reshape(w.B, w.H_kv, w.N * w.Cp, w.d)
    Kc[:, :, where] += 240.0 * u                                  # logit ~ (1/sqrt(128)) * 4 * 240 = 85 nats
    inp["Q_dec"], inp["Kcache"] = W.f32_to_bf16_bits(Q), W.f32_to_bf16_bits(Kc.reshape(w.B, w.H_kv, w.N, w.Cp, w.d))
    _attn_case(B, w, inp, [1, 2])


@pytest.mark.parametrize("kw", [
    dict(N=64, C=40, K=8, keep=0.5, d=128, H=4, H_kv=4, L_q=32, L_d=64),              # the C4 chunk count
    dict(N=100, C=24, K=33, keep=1.0, d=64, H=4, H_kv=2, L_q=16, L_d=40),             # ragged 4th id register, K > 32
    dict(N=128, C=16, K=5, keep=1.0, d=128, H=14, H_kv=2, L_q=40, L_d=8),             # the fold's bound; G*L_q = 280: score partials
    dict(N=129, C=16, K=5, keep=1.0, d=128, H=2, H_kv=2, L_q=16, L_d=8),              # just beyond it: the top-K kernel runs
    dict(N=1, C=300, K=1, keep=0.3, d=128, H=2, H_kv=1, L_q=8, L_d=24),               # one chunk
])
def test_step_topk_inside_attention_matches_topk_kernel(B, kw):
    """pdllm_step chooses the chunks inside the attention kernel when N <= 128 (a2 folded into a4); with stage events
    or a gather-index export the separate top-K kernel runs.  Both must give the oracle's ids and bit-identical
    scores, ids, O and LSE -- also with exact score ties (duplicated chunks), which go to the lower index."""
    w, inp = _inputs("tiny", **kw)
    if w.N >= 8:                                                  # chunks 5 and 6 become copies of 2 and 1: exact ties
        for name in ("Kcache", "Vcache"):
            inp[name][:, :, 5] = inp[name][:, :, 2]
            inp[name][:, :, 6] = inp[name][:, :, 1]
    dev = to_device(inp)
    shape = B.Shape.of(w)
    ref = oracle.step(inp["Q_dec"], inp["Kcache"], inp["Vcache"], inp["keep"], inp["K_dec"], inp["V_dec"], w.K, w.L_q)
    args = (shape, dev["Q_dec"], dev["Kcache"], dev["Vcache"], dev["keep"], dev["K_dec"], dev["V_dec"])
    for S in (1, 3):
        ws = B.alloc_workspace(shape, S)
        folded = B.step(*args, n_splits=S, workspace=ws)
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(5)]
        for e in ev:
            e.record()
        apart = B.step(*args, n_splits=S, workspace=ws, events=ev)
        gi_ref = oracle.gather_idx(ref["ids"], inp["keep"], w.N, w.C)
        gidx = torch.empty(gi_ref.shape, dtype=torch.int32, device="cuda")
        exported = B.step(*args, n_splits=S, workspace=ws, gather_idx_out=gidx)
        torch.cuda.synchronize()
        check_exact(folded["chunk_ids"], ref["ids"])
        check_close(folded["scores"], ref["scores"], SCORE_ABS, what="scores")
        check_O(folded["O"], ref["O"]); check_close(folded["LSE"], ref["LSE"], LSE_ABS)
        for other, what in ((apart, "stage events"), (exported, "gather export")):
            assert torch.equal(folded["chunk_ids"], other["chunk_ids"]), what
            assert torch.equal(folded["scores"].view(torch.int32), other["scores"].view(torch.int32)), what
            assert torch.equal(folded["O"].view(torch.int16), other["O"].view(torch.int16)), what
            assert torch.equal(folded["LSE"].view(torch.int32), other["LSE"].view(torch.int32)), what
        check_exact(gidx, gi_ref, "gather_idx")
