"""Pins for oracle steps 3-6 (attention, Split-S, LSE combine) against what the paper and
the mathematics fix (SURVEY 8(c) "What pins each part").  CPU only.

Nothing here retypes the oracle's loops: the comparators are a separately coded numpy
dense attention, torch's SDPA in fp64, scipy's logsumexp, closed forms and a pure-Python
brute force.
"""
import itertools
import math

import numpy as np
import pytest
import torch
from scipy.special import logsumexp

from oracle import oracle
from paper_2606_10537_b200 import workloads as W

TOL = 1e-12


def rand_case(seed, B=2, H=4, H_kv=2, d=8, N=5, C=6, K=3, Bk=4, L=7, L_s=3, sigma=1.0):
    """Small random problem with all dimensions distinct (so a transposed operand or a
    swapped index cannot go unnoticed)."""
    r = np.random.default_rng(seed)
    bf = lambda *s: W.f32_to_bf16_bits((sigma * r.standard_normal(s)).astype(np.float32))
    Cp = C + 1
    keep = None
    if Bk != Cp:
        keep = np.zeros((B, H_kv, N, Bk), np.int32)
        for idx in np.ndindex(B, H_kv, N):
            keep[idx][1:] = np.sort(r.choice(np.arange(1, Cp), Bk - 1, replace=False))
    ids = np.stack([np.sort(r.choice(N, K, replace=False)) for _ in range(B * H_kv)]).reshape(B, H_kv, K).astype(np.int32)
    return dict(Q_dec=bf(B, H, L, d), Kcache=bf(B, H_kv, N, Cp, d), Vcache=bf(B, H_kv, N, Cp, d),
                K_dec=bf(B, H_kv, L_s, d), V_dec=bf(B, H_kv, L_s, d), keep=keep, ids=ids)


def concat_numpy(c, b, g):
    """[selected prefix rows under keep || decode rows] for KV head (b,g), by fancy indexing."""
    Kc = oracle.bf16_to_f64(c["Kcache"][b, g]); Vc = oracle.bf16_to_f64(c["Vcache"][b, g])
    N, Cp, d = Kc.shape
    rows = []
    for n in c["ids"][b, g]:
        slots = np.arange(Cp) if c["keep"] is None else c["keep"][b, g, n]
        rows += [n * Cp + s for s in slots]
    Kx = np.concatenate([Kc.reshape(N * Cp, d)[rows], oracle.bf16_to_f64(c["K_dec"][b, g])])
    Vx = np.concatenate([Vc.reshape(N * Cp, d)[rows], oracle.bf16_to_f64(c["V_dec"][b, g])])
    return Kx, Vx


def dense_numpy(q, Kx, Vx, scale):
    """Separately coded dense softmax attention: matrix form, scipy logsumexp."""
    z = scale * (q @ Kx.T)
    lse = logsumexp(z, axis=1)
    return np.exp(z - lse[:, None]) @ Vx, lse


def run(c, **kw):
    return oracle.attn(c["Q_dec"], c["Kcache"], c["Vcache"], c["ids"], c["keep"], c["K_dec"], c["V_dec"], **kw)


def test_full_selection_equals_dense_attention_over_whole_prefix():
    # NS / P:116: K = N with a full mask must equal dense attention over the whole cached prefix.
    c = rand_case(1, N=4, K=4, C=5, Bk=6)
    c["ids"] = np.tile(np.arange(4, dtype=np.int32), (2, 2, 1))
    O, LSE = run(c)
    B, H, L, d = c["Q_dec"].shape
    G = H // c["Kcache"].shape[1]
    for b, h in np.ndindex(B, H):
        g = h // G
        Kall = np.concatenate([oracle.bf16_to_f64(c["Kcache"][b, g]).reshape(-1, d), oracle.bf16_to_f64(c["K_dec"][b, g])])
        Vall = np.concatenate([oracle.bf16_to_f64(c["Vcache"][b, g]).reshape(-1, d), oracle.bf16_to_f64(c["V_dec"][b, g])])
        o, lse = dense_numpy(oracle.bf16_to_f64(c["Q_dec"][b, h]), Kall, Vall, 1 / math.sqrt(d))
        np.testing.assert_allclose(O[b, h], o, rtol=0, atol=TOL)
        np.testing.assert_allclose(LSE[b, h], lse, rtol=0, atol=TOL)


@pytest.mark.parametrize("Bk", [4, 7])
def test_matches_dense_numpy_and_torch_sdpa_on_explicit_concat(Bk):
    c = rand_case(2, Bk=Bk)
    O, LSE, P = run(c, want_P=True)
    B, H, L, d = c["Q_dec"].shape
    G = H // c["Kcache"].shape[1]
    np.testing.assert_allclose(P.sum(-1), 1.0, rtol=0, atol=TOL)          # softmax rows sum to 1
    assert (P >= 0).all()
    for b, h in np.ndindex(B, H):
        Kx, Vx = concat_numpy(c, b, h // G)
        q = oracle.bf16_to_f64(c["Q_dec"][b, h])
        o, lse = dense_numpy(q, Kx, Vx, 1 / math.sqrt(d))
        np.testing.assert_allclose(O[b, h], o, rtol=0, atol=TOL)
        np.testing.assert_allclose(LSE[b, h], lse, rtol=0, atol=TOL)
        t = torch.nn.functional.scaled_dot_product_attention(
            torch.from_numpy(q)[None], torch.from_numpy(Kx)[None], torch.from_numpy(Vx)[None])
        np.testing.assert_allclose(O[b, h], t[0].numpy(), rtol=0, atol=TOL)


def test_gqa_maps_consecutive_query_heads_to_one_kv_head():
    # R4: kv(h) = h // G.  Heads 0,1 must read KV head 0 and heads 2,3 KV head 1.
    c = rand_case(3, B=1, H=4, H_kv=2)
    O, _ = run(c)
    for h in range(4):
        Kx, Vx = concat_numpy(c, 0, h // 2)
        o, _ = dense_numpy(oracle.bf16_to_f64(c["Q_dec"][0, h]), Kx, Vx, 1 / math.sqrt(8))
        np.testing.assert_allclose(O[0, h], o, rtol=0, atol=TOL)
    Kx_wrong, Vx_wrong = concat_numpy(c, 0, 1)
    o_wrong, _ = dense_numpy(oracle.bf16_to_f64(c["Q_dec"][0, 1]), Kx_wrong, Vx_wrong, 1 / math.sqrt(8))
    assert np.abs(O[0, 1] - o_wrong).max() > 1e-3


def test_closed_forms():
    c = rand_case(4)
    B, H, L, d = c["Q_dec"].shape
    S_kv = c["ids"].shape[-1] * c["keep"].shape[-1] + c["K_dec"].shape[2]
    # Q = 0  =>  uniform softmax: O = mean of the concatenated V rows, LSE = log S_kv
    z = dict(c, Q_dec=np.zeros_like(c["Q_dec"]))
    O, LSE = run(z)
    np.testing.assert_allclose(LSE, math.log(S_kv), rtol=0, atol=TOL)
    for b, h in np.ndindex(B, H):
        _, Vx = concat_numpy(c, b, h // 2)
        np.testing.assert_allclose(O[b, h], np.tile(Vx.mean(0), (L, 1)), rtol=0, atol=TOL)
    # all V rows equal v  =>  O = v whatever the logits
    v = W.f32_to_bf16_bits(np.linspace(-1, 1, d, dtype=np.float32))
    same = dict(c, Vcache=np.broadcast_to(v, c["Vcache"].shape).copy(), V_dec=np.broadcast_to(v, c["V_dec"].shape).copy())
    O, _ = run(same)
    np.testing.assert_allclose(O, np.broadcast_to(oracle.bf16_to_f64(v), O.shape), rtol=0, atol=1e-13)
    # explicit scale is honoured: scale = 0 is the uniform case again
    O0, LSE0 = run(c, scale=0.0)
    np.testing.assert_allclose(LSE0, math.log(S_kv), rtol=0, atol=TOL)


def test_one_dominant_key_returns_its_value_row():
    # one decode key aligned with q and scaled so that its logit is ~ +50 above the rest
    c = rand_case(5, B=1, H=1, H_kv=1, L=1, sigma=0.05)
    q = oracle.bf16_to_f64(c["Q_dec"][0, 0, 0])
    big = (50.0 * math.sqrt(8) / (q @ q)) * q
    c["K_dec"][0, 0, 1] = W.f32_to_bf16_bits(big.astype(np.float32))
    O, LSE = run(c)
    np.testing.assert_allclose(O[0, 0, 0], oracle.bf16_to_f64(c["V_dec"][0, 0, 1]), rtol=0, atol=1e-15 + 1e-13)
    kq = oracle.bf16_to_f64(c["K_dec"][0, 0, 1]) @ q / math.sqrt(8)
    assert abs(LSE[0, 0, 0] - kq) < 1e-12


def test_invariant_under_permutation_of_chunk_ids_and_monotone_lse():
    c = rand_case(6)
    O, LSE = run(c)
    p = dict(c, ids=c["ids"][:, :, ::-1].copy())           # same set, other concatenation order
    Op, LSEp = run(p)
    np.testing.assert_allclose(Op, O, rtol=0, atol=TOL)
    np.testing.assert_allclose(LSEp, LSE, rtol=0, atol=TOL)
    # adding a chunk can only add attention mass: LSE strictly grows
    extra = np.array([[sorted(set(range(5)) - set(c["ids"][b, g]))[0] for g in range(2)] for b in range(2)], np.int32)
    more = dict(c, ids=np.concatenate([c["ids"], extra[..., None]], -1))
    _, LSEm = run(more)
    assert (LSEm > LSE).all()
    # a duplicated chunk id is a literal double concatenation (R16): its rows count twice
    dup = dict(c, ids=np.concatenate([c["ids"], c["ids"][..., :1]], -1))
    _, LSEd = run(dup)
    assert (LSEd > LSE).all() and (LSEd < LSE + math.log(2) + 1e-12).all()


def test_brute_force_tiny_every_term_written_out():
    # B = H = 1, d = 3, S_kv = 2*2 + 2 = 6, pure Python floats
    c = rand_case(7, B=1, H=1, H_kv=1, d=3, N=3, C=2, K=2, Bk=2, L=2, L_s=2)
    O, LSE, P = run(c, want_P=True)
    f = lambda a: [[float(x) for x in row] for row in oracle.bf16_to_f64(a)]
    Kc, Vc = [f(c["Kcache"][0, 0, n]) for n in range(3)], [f(c["Vcache"][0, 0, n]) for n in range(3)]
    keys, vals = [], []
    for k in range(2):
        n = int(c["ids"][0, 0, k])
        for t in range(2):
            slot = int(c["keep"][0, 0, n, t])
            keys.append(Kc[n][slot]); vals.append(Vc[n][slot])
    keys += f(c["K_dec"][0, 0]); vals += f(c["V_dec"][0, 0])
    assert len(keys) == 6
    for i, q in enumerate(f(c["Q_dec"][0, 0])):
        s = [sum(q[x] * k[x] for x in range(3)) / math.sqrt(3) for k in keys]
        den = sum(math.exp(x) for x in s)
        p = [math.exp(x) / den for x in s]
        for j in range(6):
            assert abs(P[0, 0, i, j] - p[j]) < 1e-14
        for x in range(3):
            assert abs(O[0, 0, i, x] - sum(p[j] * vals[j][x] for j in range(6))) < 1e-14
        assert abs(LSE[0, 0, i] - math.log(den)) < 1e-14


def test_bos_row_of_every_selected_chunk_is_attended_once():
    # BOS is a real cached token (slot 0).  Put all the attention mass on BOS keys.
    c = rand_case(8, B=1, H=1, H_kv=1, L=1, K=2, sigma=0.05)
    q = oracle.bf16_to_f64(c["Q_dec"][0, 0, 0])
    big = W.f32_to_bf16_bits(((40.0 * math.sqrt(8) / (q @ q)) * q).astype(np.float32))
    c["Kcache"][0, 0, :, 0, :] = big                       # every chunk's BOS key
    _, _, P = run(c, want_P=True)
    Bk = c["keep"].shape[-1]
    mass = P[0, 0, 0].reshape(-1)[[0, Bk]]
    np.testing.assert_allclose(mass, 0.5, atol=1e-9)         # two selected chunks -> two BOS rows share the mass


@pytest.mark.parametrize("S", [1, 2, 3, 4, 7, 64, 1000])
def test_split_s_is_an_exact_reassociation(S):
    # partial outputs merged by log-sum-exp; the result must not depend on S.
    # S = 64 and 1000 exceed S_kv = 15: most ranges are empty (R10).
    c = rand_case(9)
    O1, LSE1 = run(c)
    Os, LSEs = run(c, n_splits=S)
    np.testing.assert_allclose(Os, O1, rtol=0, atol=TOL)
    np.testing.assert_allclose(LSEs, LSE1, rtol=0, atol=TOL)


def test_lse_combine_alone():
    r = np.random.default_rng(10)
    S, rows, d = 5, 11, 4
    Op = r.standard_normal((S, rows, d)); lp = 3 * r.standard_normal((S, rows))
    lp[2] = -np.inf                                        # an empty split
    lp[:, 4] = -np.inf                                     # a row with no mass at all
    O, LSE = oracle.lse_combine(Op, lp)
    with np.errstate(divide="ignore", invalid="ignore"):
        ref_lse = logsumexp(lp, axis=0)
        w = np.exp(lp - ref_lse)
    w[:, 4] = 0.0
    np.testing.assert_allclose(LSE, ref_lse, rtol=0, atol=TOL)
    np.testing.assert_allclose(O, (w[..., None] * np.where(np.isfinite(lp)[..., None], Op, 0.0)).sum(0), rtol=0, atol=TOL)
    assert LSE[4] == -np.inf and (O[4] == 0).all()
    # combining a single partial is the identity
    O1, L1 = oracle.lse_combine(Op[:1], lp[:1])
    np.testing.assert_array_equal(O1[np.isfinite(lp[0])], Op[0][np.isfinite(lp[0])])
    np.testing.assert_array_equal(L1, lp[0])


def test_head_mask_samples_heads_without_changing_them():
    c = rand_case(11)
    O, LSE = run(c)
    hm = np.zeros((2, 4), np.uint8); hm[1, 2] = 1
    Om, Lm = run(c, head_mask=hm)
    np.testing.assert_array_equal(Om[1, 2], O[1, 2])
    assert np.isnan(Om[0]).all() and np.isnan(Lm[1, 3]).all()
