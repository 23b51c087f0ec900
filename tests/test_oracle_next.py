"""Pins of the oracle functions for the rows after the hot path (oracle/pdllm_oracle_next.c):
token eviction scores + top-B (NEXT-1), chunk-prefill attention (NEXT-2), compact cache + pooled-key scorer (NEXT-3).
Each pin is something other than the function itself: closed forms, invariants, brute force with every term written
out, subset enumeration, a separately coded numpy / library form, or a special case that reduces to an oracle routine
that is pinned elsewhere.  No GPU."""
import itertools

import numpy as np
import pytest
import torch

from oracle import oracle
from paper_2606_10537_b200 import workloads as W


def bits(x):
    return W.f32_to_bf16_bits(np.asarray(x, np.float32))


def f64(b):
    return oracle.bf16_to_f64(b)


def rand_case(seed, B=2, H=4, H_kv=2, d=16, N=3, C=9, L_q=5, sigma=1.0):
    r = np.random.default_rng(seed)
    Q = bits(sigma * r.standard_normal((B, H, L_q + 2, d)))
    Kc = bits(sigma * r.standard_normal((B, H_kv, N, C + 1, d)))
    return Q, Kc


# --------------------------------------------------------------------------- NEXT-1 token scores (Eq. 5; R22)
def test_token_scores_columns_sum_to_number_of_scoring_rows():
    """Each scoring row spends a softmax mass of exactly 1 inside the chunk: the slots of a chunk sum to G * L_q."""
    Q, Kc = rand_case(1)
    e = oracle.token_scores(Q, Kc, 5)
    np.testing.assert_allclose(e.sum(-1), 2 * 5, rtol=0, atol=1e-12)
    assert (e > 0).all()


def test_token_scores_zero_queries_give_uniform_mass():
    Q, Kc = rand_case(2)
    e = oracle.token_scores(np.zeros_like(Q), Kc, 5)
    np.testing.assert_allclose(e, 2 * 5 / 10.0, rtol=0, atol=1e-13)


def test_token_scores_matrix_form_with_library_softmax():
    """Separately coded: scipy softmax over the chunk axis of the logit matrix, summed over the group's rows."""
    from scipy.special import softmax
    Q, Kc = rand_case(3, B=1, H=6, H_kv=2, d=8, N=4, C=12, L_q=3)
    L_q, scale = 3, 0.37
    e = oracle.token_scores(Q, Kc, L_q, scale=scale)
    q, k = f64(Q)[:, :, :L_q], f64(Kc)
    for g in range(2):
        rows = q[0, 3 * g:3 * g + 3].reshape(-1, 8)                        # the G * L_q rows of group g
        for n in range(4):
            p = softmax(scale * rows @ k[0, g, n].T, axis=1)
            np.testing.assert_allclose(e[0, g, n], p.sum(0), rtol=1e-12, atol=1e-14)


def test_token_scores_brute_force_every_term():
    Q, Kc = rand_case(4, B=1, H=2, H_kv=1, d=3, N=2, C=3, L_q=2)
    e = oracle.token_scores(Q, Kc, 2, scale=0.5)
    q, k = f64(Q), f64(Kc)
    for n in range(2):
        want = [0.0] * 4
        for h in range(2):
            for i in range(2):
                z = [0.5 * sum(q[0, h, i, c] * k[0, 0, n, j, c] for c in range(3)) for j in range(4)]
                tot = sum(np.exp(v) for v in z)
                for j in range(4):
                    want[j] += np.exp(z[j]) / tot
        np.testing.assert_allclose(e[0, 0, n], want, rtol=1e-13)


def test_token_scores_reduce_to_the_chunk_score_for_one_row():
    """One scoring row (G = L_q = 1): Attn(q, c_j) = exp(scale q.k_j - log-mass), and the log-mass of the chunk is
    exactly the R1 chunk score that oracle_scores computes (pinned in test_oracle_scores_topk.py)."""
    Q, Kc = rand_case(5, B=2, H=3, H_kv=3, d=16, N=4, C=20, L_q=1)
    e = oracle.token_scores(Q, Kc, 1)
    sc = oracle.scores(Q, Kc, 1)
    z = np.einsum("bhd,bhnjd->bhnj", f64(Q)[:, :, 0], f64(Kc)) / np.sqrt(16)
    np.testing.assert_allclose(e, np.exp(z - sc[..., None]), rtol=1e-12)


def test_token_scores_use_only_the_scoring_rows_and_the_right_kv_head():
    Q, Kc = rand_case(6, B=1, H=4, H_kv=2, d=8, N=2, C=6, L_q=3)
    e = oracle.token_scores(Q, Kc, 3)
    Q2 = Q.copy(); Q2[:, :, 3:] = bits(np.full(Q2[:, :, 3:].shape, 7.0))       # rows beyond L_q are not scoring rows
    np.testing.assert_array_equal(oracle.token_scores(Q2, Kc, 3), e)
    Q3 = Q.copy(); Q3[0, 0, 0] = bits(np.ones(8))                               # head 0 belongs to KV head 0 only (R4)
    e3 = oracle.token_scores(Q3, Kc, 3)
    assert not np.allclose(e3[0, 0], e[0, 0]) and np.array_equal(e3[0, 1], e[0, 1])


# --------------------------------------------------------------------------- NEXT-1 top-B (R7)
@pytest.mark.parametrize("C,Bk", [(6, 1), (6, 3), (7, 4), (5, 6), (8, 5)])
def test_topb_subset_enumeration(C, Bk):
    """The kept set is the max-sum (Bk-1)-subset of slots 1..C, lexicographically smallest under ties, plus slot 0."""
    r = np.random.default_rng(C * 10 + Bk)
    e = np.round(r.standard_normal((12, C + 1)) * 2) / 2                         # coarse grid: many exact ties
    e[:, 0] = -100.0                                                             # BOS is kept whatever its score
    got = oracle.topb(e, Bk)
    for row in range(12):
        best = max(itertools.combinations(range(1, C + 1), Bk - 1),
                   key=lambda s: (sum(e[row, j] for j in s), tuple(-j for j in s)))
        assert got[row].tolist() == [0] + list(best)


def test_topb_ties_nan_inf_and_bounds():
    C = 9
    e = np.zeros((5, C + 1))
    e[0] = 1.0                                         # all equal: lowest slots win
    e[1, 2::3] = 2.0
    e[2] = np.nan                                      # NaN == -inf everywhere: lowest slots
    e[3] = -np.inf; e[3, [4, 8]] = 0.5
    e[4] = np.arange(C + 1)[::-1]; e[4, 3] = np.nan; e[4, 9] = np.inf
    got = oracle.topb(e, 4)
    assert got[0].tolist() == [0, 1, 2, 3]
    assert got[1].tolist() == [0, 2, 5, 8]
    assert got[2].tolist() == [0, 1, 2, 3]
    assert got[3].tolist() == [0, 1, 4, 8]
    assert got[4].tolist() == [0, 1, 2, 9]
    assert oracle.topb(e, C + 1)[2].tolist() == list(range(C + 1))              # Bk = C + 1 keeps everything
    assert oracle.topb(e, 1).tolist() == [[0]] * 5


def test_topb_recovers_planted_tokens():
    """Generator sanity for the NEXT-1 workloads: tokens whose keys were shifted toward the queries are the kept ones."""
    w = W.small_variant(W.CONFIGS["tiny"], token_alpha=24.0)
    inp = W.make_inputs(w)
    e = oracle.token_scores(inp["Q_dec"], inp["Kcache"], w.L_q)
    np.testing.assert_array_equal(oracle.topb(e, w.Bk), inp["keep"])


# --------------------------------------------------------------------------- NEXT-2 chunk-prefill attention (Eq. 2)
def test_prefill_attn_matches_library_sdpa_fp64():
    r = np.random.default_rng(11)
    S, H, H_kv, T, d = 3, 4, 2, 13, 8
    Q, K, V = (bits(r.standard_normal(s)) for s in ((S, H, T, d), (S, H_kv, T, d), (S, H_kv, T, d)))
    O, LSE = oracle.prefill_attn(Q, K, V)
    q, k, v = (torch.from_numpy(f64(x)) for x in (Q, K, V))
    ref = torch.nn.functional.scaled_dot_product_attention(q, k.repeat_interleave(2, 1), v.repeat_interleave(2, 1))
    np.testing.assert_allclose(O, ref.numpy(), rtol=1e-12, atol=1e-13)
    z = torch.einsum("shid,shjd->shij", q, k.repeat_interleave(2, 1)) / np.sqrt(d)
    np.testing.assert_allclose(LSE, torch.logsumexp(z, -1).numpy(), rtol=1e-12)


def test_prefill_attn_closed_forms_and_independence():
    r = np.random.default_rng(12)
    S, H, T, d = 2, 2, 7, 4
    Q, K, V = (bits(r.standard_normal((S, H, T, d))) for _ in range(3))
    O, LSE = oracle.prefill_attn(np.zeros_like(Q), K, V)                         # Q = 0: mean of V, LSE = log T
    np.testing.assert_allclose(O, np.broadcast_to(f64(V).mean(2, keepdims=True), O.shape), atol=1e-13)
    np.testing.assert_allclose(LSE, np.log(T), atol=1e-13)
    O0, L0 = oracle.prefill_attn(Q, K, V)
    K2, V2 = K.copy(), V.copy()
    K2[1], V2[1] = bits(r.standard_normal((H, T, d))), bits(r.standard_normal((H, T, d)))
    O1, L1 = oracle.prefill_attn(Q, K2, V2)                                      # sequences never see each other
    np.testing.assert_array_equal(O0[0], O1[0]); np.testing.assert_array_equal(L0[0], L1[0])
    assert not np.allclose(O0[1], O1[1])
    perm = r.permutation(T)                                                      # bidirectional, no mask, no positions:
    O2, L2 = oracle.prefill_attn(Q, K[:, :, perm], V[:, :, perm])                # key order is immaterial
    np.testing.assert_allclose(O2, O0, rtol=1e-12, atol=1e-14); np.testing.assert_allclose(L2, L0, rtol=1e-13)


def test_prefill_attn_equals_decode_oracle_on_a_one_chunk_cache():
    """The sequence [BOS; c; q; m] attending to itself is oracle_attn with the chunk as the only cached chunk (kept
    whole) and the [q; m] rows as the decode block -- ties NEXT-2 to the hot path's pinned oracle."""
    r = np.random.default_rng(13)
    H, H_kv, C, Lqm, d = 4, 2, 10, 5, 8
    T = C + 1 + Lqm
    Q, K, V = bits(r.standard_normal((1, H, T, d))), bits(r.standard_normal((1, H_kv, T, d))), bits(r.standard_normal((1, H_kv, T, d)))
    O, LSE = oracle.prefill_attn(Q, K, V)
    Kc, Vc = K[:, :, None, :C + 1], V[:, :, None, :C + 1]
    ids = np.zeros((1, H_kv, 1), np.int32)
    O2, L2 = oracle.attn(Q, np.ascontiguousarray(Kc), np.ascontiguousarray(Vc), ids, None,
                         np.ascontiguousarray(K[:, :, C + 1:]), np.ascontiguousarray(V[:, :, C + 1:]))
    np.testing.assert_allclose(O, O2, rtol=1e-12, atol=1e-14); np.testing.assert_allclose(LSE, L2, rtol=1e-13)


# --------------------------------------------------------------------------- NEXT-3 compact cache
def test_compact_kv_is_the_identity_on_attention():
    """Attention over the compact cache (one 'chunk' holding the gathered rows, no keep list) equals attention over
    the original cache with the chunk ids and keep lists -- bit for bit in fp64, the row order being the same."""
    w = W.small_variant(W.CONFIGS["tiny"], H=4, H_kv=2, C=40, N=6, K=3)
    inp = W.make_inputs(w)
    ids = inp["planted"]
    gi = oracle.gather_idx(ids, inp["keep"], w.N, w.C)
    Kc, Vc = oracle.compact_kv(inp["Kcache"], inp["Vcache"], gi)
    flatK = inp["Kcache"].reshape(w.B, w.H_kv, w.N * w.Cp, w.d)
    for b, g, r in [(0, 0, 0), (0, 1, 17), (0, 1, w.S_pre - 1)]:
        np.testing.assert_array_equal(Kc[b, g, r], flatK[b, g, gi[b, g, r]])
    O, LSE = oracle.attn(inp["Q_dec"], inp["Kcache"], inp["Vcache"], ids, inp["keep"], inp["K_dec"], inp["V_dec"])
    one = np.zeros((w.B, w.H_kv, 1), np.int32)
    O2, L2 = oracle.attn(inp["Q_dec"], Kc[:, :, None], Vc[:, :, None], one, None, inp["K_dec"], inp["V_dec"])
    np.testing.assert_array_equal(O, O2); np.testing.assert_array_equal(LSE, L2)


# --------------------------------------------------------------------------- NEXT-3 pooled-key scorer (R23)
def test_pooled_keys_numpy_mean():
    Q, Kc = rand_case(21)
    np.testing.assert_allclose(oracle.pooled_keys(Kc), f64(Kc).mean(3), rtol=1e-14, atol=1e-15)


def test_pooled_score_is_a_jensen_lower_bound_of_the_chunk_score_tight_for_constant_chunks():
    Q, Kc = rand_case(22, B=2, H=4, H_kv=2, d=16, N=5, C=11, L_q=4)
    pooled = oracle.pooled_scores(Q, oracle.pooled_keys(Kc), 11, 4)
    full = oracle.scores(Q, Kc, 4)
    assert (pooled <= full + 1e-12).all() and (full - pooled).max() > 1e-3
    Kconst = np.ascontiguousarray(np.broadcast_to(Kc[:, :, :, :1], Kc.shape))    # every slot of a chunk holds the same key
    np.testing.assert_allclose(oracle.pooled_scores(Q, oracle.pooled_keys(Kconst), 11, 4), oracle.scores(Q, Kconst, 4),
                               rtol=1e-12)


def test_pooled_score_matrix_form_and_zero_queries():
    Q, Kc = rand_case(23, B=1, H=6, H_kv=2, d=8, N=3, C=7, L_q=2)
    kbar = oracle.pooled_keys(Kc)
    got = oracle.pooled_scores(Q, kbar, 7, 2, scale=0.2)
    qbar = f64(Q)[0, :, :2].reshape(2, 6, 8).mean(1)                             # mean of the G * L_q rows of each group
    want = np.log(8.0) + 0.2 * np.einsum("gd,gnd->gn", qbar, kbar[0])
    np.testing.assert_allclose(got[0], want, rtol=1e-12)
    np.testing.assert_allclose(oracle.pooled_scores(np.zeros_like(Q), kbar, 7, 2), np.log(8.0), atol=1e-14)
