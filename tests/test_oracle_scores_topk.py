"""Pins for oracle steps 1-3 (chunk scores, top-K, gather indices).  CPU only.

The chunk score is OUR reading (R1: mean log attention mass; the paper's own score is a
model NLL, Eq. 3-4, uncomputable without weights) -- "parity unpinned by the paper".  Its
arithmetic is pinned here by closed forms, the chain rule against step 5, a brute force,
and by recovering planted chunks.
"""
import itertools
import math

import numpy as np
import pytest
from scipy.special import logsumexp

from oracle import oracle
from paper_2606_10537_b200 import workloads as W


def bf(r, *s, sigma=1.0):
    return W.f32_to_bf16_bits((sigma * r.standard_normal(s)).astype(np.float32))


# --------------------------------------------------------------------------- scores
def test_zero_query_scores_log_chunk_rows():
    r = np.random.default_rng(0)
    Q = np.zeros((1, 2, 3, 8), np.uint16)
    s = oracle.scores(Q, bf(r, 1, 2, 4, 6, 8), L_q=3)
    np.testing.assert_allclose(s, math.log(6), rtol=0, atol=1e-14)     # log(C+1), BOS counted (R3)


def test_chain_rule_against_attention_lse():
    # log sum_n exp(row_lse[h,i,n]) is the LSE of dense attention over the prefix alone; step 5
    # run with K = N, full mask and one decode key gives log(exp(that) + exp(s_dec)).
    r = np.random.default_rng(1)
    B, H, H_kv, d, N, C, L_q = 2, 4, 2, 8, 5, 6, 3
    Q = bf(r, B, H, L_q, d); Kc = bf(r, B, H_kv, N, C + 1, d); Vc = bf(r, B, H_kv, N, C + 1, d)
    Kd = bf(r, B, H_kv, 1, d); Vd = bf(r, B, H_kv, 1, d)
    _, rl = oracle.scores(Q, Kc, L_q, want_row_lse=True)
    ids = np.tile(np.arange(N, dtype=np.int32), (B, H_kv, 1))
    _, LSE = oracle.attn(Q, Kc, Vc, ids, None, Kd, Vd)
    G = H // H_kv
    for b, h, i in np.ndindex(B, H, L_q):
        s_dec = oracle.bf16_to_f64(Q[b, h, i]) @ oracle.bf16_to_f64(Kd[b, h // G, 0]) / math.sqrt(d)
        np.testing.assert_allclose(np.logaddexp(logsumexp(rl[b, h, i]), s_dec), LSE[b, h, i], rtol=0, atol=1e-12)


def test_scores_against_numpy_matrix_form_and_group_mean():
    r = np.random.default_rng(2)
    B, H, H_kv, d, N, C, L_q, Lrows = 2, 6, 2, 8, 4, 5, 3, 7
    Q = bf(r, B, H, Lrows, d); Kc = bf(r, B, H_kv, N, C + 1, d)
    s, rl = oracle.scores(Q, Kc, L_q, want_row_lse=True)               # scores the first L_q of Lrows rows in place (R8)
    G = H // H_kv
    qf, kf = oracle.bf16_to_f64(Q), oracle.bf16_to_f64(Kc)
    for b, g, n in np.ndindex(B, H_kv, N):
        per_head = []
        for h in range(g * G, (g + 1) * G):
            z = qf[b, h, :L_q] @ kf[b, g, n].T / math.sqrt(d)
            ell = logsumexp(z, axis=1)
            np.testing.assert_allclose(rl[b, h, :, n], ell, rtol=0, atol=1e-13)
            per_head.append(ell.mean())
        np.testing.assert_allclose(s[b, g, n], np.mean(per_head), rtol=0, atol=1e-13)   # mean over G*L_q rows (R2)
    # explicit scale
    s2 = oracle.scores(Q, Kc, L_q, scale=0.0)
    np.testing.assert_allclose(s2, math.log(C + 1), atol=1e-14)


def test_scores_brute_force_tiny():
    r = np.random.default_rng(3)
    Q = bf(r, 1, 1, 2, 3); Kc = bf(r, 1, 1, 2, 3, 3)
    s = oracle.scores(Q, Kc, L_q=2)
    q = [[float(x) for x in row] for row in oracle.bf16_to_f64(Q[0, 0])]
    for n in range(2):
        k = [[float(x) for x in row] for row in oracle.bf16_to_f64(Kc[0, 0, n])]
        tot = 0.0
        for i in range(2):
            tot += math.log(sum(math.exp(sum(q[i][c] * k[j][c] for c in range(3)) / math.sqrt(3)) for j in range(3)))
        assert abs(s[0, 0, n] - tot / 2) < 1e-14


def test_planted_chunks_are_recovered_with_a_clear_gap_on_config_tiny():
    w = W.CONFIGS["tiny"]
    x = W.make_inputs(w, threads=1)
    s = oracle.scores(x["Q_dec"], x["Kcache"], w.L_q)
    ids = oracle.topk(s, w.K)
    np.testing.assert_array_equal(ids, x["planted"])
    srt = np.sort(s, axis=-1)[..., ::-1]
    assert (srt[..., w.K - 1] - srt[..., w.K] >= 2e-3).all()               # R6/R20: gap to rank K+1


# --------------------------------------------------------------------------- top-K
def brute_topk(row, K):
    row = [(-math.inf if v != v else v) for v in row]
    best = None
    for sub in itertools.combinations(range(len(row)), K):                  # lexicographic order of sorted id lists
        tot = sum(row[i] for i in sub if row[i] != -math.inf), sum(1 for i in sub if row[i] == -math.inf)
        key = (-tot[1], tot[0])                                             # fewest -inf first, then the largest sum
        if best is None or key > best[0]:
            best = (key, sub)                                               # strict '>' keeps the lexicographically smallest
    return list(best[1])


@pytest.mark.parametrize("seed", range(6))
def test_topk_equals_max_sum_subset_enumeration(seed):
    r = np.random.default_rng(seed)
    N = int(r.integers(2, 11)); K = int(r.integers(1, N + 1))
    s = r.standard_normal((7, N))
    if seed % 2:
        s = np.round(s * 2) / 2                                             # many exact ties
    ids = oracle.topk(s, K)
    for row, got in zip(s, ids):
        assert list(got) == brute_topk(list(row), K)
        assert list(got) == sorted(got)


def test_topk_crafted_ties_edges_and_non_finite():
    assert list(oracle.topk(np.array([[1.0, 1.0, 1.0, 1.0]]), 2)[0]) == [0, 1]         # ties -> lower index
    assert list(oracle.topk(np.array([[0.0, 2.0, 2.0, 1.0, 2.0]]), 2)[0]) == [1, 2]
    assert list(oracle.topk(np.array([[3.0, 1.0, 2.0]]), 3)[0]) == [0, 1, 2]           # K = N
    assert list(oracle.topk(np.array([[3.0, 9.0, 2.0]]), 1)[0]) == [1]                 # K = 1
    assert list(oracle.topk(np.array([[np.nan, -1.0, np.nan, -np.inf]]), 2)[0]) == [0, 1]   # NaN == -inf < -1; ties -> lower
    assert list(oracle.topk(np.array([[-np.inf, 5.0, np.nan]]), 2)[0]) == [0, 1]
    # emitted ascending by index even when the scores are descending the other way
    assert list(oracle.topk(np.array([[1.0, 5.0, 9.0]]), 2)[0]) == [1, 2]
    # float32 scores are widened exactly: a 1-ulp fp32 difference decides
    a = np.array([[1.0, np.nextafter(np.float32(1.0), np.float32(2.0)), 1.0]], np.float32)
    assert list(oracle.topk(a, 1)[0]) == [1]


# --------------------------------------------------------------------------- gather
def test_gather_idx_nested_loops_bos_once_and_ascending():
    r = np.random.default_rng(5)
    B, H_kv, N, C, K, Bk = 2, 3, 6, 9, 3, 5
    keep = np.zeros((B, H_kv, N, Bk), np.int32)
    for idx in np.ndindex(B, H_kv, N):
        keep[idx][1:] = np.sort(r.choice(np.arange(1, C + 1), Bk - 1, replace=False))
    ids = np.stack([np.sort(r.choice(N, K, replace=False)) for _ in range(B * H_kv)]).reshape(B, H_kv, K).astype(np.int32)
    gi = oracle.gather_idx(ids, keep, N, C)
    Cp = C + 1
    for b in range(B):
        for g in range(H_kv):
            want = []
            for k in range(K):
                for t in range(Bk):
                    want.append(int(ids[b, g, k]) * Cp + int(keep[b, g, ids[b, g, k], t]))
            assert list(gi[b, g]) == want
            assert all(x < y for x, y in zip(want, want[1:]))                         # strictly ascending
            bos = [x for x in want if x % Cp == 0]
            assert bos == [int(n) * Cp for n in ids[b, g]]                            # BOS row of each chunk, once
    full = oracle.gather_idx(ids, None, N, C)                                          # keep = NULL: all Cp slots
    assert full.shape == (B, H_kv, K * Cp)
    for b, g in np.ndindex(B, H_kv):
        assert list(full[b, g]) == [int(n) * Cp + t for n in ids[b, g] for t in range(Cp)]


def test_step_composes_the_stages():
    w = W.small_variant(W.CONFIGS["tiny"], N=4, C=16, L_q=4, L_d=4)
    x = W.make_inputs(w, threads=1)
    out = oracle.step(x["Q_dec"], x["Kcache"], x["Vcache"], x["keep"], x["K_dec"], x["V_dec"], w.K, w.L_q)
    np.testing.assert_array_equal(out["ids"], oracle.topk(oracle.scores(x["Q_dec"], x["Kcache"], w.L_q), w.K))
    O, LSE = oracle.attn(x["Q_dec"], x["Kcache"], x["Vcache"], out["ids"], x["keep"], x["K_dec"], x["V_dec"])
    np.testing.assert_array_equal(out["O"], O)
    assert out["gather_idx"].shape == (w.B, w.H_kv, w.S_pre)
