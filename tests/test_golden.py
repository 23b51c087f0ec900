"""Golden fixtures (tests/golden/): what the paper prints about the cache layout / budget, and the oracle's own
stored results on config "tiny" (regression guard; written by tests/golden/make_golden.py from oracle/ only)."""
import os
import re
import sys

import numpy as np

from oracle import oracle
from paper_2606_10537_b200 import workloads as W

HERE = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def read_kv(name):
    out = {}
    for line in open(os.path.join(HERE, name)):
        line = line.split("#", 1)[0].strip()
        if line:
            k, v = line.split("=", 1)
            out[k.strip()] = v.strip()
    return out


def test_paper_shape_facts_match_the_cache_layout():
    f = {k: int(v) for k, v in read_kv("paper_shape_facts.txt").items()}
    # P:213 / P:223: an 8K prompt = 8 chunks of 1024 tokens, one BOS per chunk -> Cp = C + 1 rows per chunk (R14)
    w = W.small_variant(W.CONFIGS["dream16k"], N=f["chunks_in_8k_prompt"], C=f["chunk_tokens"], K=f["selected_budget_topk"],
                        keep=1.0)
    assert w.Cp == f["chunk_tokens"] + 1
    assert w.N * w.Cp == f["chunks_in_8k_prompt"] * f["chunk_tokens"] + f["chunks_in_8k_prompt"]
    assert f["chunk_bos_tokens_in_8k_prompt"] == f["chunks_in_8k_prompt"] + 1      # + the sequence's own first token
    # K x C = 4 x 1024 selected prefix tokens; with the BOS rows the oracle gathers K*(C+1) rows
    assert w.K * w.C == f["selected_budget_tokens"]
    ids = np.arange(w.K, dtype=np.int32).reshape(1, 1, w.K) * 2
    gi = oracle.gather_idx(ids, None, w.N, w.C)
    assert gi.shape[-1] == f["selected_budget_tokens"] + f["selected_budget_topk"]
    bos_rows = [int(r) for r in gi[0, 0] if r % w.Cp == 0]
    assert bos_rows == [int(i) * w.Cp for i in ids[0, 0]]                           # one BOS row per selected chunk
    # the paper's decode-kernel shape is expressible: GQA 32/8, L_d = 32, S = 4
    assert f["fig5b_query_heads"] % f["fig5b_kv_heads"] == 0 and f["fig5b_splits"] == 4 and f["fig5b_decode_tokens"] == 32
    # NEXT-4 workloads (R25): the Fig. 5(b) shape with the paper's query window, strict R8 rows
    for name in ("fig5b_8k", "fig5b_16k", "fig5b_32k"):
        x = W.EXTRA[name]
        assert (x.H, x.H_kv, x.L_d, x.L_q) == (f["fig5b_query_heads"], f["fig5b_kv_heads"], f["fig5b_decode_tokens"], f["query_window_tokens"])
        assert x.strict and x.L == x.L_d and x.L_s == x.L_q + x.L_d and x.G * x.L == 128 and x.C == f["chunk_tokens"]
    # top-B = 512 of C = 1024 is config C3's 50 % keep: Bk = 1 + B
    c3 = W.CONFIGS["dream16k"]
    assert c3.C == f["chunk_tokens"] and c3.Bk == 1 + f["top_b_tokens"]
    assert f["timing_pseudo_label_tokens"] == 16 and f["timing_generated_tokens"] == f["fig5b_decode_tokens"]


def test_oracle_reproduces_its_stored_results_on_tiny():
    sys.path.insert(0, HERE)
    import make_golden
    want = read_kv("tiny_oracle_expected.txt")
    got = {}
    for line in make_golden.compute().splitlines():
        if not line.startswith("#"):
            k, v = line.split("=", 1)
            got[k.strip()] = v.strip()
    assert got["inputs_sha256"] == want["inputs_sha256"], "the seeded input generator changed"
    assert got["chunk_ids"] == want["chunk_ids"] and got["gather_idx_head0"] == want["gather_idx_head0"]
    for k in ("scores", "LSE_row0_per_head", "O_head0_row0_first8", "O_abs_sum", "LSE_sum"):
        a = np.array([float(x) for x in re.split(r"\s+", got[k])])
        b = np.array([float(x) for x in re.split(r"\s+", want[k])])
        np.testing.assert_allclose(a, b, rtol=1e-10, atol=1e-12, err_msg=k)
