"""Seeded random shapes through pdllm_step against the fp64 oracle: head dims, GQA factors, ragged chunk sizes around the
tile sizes, keep fractions, window / block lengths (incl. no decode block), K up to N, and split counts from auto to more
than there are KV tiles.  The shapes the hand-picked cases of test_gpu_parity.py do not name."""
import numpy as np
import pytest
import torch

from oracle import oracle
from paper_2606_10537_b200 import workloads as W

from gpu_util import LSE_ABS, SCORE_ABS, check_close, check_exact, check_O, to_device

pytestmark = pytest.mark.gpu


def _random_case(rng):
    H_kv = int(rng.choice([1, 2, 3, 4]))
    G = int(rng.choice([1, 1, 2, 4, 7]))
    N = int(rng.integers(1, 20))
    kw = dict(B=int(rng.choice([1, 1, 2, 3])), H=H_kv * G, H_kv=H_kv, d=int(rng.choice([64, 128])), N=N,
              C=int(rng.choice([1, 7, 16, 63, 64, 127, 128, 129, 200, 255, 256, 300, 511, 512])),
              K=int(rng.integers(1, min(N, 64) + 1)), keep=float(rng.choice([1.0, 1.0, 0.5, 0.25, 0.1])),
              L_q=int(rng.integers(1, 140)), L_d=int(rng.integers(0, 200)))
    return kw, int(rng.choice([0, 1, 2, 3, 5, 64]))


@pytest.mark.parametrize("seed", [11, 12, 13, 14])
def test_step_random_shapes(seed):
    from paper_2606_10537_b200 import binding as B
    B.lib()
    rng = np.random.default_rng(seed)
    for case in range(12):
        kw, S = _random_case(rng)
        w = W.small_variant(W.CONFIGS["tiny"], **kw)
        inp = W.make_inputs(w)
        dev = to_device(inp)
        what = f"seed {seed} case {case}: {kw}, n_splits {S}"
        out = B.step(B.Shape.of(w), dev["Q_dec"], dev["Kcache"], dev["Vcache"], dev["keep"], dev["K_dec"], dev["V_dec"],
                     n_splits=S)
        torch.cuda.synchronize()
        ref = oracle.step(inp["Q_dec"], inp["Kcache"], inp["Vcache"], inp["keep"], inp["K_dec"], inp["V_dec"], w.K, w.L_q)
        tol = SCORE_ABS * max(1.0, float(np.abs(ref["scores"]).max()) / 100.0)          # DESIGN.md R12b
        check_close(out["scores"], ref["scores"], tol, what=f"scores ({what})")
        # random inputs leave no guaranteed gap between the K-th and the (K+1)-th chunk: the selection rule is checked on
        # the GPU's own fp32 scores (both sides decide on the same values), the attention against the oracle on those ids
        ids = oracle.topk(out["scores"].double().cpu().numpy(), w.K)
        check_exact(out["chunk_ids"], ids, f"ids ({what})")
        O_ref, LSE_ref = oracle.attn(inp["Q_dec"], inp["Kcache"], inp["Vcache"], ids, inp["keep"], inp["K_dec"], inp["V_dec"])
        check_O(out["O"], O_ref, what=f"O ({what})")
        check_close(out["LSE"], LSE_ref, LSE_ABS, what=f"LSE ({what})")


@pytest.mark.parametrize("seed", [21, 22])
def test_next_rows_random_shapes(seed):
    """The rows after the hot path on random shapes: token scores (incl. chunks of 128 t + 1 slots: grouped tail steps),
    top-B (decided on the GPU's own scores), compact cache + TMA-tile attention with the device-made keep list, pooled
    keys / scores, chunk-prefill attention."""
    from paper_2606_10537_b200 import binding as B
    from gpu_util import dev_bf16, dev_i32
    B.lib()
    rng = np.random.default_rng(seed)
    for case in range(10):
        H_kv = int(rng.choice([1, 2, 3, 4]))
        G = int(rng.choice([1, 1, 2, 4, 7]))
        C = int(rng.choice([1, 7, 16, 63, 64, 127, 128, 129, 200, 255, 256, 257, 384, 512, 1024]))
        N = int(rng.integers(1, 40 if C <= 257 else 12))
        kw = dict(B=int(rng.choice([1, 1, 2, 3])), H=H_kv * G, H_kv=H_kv, d=int(rng.choice([64, 128])), N=N, C=C,
                  K=int(rng.integers(1, min(N, 64) + 1)), keep=float(rng.choice([1.0, 0.5, 0.25, 0.1])),
                  L_q=int(rng.integers(1, 140)), L_d=int(rng.integers(0, 200)))
        what = f"seed {seed} case {case}: {kw}"
        w = W.small_variant(W.CONFIGS["tiny"], **kw)
        inp = W.make_inputs(w)
        dev = to_device(inp)
        shape = B.Shape.of(w)
        # NEXT-1
        e = B.score_tokens(shape, dev["Q_dec"], dev["Kcache"])
        torch.cuda.synchronize()
        e_ref = oracle.token_scores(inp["Q_dec"], inp["Kcache"], w.L_q)
        worst = float((np.abs(e.double().cpu().numpy() - e_ref) - (1e-4 * np.abs(e_ref) + 1e-6 * w.G * w.L_q)).max())
        assert worst <= 0, f"token scores gate (DESIGN.md R12b) exceeded by {worst:.3e} ({what})"
        keep = B.select_topb(shape, e)
        torch.cuda.synchronize()
        check_exact(keep, oracle.topb(e.double().cpu().numpy(), w.Bk), f"top-B ({what})")
        # NEXT-3 with the device-made keep list
        ids = inp["planted"]
        thinned = w.Bk != w.Cp
        Kc, Vc = B.compact_kv(shape, dev["Kcache"], dev["Vcache"], dev_i32(ids), keep if thinned else None)
        O, LSE = B.static_attn(B.DenseShape.static_of(shape), dev["Q_dec"], Kc, Vc, dev["K_dec"], dev["V_dec"],
                               n_splits=int(rng.choice([0, 1, 2, 3, 7])))
        torch.cuda.synchronize()
        O_ref, LSE_ref = oracle.attn(inp["Q_dec"], inp["Kcache"], inp["Vcache"], ids, keep.cpu().numpy() if thinned else None,
                                     inp["K_dec"], inp["V_dec"])
        check_O(O, O_ref, what=f"static O ({what})")
        check_close(LSE, LSE_ref, LSE_ABS, what=f"static LSE ({what})")
        kbar = B.pool_keys(shape, dev["Kcache"])
        got = B.score_chunks_pooled(shape, dev["Q_dec"], kbar)
        torch.cuda.synchronize()
        check_close(kbar, oracle.pooled_keys(inp["Kcache"]), 1e-5, what=f"pooled keys ({what})")
        check_close(got, oracle.pooled_scores(inp["Q_dec"], kbar.double().cpu().numpy(), w.C, w.L_q), 1e-4,
                    what=f"pooled scores ({what})")
        # NEXT-2
        T, Sq = int(rng.integers(1, 400)), int(rng.choice([1, 2, 3]))
        Qp, Kp, Vp = (W.f32_to_bf16_bits(rng.standard_normal(s_, dtype=np.float32))
                      for s_ in ((Sq, w.H, T, w.d), (Sq, w.H_kv, T, w.d), (Sq, w.H_kv, T, w.d)))
        Op, Lp = B.prefill_attn(B.DenseShape(Sq, w.H, w.H_kv, w.d, T, T, 0), dev_bf16(Qp), dev_bf16(Kp), dev_bf16(Vp),
                                n_splits=int(rng.choice([0, 1, 2])))
        torch.cuda.synchronize()
        Op_ref, Lp_ref = oracle.prefill_attn(Qp, Kp, Vp)
        check_O(Op, Op_ref, what=f"prefill O ({what})")
        check_close(Lp, Lp_ref, LSE_ABS, what=f"prefill LSE ({what})")


@pytest.mark.parametrize("kw,S", [
    (dict(B=1, H=2, H_kv=2, d=64, N=4096, C=15, K=64, keep=1.0, L_q=16, L_d=16), 0),     # N and K at the header's bounds
    (dict(B=1, H=4, H_kv=2, d=128, N=4096, C=7, K=33, keep=0.5, L_q=40, L_d=8), 2),      # 8-row chunks, thinned, GQA
    (dict(B=1, H=2, H_kv=1, d=128, N=2, C=8191, K=2, keep=1.0, L_q=8, L_d=24), 0),       # the longest chunk top-B takes: 128 KV tiles
    (dict(B=1, H=1, H_kv=1, d=64, N=3, C=8191, K=1, keep=0.37, L_q=130, L_d=0), 5),      # no decode block, two M tiles of scoring rows
])
def test_sizes_at_the_bounds(kw, S):
    """The largest chunk count, selection size and chunk length the header allows, through the step and NEXT-1."""
    from paper_2606_10537_b200 import binding as B
    B.lib()
    w = W.small_variant(W.CONFIGS["tiny"], **kw)
    inp = W.make_inputs(w)
    dev = to_device(inp)
    shape = B.Shape.of(w)
    out = B.step(shape, dev["Q_dec"], dev["Kcache"], dev["Vcache"], dev["keep"], dev["K_dec"], dev["V_dec"], n_splits=S)
    torch.cuda.synchronize()
    ref = oracle.step(inp["Q_dec"], inp["Kcache"], inp["Vcache"], inp["keep"], inp["K_dec"], inp["V_dec"], w.K, w.L_q)
    check_close(out["scores"], ref["scores"], SCORE_ABS, what="scores")
    ids = oracle.topk(out["scores"].double().cpu().numpy(), w.K)
    check_exact(out["chunk_ids"], ids)
    O_ref, LSE_ref = oracle.attn(inp["Q_dec"], inp["Kcache"], inp["Vcache"], ids, inp["keep"], inp["K_dec"], inp["V_dec"])
    check_O(out["O"], O_ref)
    check_close(out["LSE"], LSE_ref, LSE_ABS)
    e = B.score_tokens(shape, dev["Q_dec"], dev["Kcache"])
    torch.cuda.synchronize()
    e_ref = oracle.token_scores(inp["Q_dec"], inp["Kcache"], w.L_q)
    worst = float((np.abs(e.double().cpu().numpy() - e_ref) - (1e-4 * np.abs(e_ref) + 1e-6 * w.G * w.L_q)).max())
    assert worst <= 0, f"token scores gate exceeded by {worst:.3e}"
    keep = B.select_topb(shape, e)
    torch.cuda.synchronize()
    check_exact(keep, oracle.topb(e.double().cpu().numpy(), w.Bk), "top-B")
