"""ctypes front-end of the fp64 CPU oracle (oracle/pdllm_oracle.c).

TEST INFRASTRUCTURE, NOT PRODUCT CODE: only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this module.  It does
not import, and is not imported by, paper_2606_10537_b200 (the CUDA path).

All tensors are numpy arrays; bf16 tensors are uint16 bit patterns.  Every
function cites the passage it follows in pdllm_oracle.c.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "pdllm_oracle.c"
_SRC_NEXT = _HERE / "pdllm_oracle_next.c"      # the rows after the hot path
_LIB = _HERE / "libpdllm_oracle.so"
_lib = None


def build(force: bool = False) -> Path:
    """Compile the oracle with gcc (-O2, OpenMP over (b,h) only; no SIMD intrinsics, no tuning)."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < max(_SRC.stat().st_mtime, _SRC_NEXT.stat().st_mtime):
        cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", str(_SRC), str(_SRC_NEXT), "-o", str(_LIB), "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(str(_LIB))
    return _lib


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def _p(a, ctype):
    return None if a is None else a.ctypes.data_as(ctypes.POINTER(ctype))


def _u16(a):
    a = np.ascontiguousarray(a)
    assert a.dtype == np.uint16, "bf16 tensors are passed as uint16 bit patterns"
    return a


def bf16_to_f64(bits: np.ndarray) -> np.ndarray:
    """Exact widening of bf16 bit patterns (test helper; the C oracle widens on its own)."""
    return (bits.astype(np.uint32) << 16).view(np.float32).astype(np.float64)


def scores(Q, Kcache, L_q, scale=None, want_row_lse=False):
    """Step 1 (R1; Eq. 5).  Q uint16 [B,H,Lrows,d] (first L_q rows used),
    Kcache uint16 [B,H_kv,N,C+1,d] -> scores f64 [B,H_kv,N] (and row_lse f64 [B,H,L_q,N])."""
    Q = _u16(Q); Kcache = _u16(Kcache)
    B, H, Lr, d = Q.shape
    _, H_kv, N, Cp, _ = Kcache.shape
    scale = 1.0 / np.sqrt(d) if scale is None else scale
    out = np.empty((B, H_kv, N), np.float64)
    rl = np.empty((B, H, L_q, N), np.float64) if want_row_lse else None
    rc = _load().oracle_scores(_p(Q, ctypes.c_uint16), ctypes.c_int64(H * Lr * d), ctypes.c_int64(Lr * d),
                               _p(Kcache, ctypes.c_uint16), B, H, H_kv, d, N, Cp - 1, L_q,
                               ctypes.c_double(scale), _p(out, ctypes.c_double), _p(rl, ctypes.c_double))
    assert rc == 0, rc
    return (out, rl) if want_row_lse else out


def topk(scores_, K):
    """Step 2 (R6).  scores [..., N] (any float dtype, widened exactly) -> int32 [..., K] ascending."""
    s = np.ascontiguousarray(scores_, dtype=np.float64)
    N = s.shape[-1]
    rows = s.size // N
    ids = np.empty(s.shape[:-1] + (K,), np.int32)
    rc = _load().oracle_topk(_p(s, ctypes.c_double), ctypes.c_int64(rows), N, K, _p(ids, ctypes.c_int32))
    assert rc == 0, rc
    return ids


def gather_idx(ids, keep, N, C):
    """Step 3 (R7).  ids int32 [B,H_kv,K]; keep int32 [B,H_kv,N,Bk] or None -> int32 [B,H_kv,K*Bk]."""
    ids = np.ascontiguousarray(ids, dtype=np.int32)
    B, H_kv, K = ids.shape
    Bk = C + 1 if keep is None else keep.shape[-1]
    if keep is not None:
        keep = np.ascontiguousarray(keep, dtype=np.int32)
    out = np.empty((B, H_kv, K * Bk), np.int32)
    rc = _load().oracle_gather_idx(_p(ids, ctypes.c_int32), _p(keep, ctypes.c_int32), B, H_kv, N, C, K, Bk,
                                   _p(out, ctypes.c_int32))
    assert rc == 0, rc
    return out


def attn(Q_dec, Kcache, Vcache, ids, keep, K_dec, V_dec, scale=None, n_splits=1, head_mask=None, want_P=False):
    """Steps 3-5 and, for n_splits > 1, step 6.
    Returns O f64 [B,H,L,d], LSE f64 [B,H,L] (and P f64 [B,H,L,S_kv] if want_P).
    Heads with head_mask == 0 are left as NaN."""
    Q_dec = _u16(Q_dec); Kcache = _u16(Kcache); Vcache = _u16(Vcache); K_dec = _u16(K_dec); V_dec = _u16(V_dec)
    ids = np.ascontiguousarray(ids, dtype=np.int32)
    B, H, L, d = Q_dec.shape
    _, H_kv, N, Cp, _ = Kcache.shape
    K = ids.shape[-1]
    L_s = K_dec.shape[2]
    Bk = Cp if keep is None else keep.shape[-1]
    if keep is not None:
        keep = np.ascontiguousarray(keep, dtype=np.int32)
    scale = 1.0 / np.sqrt(d) if scale is None else scale
    O = np.full((B, H, L, d), np.nan, np.float64)
    LSE = np.full((B, H, L), np.nan, np.float64)
    P = np.zeros((B, H, L, K * Bk + L_s), np.float64) if want_P else None
    hm = None if head_mask is None else np.ascontiguousarray(head_mask, dtype=np.uint8)
    rc = _load().oracle_attn(_p(Q_dec, ctypes.c_uint16), _p(Kcache, ctypes.c_uint16), _p(Vcache, ctypes.c_uint16),
                             _p(ids, ctypes.c_int32), _p(keep, ctypes.c_int32),
                             _p(K_dec, ctypes.c_uint16), _p(V_dec, ctypes.c_uint16),
                             B, H, H_kv, d, N, Cp - 1, K, Bk, L, L_s, ctypes.c_double(scale), int(n_splits),
                             _p(hm, ctypes.c_uint8), _p(O, ctypes.c_double), _p(LSE, ctypes.c_double),
                             _p(P, ctypes.c_double))
    assert rc == 0, rc
    return (O, LSE, P) if want_P else (O, LSE)


def lse_combine(O_part, lse_part):
    """Step 6's merge alone.  O_part [S,...,d], lse_part [S,...] -> O [...,d], LSE [...]."""
    O_part = np.ascontiguousarray(O_part, dtype=np.float64)
    lse_part = np.ascontiguousarray(lse_part, dtype=np.float64)
    S, d = O_part.shape[0], O_part.shape[-1]
    rows = lse_part.size // S
    O = np.empty(O_part.shape[1:], np.float64)
    LSE = np.empty(lse_part.shape[1:], np.float64)
    rc = _load().oracle_lse_combine(_p(O_part, ctypes.c_double), _p(lse_part, ctypes.c_double), S,
                                    ctypes.c_int64(rows), d, _p(O, ctypes.c_double), _p(LSE, ctypes.c_double))
    assert rc == 0, rc
    return O, LSE


def step(Q_dec, Kcache, Vcache, keep, K_dec, V_dec, K, L_q, scale=None, head_mask=None):
    """The whole per-step path: scores -> top-K -> gather -> concat -> naive attention."""
    sc = scores(Q_dec, Kcache, L_q, scale)
    ids = topk(sc, K)
    _, H_kv, N, Cp, _ = Kcache.shape
    gi = gather_idx(ids, keep, N, Cp - 1)
    O, LSE = attn(Q_dec, Kcache, Vcache, ids, keep, K_dec, V_dec, scale, head_mask=head_mask)
    return dict(scores=sc, ids=ids, gather_idx=gi, O=O, LSE=LSE)


# ---------------------------------------------------------------------------------------------------------------
# rows after the hot path; pdllm_oracle_next.c
def token_scores(Q, Kcache, L_q, scale=None):
    """NEXT-1 (Eq. 5, query->chunk term; R22).  -> e f64 [B,H_kv,N,C+1], each chunk's slots summing to G*L_q."""
    Q = _u16(Q); Kcache = _u16(Kcache)
    B, H, Lr, d = Q.shape
    _, H_kv, N, Cp, _ = Kcache.shape
    scale = 1.0 / np.sqrt(d) if scale is None else scale
    e = np.empty((B, H_kv, N, Cp), np.float64)
    rc = _load().oracle_token_scores(_p(Q, ctypes.c_uint16), ctypes.c_int64(H * Lr * d), ctypes.c_int64(Lr * d),
                                     _p(Kcache, ctypes.c_uint16), B, H, H_kv, d, N, Cp - 1, L_q, ctypes.c_double(scale),
                                     _p(e, ctypes.c_double))
    assert rc == 0, rc
    return e


def topb(e, Bk):
    """NEXT-1 (R7).  e [..., C+1] (any float dtype, widened exactly) -> keep int32 [..., Bk]: slot 0 + the
    Bk-1 best of slots 1..C, ties to the lower slot, ascending."""
    e = np.ascontiguousarray(e, dtype=np.float64)
    Cp = e.shape[-1]
    keep = np.empty(e.shape[:-1] + (Bk,), np.int32)
    rc = _load().oracle_topb(_p(e, ctypes.c_double), ctypes.c_int64(e.size // Cp), Cp - 1, Bk, _p(keep, ctypes.c_int32))
    assert rc == 0, rc
    return keep


def prefill_attn(Q, K, V, scale=None):
    """NEXT-2 (Eq. 2).  Q uint16 [S,H,T,d], K,V uint16 [S,H_kv,T,d] -> O f64 [S,H,T,d], LSE f64 [S,H,T]."""
    Q = _u16(Q); K = _u16(K); V = _u16(V)
    S, H, T, d = Q.shape
    H_kv = K.shape[1]
    scale = 1.0 / np.sqrt(d) if scale is None else scale
    O = np.empty((S, H, T, d), np.float64)
    LSE = np.empty((S, H, T), np.float64)
    rc = _load().oracle_prefill_attn(_p(Q, ctypes.c_uint16), _p(K, ctypes.c_uint16), _p(V, ctypes.c_uint16), S, H, H_kv, T, d,
                                     ctypes.c_double(scale), _p(O, ctypes.c_double), _p(LSE, ctypes.c_double))
    assert rc == 0, rc
    return O, LSE


def compact_kv(Kcache, Vcache, gather_idx_):
    """NEXT-3.  Kcache,Vcache uint16 [B,H_kv,N,C+1,d]; gather_idx int32 [B,H_kv,S_pre]
    -> Kc, Vc uint16 [B,H_kv,S_pre,d] (bit copies of the selected rows)."""
    Kcache = _u16(Kcache); Vcache = _u16(Vcache)
    gi = np.ascontiguousarray(gather_idx_, dtype=np.int32)
    B, H_kv, N, Cp, d = Kcache.shape
    S_pre = gi.shape[-1]
    Kc = np.empty((B, H_kv, S_pre, d), np.uint16)
    Vc = np.empty((B, H_kv, S_pre, d), np.uint16)
    rc = _load().oracle_compact_kv(_p(Kcache, ctypes.c_uint16), _p(Vcache, ctypes.c_uint16), _p(gi, ctypes.c_int32), B, H_kv,
                                   ctypes.c_int64(N * Cp), S_pre, d, _p(Kc, ctypes.c_uint16), _p(Vc, ctypes.c_uint16))
    assert rc == 0, rc
    return Kc, Vc


def pooled_keys(Kcache):
    """NEXT-3 (R23).  -> kbar f64 [B,H_kv,N,d], the mean of each chunk's C+1 cached keys."""
    Kcache = _u16(Kcache)
    B, H_kv, N, Cp, d = Kcache.shape
    kbar = np.empty((B, H_kv, N, d), np.float64)
    rc = _load().oracle_pooled_keys(_p(Kcache, ctypes.c_uint16), B, H_kv, N, Cp - 1, d, _p(kbar, ctypes.c_double))
    assert rc == 0, rc
    return kbar


def pooled_scores(Q, kbar, C, L_q, scale=None):
    """NEXT-3 (R23).  Q uint16 [B,H,Lrows,d]; kbar [B,H_kv,N,d] (widened to f64) -> f64 [B,H_kv,N]."""
    Q = _u16(Q)
    kbar = np.ascontiguousarray(kbar, dtype=np.float64)
    B, H, Lr, d = Q.shape
    _, H_kv, N, _ = kbar.shape
    scale = 1.0 / np.sqrt(d) if scale is None else scale
    out = np.empty((B, H_kv, N), np.float64)
    rc = _load().oracle_pooled_scores(_p(Q, ctypes.c_uint16), ctypes.c_int64(H * Lr * d), ctypes.c_int64(Lr * d),
                                      _p(kbar, ctypes.c_double), B, H, H_kv, d, N, C, L_q, ctypes.c_double(scale),
                                      _p(out, ctypes.c_double))
    assert rc == 0, rc
    return out


if os.environ.get("PDLLM_ORACLE_BUILD"):
    build(force=True)
