"""Thin ctypes binding of libpdllm.so (include/pdllm.h): argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI; torch is used for device
memory and streams.  There is no CPU fallback: if the library cannot be built/loaded, or a call
is made without a CUDA device, this module raises.

Function names mirror the C entry points (pdllm_score_chunks -> score_chunks, ...).  bf16 tensors
are torch.bfloat16 CUDA tensors, dense row-major in the shapes of the header.
"""
from __future__ import annotations

import ctypes
from dataclasses import dataclass
from pathlib import Path

_PKG = Path(__file__).resolve().parent
_LIB_PATH = _PKG / "libpdllm.so"
_lib = None
FOLD_MAX_N = 128            # include/pdllm.h PDLLM_FOLD_MAX_N: up to this many chunks pdllm_step runs a2 inside the a4 kernel

EXPORTS = [
    "pdllm_version", "pdllm_strerror", "pdllm_auto_splits", "pdllm_workspace_bytes",
    "pdllm_step_host_scratch_bytes", "pdllm_score_chunks", "pdllm_select_topk", "pdllm_gather_idx",
    "pdllm_sparse_attn", "pdllm_lse_combine", "pdllm_step", "pdllm_step_profiled", "pdllm_step_host",
    # rows after the hot path
    "pdllm_compact_kv", "pdllm_dense_auto_splits", "pdllm_dense_workspace_bytes", "pdllm_static_attn",
    "pdllm_pool_keys", "pdllm_score_chunks_pooled", "pdllm_prefill_attn",
    "pdllm_score_tokens_workspace_bytes", "pdllm_score_tokens", "pdllm_select_topb",
    # the call that allocates nothing (scratch in a fixed device array inside the library)
    "pdllm_sparse_attn_noalloc",
]
NOALLOC_SCRATCH_BYTES = 32 << 20        # include/pdllm.h PDLLM_NOALLOC_SCRATCH_BYTES
ERR_SCRATCH_LIMIT = -8                  # include/pdllm.h PDLLM_ERR_SCRATCH_LIMIT


class PdllmShape(ctypes.Structure):
    _fields_ = [(n, ctypes.c_int32) for n in ("B", "H", "H_kv", "d", "N", "C", "K", "Bk", "L_q", "L", "L_s")] + [
        ("scale", ctypes.c_float)]


class PdllmDenseShape(ctypes.Structure):
    _fields_ = [(n, ctypes.c_int32) for n in ("B", "H", "H_kv", "d", "S_pre", "L", "L_s")] + [("scale", ctypes.c_float)]


class PdllmSideStream(ctypes.Structure):
    _fields_ = [(n, ctypes.c_void_p) for n in ("stream", "ev_fork", "ev_join")]


class PdllmStageEvents(ctypes.Structure):
    _fields_ = [(n, ctypes.c_void_p) for n in ("begin", "after_score", "after_topk", "after_attn", "end")]


@dataclass(frozen=True)
class Shape:
    B: int
    H: int
    H_kv: int
    d: int
    N: int
    C: int
    K: int
    Bk: int
    L_q: int
    L: int
    L_s: int
    scale: float = 0.0      # <= 0: 1/sqrt(d)

    def c(self) -> PdllmShape:
        return PdllmShape(self.B, self.H, self.H_kv, self.d, self.N, self.C, self.K, self.Bk, self.L_q, self.L,
                          self.L_s, self.scale)

    @staticmethod
    def of(w) -> "Shape":
        """From a workloads.Workload."""
        return Shape(w.B, w.H, w.H_kv, w.d, w.N, w.C, w.K, w.Bk, w.L_q, w.L, w.L_s, 0.0)


@dataclass(frozen=True)
class DenseShape:
    """pdllm_dense_shape: attention over contiguous K/V (compact static cache, chunk prefill)."""
    B: int
    H: int
    H_kv: int
    d: int
    S_pre: int
    L: int
    L_s: int
    scale: float = 0.0

    def c(self) -> PdllmDenseShape:
        return PdllmDenseShape(self.B, self.H, self.H_kv, self.d, self.S_pre, self.L, self.L_s, self.scale)

    @staticmethod
    def static_of(shape: "Shape") -> "DenseShape":
        """The compact-cache attention that corresponds to a Shape (S_pre = K * Bk)."""
        return DenseShape(shape.B, shape.H, shape.H_kv, shape.d, shape.K * shape.Bk, shape.L, shape.L_s, shape.scale)


class PdllmError(RuntimeError):
    pass


def lib() -> ctypes.CDLL:
    """Load (building first if the .so is missing or stale and nvcc is present) the C-ABI library."""
    global _lib
    if _lib is not None:
        return _lib
    from . import build as _build
    try:
        _build.build()
    except Exception as e:  # stale-check / nvcc problems: fall through to whatever .so exists
        if not _LIB_PATH.exists():
            raise PdllmError(f"libpdllm.so is missing and could not be built: {e}") from e
    L = ctypes.CDLL(str(_LIB_PATH))
    vp, i32, i64, sz = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_size_t
    shp = ctypes.POINTER(PdllmShape)
    L.pdllm_version.restype = ctypes.c_int
    L.pdllm_strerror.restype = ctypes.c_char_p
    L.pdllm_strerror.argtypes = [ctypes.c_int]
    L.pdllm_auto_splits.restype = i32
    L.pdllm_auto_splits.argtypes = [shp, i32]
    L.pdllm_workspace_bytes.restype = sz
    L.pdllm_workspace_bytes.argtypes = [shp, i32, i32]
    L.pdllm_step_host_scratch_bytes.restype = sz
    L.pdllm_step_host_scratch_bytes.argtypes = [shp, i32, i32]
    L.pdllm_score_chunks.argtypes = [shp, vp, i64, i64, vp, vp, vp]
    L.pdllm_select_topk.argtypes = [shp, vp, vp, vp]
    L.pdllm_gather_idx.argtypes = [shp, vp, vp, vp, vp]
    L.pdllm_sparse_attn.argtypes = [shp, vp, vp, vp, vp, vp, vp, vp, i32, vp, vp, vp, vp, sz, vp]
    L.pdllm_sparse_attn_noalloc.argtypes = [shp, vp, vp, vp, vp, vp, vp, vp, i32, vp, vp, vp, vp]
    L.pdllm_lse_combine.argtypes = [vp, vp, i32, i64, i32, vp, vp, vp]
    L.pdllm_step.argtypes = [shp, vp, vp, vp, vp, vp, vp, i32, vp, vp, vp, vp, vp, vp, sz, vp]
    L.pdllm_step_profiled.argtypes = [shp, vp, vp, vp, vp, vp, vp, i32, vp, vp, vp, vp, vp, vp, sz,
                                      ctypes.POINTER(PdllmStageEvents), vp]
    L.pdllm_step_host.argtypes = [shp, vp, vp, vp, vp, vp, vp, i32, vp, vp, vp, vp, sz, ctypes.POINTER(PdllmSideStream), vp]
    dshp = ctypes.POINTER(PdllmDenseShape)
    L.pdllm_compact_kv.argtypes = [shp, vp, vp, vp, vp, vp, vp, vp]
    L.pdllm_dense_auto_splits.restype = i32
    L.pdllm_dense_auto_splits.argtypes = [dshp, i32]
    L.pdllm_dense_workspace_bytes.restype = sz
    L.pdllm_dense_workspace_bytes.argtypes = [dshp, i32, i32]
    L.pdllm_static_attn.argtypes = [dshp, vp, vp, vp, vp, vp, i32, vp, vp, vp, sz, vp]
    L.pdllm_prefill_attn.argtypes = [dshp, vp, vp, vp, i32, vp, vp, vp, sz, vp]
    L.pdllm_pool_keys.argtypes = [shp, vp, vp, vp]
    L.pdllm_score_chunks_pooled.argtypes = [shp, vp, i64, i64, vp, vp, vp]
    L.pdllm_score_tokens_workspace_bytes.restype = sz
    L.pdllm_score_tokens_workspace_bytes.argtypes = [shp]
    L.pdllm_score_tokens.argtypes = [shp, vp, i64, i64, vp, vp, vp, sz, vp]
    L.pdllm_select_topb.argtypes = [shp, vp, vp, vp]
    L.pdllm_score_tokens.restype = ctypes.c_int
    L.pdllm_select_topb.restype = ctypes.c_int
    for n in ("pdllm_compact_kv", "pdllm_static_attn", "pdllm_prefill_attn", "pdllm_pool_keys", "pdllm_score_chunks_pooled"):
        getattr(L, n).restype = ctypes.c_int
    for n in ("pdllm_score_chunks", "pdllm_select_topk", "pdllm_gather_idx", "pdllm_sparse_attn", "pdllm_lse_combine",
              "pdllm_step", "pdllm_step_profiled", "pdllm_step_host"):
        getattr(L, n).restype = ctypes.c_int
    L.pdllm_sparse_attn_noalloc.restype = ctypes.c_int
    _lib = L
    return L


def _check(rc: int):
    if rc != 0:
        raise PdllmError(f"pdllm error {rc}: {lib().pdllm_strerror(rc).decode()}")


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise PdllmError("no CUDA device: the pdllm hot path has no CPU fallback")
    return torch


def _ptr(t):
    return None if t is None else ctypes.c_void_p(t.data_ptr())


def _stream(stream=None):
    torch = _torch()
    s = torch.cuda.current_stream() if stream is None else stream
    return ctypes.c_void_p(s.cuda_stream)


def num_sms() -> int:
    torch = _torch()
    return torch.cuda.get_device_properties(torch.cuda.current_device()).multi_processor_count


def version() -> int:
    return lib().pdllm_version()


def auto_splits(shape: Shape, sms: int = 148) -> int:
    return lib().pdllm_auto_splits(ctypes.byref(shape.c()), sms)


def workspace_bytes(shape: Shape, n_splits: int = 0, sms: int = 148) -> int:
    return lib().pdllm_workspace_bytes(ctypes.byref(shape.c()), n_splits, sms)


def step_host_scratch_bytes(shape: Shape, n_splits: int = 0, sms: int = 148) -> int:
    return lib().pdllm_step_host_scratch_bytes(ctypes.byref(shape.c()), n_splits, sms)


def score_chunks(shape: Shape, Q, Kcache, scores=None, stream=None):
    """Q: bf16 [B,H,rows>=L_q,d] (the first L_q rows of every head are scored); returns scores fp32 [B,H_kv,N]."""
    torch = _torch()
    if scores is None:
        scores = torch.empty((shape.B, shape.H_kv, shape.N), dtype=torch.float32, device=Q.device)
    assert Q.is_contiguous() and Kcache.is_contiguous()
    _check(lib().pdllm_score_chunks(ctypes.byref(shape.c()), _ptr(Q), Q.stride(0), Q.stride(1), _ptr(Kcache),
                                    _ptr(scores), _stream(stream)))
    return scores


def select_topk(shape: Shape, scores, chunk_ids=None, stream=None):
    torch = _torch()
    if chunk_ids is None:
        chunk_ids = torch.empty((shape.B, shape.H_kv, shape.K), dtype=torch.int32, device=scores.device)
    _check(lib().pdllm_select_topk(ctypes.byref(shape.c()), _ptr(scores), _ptr(chunk_ids), _stream(stream)))
    return chunk_ids


def gather_idx(shape: Shape, chunk_ids, token_keep_idx=None, out=None, stream=None):
    torch = _torch()
    if out is None:
        out = torch.empty((shape.B, shape.H_kv, shape.K * shape.Bk), dtype=torch.int32, device=chunk_ids.device)
    _check(lib().pdllm_gather_idx(ctypes.byref(shape.c()), _ptr(chunk_ids), _ptr(token_keep_idx), _ptr(out),
                                  _stream(stream)))
    return out


def alloc_workspace(shape: Shape, n_splits: int = 0, device=None):
    torch = _torch()
    nbytes = workspace_bytes(shape, n_splits, num_sms())
    return torch.empty((max(nbytes, 16),), dtype=torch.uint8, device=device or "cuda")


def sparse_attn(shape: Shape, Q_dec, Kcache, Vcache, chunk_ids, token_keep_idx, K_dec, V_dec, n_splits=0,
                O=None, LSE=None, gather_idx_out=None, workspace=None, stream=None):
    torch = _torch()
    if O is None:
        O = torch.empty((shape.B, shape.H, shape.L, shape.d), dtype=torch.bfloat16, device=Q_dec.device)
    if LSE is None:
        LSE = torch.empty((shape.B, shape.H, shape.L), dtype=torch.float32, device=Q_dec.device)
    if workspace is None:
        workspace = alloc_workspace(shape, n_splits, Q_dec.device)
    _check(lib().pdllm_sparse_attn(ctypes.byref(shape.c()), _ptr(Q_dec), _ptr(Kcache), _ptr(Vcache), _ptr(chunk_ids),
                                   _ptr(token_keep_idx), _ptr(K_dec), _ptr(V_dec), n_splits, _ptr(O), _ptr(LSE),
                                   _ptr(gather_idx_out), _ptr(workspace), workspace.numel(), _stream(stream)))
    return O, LSE


def sparse_attn_noalloc(shape: Shape, Q_dec, Kcache, Vcache, chunk_ids, token_keep_idx, K_dec, V_dec, O, LSE, n_splits=0,
                        gather_idx_out=None, stream=None):
    """pdllm_sparse_attn without a workspace: the scratch is a fixed device array inside the library
    (NOALLOC_SCRATCH_BYTES); nothing is allocated here either -- O and LSE are the caller's.  Calls that overlap on one
    GPU race on that array."""
    _check(lib().pdllm_sparse_attn_noalloc(ctypes.byref(shape.c()), _ptr(Q_dec), _ptr(Kcache), _ptr(Vcache),
                                           _ptr(chunk_ids), _ptr(token_keep_idx), _ptr(K_dec), _ptr(V_dec), n_splits,
                                           _ptr(O), _ptr(LSE), _ptr(gather_idx_out), _stream(stream)))
    return O, LSE


def lse_combine(O_part, lse_part, O=None, LSE=None, stream=None):
    """O_part fp32 [S,rows,d], lse_part fp32 [S,rows] -> O bf16 [rows,d], LSE fp32 [rows]."""
    torch = _torch()
    S, rows, d = O_part.shape
    if O is None:
        O = torch.empty((rows, d), dtype=torch.bfloat16, device=O_part.device)
    if LSE is None:
        LSE = torch.empty((rows,), dtype=torch.float32, device=O_part.device)
    _check(lib().pdllm_lse_combine(_ptr(O_part), _ptr(lse_part), S, rows, d, _ptr(O), _ptr(LSE), _stream(stream)))
    return O, LSE


def step(shape: Shape, Q_dec, Kcache, Vcache, token_keep_idx, K_dec, V_dec, n_splits=0, scores=None, chunk_ids=None,
         O=None, LSE=None, gather_idx_out=None, workspace=None, stream=None, events=None):
    """One denoising step's attention: score_chunks -> select_topk -> sparse_attn (-> combine).

    events: optional 5 torch.cuda.Event(enable_timing=True), each recorded at least once before (torch creates the
    cudaEvent_t lazily); pdllm_step_profiled records them at the stage boundaries (begin, after_score, after_topk,
    after_attn, end) on the stream."""
    torch = _torch()
    dev = Q_dec.device
    if scores is None:
        scores = torch.empty((shape.B, shape.H_kv, shape.N), dtype=torch.float32, device=dev)
    if chunk_ids is None:
        chunk_ids = torch.empty((shape.B, shape.H_kv, shape.K), dtype=torch.int32, device=dev)
    if O is None:
        O = torch.empty((shape.B, shape.H, shape.L, shape.d), dtype=torch.bfloat16, device=dev)
    if LSE is None:
        LSE = torch.empty((shape.B, shape.H, shape.L), dtype=torch.float32, device=dev)
    if workspace is None:
        workspace = alloc_workspace(shape, n_splits, dev)
    args = (ctypes.byref(shape.c()), _ptr(Q_dec), _ptr(Kcache), _ptr(Vcache), _ptr(token_keep_idx),
            _ptr(K_dec), _ptr(V_dec), n_splits, _ptr(scores), _ptr(chunk_ids), _ptr(O), _ptr(LSE),
            _ptr(gather_idx_out), _ptr(workspace), workspace.numel())
    if events is None:
        _check(lib().pdllm_step(*args, _stream(stream)))
    else:
        ev = PdllmStageEvents(*[ctypes.c_void_p(e.cuda_event) for e in events])
        _check(lib().pdllm_step_profiled(*args, ctypes.byref(ev), _stream(stream)))
    return dict(scores=scores, chunk_ids=chunk_ids, O=O, LSE=LSE)


class SideStream:
    """A caller-owned side stream + fork / join events for step_host (the library keeps none of its own)."""

    def __init__(self, device=None):
        torch = _torch()
        self.stream = torch.cuda.Stream(device=device)
        self.ev_fork, self.ev_join = torch.cuda.Event(), torch.cuda.Event()
        for e in (self.ev_fork, self.ev_join):      # torch creates the cudaEvent_t on first record
            e.record(self.stream)

    def c(self) -> PdllmSideStream:
        return PdllmSideStream(self.stream.cuda_stream, self.ev_fork.cuda_event, self.ev_join.cuda_event)


def step_host(shape: Shape, h_Q_dec, h_K_dec, h_V_dec, d_Kcache, d_Vcache, d_token_keep_idx, n_splits, h_O, h_LSE,
              h_chunk_ids, d_scratch, side: "SideStream | None" = None, stream=None):
    """pdllm_step with HOST (pinned) per-step tensors: H2D copies, the step, D2H copies, all ordered on `stream`;
    with `side` the K_dec / V_dec copies run on that stream underneath the scoring kernel."""
    sd = ctypes.byref(side.c()) if side is not None else None
    _check(lib().pdllm_step_host(ctypes.byref(shape.c()), _ptr(h_Q_dec), _ptr(h_K_dec), _ptr(h_V_dec), _ptr(d_Kcache),
                                 _ptr(d_Vcache), _ptr(d_token_keep_idx), n_splits, _ptr(h_O), _ptr(h_LSE),
                                 _ptr(h_chunk_ids), _ptr(d_scratch), d_scratch.numel(), sd, _stream(stream)))


# ---------------------------------------------------------------------------------------------------------------
# rows after the hot path
def compact_kv(shape: Shape, Kcache, Vcache, chunk_ids, token_keep_idx=None, Kcompact=None, Vcompact=None, stream=None):
    """NEXT-3: the selected, token-thinned rows copied once -> (Kcompact, Vcompact) bf16 [B,H_kv,K*Bk,d]."""
    torch = _torch()
    shp = (shape.B, shape.H_kv, shape.K * shape.Bk, shape.d)
    if Kcompact is None:
        Kcompact = torch.empty(shp, dtype=torch.bfloat16, device=Kcache.device)
    if Vcompact is None:
        Vcompact = torch.empty(shp, dtype=torch.bfloat16, device=Kcache.device)
    _check(lib().pdllm_compact_kv(ctypes.byref(shape.c()), _ptr(Kcache), _ptr(Vcache), _ptr(chunk_ids), _ptr(token_keep_idx),
                                  _ptr(Kcompact), _ptr(Vcompact), _stream(stream)))
    return Kcompact, Vcompact


def dense_auto_splits(ds: DenseShape, sms: int = 148) -> int:
    return lib().pdllm_dense_auto_splits(ctypes.byref(ds.c()), sms)


def dense_workspace_bytes(ds: DenseShape, n_splits: int = 0, sms: int = 148) -> int:
    return lib().pdllm_dense_workspace_bytes(ctypes.byref(ds.c()), n_splits, sms)


def alloc_dense_workspace(ds: DenseShape, n_splits: int = 0, device=None):
    torch = _torch()
    return torch.empty((max(dense_workspace_bytes(ds, n_splits, num_sms()), 16),), dtype=torch.uint8, device=device or "cuda")


def static_attn(ds: DenseShape, Q_dec, Kcompact, Vcompact, K_dec, V_dec, n_splits=0, O=None, LSE=None, workspace=None,
                stream=None):
    """NEXT-3: attention over [compact static cache || decode rows], K/V fetched as TMA tiles."""
    torch = _torch()
    if O is None:
        O = torch.empty((ds.B, ds.H, ds.L, ds.d), dtype=torch.bfloat16, device=Q_dec.device)
    if LSE is None:
        LSE = torch.empty((ds.B, ds.H, ds.L), dtype=torch.float32, device=Q_dec.device)
    if workspace is None:
        workspace = alloc_dense_workspace(ds, n_splits, Q_dec.device)
    _check(lib().pdllm_static_attn(ctypes.byref(ds.c()), _ptr(Q_dec), _ptr(Kcompact), _ptr(Vcompact), _ptr(K_dec), _ptr(V_dec),
                                   n_splits, _ptr(O), _ptr(LSE), _ptr(workspace), workspace.numel(), _stream(stream)))
    return O, LSE


def prefill_attn(ds: DenseShape, Q, K, V, n_splits=0, O=None, LSE=None, workspace=None, stream=None):
    """NEXT-2: bidirectional attention of ds.B independent sequences of T = ds.S_pre = ds.L rows (ds.L_s == 0)."""
    torch = _torch()
    if O is None:
        O = torch.empty((ds.B, ds.H, ds.L, ds.d), dtype=torch.bfloat16, device=Q.device)
    if LSE is None:
        LSE = torch.empty((ds.B, ds.H, ds.L), dtype=torch.float32, device=Q.device)
    if workspace is None:
        workspace = alloc_dense_workspace(ds, n_splits, Q.device)
    _check(lib().pdllm_prefill_attn(ctypes.byref(ds.c()), _ptr(Q), _ptr(K), _ptr(V), n_splits, _ptr(O), _ptr(LSE),
                                    _ptr(workspace), workspace.numel(), _stream(stream)))
    return O, LSE


def pool_keys(shape: Shape, Kcache, kbar=None, stream=None):
    """NEXT-3 (R23): mean key of every chunk -> fp32 [B,H_kv,N,d]."""
    torch = _torch()
    if kbar is None:
        kbar = torch.empty((shape.B, shape.H_kv, shape.N, shape.d), dtype=torch.float32, device=Kcache.device)
    _check(lib().pdllm_pool_keys(ctypes.byref(shape.c()), _ptr(Kcache), _ptr(kbar), _stream(stream)))
    return kbar


def score_chunks_pooled(shape: Shape, Q, kbar, scores=None, stream=None):
    """NEXT-3 (R23): log(C+1) + scale * <mean scoring row, mean key> -> fp32 [B,H_kv,N]."""
    torch = _torch()
    if scores is None:
        scores = torch.empty((shape.B, shape.H_kv, shape.N), dtype=torch.float32, device=Q.device)
    _check(lib().pdllm_score_chunks_pooled(ctypes.byref(shape.c()), _ptr(Q), Q.stride(0), Q.stride(1), _ptr(kbar),
                                           _ptr(scores), _stream(stream)))
    return scores


def score_tokens(shape: Shape, Q, Kcache, token_scores=None, workspace=None, stream=None):
    """NEXT-1: token eviction scores (Eq. 5, query->chunk) -> fp32 [B,H_kv,N,C+1]."""
    torch = _torch()
    if token_scores is None:
        token_scores = torch.empty((shape.B, shape.H_kv, shape.N, shape.C + 1), dtype=torch.float32, device=Q.device)
    if workspace is None:
        nbytes = lib().pdllm_score_tokens_workspace_bytes(ctypes.byref(shape.c()))
        workspace = torch.empty((max(nbytes, 16),), dtype=torch.uint8, device=Q.device)
    assert Q.is_contiguous() and Kcache.is_contiguous()
    _check(lib().pdllm_score_tokens(ctypes.byref(shape.c()), _ptr(Q), Q.stride(0), Q.stride(1), _ptr(Kcache),
                                    _ptr(token_scores), _ptr(workspace), workspace.numel(), _stream(stream)))
    return token_scores


def select_topb(shape: Shape, token_scores, token_keep_idx=None, stream=None):
    """NEXT-1: per chunk BOS + the Bk-1 best slots, ascending -> int32 [B,H_kv,N,Bk]."""
    torch = _torch()
    if token_keep_idx is None:
        token_keep_idx = torch.empty((shape.B, shape.H_kv, shape.N, shape.Bk), dtype=torch.int32, device=token_scores.device)
    _check(lib().pdllm_select_topb(ctypes.byref(shape.c()), _ptr(token_scores), _ptr(token_keep_idx), _stream(stream)))
    return token_keep_idx
