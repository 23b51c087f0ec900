"""pdllm_sparse_attn_noalloc: the entry point that allocates nothing (its scratch is a fixed device array inside the
library, include/pdllm.h PDLLM_NOALLOC_SCRATCH_BYTES) against the existing path pdllm_sparse_attn, which gets a
caller-allocated workspace.  Collected last on purpose (the suite runs with pytest -x)."""
import ctypes
import re
from pathlib import Path

import pytest
import torch

from paper_2606_10537_b200 import binding as B
from paper_2606_10537_b200 import workloads as W

from gpu_util import LSE_ABS, check_close, check_O, dev_i32, host_bf16_as_f64, to_device

ROOT = Path(__file__).resolve().parents[1]


def test_limit_matches_the_header_and_oversized_requests_are_refused():
    """Host-side only (nothing reaches a device): the binding's constants are the header's, and an explicit split count
    whose partials exceed the fixed array is refused with the dedicated status before any pointer is looked at."""
    hdr = (ROOT / "include" / "pdllm.h").read_text()
    m = re.search(r"#define\s+PDLLM_NOALLOC_SCRATCH_BYTES\s+\((\d+)u\s*<<\s*(\d+)\)", hdr)
    assert m and int(m.group(1)) << int(m.group(2)) == B.NOALLOC_SCRATCH_BYTES
    assert int(re.search(r"PDLLM_ERR_SCRATCH_LIMIT\s*=\s*(-\d+)", hdr).group(1)) == B.ERR_SCRATCH_LIMIT
    lib = B.lib()
    assert b"PDLLM_NOALLOC_SCRATCH_BYTES" in lib.pdllm_strerror(B.ERR_SCRATCH_LIMIT)
    shape = B.Shape.of(W.CONFIGS["sparse32k"])            # 49152 output rows: 25 MB of fp32 partials per split
    need = lib.pdllm_workspace_bytes(ctypes.byref(shape.c()), 2, 148)
    assert need > B.NOALLOC_SCRATCH_BYTES
    rc = lib.pdllm_sparse_attn_noalloc(ctypes.byref(shape.c()), None, None, None, None, None, None, None, 2, None, None,
                                       None, None)
    assert rc == B.ERR_SCRATCH_LIMIT
    assert lib.pdllm_workspace_bytes(ctypes.byref(shape.c()), 1, 148) <= B.NOALLOC_SCRATCH_BYTES   # one split always fits


def test_noalloc_refuses_to_run_under_the_debug_switch(monkeypatch):
    """PDLLM_DEBUG_VALIDATE=1 makes the workspace path allocate a flag and synchronise; the call that must not allocate
    says so (host-side, before anything reaches a device) instead of skipping the check silently."""
    lib = B.lib()
    shape = B.Shape.of(W.CONFIGS["tiny"])
    monkeypatch.setenv("PDLLM_DEBUG_VALIDATE", "1")
    rc = lib.pdllm_sparse_attn_noalloc(ctypes.byref(shape.c()), None, None, None, None, None, None, None, 1, None, None,
                                       None, None)
    assert rc == -5 and b"unsupported" in lib.pdllm_strerror(rc)
    monkeypatch.setenv("PDLLM_DEBUG_VALIDATE", "0")
    rc = lib.pdllm_sparse_attn_noalloc(ctypes.byref(shape.c()), None, None, None, None, None, None, None, 1 << 20, None,
                                       None, None, None)
    assert rc != -5                                       # (an absurd split count: refused for its size or shape, not the switch)


def _case(w, S):
    inp = W.make_inputs(w)
    dev = to_device(inp)
    ids = dev_i32(inp["planted"])
    shape = B.Shape.of(w)
    args = (shape, dev["Q_dec"], dev["Kcache"], dev["Vcache"], ids, dev["keep"], dev["K_dec"], dev["V_dec"])
    O_ref, LSE_ref = B.sparse_attn(*args, n_splits=S)     # the existing path: workspace allocated by the binding
    O = torch.full((w.B, w.H, w.L, w.d), float("nan"), dtype=torch.bfloat16, device="cuda")
    LSE = torch.full((w.B, w.H, w.L), float("nan"), dtype=torch.float32, device="cuda")
    return args, S, O_ref, LSE_ref, O, LSE


def _compare(O, LSE, O_ref, LSE_ref, what):
    # the tolerance of the parity tests (R12); the two paths run the same kernels, so they agree to the bit
    check_O(O, host_bf16_as_f64(O_ref), what=f"O ({what})")
    check_close(LSE, LSE_ref.double().cpu().numpy(), LSE_ABS, what=f"LSE ({what})")
    assert torch.equal(O.view(torch.int16), O_ref.view(torch.int16)), f"O differs from the workspace path ({what})"
    assert torch.equal(LSE.view(torch.int32), LSE_ref.view(torch.int32)), f"LSE differs from the workspace path ({what})"


@pytest.mark.gpu
def test_noalloc_matches_the_workspace_path_on_calls_in_a_row():
    """Two calls in a row on different shapes and split counts (the second finds the first one's partials and a used
    work-item counter in the shared array), then the second once more with the device's free memory read around it."""
    B.lib()
    first = _case(W.small_variant(W.CONFIGS["tiny"], C=300, H=8, H_kv=2, d=128, N=6, K=3, keep=0.5, L_q=40, L_d=216), 3)
    second = _case(W.small_variant(W.CONFIGS["tiny"], C=200, H=4, H_kv=4, d=64, N=9, K=4, keep=1.0, L_q=16, L_d=150), 2)
    torch.cuda.synchronize()
    for what, (args, S, O_ref, LSE_ref, O, LSE) in (("first call, 3 splits", first), ("second call, 2 splits", second)):
        B.sparse_attn_noalloc(*args, O, LSE, n_splits=S)
    torch.cuda.synchronize()
    for what, (args, S, O_ref, LSE_ref, O, LSE) in (("first call, 3 splits", first), ("second call, 2 splits", second)):
        _compare(O, LSE, O_ref, LSE_ref, what)

    args, S, O_ref, LSE_ref, O, LSE = second
    O.fill_(float("nan"))
    LSE.fill_(float("nan"))
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    B.sparse_attn_noalloc(*args, O, LSE, n_splits=S)
    B.sparse_attn_noalloc(*args, O, LSE, n_splits=0)      # the auto choice, bounded by what the array holds
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before, "device memory was allocated or freed by the call"
    O_auto, LSE_auto = B.sparse_attn(*args, n_splits=0)
    torch.cuda.synchronize()
    _compare(O, LSE, O_auto, LSE_auto, "third call, auto splits")


@pytest.mark.gpu
def test_noalloc_refuses_an_oversized_request_with_real_pointers():
    """With valid device buffers the oversized request is still refused, the outputs stay untouched, and the call
    keeps working afterwards."""
    B.lib()
    w = W.small_variant(W.CONFIGS["tiny"], B=2, C=64, H=32, H_kv=32, d=128, N=4, K=2, keep=1.0, L_q=16, L_d=1008)
    shape = B.Shape.of(w)                                 # 65536 output rows: 33.6 MB of fp32 partials per split
    assert B.lib().pdllm_workspace_bytes(ctypes.byref(shape.c()), 2, 148) > B.NOALLOC_SCRATCH_BYTES
    args, S, O_ref, LSE_ref, O, LSE = _case(w, 1)
    with pytest.raises(B.PdllmError, match="PDLLM_NOALLOC_SCRATCH_BYTES"):
        B.sparse_attn_noalloc(*args, O, LSE, n_splits=2)
    torch.cuda.synchronize()
    assert torch.isnan(LSE).all(), "a refused call wrote to its outputs"
    B.sparse_attn_noalloc(*args, O, LSE, n_splits=0)      # auto: falls back to the one split the array holds
    torch.cuda.synchronize()
    _compare(O, LSE, O_ref, LSE_ref, "auto splits capped by the array")
