"""CPU-side checks of the boundary: the C-ABI library builds, loads without a GPU and exports every
symbol include/pdllm.h declares; host-only helpers (split choice, workspace sizes, validation)."""
import ctypes
import re
from pathlib import Path

import pytest

from paper_2606_10537_b200 import binding as B
from paper_2606_10537_b200 import workloads as W

ROOT = Path(__file__).resolve().parents[1]


def declared_symbols():
    hdr = (ROOT / "include" / "pdllm.h").read_text()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    return sorted(set(re.findall(r"\b(pdllm_[a-z_0-9]+)\s*\(", hdr)))


def test_library_exports_every_declared_symbol():
    lib = B.lib()
    names = declared_symbols()
    assert len(names) >= 12
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(B.EXPORTS) == names


def test_header_constants_match_the_binding():
    hdr = (ROOT / "include" / "pdllm.h").read_text()
    assert int(re.search(r"#define\s+PDLLM_FOLD_MAX_N\s+(\d+)", hdr).group(1)) == B.FOLD_MAX_N


def test_version_and_strerror():
    lib = B.lib()
    assert lib.pdllm_version() >= 100
    for rc in range(0, -8, -1):
        assert lib.pdllm_strerror(rc)


@pytest.mark.parametrize("name,expect_min,expect_max", [("tiny", 1, 1), ("llada8k", 2, 5), ("dream16k", 2, 5),
                                                        ("sparse32k", 1, 1)])
def test_auto_splits(name, expect_min, expect_max):
    """a6: C4 has 384 M tiles >= 2*148 slots -> S = 1; C2/C3 (96 / 84 tiles) need a few splits."""
    s = B.auto_splits(B.Shape.of(W.CONFIGS[name]), 148)
    assert expect_min <= s <= expect_max, s


@pytest.mark.parametrize("name", ["fig5b", "fig5b_8k", "fig5b_16k", "fig5b_32k"])
def test_auto_splits_fig5b_shapes_fill_one_wave(name):
    """The Fig. 5(b) decode shapes are 8 KV groups of one query tile: the split count is what turns them into about one
    wave of work items (8 * S <= 148 SMs), far beyond the paper's S = 4 (measured: profiles/r2_splitsweep_dream16k.md)."""
    s = B.auto_splits(B.Shape.of(W.EXTRA[name]), 148)
    assert 11 <= s <= 18, s
    # a big batch needs none: its work items fill the SMs by themselves and its partials would go through HBM
    big = W.small_variant(W.CONFIGS["sparse32k"], B=8, N=16, C=1024, K=16, keep=1.0, L_q=64, L_d=512)
    assert B.auto_splits(B.Shape.of(big), 148) == 1


def test_workspace_bytes():
    w = W.CONFIGS["sparse32k"]
    sh = B.Shape.of(w)
    assert B.workspace_bytes(sh, 1, 148) == 256          # the persistent kernel's work-item counter
    rows = w.B * w.H * w.L
    got = B.workspace_bytes(sh, 2, 148)
    assert got >= 256 + 2 * rows * (w.d + 1) * 4 and got <= 256 + 2 * rows * (w.d + 1) * 4 + 1024
    # more splits than KV tiles are capped (no empty split, R10)
    tiles = -(-w.S_kv // 128)
    assert B.workspace_bytes(sh, 1000, 148) == B.workspace_bytes(sh, tiles, 148)
    assert B.step_host_scratch_bytes(sh, 1, 148) > 2 * rows * w.d * 2


def test_invalid_shapes_rejected_without_gpu():
    lib = B.lib()
    bad = B.Shape(1, 4, 3, 64, 8, 64, 2, 33, 16, 48, 48)          # H % H_kv != 0
    assert B.workspace_bytes(bad, 2, 148) == 0
    null = ctypes.c_void_p(0)
    rc = lib.pdllm_select_topk(ctypes.byref(bad.c()), null, null, null)
    assert rc == -1                                               # NULL pointers are reported first
    good = B.Shape.of(W.CONFIGS["tiny"])
    one = ctypes.c_void_p(16)
    assert lib.pdllm_select_topk(ctypes.byref(bad.c()), one, one, null) == -3
    d96 = B.Shape(1, 4, 4, 96, 8, 64, 2, 33, 16, 48, 48)
    assert lib.pdllm_gather_idx(ctypes.byref(d96.c()), one, one, one, null) == -3
    assert lib.pdllm_lse_combine(one, one, 0, 10, 128, one, one, null) == -3
    assert lib.pdllm_sparse_attn(ctypes.byref(good.c()), one, one, one, one, one, one, one, -1, one, one, null, null, 0,
                                 null) == -3


def test_binding_refuses_to_run_without_cuda():
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA present")
    with pytest.raises(B.PdllmError):
        B.score_chunks(B.Shape.of(W.CONFIGS["tiny"]), torch.zeros(1), torch.zeros(1))
