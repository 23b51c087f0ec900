"""Helpers of the GPU parity tests: host<->device marshalling and the tolerance gates of
DESIGN.md / SURVEY 8(c) R12.  No method arithmetic here."""
import numpy as np
import torch

from paper_2606_10537_b200 import binding

# R12 (BASELINE.json north_star: max-abs 2e-2 / max-rel 1e-2 on O, 1e-3 on LSE for bf16 inputs)
O_ABS, O_REL, O_NORM_REL, LSE_ABS, SCORE_ABS = 2e-2, 1e-2, 1e-2, 1e-3, 1e-3


def dev_bf16(bits: np.ndarray) -> torch.Tensor:
    """uint16 bf16 bit patterns -> torch.bfloat16 CUDA tensor (bit-exact)."""
    return torch.from_numpy(np.ascontiguousarray(bits).view(np.int16)).cuda().view(torch.bfloat16)


def dev_i32(a):
    return None if a is None else torch.from_numpy(np.ascontiguousarray(a, dtype=np.int32)).cuda()


def dev_f32(a):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()


def host_bf16_as_f64(t: torch.Tensor) -> np.ndarray:
    bits = t.detach().contiguous().view(torch.int16).cpu().numpy().view(np.uint16)
    return (bits.astype(np.uint32) << 16).view(np.float32).astype(np.float64)


def to_device(inp: dict) -> dict:
    return dict(Q_dec=dev_bf16(inp["Q_dec"]), Kcache=dev_bf16(inp["Kcache"]), Vcache=dev_bf16(inp["Vcache"]),
                K_dec=dev_bf16(inp["K_dec"]), V_dec=dev_bf16(inp["V_dec"]), keep=dev_i32(inp["keep"]))


def shape_of(inp: dict, K: int, L_q: int) -> binding.Shape:
    B, H, L, d = inp["Q_dec"].shape
    _, H_kv, N, Cp, _ = inp["Kcache"].shape
    Bk = Cp if inp["keep"] is None else inp["keep"].shape[-1]
    return binding.Shape(B, H, H_kv, d, N, Cp - 1, K, Bk, L_q, L, inp["K_dec"].shape[2])


def check_O(O_gpu: torch.Tensor, O_ref: np.ndarray, mask=None, what="O"):
    """R12: every element |d| <= 2e-2 + 1e-2 |ref|, and max|d| / max|ref| <= 1e-2."""
    got = host_bf16_as_f64(O_gpu)
    if mask is not None:
        got, O_ref = got[mask], O_ref[mask]
    assert np.isfinite(got).all(), f"{what}: non-finite GPU values"
    diff = np.abs(got - O_ref)
    lim = O_ABS + O_REL * np.abs(O_ref)
    worst = float((diff - lim).max())
    assert worst <= 0, f"{what}: element-wise gate exceeded by {worst:.3e} (max|d|={diff.max():.3e})"
    ratio = diff.max() / max(np.abs(O_ref).max(), 1e-30)
    assert ratio <= O_NORM_REL, f"{what}: max|d|/max|ref| = {ratio:.3e}"
    return float(diff.max()), float(ratio)


def check_close(got: torch.Tensor, ref: np.ndarray, tol: float, mask=None, what="LSE"):
    g = got.detach().double().cpu().numpy()
    if mask is not None:
        g, ref = g[mask], ref[mask]
    both_ninf = np.isneginf(g) & np.isneginf(ref)
    d = np.where(both_ninf, 0.0, np.abs(g - ref))
    assert np.isfinite(d).all(), f"{what}: non-finite difference"
    assert d.max() <= tol, f"{what}: max|d| = {d.max():.3e} > {tol}"
    return float(d.max())


def check_exact(got: torch.Tensor, ref: np.ndarray, what="ids"):
    g = got.detach().cpu().numpy()
    assert g.shape == ref.shape and (g == ref).all(), f"{what}: mismatch at {np.argwhere(g != ref)[:5].tolist()}"
