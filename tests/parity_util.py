"""Shared helpers of the GPU parity tests: tolerances (BASELINE.json north_star) and host<->device marshalling.

Tolerances (bf16 inputs, fp32 accumulation; R17 applies the same numbers to fp32 inputs):
  per-row KL   |err| <= 2e-3 + 1e-2*|ref|
  lse          |err| <= 1e-3
  gradients    cosine similarity >= 0.999 and max|g - ref| / max|ref| <= 3e-2   (R16), evaluated PER (batch, head):
               a head with small gradients must not hide behind a head with large ones (check_grad_heads)
"""
from __future__ import annotations

import numpy as np

KL_ATOL, KL_RTOL = 2e-3, 1e-2
LSE_ATOL = 1e-3
GRAD_COS, GRAD_MAXREL = 0.999, 3e-2
GRAD_ZERO_ATOL = 1e-4


def to_torch(a: np.ndarray, device="cuda"):
    """numpy (uint16 bf16 bits | float16 | float32) -> torch tensor on `device` (bfloat16 | float16 | float32)."""
    import torch

    if a.dtype == np.uint16:
        return torch.from_numpy(a.view(np.int16).copy()).view(torch.bfloat16).to(device)
    return torch.from_numpy(np.ascontiguousarray(a)).to(device)


def to_f64(t) -> np.ndarray:
    """torch tensor (any float dtype, any device) -> numpy float64, exact widening."""
    import torch

    return t.detach().to("cpu").to(torch.float64).numpy()


def bits_to_f64(a: np.ndarray) -> np.ndarray:
    if a.dtype == np.uint16:
        return (a.astype(np.uint32) << np.uint32(16)).view(np.float32).astype(np.float64)
    return a.astype(np.float64)


def check_fwd(got_kl, got_l1, got_l2, ref, what=""):
    kl, l1, l2 = (np.asarray(x, dtype=np.float64) for x in (got_kl, got_l1, got_l2))
    assert np.isfinite(kl).all() and np.isfinite(l1).all() and np.isfinite(l2).all(), f"{what}: non-finite output"
    e1 = np.abs(l1 - ref["lse1"]).max(initial=0.0)
    e2 = np.abs(l2 - ref["lse2"]).max(initial=0.0)
    assert e1 <= LSE_ATOL, f"{what}: lse1 max err {e1:.3e} > {LSE_ATOL}"
    assert e2 <= LSE_ATOL, f"{what}: lse2 max err {e2:.3e} > {LSE_ATOL}"
    err = np.abs(kl - ref["kl"])
    bound = KL_ATOL + KL_RTOL * np.abs(ref["kl"])
    worst = (err - bound).max(initial=-1.0)
    assert worst <= 0, f"{what}: KL err exceeds 2e-3+1e-2|ref| by {worst:.3e} (max err {err.max():.3e})"
    return {"kl_err": float(err.max(initial=0.0)), "lse_err": float(max(e1, e2))}


def grad_metrics(got, ref):
    got = np.asarray(got, dtype=np.float64).ravel()
    ref = np.asarray(ref, dtype=np.float64).ravel()
    nr = np.linalg.norm(ref)
    ng = np.linalg.norm(got)
    if nr == 0.0:
        # the exact gradient vanishes identically (e.g. NK = 1: P1 = P2 = 1): cosine is undefined, so the bar is
        # absolute -- |got| <= GRAD_ZERO_ATOL, the size of an fp32 rounding of P (1e-6) times O(10) operands
        amax = float(np.abs(got).max(initial=0.0))
        return (1.0 if amax <= GRAD_ZERO_ATOL else 0.0), 0.0
    cos = float(got @ ref / (ng * nr)) if ng > 0 else 0.0
    rel = float(np.abs(got - ref).max() / np.abs(ref).max())
    return cos, rel


def check_grad(got, ref, what=""):
    assert np.isfinite(np.asarray(got, dtype=np.float64)).all(), f"{what}: non-finite gradient"
    cos, rel = grad_metrics(got, ref)
    assert cos >= GRAD_COS, f"{what}: cosine {cos:.6f} < {GRAD_COS}"
    assert rel <= GRAD_MAXREL, f"{what}: max|err|/max|ref| {rel:.3e} > {GRAD_MAXREL}"
    return cos, rel


def check_grad_heads(got, ref, what=""):
    """The gradient bars applied to every (batch, head) slice of [..., N, d] tensors separately; returns the worst
    (min cosine, max relative error) over the heads."""
    got = np.asarray(got, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    assert got.shape == ref.shape, f"{what}: shape {got.shape} vs {ref.shape}"
    if got.ndim <= 2:
        return check_grad(got, ref, what)
    g3 = got.reshape((-1,) + got.shape[-2:])
    r3 = ref.reshape((-1,) + ref.shape[-2:])
    worst_cos, worst_rel = 1.0, 0.0
    for i in range(g3.shape[0]):
        cos, rel = check_grad(g3[i], r3[i], f"{what} [head {i}]")
        worst_cos, worst_rel = min(worst_cos, cos), max(worst_rel, rel)
    return worst_cos, worst_rel
