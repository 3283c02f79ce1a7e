"""GPU parity on inputs built to break the forward's running-reference logic and the kernels' tail handling.

The forward keeps a per-row softmax reference that is NOT recomputed on every tile ("lazy reference": Eq.8-10,
PAPER.md:149-154/:196-206, hold for any reference as long as (l, acc) are relative to it); it is only raised -- and
(l1, l2, acc) rescaled as Alg.1 lines 8-12 do -- when a tile shows that the reference is stale.  With i.i.d. N(0,1) logits that
path is never taken after a row's first tile, so these cases plant it: a key in a LATE tile whose logit sits +25 / +60 / +140
log2-units above everything the row has seen, at column positions that cover every column residue of the kernel's per-thread
32-column groups (the columns evaluated by the FMA-pipe polynomial as well as the MUFU ones), for P1 only, P2 only and both,
causal and not, through the default kernel and through split-K.  Everything is compared with the float64 definition
element by element at the north-star tolerances; the backward runs on the same inputs (its P = exp(s - lse) sees the same spikes).

Second family: logits shifted far negative (lse < -100) with ragged NK, so that a zero-filled TMA tail row would give
P = exp(0 - lse) = inf -- every kernel has to mask those rows, including the ones whose tail rows feed a contraction.
"""
from __future__ import annotations

import numpy as np
import pytest

import workloads as W
from oracle.streamkl_oracle import attention_kl
from parity_util import bits_to_f64, check_fwd, check_grad_heads, to_f64, to_torch

pytestmark = pytest.mark.gpu

LOG2E = 1.4426950408889634


def _bf16_round(a: np.ndarray) -> np.ndarray:
    """float32 -> bf16 bits (round to nearest even), as workloads.py does for the seeded inputs."""
    return W.f32_to_bf16_bits(np.ascontiguousarray(a, dtype=np.float32))


def _planted(cfg: W.Config, which: str, jump_log2: float, row: int, key: int):
    """cfg's seeded inputs with key `key` of every head replaced by lam * Q_t[row] for the distributions in `which`
    ('1', '2' or '12'): logit(row, key) = c_t lam |q|^2, chosen `jump_log2` log2-units above the typical row maximum."""
    inp = W.all_inputs(cfg)
    out = {k: v.copy() for k, v in inp.items()}
    for t, d, c in (("1", cfg.d1, cfg.c1), ("2", cfg.d2, cfg.c2)):
        if t not in which:
            continue
        q = bits_to_f64(inp["Q" + t])[:, :, row, :]                         # [B,H,d]
        n2 = (q * q).sum(-1, keepdims=True)
        lam = (jump_log2 + 8.0) / (c * LOG2E * n2)                           # +8: above the ~5-sigma maximum of N(0,1) logits
        out["K" + t][:, :, key, :] = _bf16_round(lam * q)
    return out


def _run_and_check(cfg, inp, what, splitk=False, bwd=True, teacher=True):
    import paper_2606_20005_b200 as skl

    Q1, K1, Q2, K2 = (to_torch(inp[k]) for k in ("Q1", "K1", "Q2", "K2"))
    g = to_torch(inp["g"])
    ref = attention_kl(*(bits_to_f64(inp[k]) for k in ("Q1", "K1", "Q2", "K2")), cfg.c1, cfg.c2, cfg.causal,
                       g=inp["g"].astype(np.float64), teacher=teacher)
    kl, l1, l2 = skl.streamkl_fwd(Q1, K1, Q2, K2, cfg.c1, cfg.c2, cfg.causal)
    check_fwd(to_f64(kl), to_f64(l1), to_f64(l2), ref, what + " fwd")
    if splitk:
        for W_ in (2, 3):
            ks, l1s, l2s = skl.streamkl_fwd_splitk(Q1, K1, Q2, K2, cfg.c1, cfg.c2, cfg.causal, splits=W_)
            check_fwd(to_f64(ks), to_f64(l1s), to_f64(l2s), ref, f"{what} split-K W={W_}")
    if bwd:
        grads = skl.streamkl_bwd(Q1, K1, Q2, K2, cfg.c1, cfg.c2, cfg.causal, kl, l1, l2, g, teacher=teacher)
        for name, t in zip(("dQ1", "dK1", "dQ2", "dK2"), grads):
            if t is not None:
                check_grad_heads(to_f64(t), ref[name], f"{what} {name}")
    return ref


@pytest.mark.parametrize("jump", [25.0, 60.0, 140.0])
@pytest.mark.parametrize("which", ["1", "2", "12"])
@pytest.mark.parametrize("causal", [False, True])
def test_late_spike_raises_a_stale_reference(jump, which, causal):
    """A spike in key tile 5 of 7 (and, for the causal case, visible to the planted row and every later row), swept over
    eight column positions that cover all residues mod 8 and three of the four 32-column groups."""
    d2 = 64 if which == "1" else 128
    for col in (0, 1, 2, 5, 39, 44, 70, 127):
        cfg = W.Config(60, "spike", 1, 2, 384, 900, 128, d2, "bf16", causal)
        key = 5 * 128 + col
        row = 383 if causal else 17            # causal: row 383 sees keys <= 383 + 516 = 899
        inp = _planted(cfg, which, jump, row, key)
        ref = _run_and_check(cfg, inp, f"spike +{jump} P{which} col {col} causal={causal}", splitk=(col in (1, 44)), bwd=(col in (0, 39)))
        # the planted row is (nearly) one-hot in the planted distribution: its lse equals the planted logit
        t = which[0]
        assert ref["lse" + t][0, 0, row] > (jump + 4.0) / LOG2E


def test_spike_in_first_tile_then_everything_far_below():
    """The mirror case: the maximum comes first and every later logit underflows relative to it (exp2(x), x < -126)."""
    cfg = W.Config(61, "spike-first", 1, 2, 256, 1024, 128, 128, "bf16", False)
    for col in (0, 3, 9, 64):
        inp = _planted(cfg, "12", 160.0, 5, col)
        _run_and_check(cfg, inp, f"first-tile spike col {col}", splitk=True)


def test_two_spikes_of_increasing_height():
    """Two raises in one row (tile 2: +30, tile 6: +90) -- the rescale factors compose (Eq.10)."""
    cfg = W.Config(62, "two-spikes", 1, 2, 256, 1024, 128, 64, "bf16", False)
    inp = _planted(cfg, "12", 30.0, 40, 2 * 128 + 8)
    base = W.all_inputs(cfg)
    for t, d, c in (("1", cfg.d1, cfg.c1), ("2", cfg.d2, cfg.c2)):
        q = bits_to_f64(base["Q" + t])[:, :, 40, :]
        lam = 98.0 / (c * LOG2E * (q * q).sum(-1, keepdims=True))
        inp["K" + t][:, :, 6 * 128 + 33, :] = _bf16_round(lam * q)
    _run_and_check(cfg, inp, "two spikes", splitk=True)


@pytest.mark.parametrize("NK", [200, 515, 1000])
@pytest.mark.parametrize("causal", [False, True])
def test_strongly_negative_logits_and_ragged_key_tails(NK, causal):
    """Every logit ~ -150 nats (lse < -100) and NK % 128 != 0: exp(0 - lse) of a zero-filled tail key overflows fp32.  Forward,
    split-K, Setting-2 backward and both Setting-1 strategies (the fused kernel contracts over its owned key tile)."""
    import paper_2606_20005_b200 as skl

    NQ = min(NK, 300)
    cfg = W.Config(63, "negshift", 1, 2, NQ, NK, 128, 64, "bf16", causal)
    inp = W.all_inputs(cfg)
    out = {k: v.copy() for k, v in inp.items()}
    for t, d, c in (("1", cfg.d1, cfg.c1), ("2", cfg.d2, cfg.c2)):
        shift = np.sqrt(150.0 / c) / np.sqrt(d)                            # (q + s e).(k - s e) ~ q.k - s^2 d  = -150 / c
        out["Q" + t] = _bf16_round(bits_to_f64(inp["Q" + t]) + shift)
        out["K" + t] = _bf16_round(bits_to_f64(inp["K" + t]) - shift)
    ref = _run_and_check(cfg, out, f"negative shift NK={NK}", splitk=True, teacher=True)
    assert ref["lse1"].max() < -100.0 and ref["lse2"].max() < -100.0
    Q1, K1, Q2, K2 = (to_torch(out[k]) for k in ("Q1", "K1", "Q2", "K2"))
    g = to_torch(out["g"])
    kl, l1, l2 = skl.streamkl_fwd(Q1, K1, Q2, K2, cfg.c1, cfg.c2, cfg.causal)
    try:
        for mode in (skl.STREAMKL_BWD_FUSED, skl.STREAMKL_BWD_SEPARATE, skl.STREAMKL_BWD_AUTO):
            skl.streamkl_set_bwd_mode(mode)
            _, _, dQ2, dK2 = skl.streamkl_bwd(Q1, K1, Q2, K2, cfg.c1, cfg.c2, cfg.causal, kl, l1, l2, g, teacher=False)
            check_grad_heads(to_f64(dQ2), ref["dQ2"], f"negshift mode {mode} dQ2")
            check_grad_heads(to_f64(dK2), ref["dK2"], f"negshift mode {mode} dK2")
    finally:
        skl.streamkl_set_bwd_mode(skl.STREAMKL_BWD_AUTO)
