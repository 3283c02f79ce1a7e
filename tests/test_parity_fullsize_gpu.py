"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (same entry points, same
shapes, whole batch in one call), against the float64 oracle on outputs the oracle can compute one by one:

  * kl / lse1 / lse2 / dQ rows: a sample of query rows per sampled head (first, last, every 128/256-row tile boundary
    +-1 near both ends, seeded random rows) -- `attention_kl_rows` is exact for any row subset.
  * dK: the whole head for cfg 2/3/5 (one head each).  cfg 4 (the bench workload; ">= 2 whole heads, first
    and last -- needed for dK, which sums over all rows"): heads 0 and 31 in full -- every kl / lse / dQ row and all of
    dK1, dK2, i.e. also the early key tiles whose K-owner CTAs stream all 1024 query tiles.  The oracle is called block by
    block on the causal prefix the block can see (rows r0..r1-1 of a causal NQ = NK head see keys < r1 only: passing
    Q[:r1], K[:r1] to the unmodified definition gives the same rows and the same dK contributions, the masked remainder
    contributes exact zeros), several blocks at a time on the host's threads.
  * properties that hold at any size, on EVERY head: all outputs finite, KL >= -2e-3 (R14), column sums of dK vanish
    (sum_j dS[i,j] = 0 per row).
Tolerances are parity_util's (BASELINE.json north_star).
"""
from __future__ import annotations

import os
from concurrent.futures import ThreadPoolExecutor

import numpy as np
import pytest

import workloads as W
from oracle.streamkl_oracle import attention_kl_head, attention_kl_rows
from parity_util import GRAD_COS, GRAD_MAXREL, KL_ATOL, KL_RTOL, LSE_ATOL, grad_metrics, to_f64, to_torch

pytestmark = pytest.mark.gpu


def gen_all(cfg: W.Config):
    heads = [(b, h) for b in range(cfg.B) for h in range(cfg.H)]
    with ThreadPoolExecutor(max_workers=min(16, os.cpu_count() or 1)) as ex:
        per = list(ex.map(lambda bh: W.head_inputs(cfg, *bh), heads))
    out = {}
    for k in ("Q1", "K1", "Q2", "K2", "g"):
        a = np.stack([p[k] for p in per])
        out[k] = a.reshape((cfg.B, cfg.H) + a.shape[1:])
    return out, per


def sample_rows(NQ: int, n_random: int, seed: int) -> np.ndarray:
    edge = [0, 1, 63, 64, 65, 127, 128, 129, 255, 256, 257]
    rows = set(r for r in edge if r < NQ) | set(NQ - 1 - r for r in edge if r < NQ)
    rng = np.random.default_rng(seed)
    rows |= set(int(x) for x in rng.integers(0, NQ, size=n_random))
    return np.array(sorted(rows), dtype=np.int64)


def run_gpu(cfg: W.Config, inp):
    import torch

    import paper_2606_20005_b200 as skl

    Q1, K1, Q2, K2 = (to_torch(inp[k]) for k in ("Q1", "K1", "Q2", "K2"))
    g = to_torch(inp["g"])
    kl, l1, l2 = skl.streamkl_fwd(Q1, K1, Q2, K2, cfg.c1, cfg.c2, cfg.causal)
    assert skl.streamkl_last_launch_count() >= 1
    dQ1, dK1, dQ2, dK2 = skl.streamkl_bwd(Q1, K1, Q2, K2, cfg.c1, cfg.c2, cfg.causal, kl, l1, l2, g, teacher=cfg.teacher_grads)
    assert skl.streamkl_last_launch_count() >= 2
    torch.cuda.synchronize()
    return kl, l1, l2, dQ1, dK1, dQ2, dK2


def check_rows(cfg, head_inp, hidx, rows, kl, l1, l2, dQ1, dQ2):
    """Sampled query rows of head `hidx` (flat b*H+h) against the definition."""
    Q1, K1, Q2, K2 = (W.widen_f64(head_inp[k]) for k in ("Q1", "K1", "Q2", "K2"))
    ref = attention_kl_rows(Q1, K1, Q2, K2, cfg.c1, cfg.c2, cfg.causal, rows, head_inp["g"].astype(np.float64), cfg.teacher_grads)
    b, h = divmod(hidx, cfg.H)
    got_kl, got_l1, got_l2 = (to_f64(t[b, h])[rows] for t in (kl, l1, l2))
    assert np.abs(got_l1 - ref["lse1"]).max() <= LSE_ATOL, f"cfg{cfg.idx} head {hidx}: lse1"
    assert np.abs(got_l2 - ref["lse2"]).max() <= LSE_ATOL, f"cfg{cfg.idx} head {hidx}: lse2"
    assert (np.abs(got_kl - ref["kl"]) <= KL_ATOL + KL_RTOL * np.abs(ref["kl"])).all(), f"cfg{cfg.idx} head {hidx}: kl"
    rt = __import__("torch").from_numpy(rows).to(dQ2.device)
    for name, t in (("dQ2", dQ2), ("dQ1", dQ1)):
        if t is None:
            continue
        cos, rel = grad_metrics(to_f64(t[b, h][rt]), ref[name])
        assert cos >= GRAD_COS and rel <= GRAD_MAXREL, f"cfg{cfg.idx} head {hidx} {name} rows: cos {cos:.6f} rel {rel:.3e}"
    return ref


def check_global_properties(cfg, kl, l1, l2, grads):
    import torch

    for t in (kl, l1, l2) + tuple(x for x in grads if x is not None):
        assert bool(torch.isfinite(t.float() if t.dtype != torch.float32 else t).all()), f"cfg{cfg.idx}: non-finite output"
    assert float(kl.min()) >= -2e-3, f"cfg{cfg.idx}: KL < 0 beyond rounding"
    dQ1, dK1, dQ2, dK2 = grads
    for name, dK in (("dK2", dK2), ("dK1", dK1)):
        if dK is None:
            continue
        col = dK.float().sum(dim=2).abs().amax(dim=-1)            # [B,H]
        scale = dK.float().abs().sum(dim=2).amax(dim=-1)
        assert bool((col <= 2e-2 * scale + 1e-6).all()), f"cfg{cfg.idx}: column sums of {name} do not vanish"


def whole_head_dk(cfg, head_inp, hidx, dK1, dK2):
    Q1, K1, Q2, K2 = (W.widen_f64(head_inp[k]) for k in ("Q1", "K1", "Q2", "K2"))
    ref = attention_kl_head(Q1, K1, Q2, K2, cfg.c1, cfg.c2, cfg.causal, head_inp["g"].astype(np.float64), cfg.teacher_grads)
    b, h = divmod(hidx, cfg.H)
    for name, t in (("dK2", dK2), ("dK1", dK1)):
        if t is None:
            continue
        cos, rel = grad_metrics(to_f64(t[b, h]), ref[name])
        assert cos >= GRAD_COS and rel <= GRAD_MAXREL, f"cfg{cfg.idx} head {hidx} {name}: cos {cos:.6f} rel {rel:.3e}"


def whole_head_causal_by_prefix_blocks(cfg, head_inp, hidx, kl, l1, l2, dQ1, dK1, dQ2, dK2, row_block=256, workers=8):
    """Every output of head `hidx` of a causal NQ = NK config against the definition (see the module docstring)."""
    import torch

    assert cfg.causal and cfg.NQ == cfg.NK
    Q1, K1, Q2, K2 = (W.widen_f64(head_inp[k]) for k in ("Q1", "K1", "Q2", "K2"))
    g = head_inp["g"].astype(np.float64)
    N = cfg.NQ
    ref = {"kl": np.empty(N), "lse1": np.empty(N), "lse2": np.empty(N), "dQ2": np.empty((N, cfg.d2)), "dK2": np.zeros((N, cfg.d2))}
    if cfg.teacher_grads:
        ref["dQ1"] = np.empty((N, cfg.d1))
        ref["dK1"] = np.zeros((N, cfg.d1))

    def block(r0):
        r1 = min(N, r0 + row_block)
        rows = np.arange(r0, r1)
        return r0, r1, attention_kl_rows(Q1[:r1], K1[:r1], Q2[:r1], K2[:r1], cfg.c1, cfg.c2, True, rows, g[:r1], cfg.teacher_grads)

    with ThreadPoolExecutor(max_workers=workers) as ex:
        for r0, r1, part in ex.map(block, range(0, N, row_block)):
            for k in ("kl", "lse1", "lse2", "dQ2") + (("dQ1",) if cfg.teacher_grads else ()):
                ref[k][r0:r1] = part[k]
            ref["dK2"][:r1] += part["dK2_part"]
            if cfg.teacher_grads:
                ref["dK1"][:r1] += part["dK1_part"]
    b, h = divmod(hidx, cfg.H)
    got_kl, got_l1, got_l2 = (to_f64(t[b, h]) for t in (kl, l1, l2))
    assert np.abs(got_l1 - ref["lse1"]).max() <= LSE_ATOL, f"cfg{cfg.idx} head {hidx}: lse1 (all rows)"
    assert np.abs(got_l2 - ref["lse2"]).max() <= LSE_ATOL, f"cfg{cfg.idx} head {hidx}: lse2 (all rows)"
    assert (np.abs(got_kl - ref["kl"]) <= KL_ATOL + KL_RTOL * np.abs(ref["kl"])).all(), f"cfg{cfg.idx} head {hidx}: kl (all rows)"
    res = {}
    for name, t in (("dQ2", dQ2), ("dK2", dK2), ("dQ1", dQ1), ("dK1", dK1)):
        if t is None:
            continue
        cos, rel = grad_metrics(to_f64(t[b, h]), ref[name])
        assert cos >= GRAD_COS and rel <= GRAD_MAXREL, f"cfg{cfg.idx} head {hidx} {name} (whole head): cos {cos:.6f} rel {rel:.3e}"
        if name.startswith("dK"):   # the longest K-owner loops: the first key tiles, seen by every query row
            cos, rel = grad_metrics(to_f64(t[b, h][:256]), ref[name][:256])
            assert cos >= GRAD_COS and rel <= GRAD_MAXREL, f"cfg{cfg.idx} head {hidx} {name} first 256 keys: cos {cos:.6f} rel {rel:.3e}"
        res[name] = (cos, rel)
    return res


def fullsize_case(idx, row_heads, n_random: int, dk_whole_head=None, dk_tail_rows: int = 0, whole_heads=()):
    cfg = idx if isinstance(idx, W.Config) else W.CONFIGS[idx]
    idx = cfg.idx
    inp, per = gen_all(cfg)
    kl, l1, l2, dQ1, dK1, dQ2, dK2 = run_gpu(cfg, inp)
    check_global_properties(cfg, kl, l1, l2, (dQ1, dK1, dQ2, dK2))
    for hidx in row_heads:
        check_rows(cfg, per[hidx], hidx, sample_rows(cfg.NQ, n_random, 1000 * idx + hidx), kl, l1, l2, dQ1, dQ2)
    if dk_whole_head is not None:
        whole_head_dk(cfg, per[dk_whole_head], dk_whole_head, dK1, dK2)
    for hidx in whole_heads:
        whole_head_causal_by_prefix_blocks(cfg, per[hidx], hidx, kl, l1, l2, dQ1, dK1, dQ2, dK2)
    if dk_tail_rows:
        assert cfg.causal and cfg.NQ == cfg.NK
        hidx = row_heads[-1]
        acc = {}
        for r0 in range(cfg.NQ - dk_tail_rows, cfg.NQ, 256):   # 256-row groups bound the materialised [R,NK] float64 arrays
            ref = check_rows(cfg, per[hidx], hidx, np.arange(r0, min(cfg.NQ, r0 + 256)), kl, l1, l2, dQ1, dQ2)
            for name in ("dK2", "dK1"):
                if name + "_part" in ref:
                    acc[name] = acc.get(name, 0.0) + ref[name + "_part"][cfg.NK - dk_tail_rows:]
        b, h = divmod(hidx, cfg.H)
        for name, t in (("dK2", dK2), ("dK1", dK1)):
            if t is None:
                continue
            cos, rel = grad_metrics(to_f64(t[b, h][cfg.NK - dk_tail_rows:]), acc[name])
            assert cos >= GRAD_COS and rel <= GRAD_MAXREL, f"cfg{cfg.idx} head {hidx} {name} tail keys: cos {cos:.6f} rel {rel:.3e}"


def test_cfg2_fullsize():
    """B=1,H=32,4096^2,d=128/128,causal, near-identical distributions: rows of 3 heads + whole-head dK of head 31."""
    fullsize_case(2, row_heads=[0, 15, 31], n_random=48, dk_whole_head=31)


def test_cfg3_fullsize():
    """B=1,H=32,16384^2,d=128/64,causal, student gradients only: rows of 3 heads + whole-head dK2 of head 7."""
    fullsize_case(3, row_heads=[0, 16, 31], n_random=40, dk_whole_head=7)


def test_cfg4_fullsize():
    """B=1,H=32,65536^2,d=128/128,causal (the bench workload): sampled rows of heads 7 and 20; heads 0 and 31 WHOLE (every
    kl/lse/dQ row, all of dK1 and dK2 -- SURVEY 8(c) C4), plus the global properties on every head."""
    fullsize_case(4, row_heads=[7, 20], n_random=40, whole_heads=(0, 31))


def test_cfg5_fullsize():
    """B=4,H=16,2048x131072,d=128/64,no mask, Q1 x4 (peaky): rows of 3 heads + whole-head dK of head 63 (last b, last h)."""
    fullsize_case(5, row_heads=[0, 37, 63], n_random=24, dk_whole_head=63)


def test_long_context_narrow_student_under_auto_runs_the_one_visit_pass():
    """cfg 3's recipe (frozen teacher d1 = 128, student d2 = 64, causal) at 32K: the size from which AUTO selects the one-visit student
    pass for Setting 1 (profiles/r03_bwd_strategies_large.md).  Sampled rows of both heads, the dK2 of the last 512 keys, the global
    properties -- and the workspace AUTO asks for shows which strategy ran."""
    import paper_2606_20005_b200 as skl

    cfg = W.shrink(W.CONFIGS[3], H=2, NQ=32768, NK=32768)
    stats_only = cfg.B * cfg.H * cfg.NQ * 16
    assert skl.streamkl_bwd_workspace_bytes(cfg.B, cfg.H, cfg.NQ, cfg.NK, cfg.d1, cfg.d2, False) == stats_only + cfg.B * cfg.H * cfg.NQ * 64 * 4
    fullsize_case(cfg, row_heads=[0, 1], n_random=32, dk_tail_rows=512)
