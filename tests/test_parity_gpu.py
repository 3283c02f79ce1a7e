"""GPU parity: the CUDA path (through the C ABI, via the thin binding) against the float64 oracle, element by
element, on the same seeded inputs.  Sizes span several 128/256-row tiles and ragged tails; the five BASELINE
configs appear shrunk here (the oracle finishes in seconds) and at full size in test_parity_fullsize_gpu.py."""
from __future__ import annotations

import numpy as np
import pytest

import workloads as W
from oracle.streamkl_oracle import attention_kl
from parity_util import bits_to_f64, check_fwd, check_grad, check_grad_heads, to_f64, to_torch

pytestmark = pytest.mark.gpu


def run_case(cfg: W.Config, teacher=None, check_bwd=True):
    import paper_2606_20005_b200 as skl

    teacher = cfg.teacher_grads if teacher is None else teacher
    inp = W.all_inputs(cfg)
    Q1, K1, Q2, K2 = (to_torch(inp[k]) for k in ("Q1", "K1", "Q2", "K2"))
    g = to_torch(inp["g"])
    ref = attention_kl(*(bits_to_f64(inp[k]) for k in ("Q1", "K1", "Q2", "K2")), cfg.c1, cfg.c2, cfg.causal,
                       g=inp["g"].astype(np.float64), teacher=teacher)
    kl, l1, l2 = skl.streamkl_fwd(Q1, K1, Q2, K2, cfg.c1, cfg.c2, cfg.causal)
    assert skl.streamkl_last_launch_count() >= 1
    stats = check_fwd(to_f64(kl), to_f64(l1), to_f64(l2), ref, cfg.name)
    assert (to_f64(kl) >= -2e-3).all(), "KL >= 0 up to rounding (R14: not clamped)"
    if not check_bwd:
        return stats
    dQ1, dK1, dQ2, dK2 = skl.streamkl_bwd(Q1, K1, Q2, K2, cfg.c1, cfg.c2, cfg.causal, kl, l1, l2, g, teacher=teacher)
    assert skl.streamkl_last_launch_count() >= 1
    check_grad_heads(to_f64(dQ2), ref["dQ2"], cfg.name + " dQ2")
    check_grad_heads(to_f64(dK2), ref["dK2"], cfg.name + " dK2")
    if teacher:
        check_grad_heads(to_f64(dQ1), ref["dQ1"], cfg.name + " dQ1")
        check_grad_heads(to_f64(dK1), ref["dK1"], cfg.name + " dK1")
    else:
        assert dQ1 is None and dK1 is None
    if cfg.dtype == "bf16" and cfg.d1 in (64, 128) and cfg.d2 in (64, 128):
        # the default (AUTO) picks the one-visit kernels for NQ <= 512 and the owner kernels beyond: run the OTHER strategy too
        other = skl.STREAMKL_BWD_SEPARATE if cfg.NQ <= (256 if teacher else 512) else skl.STREAMKL_BWD_FUSED
        skl.streamkl_set_bwd_mode(other)
        try:
            g1, k1, g2, k2 = skl.streamkl_bwd(Q1, K1, Q2, K2, cfg.c1, cfg.c2, cfg.causal, kl, l1, l2, g, teacher=teacher)
        finally:
            skl.streamkl_set_bwd_mode(skl.STREAMKL_BWD_AUTO)
        check_grad_heads(to_f64(g2), ref["dQ2"], f"{cfg.name} mode {other} dQ2")
        check_grad_heads(to_f64(k2), ref["dK2"], f"{cfg.name} mode {other} dK2")
        if teacher:
            check_grad_heads(to_f64(g1), ref["dQ1"], f"{cfg.name} mode {other} dQ1")
            check_grad_heads(to_f64(k1), ref["dK1"], f"{cfg.name} mode {other} dK1")
    return stats


def test_cfg1_tiny_exact_shape():
    """BASELINE config 1 as specified: fp32, 256x256, d=64/64, no mask, dkl=1, student grads."""
    run_case(W.CONFIGS[1])


def test_cfg2_shrunk_near_identical():
    """cfg-2 recipe (Q2=Q1+0.1eps: small KL, cancellation in acc/l1 - lse1 + lse2), 2 heads, N=1024, all four grads."""
    run_case(W.shrink(W.CONFIGS[2], H=2, NQ=1024, NK=1024))


def test_cfg3_shrunk_indexer():
    """cfg-3 recipe: d1=128 teacher frozen, d2=64 student, causal; ragged N (not a tile multiple)."""
    run_case(W.shrink(W.CONFIGS[3], H=2, NQ=1500, NK=1500))


def test_cfg4_shrunk_long():
    run_case(W.shrink(W.CONFIGS[4], H=3, NQ=1280, NK=1280))


def test_cfg5_shrunk_skewed():
    """cfg-5 recipe: non-causal, NQ << NK, Q1 scaled by 4 (large running-max jumps stress the rescaling of acc)."""
    run_case(W.shrink(W.CONFIGS[5], B=2, H=2, NQ=320, NK=4096))


@pytest.mark.parametrize("d1,d2", [(64, 64), (64, 128), (128, 64), (128, 128)])
@pytest.mark.parametrize("causal", [False, True])
def test_all_head_dim_pairs_ragged(d1, d2, causal):
    cfg = W.Config(20 + d1 // 64 * 2 + d2 // 64, "ragged", 1, 2, 333, 777, d1, d2, "bf16", causal)
    run_case(cfg)


@pytest.mark.parametrize("NQ,NK,causal", [(1, 1, False), (1, 1, True), (1, 300, False), (1, 300, True), (300, 1, False),
                                         (129, 129, True), (257, 513, True), (64, 64, True), (127, 63, False)])
def test_degenerate_sizes(NQ, NK, causal):
    """NK=1 or causal row 0: KL=0, lse_t=s_t[0]; single rows; sizes straddling one tile."""
    cfg = W.Config(40, "degenerate", 1, 2, NQ, NK, 128, 64, "bf16", causal)
    run_case(cfg)


def test_simt_path_other_head_dims_bf16():
    """Head dims that are not multiples of 8 (up to 256) run the fp32 SIMT kernels."""
    run_case(W.Config(41, "simt-bf16", 1, 2, 200, 300, 44, 84, "bf16", True))
    run_case(W.Config(48, "simt-bf16-wide", 1, 2, 150, 260, 164, 196, "bf16", False))


def test_simt_path_fp32_causal_teacher():
    run_case(W.Config(42, "simt-f32", 2, 1, 150, 260, 32, 64, "f32", True))


def test_identical_logits_give_zero_kl_and_zero_grads():
    """Closed form: Q2=2*Q1 (exact in bf16), K2=K1, c2=c1/2 => same logits => KL=0, grads 0, lse1=lse2."""
    import torch

    import paper_2606_20005_b200 as skl

    cfg = W.Config(43, "same", 1, 2, 384, 640, 128, 128, "bf16", True)
    inp = W.all_inputs(cfg)
    Q1, K1 = to_torch(inp["Q1"]), to_torch(inp["K1"])
    Q2, K2 = (Q1 * 2).contiguous(), K1.clone()
    g = to_torch(inp["g"])
    kl, l1, l2 = skl.streamkl_fwd(Q1, K1, Q2, K2, cfg.c1, cfg.c1 / 2, True)
    assert torch.equal(l1, l2)
    assert kl.abs().max().item() <= 1e-5
    dQ1, dK1, dQ2, dK2 = skl.streamkl_bwd(Q1, K1, Q2, K2, cfg.c1, cfg.c1 / 2, True, kl, l1, l2, g, teacher=True)
    for t in (dQ1, dK1, dQ2, dK2):
        assert t.float().abs().max().item() <= 1e-4


def test_uniform_p2_closed_form():
    """Q2=0 => P2 uniform over the nV visible keys: lse2 = log nV, KL = log nV - H(P1)  (R18)."""
    import torch

    import paper_2606_20005_b200 as skl

    cfg = W.Config(44, "p2uniform", 1, 1, 256, 512, 64, 64, "bf16", True)
    inp = W.all_inputs(cfg)
    Q1, K1, K2 = to_torch(inp["Q1"]), to_torch(inp["K1"]), to_torch(inp["K2"])
    Q2 = torch.zeros_like(to_torch(inp["Q2"]))
    kl, l1, l2 = skl.streamkl_fwd(Q1, K1, Q2, K2, cfg.c1, cfg.c2, True)
    nV = np.arange(cfg.NQ) + (cfg.NK - cfg.NQ) + 1
    assert np.abs(to_f64(l2)[0, 0] - np.log(nV)).max() <= 1e-4
    S1 = cfg.c1 * bits_to_f64(inp["Q1"])[0, 0] @ bits_to_f64(inp["K1"])[0, 0].T
    vis = np.arange(cfg.NK)[None, :] < nV[:, None]
    S1 = np.where(vis, S1, -np.inf)
    logP1 = S1 - np.log(np.exp(S1 - S1.max(1, keepdims=True)).sum(1, keepdims=True)) - S1.max(1, keepdims=True)
    H = -(np.where(vis, np.exp(logP1) * np.where(vis, logP1, 0.0), 0.0)).sum(1)
    assert np.abs(to_f64(kl)[0, 0] - (np.log(nV) - H)).max() <= 2e-3


def test_dk_column_sums_vanish():
    """Invariant: sum_j dS[i,j] = 0 per row  =>  sum_j dK_t[j,:] = 0, seen at the boundary."""
    import paper_2606_20005_b200 as skl

    cfg = W.Config(45, "colsum", 1, 2, 512, 768, 128, 64, "bf16", True)
    inp = W.all_inputs(cfg)
    Q1, K1, Q2, K2 = (to_torch(inp[k]) for k in ("Q1", "K1", "Q2", "K2"))
    g = to_torch(inp["g"])
    kl, l1, l2 = skl.streamkl_fwd(Q1, K1, Q2, K2, cfg.c1, cfg.c2, True)
    dQ1, dK1, dQ2, dK2 = skl.streamkl_bwd(Q1, K1, Q2, K2, cfg.c1, cfg.c2, True, kl, l1, l2, g, teacher=True)
    for dK in (dK1, dK2):
        col = dK.float().sum(dim=2).abs().max().item()
        scale = dK.float().abs().sum(dim=2).max().item()
        assert col <= 2e-2 * scale


def test_empty_batch_is_a_noop():
    import torch

    import paper_2606_20005_b200 as skl

    z = lambda n, d: torch.empty((0, 4, n, d), dtype=torch.bfloat16, device="cuda")
    kl, l1, l2 = skl.streamkl_fwd(z(16, 64), z(32, 64), z(16, 64), z(32, 64), 0.125, 0.125, False)
    assert kl.shape == (0, 4, 16) and skl.streamkl_last_launch_count() == 0


def test_host_entry_point_matches_device_path():
    """streamkl_fwd_bwd_host (HOST buffers, copies inside) gives bit-identical results to the device entry points."""
    import paper_2606_20005_b200 as skl

    cfg = W.shrink(W.CONFIGS[3], H=2, NQ=512, NK=512)
    inp = W.all_inputs(cfg)
    skl.streamkl_set_bwd_mode(skl.STREAMKL_BWD_SEPARATE)   # bit-for-bit comparison: the atomic-free strategy
    out = skl.streamkl_fwd_bwd_host(inp["Q1"], inp["K1"], inp["Q2"], inp["K2"], cfg.c1, cfg.c2, cfg.causal, inp["g"], teacher=False)
    Q1, K1, Q2, K2 = (to_torch(inp[k]) for k in ("Q1", "K1", "Q2", "K2"))
    kl, l1, l2 = skl.streamkl_fwd(Q1, K1, Q2, K2, cfg.c1, cfg.c2, cfg.causal)
    _, _, dQ2, dK2 = skl.streamkl_bwd(Q1, K1, Q2, K2, cfg.c1, cfg.c2, cfg.causal, kl, l1, l2, to_torch(inp["g"]))
    assert np.array_equal(out["kl"], kl.cpu().numpy())
    assert np.array_equal(bits_to_f64(out["dQ2"]), to_f64(dQ2))
    assert np.array_equal(bits_to_f64(out["dK2"]), to_f64(dK2))
    kl_h, l1_h, l2_h = skl.streamkl_fwd_host(inp["Q1"], inp["K1"], inp["Q2"], inp["K2"], cfg.c1, cfg.c2, cfg.causal)
    assert np.array_equal(kl_h, out["kl"]) and np.array_equal(l1_h, out["lse1"]) and np.array_equal(l2_h, out["lse2"])
    skl.streamkl_set_bwd_mode(skl.STREAMKL_BWD_AUTO)


def test_host_entry_point_pipelined_head_groups_match_device_path():
    """cfg 2 at full size (32 heads, 136 MB of inputs): the host entry point splits the batch into head groups and overlaps
    copies with kernels; every group must land where one ungrouped device call puts it, bit for bit."""
    import paper_2606_20005_b200 as skl

    cfg = W.CONFIGS[2]
    inp = W.all_inputs(cfg)
    out = skl.streamkl_fwd_bwd_host(inp["Q1"], inp["K1"], inp["Q2"], inp["K2"], cfg.c1, cfg.c2, cfg.causal, inp["g"], teacher=True)
    assert skl.streamkl_last_launch_count() > 4          # more than one group's worth of {fwd, stats, dQ, dK}
    Q1, K1, Q2, K2 = (to_torch(inp[k]) for k in ("Q1", "K1", "Q2", "K2"))
    kl, l1, l2 = skl.streamkl_fwd(Q1, K1, Q2, K2, cfg.c1, cfg.c2, cfg.causal)
    dQ1, dK1, dQ2, dK2 = skl.streamkl_bwd(Q1, K1, Q2, K2, cfg.c1, cfg.c2, cfg.causal, kl, l1, l2, to_torch(inp["g"]), teacher=True)
    assert np.array_equal(out["kl"], kl.cpu().numpy()) and np.array_equal(out["lse2"], l2.cpu().numpy())
    for name, t in (("dQ1", dQ1), ("dK1", dK1), ("dQ2", dQ2), ("dK2", dK2)):
        assert np.array_equal(bits_to_f64(out[name]), to_f64(t)), name
    skl.streamkl_host_trim()


def test_device_entry_points_are_graph_capturable_and_deterministic():
    """streamkl_fwd + streamkl_bwd only enqueue kernels on the caller's stream (no allocation, no sync): they can be
    captured into a CUDA graph, and replaying it reproduces the eager results bit for bit (tile ownership: no atomics)."""
    import torch

    import paper_2606_20005_b200 as skl

    cfg = W.shrink(W.CONFIGS[2], H=3, NQ=1100, NK=1100)
    inp = W.all_inputs(cfg)
    Q1, K1, Q2, K2 = (to_torch(inp[k]) for k in ("Q1", "K1", "Q2", "K2"))
    g = to_torch(inp["g"])
    kl, l1, l2 = skl.streamkl_fwd(Q1, K1, Q2, K2, cfg.c1, cfg.c2, True)
    eager = skl.streamkl_bwd(Q1, K1, Q2, K2, cfg.c1, cfg.c2, True, kl, l1, l2, g, teacher=True)
    ws = torch.empty(skl.streamkl_bwd_workspace_bytes(cfg.B, cfg.H, cfg.NQ, cfg.NK, cfg.d1, cfg.d2, True), dtype=torch.uint8, device="cuda")
    outs = [torch.zeros_like(t) for t in (kl, l1, l2)]
    grads = [torch.zeros_like(t) for t in eager]
    torch.cuda.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        skl.streamkl_fwd(Q1, K1, Q2, K2, cfg.c1, cfg.c2, True, *outs)
        skl.streamkl_bwd(Q1, K1, Q2, K2, cfg.c1, cfg.c2, True, outs[0], outs[1], outs[2], g, teacher=True, dQ1=grads[0],
                         dK1=grads[1], dQ2=grads[2], dK2=grads[3], workspace=ws)
    for _ in range(2):
        for t in outs + grads:
            t.zero_()
        graph.replay()
        torch.cuda.synchronize()
        assert torch.equal(outs[0], kl) and torch.equal(outs[1], l1) and torch.equal(outs[2], l2)
        for a, b in zip(grads, eager):
            assert torch.equal(a, b)


@pytest.mark.parametrize("d1,d2", [(128, 128), (128, 64), (64, 128), (64, 64)])
@pytest.mark.parametrize("causal", [False, True])
def test_setting1_fused_and_separate_strategies_agree_with_the_oracle(d1, d2, causal):
    """Setting 1 (teacher frozen) through both backward strategies: the one-visit kernel with fp32-atomic
    dQ2 and the two deterministic owner kernels; ragged sizes, several K-owner tiles, several 64-query steps."""
    import paper_2606_20005_b200 as skl

    cfg = W.Config(50 + d1 // 64 * 2 + d2 // 64, "setting1", 1, 3, 457, 901, d1, d2, "bf16", causal, teacher_grads=False)
    inp = W.all_inputs(cfg)
    Q1, K1, Q2, K2 = (to_torch(inp[k]) for k in ("Q1", "K1", "Q2", "K2"))
    g = to_torch(inp["g"])
    ref = attention_kl(*(bits_to_f64(inp[k]) for k in ("Q1", "K1", "Q2", "K2")), cfg.c1, cfg.c2, cfg.causal,
                       g=inp["g"].astype(np.float64), teacher=False)
    kl, l1, l2 = skl.streamkl_fwd(Q1, K1, Q2, K2, cfg.c1, cfg.c2, cfg.causal)
    res = {}
    try:
        for mode in (skl.STREAMKL_BWD_FUSED, skl.STREAMKL_BWD_SEPARATE):
            skl.streamkl_set_bwd_mode(mode)
            _, _, dQ2, dK2 = skl.streamkl_bwd(Q1, K1, Q2, K2, cfg.c1, cfg.c2, cfg.causal, kl, l1, l2, g, teacher=False)
            check_grad_heads(to_f64(dQ2), ref["dQ2"], f"mode {mode} dQ2")
            check_grad_heads(to_f64(dK2), ref["dK2"], f"mode {mode} dK2")
            res[mode] = (to_f64(dQ2), to_f64(dK2), skl.streamkl_last_launch_count())
    finally:
        skl.streamkl_set_bwd_mode(skl.STREAMKL_BWD_AUTO)
    assert res[skl.STREAMKL_BWD_FUSED][2] == 3 and res[skl.STREAMKL_BWD_SEPARATE][2] == 3   # {stats, fused, convert} / {stats, dQ, dK}


@pytest.mark.parametrize("d1,d2", [(128, 128), (128, 64), (64, 128), (64, 64)])
@pytest.mark.parametrize("causal", [False, True])
def test_setting2_fused_and_separate_strategies_agree_with_the_oracle(d1, d2, causal):
    """Setting 2 (teacher trainable) through both strategies: two one-visit passes (student: dS2 -> dK2, dQ2; teacher: dS1 -> dK1,
    dQ1, each dQ by fp32 atomics) and the two deterministic owner kernels; ragged sizes; mixed-sign upstream gradient."""
    import torch

    import paper_2606_20005_b200 as skl

    cfg = W.Config(70 + d1 // 64 * 2 + d2 // 64, "setting2", 1, 3, 457, 901, d1, d2, "bf16", causal)
    inp = W.all_inputs(cfg)
    gnp = (inp["g"] - 0.9).astype(np.float32)
    Q1, K1, Q2, K2 = (to_torch(inp[k]) for k in ("Q1", "K1", "Q2", "K2"))
    g = torch.from_numpy(gnp).cuda()
    ref = attention_kl(*(bits_to_f64(inp[k]) for k in ("Q1", "K1", "Q2", "K2")), cfg.c1, cfg.c2, cfg.causal,
                       g=gnp.astype(np.float64), teacher=True)
    kl, l1, l2 = skl.streamkl_fwd(Q1, K1, Q2, K2, cfg.c1, cfg.c2, cfg.causal)
    counts = {}
    try:
        for mode in (skl.STREAMKL_BWD_FUSED, skl.STREAMKL_BWD_SEPARATE):
            skl.streamkl_set_bwd_mode(mode)
            grads = skl.streamkl_bwd(Q1, K1, Q2, K2, cfg.c1, cfg.c2, cfg.causal, kl, l1, l2, g, teacher=True)
            counts[mode] = skl.streamkl_last_launch_count()
            for name, t in zip(("dQ1", "dK1", "dQ2", "dK2"), grads):
                check_grad_heads(to_f64(t), ref[name], f"mode {mode} {name}")
    finally:
        skl.streamkl_set_bwd_mode(skl.STREAMKL_BWD_AUTO)
    assert counts[skl.STREAMKL_BWD_FUSED] == 5 and counts[skl.STREAMKL_BWD_SEPARATE] == 3   # {stats, 2 x (fused, convert)} / {stats, dQ, dK}


def test_setting1_fused_mixed_sign_upstream_gradient_and_tiny_sizes():
    """dkl_rows of both signs (and zeros); NQ, NK below one tile."""
    import torch

    import paper_2606_20005_b200 as skl

    for NQ, NK in ((1, 1), (5, 300), (130, 70)):
        cfg = W.Config(58, "setting1-sign", 1, 2, NQ, NK, 128, 128, "bf16", False, teacher_grads=False)
        inp = W.all_inputs(cfg)
        gnp = inp["g"] - 1.0
        gnp[..., ::3] = 0.0
        Q1, K1, Q2, K2 = (to_torch(inp[k]) for k in ("Q1", "K1", "Q2", "K2"))
        ref = attention_kl(*(bits_to_f64(inp[k]) for k in ("Q1", "K1", "Q2", "K2")), cfg.c1, cfg.c2, False, g=gnp.astype(np.float64), teacher=False)
        kl, l1, l2 = skl.streamkl_fwd(Q1, K1, Q2, K2, cfg.c1, cfg.c2, False)
        _, _, dQ2, dK2 = skl.streamkl_bwd(Q1, K1, Q2, K2, cfg.c1, cfg.c2, False, kl, l1, l2, torch.from_numpy(gnp).cuda(), teacher=False)
        check_grad_heads(to_f64(dQ2), ref["dQ2"], f"{NQ}x{NK} dQ2")
        check_grad_heads(to_f64(dK2), ref["dK2"], f"{NQ}x{NK} dK2")


def test_one_million_keys_and_many_small_heads():
    """Index arithmetic at the extremes: NK = 2^20 + 3 keys (8 query rows: forward, split-K forward, both Setting-1 backward
    strategies, Setting-2 backward), and 1024 heads of a 130 x 190 problem in one call."""
    import paper_2606_20005_b200 as skl

    cfg = W.Config(46, "1M-keys", 1, 2, 8, (1 << 20) + 3, 128, 64, "bf16", False)
    inp = W.all_inputs(cfg)
    Q1, K1, Q2, K2 = (to_torch(inp[k]) for k in ("Q1", "K1", "Q2", "K2"))
    g = to_torch(inp["g"])
    ref = attention_kl(*(bits_to_f64(inp[k]) for k in ("Q1", "K1", "Q2", "K2")), cfg.c1, cfg.c2, False, g=inp["g"].astype(np.float64), teacher=True)
    kl, l1, l2 = skl.streamkl_fwd(Q1, K1, Q2, K2, cfg.c1, cfg.c2, False)
    check_fwd(to_f64(kl), to_f64(l1), to_f64(l2), ref, "1M fwd")
    ks, l1s, l2s = skl.streamkl_fwd_splitk(Q1, K1, Q2, K2, cfg.c1, cfg.c2, False)
    check_fwd(to_f64(ks), to_f64(l1s), to_f64(l2s), ref, "1M split-K")
    dQ1, dK1, dQ2, dK2 = skl.streamkl_bwd(Q1, K1, Q2, K2, cfg.c1, cfg.c2, False, kl, l1, l2, g, teacher=True)
    for name, t in (("dQ1", dQ1), ("dK1", dK1), ("dQ2", dQ2), ("dK2", dK2)):
        check_grad_heads(to_f64(t), ref[name], "1M " + name)
    try:
        for mode in (skl.STREAMKL_BWD_FUSED, skl.STREAMKL_BWD_SEPARATE):
            skl.streamkl_set_bwd_mode(mode)
            _, _, dQ2, dK2 = skl.streamkl_bwd(Q1, K1, Q2, K2, cfg.c1, cfg.c2, False, kl, l1, l2, g, teacher=False)
            check_grad_heads(to_f64(dQ2), ref["dQ2"], f"1M mode {mode} dQ2")
            check_grad_heads(to_f64(dK2), ref["dK2"], f"1M mode {mode} dK2")
    finally:
        skl.streamkl_set_bwd_mode(skl.STREAMKL_BWD_AUTO)
    run_case(W.Config(47, "many-heads", 32, 32, 130, 190, 64, 128, "bf16", True))
