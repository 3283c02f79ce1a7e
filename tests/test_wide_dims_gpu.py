"""GPU parity for head dims above 128 on the tensor cores (the paper fixes d = 128, and the
DeepSeek-style teacher it names, :143, has 192-wide query/key heads): the BLOCKED forward plan (K streamed in single 64-element
K-blocks) and the wide owner backward kernels (one differentiated distribution per pass when the accumulators do not fit TMEM
together).  Everything is compared with the float64 definition on the same stored bits, per head, at the north-star tolerances;
the profile of each call must show tcgen05 kernels only (no SIMT fallback)."""
from __future__ import annotations

import numpy as np
import pytest

import workloads as W
from oracle.streamkl_oracle import attention_kl
from parity_util import check_fwd, check_grad_heads, to_f64, to_torch
from test_layouts_gpu import _as_bnhd, _run

pytestmark = pytest.mark.gpu

# every padded pair class: both-in-one-pass (192/64, 64/192), two passes (d1 + d2 > 256), ring depths from 4 down to the
# 2 + 1 stages of 256/256, true dims that are not multiples of 64
WIDE_PAIRS = [(192, 64), (64, 192), (192, 128), (128, 192), (192, 192), (256, 64), (64, 256), (256, 128), (128, 256), (256, 192),
              (192, 256), (256, 256), (136, 72), (200, 248), (160, 8)]


def _kernels_of(fn):
    import torch

    import paper_2606_20005_b200 as skl

    skl.streamkl_profile_enable(True)
    try:
        fn()
        torch.cuda.synchronize()
    finally:
        skl.streamkl_profile_enable(False)
    return [n for n, _ in skl.streamkl_profile_collect()]


@pytest.mark.parametrize("d1,d2", WIDE_PAIRS)
def test_wide_head_dims_both_settings(d1, d2):
    """ragged sizes spanning several tiles, causal with NQ != NK and no mask; Setting 2 (all four gradients) and Setting 1"""
    _run(W.Config(100, f"wide{d1}x{d2}-causal", 1, 2, 333, 555, d1, d2, "bf16", True), both_modes=False)
    _run(W.Config(101, f"wide{d1}x{d2}", 1, 2, 300, 450, d1, d2, "bf16", False), teacher=False, both_modes=False)


@pytest.mark.parametrize("d1,d2", [(192, 64), (192, 128), (256, 256)])
def test_wide_head_dims_run_on_the_tensor_cores(d1, d2):
    import paper_2606_20005_b200 as skl

    cfg = W.Config(102, "wide-kernels", 1, 2, 200, 300, d1, d2, "bf16", True)
    inp = W.all_inputs(cfg)
    dev = [to_torch(inp[k]) for k in ("Q1", "K1", "Q2", "K2")]
    g = to_torch(inp["g"])
    out = {}

    def call():
        out["f"] = skl.streamkl_fwd(*dev, cfg.c1, cfg.c2, True)
        skl.streamkl_bwd(*dev, cfg.c1, cfg.c2, True, *out["f"], g, teacher=True)

    names = _kernels_of(call)
    passes = 1 if d1 + d2 <= 256 else 2
    assert names == ["streamkl_fwd_sm100_kernel", "streamkl_bwd_stats_kernel"] + ["streamkl_bwd_wide_sm100_kernel<OWNER_Q>"] * passes + [
        "streamkl_bwd_wide_sm100_kernel<OWNER_K>"] * passes, names


@pytest.mark.parametrize("causal", [False, True])
def test_wide_long_streams(causal):
    """many steps per CTA (ring wrap-around, both TMEM stage parities, several Q / K tiles per head)"""
    _run(W.Config(103, "wide-long", 1, 2, 1500, 1500, 192, 128, "bf16", causal), both_modes=False)
    _run(W.Config(104, "wide-long256", 1, 1, 1100, 2100, 256, 256, "bf16", causal), both_modes=False)


def test_wide_fp16_strided_shared_heads_relu():
    """the layout features of the narrow kernels carry over: fp16, [B,N,H,d] strides, shared K heads, student ReLU"""
    _run(W.Config(105, "wide-f16", 1, 3, 260, 520, 192, 64, "f16", True), both_modes=False)
    _run(W.Config(106, "wide-bnhd", 2, 2, 300, 300, 192, 192, "bf16", True), view=_as_bnhd, both_modes=False)
    _run(W.Config(107, "wide-gqa", 1, 4, 200, 400, 256, 128, "bf16", False), HK=2, both_modes=False)
    _run(W.Config(108, "wide-relu", 1, 2, 300, 500, 192, 64, "bf16", True), act2="relu", both_modes=False)
    _run(W.Config(109, "wide-all", 2, 4, 260, 777, 200, 72, "f16", True), HK=2, view=_as_bnhd, act2="relu", both_modes=False)


def test_wide_degenerate_sizes():
    """one key, one query, a single partial tile, NQ = 1 against many keys"""
    _run(W.Config(110, "wide-1x1", 1, 1, 1, 1, 192, 192, "bf16", False), both_modes=False)
    _run(W.Config(111, "wide-1xN", 1, 2, 1, 700, 256, 64, "bf16", True), both_modes=False)
    _run(W.Config(112, "wide-tile", 1, 1, 127, 129, 192, 256, "bf16", True), both_modes=False)


@pytest.mark.parametrize("d1,d2", [(192, 64), (256, 256)])
def test_wide_splitk(d1, d2):
    """split-K forward through the BLOCKED plan"""
    import paper_2606_20005_b200 as skl

    cfg = W.Config(113, "wide-splitk", 1, 2, 40, 5000, d1, d2, "bf16", False)
    inp = W.all_inputs(cfg)
    f = {k: W.widen_f64(inp[k]) for k in ("Q1", "K1", "Q2", "K2")}
    ref = attention_kl(f["Q1"], f["K1"], f["Q2"], f["K2"], cfg.c1, cfg.c2, False)
    dev = [to_torch(inp[k]) for k in ("Q1", "K1", "Q2", "K2")]
    for splits in (0, 3, 40):
        names = _kernels_of(lambda: check_fwd(*(to_f64(t) for t in skl.streamkl_fwd_splitk(*dev, cfg.c1, cfg.c2, False, splits=splits)), ref,
                                              f"wide split-K W={splits}"))
        assert names == ["streamkl_fwd_sm100_kernel<SPLIT>", "streamkl_fwd_splitk_reduce_kernel"], names


def test_wide_gradient_padding_columns_are_left_untouched():
    """d = 160 inside a 256-wide row: the columns between rows belong to the caller and must survive the backward"""
    import torch

    import paper_2606_20005_b200 as skl

    cfg = W.Config(114, "d160-in-256", 1, 2, 200, 300, 160, 160, "bf16", False)
    inp = W.all_inputs(cfg)
    f = {k: W.widen_f64(inp[k]) for k in ("Q1", "K1", "Q2", "K2")}
    ref = attention_kl(f["Q1"], f["K1"], f["Q2"], f["K2"], cfg.c1, cfg.c2, False, g=inp["g"].astype(np.float64), teacher=True)
    wide = {k: torch.full((cfg.B, cfg.H, inp[k].shape[2], 256), 7.0, dtype=torch.bfloat16, device="cuda") for k in ("Q1", "K1", "Q2", "K2")}
    dev = {}
    for k in wide:
        wide[k][..., :160] = to_torch(inp[k])
        dev[k] = wide[k][..., :160]
    kl, l1, l2 = skl.streamkl_fwd(dev["Q1"], dev["K1"], dev["Q2"], dev["K2"], cfg.c1, cfg.c2, False)
    check_fwd(to_f64(kl), to_f64(l1), to_f64(l2), ref, "d160-in-256 fwd")
    outs = {k: torch.full_like(wide[k], 5.0) for k in wide}
    skl.streamkl_bwd(dev["Q1"], dev["K1"], dev["Q2"], dev["K2"], cfg.c1, cfg.c2, False, kl, l1, l2, to_torch(inp["g"]), teacher=True,
                     dQ1=outs["Q1"][..., :160], dK1=outs["K1"][..., :160], dQ2=outs["Q2"][..., :160], dK2=outs["K2"][..., :160])
    for k, name in (("Q1", "dQ1"), ("K1", "dK1"), ("Q2", "dQ2"), ("K2", "dK2")):
        check_grad_heads(to_f64(outs[k][..., :160]), ref[name], name)
        assert bool((outs[k][..., 160:] == 5.0).all()), f"{name} wrote beyond its head dim"


# ---------------------------------------------------------------- NEXT-3: the two CTA-pair plans of the forward
@pytest.mark.parametrize("plan", ["multicast", "pair_mma", "persistent"])
@pytest.mark.parametrize("causal", [False, True])
@pytest.mark.parametrize("d1,d2", [(128, 128), (128, 64), (64, 64), (192, 64), (256, 256), (96, 40), (200, 136)])
def test_forward_plans_are_bit_identical(d1, d2, causal, plan):
    """STREAMKL_FWD_MULTICAST: clusters of two CTAs share one TMA-multicast K stream.  STREAMKL_FWD_PAIR_MMA (head dims above 128; the
    plan is ignored below): the pair issues one `tcgen05.mma.cta_group::2` per K-slice, M = 256, each CTA holding 64 of the 128 keys.
    STREAMKL_FWD_PERSISTENT (head dims up to 128; ignored above): one CTA per SM loops over the Q tiles.
    Same arithmetic in the same order per row, so kl / lse must equal the single-CTA plan bit for bit -- and match the oracle.  Odd
    tile counts (a pair with one tile), ragged tails, NQ != NK, shared K heads and many steps (ring wrap-around) are covered."""
    import torch

    import paper_2606_20005_b200 as skl

    code = {"multicast": skl.STREAMKL_FWD_MULTICAST, "pair_mma": skl.STREAMKL_FWD_PAIR_MMA, "persistent": skl.STREAMKL_FWD_PERSISTENT}[plan]
    # (the last shape has 400 Q tiles: more than one work item per persistent CTA, odd and even step counts, the shared counter)
    for idx, (B, H, HK, NQ, NK) in enumerate([(1, 2, 2, 333, 555), (2, 4, 2, 640, 1500), (1, 1, 1, 129, 129), (1, 2, 2, 2100, 2100),
                                              (2, 40, 40, 600, 900)]):
        cfg = W.Config(120 + idx, f"pair{d1}x{d2}", B, H, NQ, NK, d1, d2, "bf16", causal)
        inp = W.all_inputs(cfg)
        if HK != H:
            inp["K1"] = np.ascontiguousarray(inp["K1"][:, :HK])
            inp["K2"] = np.ascontiguousarray(inp["K2"][:, :HK])
        dev = [to_torch(inp[k]) for k in ("Q1", "K1", "Q2", "K2")]
        skl.streamkl_set_fwd_plan(skl.STREAMKL_FWD_PER_TILE)
        try:
            single = skl.streamkl_fwd(*dev, cfg.c1, cfg.c2, causal)
            skl.streamkl_set_fwd_plan(code)
            pair = skl.streamkl_fwd(*dev, cfg.c1, cfg.c2, causal)
            pair = skl.streamkl_fwd(*dev, cfg.c1, cfg.c2, causal, *pair)   # (twice: the persistent plan's scheduler slot is rearmed by each launch)
            torch.cuda.synchronize()
        finally:
            skl.streamkl_set_fwd_plan(skl.STREAMKL_FWD_AUTO)
        for a, b, name in zip(single, pair, ("kl", "lse1", "lse2")):
            assert torch.equal(a, b), f"{cfg.name} case {idx}: {name} differs between the plans"
        G = H // HK
        f = {k: W.widen_f64(inp[k]) for k in ("Q1", "K1", "Q2", "K2")}
        ref = attention_kl(f["Q1"], np.repeat(f["K1"], G, axis=1), f["Q2"], np.repeat(f["K2"], G, axis=1), cfg.c1, cfg.c2, causal)
        check_fwd(*(to_f64(t) for t in pair), ref, f"{cfg.name} case {idx} {plan}")


# ---------------------------------------------------------------- larger sizes, graph capture, concurrent streams
@pytest.mark.parametrize("d1,d2,teacher,causal", [(192, 64, True, True), (256, 256, False, False), (192, 128, True, True)])
def test_wide_bench_sized_head(d1, d2, teacher, causal):
    """One head at a bench-like length (N = 6000: 47 Q tiles, 94 streamed 64-row steps per owner tile, hundreds of ring
    wrap-arounds), every output row and all of dK against the oracle."""
    _run(W.Config(130, f"wide-big{d1}x{d2}", 1, 1, 6000, 6000, d1, d2, "bf16", causal), teacher=teacher, both_modes=False)


def test_wide_and_cta_pair_kernels_are_graph_capturable_and_deterministic():
    """The wide kernels (several passes) and the cluster launch of a CTA-pair plan only enqueue work on the caller's stream:
    capture fwd + bwd into a CUDA graph; replays reproduce the eager results bit for bit (tile ownership, no atomics)."""
    import torch

    import paper_2606_20005_b200 as skl

    cfg = W.Config(131, "wide-graph", 1, 2, 700, 900, 256, 192, "bf16", True)
    inp = W.all_inputs(cfg)
    Q1, K1, Q2, K2 = (to_torch(inp[k]) for k in ("Q1", "K1", "Q2", "K2"))
    g = to_torch(inp["g"])
    kl, l1, l2 = skl.streamkl_fwd(Q1, K1, Q2, K2, cfg.c1, cfg.c2, True)
    eager = skl.streamkl_bwd(Q1, K1, Q2, K2, cfg.c1, cfg.c2, True, kl, l1, l2, g, teacher=True)
    ws = torch.empty(skl.streamkl_bwd_workspace_bytes(cfg.B, cfg.H, cfg.NQ, cfg.NK, cfg.d1, cfg.d2, True), dtype=torch.uint8, device="cuda")
    outs = [torch.zeros_like(t) for t in (kl, l1, l2)]
    grads = [torch.zeros_like(t) for t in eager]
    torch.cuda.synchronize()
    skl.streamkl_set_fwd_plan(skl.STREAMKL_FWD_PAIR_MMA)   # (a wide pair: the cta_group::2 cluster launch is what gets captured)
    try:
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph):
            skl.streamkl_fwd(Q1, K1, Q2, K2, cfg.c1, cfg.c2, True, *outs)
            skl.streamkl_bwd(Q1, K1, Q2, K2, cfg.c1, cfg.c2, True, outs[0], outs[1], outs[2], g, teacher=True, dQ1=grads[0],
                             dK1=grads[1], dQ2=grads[2], dK2=grads[3], workspace=ws)
    finally:
        skl.streamkl_set_fwd_plan(skl.STREAMKL_FWD_AUTO)
    for _ in range(2):
        for t in outs + grads:
            t.zero_()
        graph.replay()
        torch.cuda.synchronize()
        assert torch.equal(outs[0], kl) and torch.equal(outs[1], l1) and torch.equal(outs[2], l2)
        for a, b in zip(grads, eager):
            assert torch.equal(a, b)


def test_concurrent_streams_do_not_interfere():
    """Two different problems (a wide one and a fixed-plan one) enqueued back to back on two streams, several rounds: each
    stream's results equal those of the same call made alone (the library keeps no cross-call device state)."""
    import torch

    import paper_2606_20005_b200 as skl

    cfgs = [W.Config(132, "cs-wide", 1, 2, 900, 900, 192, 64, "bf16", True), W.Config(133, "cs-narrow", 1, 3, 1100, 1300, 128, 128, "bf16", False)]
    devs, alone = [], []
    for cfg in cfgs:
        inp = W.all_inputs(cfg)
        d = [to_torch(inp[k]) for k in ("Q1", "K1", "Q2", "K2")] + [to_torch(inp["g"])]
        devs.append(d)
        f = skl.streamkl_fwd(*d[:4], cfg.c1, cfg.c2, cfg.causal)
        b = skl.streamkl_bwd(*d[:4], cfg.c1, cfg.c2, cfg.causal, *f, d[4], teacher=True)
        alone.append((f, b))
    torch.cuda.synchronize()
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    for _ in range(3):
        res = []
        for cfg, d, st in zip(cfgs, devs, streams):
            with torch.cuda.stream(st):
                f = skl.streamkl_fwd(*d[:4], cfg.c1, cfg.c2, cfg.causal, stream=st)
                b = skl.streamkl_bwd(*d[:4], cfg.c1, cfg.c2, cfg.causal, *f, d[4], teacher=True, stream=st)
            res.append((f, b))
        torch.cuda.synchronize()
        for (f, b), (f0, b0) in zip(res, alone):
            for x, y in zip(list(f) + list(b), list(f0) + list(b0)):
                assert torch.equal(x, y)


def test_persistent_plan_in_graphs_and_on_concurrent_streams():
    """The persistent forward keeps its scheduler state in library-owned device memory (one slot leased per launch): overlapping launches
    on two streams must reproduce the per-tile kernel bit for bit every time; under stream capture the library runs the per-tile kernel
    (a captured launch would hold its slot for the life of the graph), so replays must match as well."""
    import torch

    import paper_2606_20005_b200 as skl

    cfgs = [W.Config(134, "ps-a", 1, 24, 1500, 1500, 128, 64, "bf16", True), W.Config(135, "ps-b", 2, 10, 900, 2300, 128, 128, "bf16", False)]
    devs, want = [], []
    skl.streamkl_set_fwd_plan(skl.STREAMKL_FWD_PER_TILE)
    try:
        for cfg in cfgs:
            inp = W.all_inputs(cfg)
            d = [to_torch(inp[k]) for k in ("Q1", "K1", "Q2", "K2")]
            devs.append(d)
            want.append(skl.streamkl_fwd(*d, cfg.c1, cfg.c2, cfg.causal))
        torch.cuda.synchronize()
        skl.streamkl_set_fwd_plan(skl.STREAMKL_FWD_PERSISTENT)
        # (a) graph replays
        outs = [torch.zeros_like(t) for t in want[0]]
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph):
            skl.streamkl_fwd(*devs[0], cfgs[0].c1, cfgs[0].c2, cfgs[0].causal, *outs)
        for _ in range(3):
            for t in outs:
                t.zero_()
            graph.replay()
            torch.cuda.synchronize()
            assert all(torch.equal(a, b) for a, b in zip(outs, want[0]))
        # (b) two streams, launches interleaved and overlapping; many more launches than the library has scheduler slots (1024), queued
        # without a synchronisation in between: a slot must never be handed to a launch while an earlier one may still be using it
        streams = [torch.cuda.Stream(), torch.cuda.Stream()]
        small = W.Config(139, "ps-c", 1, 40, 1024, 1024, 64, 64, "bf16", True)
        ds = [to_torch(W.all_inputs(small)[k]) for k in ("Q1", "K1", "Q2", "K2")]
        skl.streamkl_set_fwd_plan(skl.STREAMKL_FWD_PER_TILE)
        want_small = skl.streamkl_fwd(*ds, small.c1, small.c2, small.causal)
        skl.streamkl_set_fwd_plan(skl.STREAMKL_FWD_PERSISTENT)
        outs_small = [[torch.empty_like(t) for t in want_small] for _ in range(2)]
        for i in range(2600):
            st = streams[i & 1]
            with torch.cuda.stream(st):
                skl.streamkl_fwd(*ds, small.c1, small.c2, small.causal, *outs_small[i & 1], stream=st)
            if i % 325 == 324:
                torch.cuda.synchronize()
                for o in outs_small:
                    assert all(torch.equal(a, b) for a, b in zip(o, want_small))
        for _ in range(4):
            res = []
            for cfg, d, st in zip(cfgs, devs, streams):
                with torch.cuda.stream(st):
                    res.append(skl.streamkl_fwd(*d, cfg.c1, cfg.c2, cfg.causal, stream=st))
            torch.cuda.synchronize()
            for got, exp in zip(res, want):
                assert all(torch.equal(a, b) for a, b in zip(got, exp))
    finally:
        skl.streamkl_set_fwd_plan(skl.STREAMKL_FWD_AUTO)


def test_persistent_plan_with_layout_features():
    """The persistent forward takes the same layout as the per-tile kernel: fp16, [B,N,H,d] strides, shared K heads, odd head dims, student ReLU
    -- forward and (through its saved statistics) every gradient against the oracle."""
    import paper_2606_20005_b200 as skl

    skl.streamkl_set_fwd_plan(skl.STREAMKL_FWD_PERSISTENT)
    try:
        _run(W.Config(136, "ps-all", 2, 4, 260, 777, 96, 40, "f16", True), HK=2, view=_as_bnhd, act2="relu", both_modes=False)
        _run(W.Config(137, "ps-f16", 1, 3, 457, 901, 128, 64, "f16", False), both_modes=False)
        _run(W.Config(138, "ps-bnhd", 2, 3, 300, 700, 128, 128, "bf16", True), view=_as_bnhd, both_modes=False)
    finally:
        skl.streamkl_set_fwd_plan(skl.STREAMKL_FWD_AUTO)
