"""GPU parity for SURVEY 8(f) NEXT-3 -- shapes and layouts beyond the paper's contiguous [bsz, N, 128] bf16:
strided [B,N,H,d] tensors and views of packed buffers, K heads shared by groups of query heads, fp16 inputs, and head dims
other than 64 / 128 on the tensor-core path (any multiple of 8 up to 128, zero-padded inside the kernels).  Everything is
compared with the float64 definition on the same stored bits, at the north-star tolerances, per head, through the default
strategy and the other one.  The oracle knows nothing about layouts: it is fed plain [B,H,N,d] float64 arrays (shared K heads
repeated per query head; its per-head dK summed over each group)."""
from __future__ import annotations

import numpy as np
import pytest

import workloads as W
from oracle.streamkl_oracle import attention_kl
from parity_util import check_fwd, check_grad_heads, to_f64, to_torch

pytestmark = pytest.mark.gpu


def _ref(cfg, inp, HK, teacher, g, act2=None):
    """float64 definition with K heads expanded to the query heads; dK folded back onto the HK shared heads."""
    G = cfg.H // HK
    f = {k: W.widen_f64(inp[k]) for k in ("Q1", "K1", "Q2", "K2")}
    K1 = np.repeat(f["K1"], G, axis=1)
    K2 = np.repeat(f["K2"], G, axis=1)
    ref = attention_kl(f["Q1"], K1, f["Q2"], K2, cfg.c1, cfg.c2, cfg.causal, g=g.astype(np.float64), teacher=teacher, act2=act2)
    for name in ("dK1", "dK2"):
        if name in ref:
            a = ref[name]
            ref[name] = a.reshape(cfg.B, HK, G, *a.shape[2:]).sum(axis=2)
    return ref


def _inputs(cfg, HK):
    inp = W.all_inputs(cfg)
    if HK != cfg.H:   # K tensors of the first HK heads serve as the shared heads
        inp["K1"] = np.ascontiguousarray(inp["K1"][:, :HK])
        inp["K2"] = np.ascontiguousarray(inp["K2"][:, :HK])
    return inp


def _as_bnhd(t):
    """the same values as a [B,H,N,d] VIEW of a [B,N,H,d] buffer"""
    return t.permute(0, 2, 1, 3).contiguous().permute(0, 2, 1, 3)


def _run(cfg, HK=None, teacher=True, view=None, both_modes=True, act2=None):
    import torch

    import paper_2606_20005_b200 as skl

    HK = cfg.H if HK is None else HK
    inp = _inputs(cfg, HK)
    g_np = inp["g"]
    ref = _ref(cfg, inp, HK, teacher, g_np, act2)
    dev = {k: to_torch(inp[k]) for k in ("Q1", "K1", "Q2", "K2")}
    if view is not None:
        dev = {k: view(v) for k, v in dev.items()}
    g = to_torch(g_np)
    kl, l1, l2 = skl.streamkl_fwd(dev["Q1"], dev["K1"], dev["Q2"], dev["K2"], cfg.c1, cfg.c2, cfg.causal, student_activation=act2)
    check_fwd(to_f64(kl), to_f64(l1), to_f64(l2), ref, cfg.name + " fwd")
    modes = [skl.STREAMKL_BWD_AUTO] + ([skl.STREAMKL_BWD_SEPARATE, skl.STREAMKL_BWD_FUSED] if both_modes else [])
    try:
        for mode in modes:
            skl.streamkl_set_bwd_mode(mode)
            grads = skl.streamkl_bwd(dev["Q1"], dev["K1"], dev["Q2"], dev["K2"], cfg.c1, cfg.c2, cfg.causal, kl, l1, l2, g, teacher=teacher,
                                     student_activation=act2)
            for name, t, src in zip(("dQ1", "dK1", "dQ2", "dK2"), grads, (dev["Q1"], dev["K1"], dev["Q2"], dev["K2"])):
                if t is None:
                    assert not teacher and name in ("dQ1", "dK1")
                    continue
                assert t.shape == src.shape and t.stride() == src.stride() and t.dtype == src.dtype
                check_grad_heads(to_f64(t), ref[name], f"{cfg.name} mode {mode} {name}")
    finally:
        skl.streamkl_set_bwd_mode(skl.STREAMKL_BWD_AUTO)
    return ref


@pytest.mark.parametrize("causal", [False, True])
@pytest.mark.parametrize("d1,d2", [(128, 128), (128, 64), (64, 64)])
def test_bnhd_strided_views(d1, d2, causal):
    """[B,N,H,d] storage seen as [B,H,N,d] (head stride d, row stride H*d): forward, both settings' gradients written with the same strides."""
    _run(W.Config(80, "bnhd", 2, 3, 300, 700, d1, d2, "bf16", causal), view=_as_bnhd)
    _run(W.Config(81, "bnhd-long", 1, 2, 1100, 1100, d1, d2, "bf16", causal), view=_as_bnhd, teacher=False)


def test_views_of_one_packed_buffer():
    """Q1, K1, Q2, K2 as slices of ONE [B, N, 4, H, d] buffer (a fused projection's output): row stride 4*H*d."""
    import torch

    import paper_2606_20005_b200 as skl

    cfg = W.Config(82, "packed", 2, 2, 384, 384, 64, 64, "bf16", True)
    inp = W.all_inputs(cfg)
    ref = _ref(cfg, inp, cfg.H, True, inp["g"])
    buf = torch.empty((cfg.B, cfg.NQ, 4, cfg.H, 64), dtype=torch.bfloat16, device="cuda")
    for i, k in enumerate(("Q1", "K1", "Q2", "K2")):
        buf[:, :, i] = to_torch(inp[k]).permute(0, 2, 1, 3)
    Q1, K1, Q2, K2 = (buf[:, :, i].permute(0, 2, 1, 3) for i in range(4))
    assert not Q1.is_contiguous() and Q1.stride(2) == 4 * cfg.H * 64
    kl, l1, l2 = skl.streamkl_fwd(Q1, K1, Q2, K2, cfg.c1, cfg.c2, True)
    check_fwd(to_f64(kl), to_f64(l1), to_f64(l2), ref, "packed fwd")
    grads = skl.streamkl_bwd(Q1, K1, Q2, K2, cfg.c1, cfg.c2, True, kl, l1, l2, to_torch(inp["g"]), teacher=True)
    for name, t in zip(("dQ1", "dK1", "dQ2", "dK2"), grads):
        check_grad_heads(to_f64(t), ref[name], "packed " + name)


@pytest.mark.parametrize("H,HK", [(4, 2), (6, 1), (8, 4)])
@pytest.mark.parametrize("causal", [False, True])
def test_shared_k_heads(H, HK, causal):
    """Grouped-query layout: HK K heads, query head h reads K head h // (H/HK); dK sums over the group's query heads."""
    _run(W.Config(83, f"gqa{H}:{HK}", 1, H, 260, 520, 128, 64, "bf16", causal), HK=HK)
    _run(W.Config(84, f"gqa{H}:{HK}-long", 1, H, 900, 900, 128, 128, "bf16", causal), HK=HK, teacher=(HK != 1), both_modes=False)


@pytest.mark.parametrize("d1,d2", [(32, 32), (96, 96), (32, 96), (96, 128), (8, 120), (48, 80), (104, 16)])
def test_head_dims_that_are_multiples_of_8(d1, d2):
    """Head dims other than 64 / 128 run on the tensor cores zero-padded to 64 / 128; gradient columns beyond d are not written."""
    import torch

    import paper_2606_20005_b200 as skl

    cfg = W.Config(85, f"d{d1}x{d2}", 1, 2, 333, 555, d1, d2, "bf16", True)
    _run(cfg)
    # no kernel of the SIMT fallback may have run: every launch of the forward is the tcgen05 kernel
    inp = W.all_inputs(cfg)
    skl.streamkl_profile_enable(True)
    skl.streamkl_fwd(*(to_torch(inp[k]) for k in ("Q1", "K1", "Q2", "K2")), cfg.c1, cfg.c2, True)
    torch.cuda.synchronize()
    skl.streamkl_profile_enable(False)
    names = [n for n, _ in skl.streamkl_profile_collect()]
    assert names == ["streamkl_fwd_sm100_kernel"], names


def test_gradient_padding_columns_are_left_untouched():
    """d = 96 inside a wider row (row stride 128): the 32 columns between rows belong to the caller and must survive the backward."""
    import torch

    import paper_2606_20005_b200 as skl

    cfg = W.Config(86, "d96-in-128", 1, 2, 200, 300, 96, 96, "bf16", False)
    inp = W.all_inputs(cfg)
    ref = _ref(cfg, inp, cfg.H, True, inp["g"])
    wide = {k: torch.full((cfg.B, cfg.H, inp[k].shape[2], 128), 7.0, dtype=torch.bfloat16, device="cuda") for k in ("Q1", "K1", "Q2", "K2")}
    dev = {}
    for k in wide:
        wide[k][..., :96] = to_torch(inp[k])
        dev[k] = wide[k][..., :96]
    kl, l1, l2 = skl.streamkl_fwd(dev["Q1"], dev["K1"], dev["Q2"], dev["K2"], cfg.c1, cfg.c2, False)
    check_fwd(to_f64(kl), to_f64(l1), to_f64(l2), ref, "d96-in-128 fwd")
    outs = {k: torch.full_like(wide[k], 5.0) for k in wide}
    for mode in (skl.STREAMKL_BWD_FUSED, skl.STREAMKL_BWD_SEPARATE):
        skl.streamkl_set_bwd_mode(mode)
        try:
            skl.streamkl_bwd(dev["Q1"], dev["K1"], dev["Q2"], dev["K2"], cfg.c1, cfg.c2, False, kl, l1, l2, to_torch(inp["g"]), teacher=True,
                             dQ1=outs["Q1"][..., :96], dK1=outs["K1"][..., :96], dQ2=outs["Q2"][..., :96], dK2=outs["K2"][..., :96])
        finally:
            skl.streamkl_set_bwd_mode(skl.STREAMKL_BWD_AUTO)
        for k, name in (("Q1", "dQ1"), ("K1", "dK1"), ("Q2", "dQ2"), ("K2", "dK2")):
            check_grad_heads(to_f64(outs[k][..., :96]), ref[name], f"mode {mode} {name}")
            assert bool((outs[k][..., 96:] == 5.0).all()), f"mode {mode}: {name} wrote beyond its head dim"


@pytest.mark.parametrize("causal", [False, True])
@pytest.mark.parametrize("d1,d2", [(128, 128), (128, 64), (96, 32)])
def test_fp16_inputs(d1, d2, causal):
    """fp16 elements on the tcgen05 path (kind::f16 with the fp16 operand format; gradients rounded to fp16)."""
    _run(W.Config(87, "fp16", 1, 3, 457, 901, d1, d2, "f16", causal))
    _run(W.Config(88, "fp16-long", 1, 2, 1300, 1300, d1, d2, "f16", causal), both_modes=False)


def test_everything_at_once():
    """fp16 + [B,N,H,d] strides + shared K heads + odd head dims + causal with NQ != NK, all strategies."""
    _run(W.Config(89, "all", 2, 4, 260, 777, 96, 40, "f16", True), HK=2, view=_as_bnhd)


def test_layout_errors_are_reported_not_launched():
    import ctypes

    import paper_2606_20005_b200 as skl

    L = skl.lib()
    lay = skl.StreamKLLayout()
    lay.dtype = skl.STREAMKL_BF16
    lay.kv_heads = 3                      # 4 query heads are not a multiple of 3 K heads
    vp = ctypes.c_void_p
    args = (vp(16), vp(16), vp(16), vp(16), 1, 4, 8, 8, 64, 64, 0.125, 0.125, 0, vp(16), vp(16), vp(16), vp(0))
    assert L.streamkl_fwd_ex(ctypes.cast(ctypes.pointer(lay), vp), *args) == -2
    lay.kv_heads = 2
    lay.q1_stride[0], lay.q1_stride[1], lay.q1_stride[2] = 4 * 8 * 64, 8 * 64, 60   # row stride < d
    assert L.streamkl_fwd_ex(ctypes.cast(ctypes.pointer(lay), vp), *args) == -2
    lay.q1_stride[2] = 68                 # not a multiple of 8 elements (16 bytes)
    assert L.streamkl_fwd_ex(ctypes.cast(ctypes.pointer(lay), vp), *args) == -3
    lay.q1_stride[2] = 64
    lay.dtype = skl.STREAMKL_F32          # fp32 runs the SIMT kernels: default layout only
    assert L.streamkl_fwd_ex(ctypes.cast(ctypes.pointer(lay), vp), *args) == -2
    lay.dtype = 9
    assert L.streamkl_fwd_ex(ctypes.cast(ctypes.pointer(lay), vp), *args) == -7


def test_expanded_k_runs_forward_and_is_refused_by_backward():
    """K2.expand over heads (head stride 0): the forward reads it like H copies; the backward would have H owner CTAs store to the
    one dK2 head, so the binding and the library refuse it instead of returning the last writer's values."""
    import paper_2606_20005_b200 as skl

    cfg = W.Config(93, "expand", 1, 4, 200, 300, 64, 64, "bf16", False)
    inp = W.all_inputs(cfg)
    Q1, K1, Q2, K2 = (to_torch(inp[k]) for k in ("Q1", "K1", "Q2", "K2"))
    K2e = K2[:, :1].expand(-1, cfg.H, -1, -1)
    kl, l1, l2 = skl.streamkl_fwd(Q1, K1, Q2, K2e, cfg.c1, cfg.c2, False)
    kl_c, l1_c, l2_c = skl.streamkl_fwd(Q1, K1, Q2, K2e.contiguous(), cfg.c1, cfg.c2, False)
    assert np.array_equal(to_f64(kl), to_f64(kl_c)) and np.array_equal(to_f64(l2), to_f64(l2_c))
    g = to_torch(np.ones((cfg.B, cfg.H, cfg.NQ), dtype=np.float32))
    with pytest.raises(ValueError, match="broadcast or self-overlapping"):
        skl.streamkl_bwd(Q1, K1, Q2, K2e, cfg.c1, cfg.c2, False, kl, l1, l2, g)


# ---------------------------------------------------------------- NEXT-4: student ReLU activation (R23)
@pytest.mark.parametrize("causal", [False, True])
@pytest.mark.parametrize("d1,d2,dtype", [(128, 64, "bf16"), (128, 128, "bf16"), (64, 64, "f16")])
def test_relu_student(d1, d2, dtype, causal):
    """s2 = relu(c2 <q2,k2>) before the student's softmax: kl / lse2 of that P2, dS2 gated by relu'; every strategy, both settings."""
    _run(W.Config(91, "relu", 1, 3, 457, 901, d1, d2, dtype, causal), act2="relu")
    _run(W.Config(92, "relu-long", 1, 2, 1300, 1300, d1, d2, dtype, causal), act2="relu", both_modes=False)


def test_relu_student_with_strides_shared_heads_and_odd_dims():
    _run(W.Config(93, "relu-all", 2, 4, 260, 777, 96, 40, "bf16", True), HK=2, view=_as_bnhd, act2="relu")


def test_relu_student_closed_form_all_logits_negative():
    """Every raw student logit < 0 (Q2 > 0, K2 < 0 elementwise): relu makes P2 uniform -- lse2 = log nV exactly, KL = log nV - H(P1),
    and the student's gradients vanish identically (the gate is 0 everywhere), while the teacher's do not."""
    import torch

    import paper_2606_20005_b200 as skl

    cfg = W.Config(94, "relu-neg", 1, 2, 300, 600, 128, 64, "bf16", True)
    inp = W.all_inputs(cfg)
    Q1, K1 = to_torch(inp["Q1"]), to_torch(inp["K1"])
    Q2, K2 = to_torch(inp["Q2"]).abs(), -to_torch(inp["K2"]).abs()
    g = to_torch(inp["g"])
    kl, l1, l2 = skl.streamkl_fwd(Q1, K1, Q2, K2, cfg.c1, cfg.c2, True, student_activation="relu")
    nV = np.arange(cfg.NQ) + (cfg.NK - cfg.NQ) + 1
    assert np.abs(to_f64(l2)[0, 0] - np.log(nV)).max() <= 1e-4
    f = {"Q1": W.widen_f64(inp["Q1"]), "K1": W.widen_f64(inp["K1"]), "Q2": to_f64(Q2), "K2": to_f64(K2)}
    ref = attention_kl(f["Q1"], f["K1"], f["Q2"], f["K2"], cfg.c1, cfg.c2, True, g=inp["g"].astype(np.float64), teacher=True, act2="relu")
    check_fwd(to_f64(kl), to_f64(l1), to_f64(l2), ref, "relu-neg fwd")
    for mode in (skl.STREAMKL_BWD_FUSED, skl.STREAMKL_BWD_SEPARATE):
        skl.streamkl_set_bwd_mode(mode)
        try:
            dQ1, dK1, dQ2, dK2 = skl.streamkl_bwd(Q1, K1, Q2, K2, cfg.c1, cfg.c2, True, kl, l1, l2, g, teacher=True, student_activation="relu")
        finally:
            skl.streamkl_set_bwd_mode(skl.STREAMKL_BWD_AUTO)
        assert float(dQ2.float().abs().max()) == 0.0 and float(dK2.float().abs().max()) == 0.0
        check_grad_heads(to_f64(dQ1), ref["dQ1"], f"mode {mode} dQ1")
        check_grad_heads(to_f64(dK1), ref["dK1"], f"mode {mode} dK1")


def test_relu_gate_follows_the_sign_of_the_raw_logit():
    """relu' = 1[<q2,k2> > 0] (R23) must be decided on the raw logit.  Here every student logit but one is a tiny positive number
    (2^-20) while one key per row has logit 40, so lse2 ~ 40: in the shifted log2 domain the tiny logits round away against
    lse2 log2e ~ 57.7 (half an ulp there is 1.9e-6), and a gate taken after the shift would switch them all off -- dS2 = 0 where the
    definition has dS2 = g (P2 - P1) ~ -g P1.  Every strategy against the oracle."""
    import paper_2606_20005_b200 as skl

    cfg = W.Config(95, "relu-gate", 1, 2, 200, 300, 64, 64, "bf16", False)
    inp = W.all_inputs(cfg)
    f = {k: W.widen_f64(inp[k]) for k in ("Q1", "K1", "Q2", "K2")}
    f["Q2"][...] = 0.0
    f["Q2"][..., 0] = 2.0 ** -10
    f["K2"][..., 0] = 2.0 ** -10                     # raw logit 2^-20 > 0 for every (i, j) ...
    f["K2"][:, :, 7, 0] = 40.0 / cfg.c2 * 2.0 ** 10  # ... but key 7: logit 40 (bf16-exact: 327680 for c2 = 1/8)
    import torch

    Q1, K1 = to_torch(inp["Q1"]), to_torch(inp["K1"])
    Q2, K2 = (torch.from_numpy(f[k]).to(torch.bfloat16).cuda() for k in ("Q2", "K2"))
    assert np.array_equal(to_f64(Q2), f["Q2"]) and np.array_equal(to_f64(K2), f["K2"])      # bf16-exact inputs
    g = to_torch(inp["g"])
    ref = attention_kl(f["Q1"], f["K1"], f["Q2"], f["K2"], cfg.c1, cfg.c2, False, g=inp["g"].astype(np.float64), teacher=True, act2="relu")
    assert np.abs(ref["dK2"][:, :, :7, 0]).min() > 0                                         # the gated-on keys do carry gradient
    kl, l1, l2 = skl.streamkl_fwd(Q1, K1, Q2, K2, cfg.c1, cfg.c2, False, student_activation="relu")
    check_fwd(to_f64(kl), to_f64(l1), to_f64(l2), ref, "relu-gate fwd")
    for mode in (skl.STREAMKL_BWD_FUSED, skl.STREAMKL_BWD_SEPARATE):
        skl.streamkl_set_bwd_mode(mode)
        try:
            grads = skl.streamkl_bwd(Q1, K1, Q2, K2, cfg.c1, cfg.c2, False, kl, l1, l2, g, teacher=True, student_activation="relu")
        finally:
            skl.streamkl_set_bwd_mode(skl.STREAMKL_BWD_AUTO)
        for name, t in zip(("dQ1", "dK1", "dQ2", "dK2"), grads):
            check_grad_heads(to_f64(t), ref[name], f"relu-gate mode {mode} {name}")
        # the entries that exist only because the tiny logits are gated ON: dK2[j != 7, 0] = -c2 2^-10 sum_i g_i P1[i,j] (about 1e-4,
        # 0.3 % of the column's largest entry, so the per-head bars above would not notice them missing) -- element by element
        keys = np.arange(cfg.NK) != 7
        got, want = to_f64(grads[3])[:, :, keys, 0], ref["dK2"][:, :, keys, 0]
        assert np.abs(got - want).max() <= 3e-2 * np.abs(want).min(), f"relu-gate mode {mode}: dK2 of the tiny-logit keys"
