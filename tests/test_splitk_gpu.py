"""GPU parity of the split-K forward (Eq.11) against the float64 definition, element by element:
small N_Q (the regime it exists for), long and ragged N_K, every head-dim pair, causal and not, split counts from 2 to
one chunk per key tile (incl. chunks that lie wholly past a row's causal frontier), and the adaptive choice."""
from __future__ import annotations

import numpy as np
import pytest

import workloads as W
from oracle.streamkl_oracle import attention_kl
from parity_util import bits_to_f64, check_fwd, to_f64, to_torch

pytestmark = pytest.mark.gpu


def run_splitk(cfg: W.Config, splits: int):
    import paper_2606_20005_b200 as skl

    inp = W.all_inputs(cfg)
    Q1, K1, Q2, K2 = (to_torch(inp[k]) for k in ("Q1", "K1", "Q2", "K2"))
    ref = attention_kl(*(bits_to_f64(inp[k]) for k in ("Q1", "K1", "Q2", "K2")), cfg.c1, cfg.c2, cfg.causal)
    kl, l1, l2 = skl.streamkl_fwd_splitk(Q1, K1, Q2, K2, cfg.c1, cfg.c2, cfg.causal, splits=splits)
    launches = skl.streamkl_last_launch_count()
    check_fwd(to_f64(kl), to_f64(l1), to_f64(l2), ref, f"{cfg.name} splits={splits}")
    # and against the default kernel: same statistics; the fp32 merge order differs, and so does which running maximum
    # an element is shifted by (a 7.6e-5-relative exp2 polynomial and fp32 lse ~ 20 give differences of a few 1e-5)
    kl0, l10, l20 = skl.streamkl_fwd(Q1, K1, Q2, K2, cfg.c1, cfg.c2, cfg.causal)
    assert np.abs(to_f64(l1) - to_f64(l10)).max() <= 1e-4 and np.abs(to_f64(l2) - to_f64(l20)).max() <= 1e-4
    assert np.abs(to_f64(kl) - to_f64(kl0)).max() <= 3e-4
    return launches


@pytest.mark.parametrize("NQ", [1, 16, 64, 200, 300])
@pytest.mark.parametrize("causal", [False, True])
def test_splitk_small_nq(NQ, causal):
    cfg = W.Config(60, "splitk", 2, 2, NQ, 4096 + 17, 128, 128, "bf16", causal)
    assert run_splitk(cfg, 7) == 2          # split kernel + reduce kernel


@pytest.mark.parametrize("d1,d2", [(64, 64), (64, 128), (128, 64)])
def test_splitk_head_dim_pairs(d1, d2):
    run_splitk(W.Config(61, "splitk-d", 1, 3, 33, 2048 + 5, d1, d2, "bf16", True), 5)


@pytest.mark.parametrize("splits", [2, 3, 1000])
def test_splitk_split_counts_up_to_one_tile_per_chunk(splits):
    """splits=1000 is clamped to one chunk per key tile; causal rows then meet empty chunks."""
    run_splitk(W.Config(62, "splitk-w", 1, 2, 48, 1024 + 40, 128, 64, "bf16", True), splits)


def test_splitk_adaptive_choice_and_peaky_logits():
    """cfg-5 recipe (Q1 x4: large running-max differences between chunks stress the Eq.11 rescaling), adaptive W."""
    import paper_2606_20005_b200 as skl

    cfg = W.shrink(W.CONFIGS[5], B=1, H=4, NQ=16, NK=16384)
    w = skl.streamkl_fwd_splitk_splits(cfg.B, cfg.H, cfg.NQ, cfg.NK)
    assert w == 148 // 4
    assert run_splitk(cfg, 0) == 2


def test_splitk_with_one_split_is_the_default_kernel():
    assert run_splitk(W.Config(63, "splitk-1", 1, 2, 16, 512, 128, 128, "bf16", False), 1) == 1


# ---------------------------------------------------------------- split-K with a layout (streamkl_fwd_splitk_ex): NEXT-1 x NEXT-3
# decode against a grouped KV cache is the paper's small-N_Q case: few query rows, K heads shared by groups
# of query heads, keys stored [B][N][H][d], fp16 or bf16, optionally the ReLU student
@pytest.mark.parametrize("NQ", [1, 16])
@pytest.mark.parametrize("G", [4, 8])
@pytest.mark.parametrize("dtype,act2", [("bf16", None), ("f16", None), ("bf16", "relu")])
def test_splitk_with_shared_k_heads_strides_fp16_and_relu(NQ, G, dtype, act2):
    import paper_2606_20005_b200 as skl
    from test_layouts_gpu import _as_bnhd, _inputs, _ref

    H, HK = 8, 8 // G
    cfg = W.Config(64, "splitk-ex", 2, H, NQ, 4096 + 17, 128, 64, dtype, True)
    inp = _inputs(cfg, HK)
    ref = _ref(cfg, inp, HK, False, inp["g"], act2)
    dev = {k: _as_bnhd(to_torch(inp[k])) for k in ("Q1", "K1", "Q2", "K2")}          # [B,H,N,d] views of [B,N,H,d] buffers
    assert dev["K1"].shape[1] == HK and (HK == 1 or not dev["K1"].is_contiguous())      # (size-1 dims make a permuted view contiguous)
    for splits in (7, 0):
        kl, l1, l2 = skl.streamkl_fwd_splitk(dev["Q1"], dev["K1"], dev["Q2"], dev["K2"], cfg.c1, cfg.c2, cfg.causal, splits=splits,
                                             student_activation=act2)
        assert skl.streamkl_last_launch_count() == 2
        check_fwd(to_f64(kl), to_f64(l1), to_f64(l2), ref, f"{cfg.name} NQ={NQ} G={G} {dtype} {act2} splits={splits}")
    # the same statistics as the unsplit kernel on the same layout (fp32 merge order differs)
    kl0, l10, l20 = skl.streamkl_fwd(dev["Q1"], dev["K1"], dev["Q2"], dev["K2"], cfg.c1, cfg.c2, cfg.causal, student_activation=act2)
    assert np.abs(to_f64(l1) - to_f64(l10)).max() <= 1e-4 and np.abs(to_f64(l2) - to_f64(l20)).max() <= 1e-4
    assert np.abs(to_f64(kl) - to_f64(kl0)).max() <= 3e-4


def test_splitk_ex_wide_head_dims_and_odd_dims():
    import paper_2606_20005_b200 as skl
    from test_layouts_gpu import _inputs, _ref

    for d1, d2 in ((192, 64), (96, 40)):
        cfg = W.Config(65, "splitk-ex-d", 1, 4, 33, 2048 + 5, d1, d2, "f16", False)
        inp = _inputs(cfg, 2)
        ref = _ref(cfg, inp, 2, False, inp["g"], None)
        dev = [to_torch(inp[k]) for k in ("Q1", "K1", "Q2", "K2")]
        kl, l1, l2 = skl.streamkl_fwd_splitk(*dev, cfg.c1, cfg.c2, False, splits=5)
        assert skl.streamkl_last_launch_count() == 2
        check_fwd(to_f64(kl), to_f64(l1), to_f64(l2), ref, f"{cfg.name} d={d1}/{d2}")
