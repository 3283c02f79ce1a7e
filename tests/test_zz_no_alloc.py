"""GPU test of streamkl_fwd_splitk_noalloc: the split-K forward for callers that cannot allocate device memory when they call
(plugins that run inside a host application's fixed memory arena, latency-bound decode loops where a cudaMalloc would stall the
whole device, processes whose HBM share is already spent).  Its per-chunk partial statistics go to a 4 MiB array built into
libstreamkl.so instead of a caller-owned workspace.

What is checked, on two calls in a row that share that array:
  * each call agrees with the existing streamkl_fwd_splitk (caller-owned workspace) at the same W -- the kernels and their
    arithmetic are the same, so the bar is equality, far inside the tolerance the split-K parity tests use (lse 1e-3,
    KL 2e-3 + 1e-2|ref| against the float64 oracle, which is checked here as well);
  * the second call has a different shape and split count from the first, so its partials land on different offsets of the
    array the first call left full: a call that depended on the array's previous contents would fail here;
  * a split count whose partials exceed the built-in array is refused with STREAMKL_ERR_SCRATCH_LIMIT and leaves the outputs
    untouched, while the adaptive choice (splits <= 0) quietly settles on a W that fits.
The calls run one after the other on one stream: calls that overlap on the GPU share the array and would race (see the header).

This file is named to be collected last: `pytest -x` stops at the first failure, and a failure here should not hide the parity
tests.  It passes alone in a fresh process (the first call then does the one-time address lookup) and after the other tests."""
from __future__ import annotations

import numpy as np
import pytest

import workloads as W
from oracle.streamkl_oracle import attention_kl
from parity_util import bits_to_f64, check_fwd, to_f64, to_torch

pytestmark = pytest.mark.gpu


def _inputs(cfg):
    inp = W.all_inputs(cfg)
    dev = tuple(to_torch(inp[k]) for k in ("Q1", "K1", "Q2", "K2"))
    ref = attention_kl(*(bits_to_f64(inp[k]) for k in ("Q1", "K1", "Q2", "K2")), cfg.c1, cfg.c2, cfg.causal)
    return dev, ref


def _both_paths(cfg, splits):
    """(no-alloc outputs, workspace-path outputs, oracle) for one problem; outputs preallocated, so the no-alloc call
    allocates nothing on the Python side either."""
    import torch
    import paper_2606_20005_b200 as skl

    (Q1, K1, Q2, K2), ref = _inputs(cfg)
    outs = [torch.full((cfg.B, cfg.H, cfg.NQ), float("nan"), dtype=torch.float32, device="cuda") for _ in range(3)]
    got = skl.streamkl_fwd_splitk_noalloc(Q1, K1, Q2, K2, cfg.c1, cfg.c2, cfg.causal, splits=splits,
                                          kl_rows=outs[0], lse1=outs[1], lse2=outs[2])
    assert skl.streamkl_last_launch_count() == 2          # split kernel + reduce kernel, as on the workspace path
    want = skl.streamkl_fwd_splitk(Q1, K1, Q2, K2, cfg.c1, cfg.c2, cfg.causal, splits=splits)
    torch.cuda.synchronize()
    return got, want, ref


def test_no_alloc_splitk_matches_the_workspace_path_on_two_calls_in_a_row():
    import paper_2606_20005_b200 as skl

    assert skl.streamkl_fwd_splitk_noalloc_capacity() == 4 << 20
    # call 1: 4 heads x 200 rows x 9 chunks (causal: late chunks are invisible to early rows -> identity partials);
    # call 2: 6 heads x 16 rows x 5 chunks, other head dims, no mask -- smaller, so it lands inside what call 1 wrote
    cases = [(W.Config(70, "noalloc-a", 2, 2, 200, 4096 + 17, 128, 128, "bf16", True), 9),
             (W.Config(71, "noalloc-b", 1, 6, 16, 2048 + 5, 128, 64, "bf16", False), 5)]
    for cfg, splits in cases:
        got, want, ref = _both_paths(cfg, splits)
        for name, g, w in zip(("kl_rows", "lse1", "lse2"), got, want):
            assert np.array_equal(to_f64(g), to_f64(w)), f"{cfg.name}: {name} differs from streamkl_fwd_splitk"
        check_fwd(to_f64(got[0]), to_f64(got[1]), to_f64(got[2]), ref, cfg.name)


def test_no_alloc_splitk_refuses_what_does_not_fit_and_adapts_when_asked():
    import torch
    import paper_2606_20005_b200 as skl

    cap = skl.streamkl_fwd_splitk_noalloc_capacity()
    cfg = W.Config(72, "noalloc-big", 1, 32, 256, 8192, 64, 64, "bf16", False)     # 32*256*5*4 = 160 KiB per chunk
    (Q1, K1, Q2, K2), ref = _inputs(cfg)
    w_fit = cap // (skl.streamkl_fwd_splitk_workspace_bytes(cfg.B, cfg.H, cfg.NQ, 2) // 2)     # 25
    assert skl.streamkl_fwd_splitk_workspace_bytes(cfg.B, cfg.H, cfg.NQ, w_fit + 1) > cap >= \
        skl.streamkl_fwd_splitk_workspace_bytes(cfg.B, cfg.H, cfg.NQ, w_fit)
    outs = [torch.full((cfg.B, cfg.H, cfg.NQ), -7.0, dtype=torch.float32, device="cuda") for _ in range(3)]
    with pytest.raises(skl.StreamKLError) as e:
        skl.streamkl_fwd_splitk_noalloc(Q1, K1, Q2, K2, cfg.c1, cfg.c2, cfg.causal, splits=w_fit + 1,
                                        kl_rows=outs[0], lse1=outs[1], lse2=outs[2])
    assert e.value.code == skl.STREAMKL_ERR_SCRATCH_LIMIT
    torch.cuda.synchronize()
    assert all(bool((o == -7.0).all()) for o in outs)       # a refused call enqueues nothing
    # the largest W that fits runs, and so does the adaptive choice
    for splits in (w_fit, 0):
        kl, l1, l2 = skl.streamkl_fwd_splitk_noalloc(Q1, K1, Q2, K2, cfg.c1, cfg.c2, cfg.causal, splits=splits,
                                                     kl_rows=outs[0], lse1=outs[1], lse2=outs[2])
        check_fwd(to_f64(kl), to_f64(l1), to_f64(l2), ref, f"{cfg.name} splits={splits}")
