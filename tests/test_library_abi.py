"""CPU-side checks of the C-ABI boundary: the library builds, loads without a GPU, exports every symbol the header
declares, validates arguments before touching the device, and refuses to compute without an sm_100 GPU
(no CPU fallback).  No compute calls are made here."""
from __future__ import annotations

import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "streamkl.h")


@pytest.fixture(scope="module")
def L():
    from paper_2606_20005_b200.build import build_library

    build_library()
    from paper_2606_20005_b200.binding import lib

    return lib()


def declared_functions():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(streamkl_[a-z0-9_]+)\s*\(", src)))


def test_header_declares_the_north_star_entry_points():
    names = declared_functions()
    for must in ("streamkl_fwd", "streamkl_bwd", "streamkl_fwd_f32", "streamkl_bwd_f32", "streamkl_bwd_workspace_bytes",
                 "streamkl_fwd_host", "streamkl_fwd_bwd_host", "streamkl_strerror", "streamkl_version"):
        assert must in names


def test_every_declared_symbol_is_exported(L):
    for name in declared_functions():
        assert hasattr(L, name), f"{name} declared in include/streamkl.h but not exported"


def test_binding_exposes_the_same_names():
    import paper_2606_20005_b200 as skl

    for name in declared_functions():
        if name.endswith("_f32") or name.endswith("_ex"):
            continue  # the binding dispatches on the tensor's dtype, strides and head counts (streamkl_fwd / streamkl_bwd)
        assert hasattr(skl, name)


def test_version_and_strerror(L):
    assert b"sm_100a" in L.streamkl_version()
    assert L.streamkl_strerror(0) == b"ok"
    msgs = {L.streamkl_strerror(c) for c in range(-8, 1)}
    assert len(msgs) == 9


def _call_fwd(L, ptrs=(16, 16, 16, 16), B=1, H=1, NQ=8, NK=8, d1=64, d2=64, c1=0.125, c2=0.125, causal=0, outs=(16, 16, 16)):
    return L.streamkl_fwd(*[ctypes.c_void_p(p) for p in ptrs], B, H, NQ, NK, d1, d2, c1, c2, causal,
                          *[ctypes.c_void_p(p) for p in outs], ctypes.c_void_p(0))


def test_argument_validation_happens_before_any_device_work(L):
    ERR_NULL, ERR_SHAPE, ERR_ALIGN, ERR_SCALE, ERR_CUDA = -1, -2, -3, -4, -6
    assert _call_fwd(L, NK=0) == ERR_SHAPE
    assert _call_fwd(L, d1=0) == ERR_SHAPE
    assert _call_fwd(L, d2=300) == ERR_SHAPE
    assert _call_fwd(L, NQ=9, NK=8, causal=1) == ERR_SHAPE      # R5: causal needs NQ <= NK
    assert _call_fwd(L, c1=0.0) == ERR_SCALE
    assert _call_fwd(L, c2=float("nan")) == ERR_SCALE
    assert _call_fwd(L, ptrs=(0, 16, 16, 16)) == ERR_NULL
    assert _call_fwd(L, ptrs=(16, 24, 16, 16)) == ERR_ALIGN
    assert _call_fwd(L, outs=(0, 16, 16)) == ERR_NULL
    assert _call_fwd(L, B=0) == 0                                 # empty batch: successful no-op
    assert _call_fwd(L, NQ=0) == 0


def test_no_gpu_means_error_not_fallback(L):
    import torch

    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    assert _call_fwd(L) == -6  # STREAMKL_ERR_CUDA: the product path never computes on the CPU
    import paper_2606_20005_b200 as skl

    a = np.zeros((1, 1, 4, 64), np.float32)
    with pytest.raises(skl.StreamKLError):
        skl.streamkl_fwd_host(a, a, a, a, 0.125, 0.125, False)


def test_bwd_teacher_pointers_must_come_in_pairs(L):
    vp = ctypes.c_void_p
    rc = L.streamkl_bwd(vp(16), vp(16), vp(16), vp(16), 1, 1, 8, 8, 64, 64, 0.125, 0.125, 0, vp(16), vp(16), vp(16), vp(16),
                        vp(16), vp(0), vp(16), vp(16), vp(0), 0, vp(0))
    assert rc == -1


def test_workspace_is_never_quadratic(L):
    small = L.streamkl_bwd_workspace_bytes(1, 32, 4096, 4096, 128, 128, 1)
    big = L.streamkl_bwd_workspace_bytes(1, 32, 65536, 65536, 128, 128, 1)
    assert big <= 16 * max(small, 1) + 4 * 32 * 65536 * 256 * 4  # O((NQ+NK) d), not O(NQ NK)


def test_bwd_workspace_follows_the_selected_strategy(L):
    """16 B of packed per-query scalars (rows padded to 64 per head) always; the fp32 dQ accumulators of the one-visit kernels
    only when that strategy will run (mode FUSED, or AUTO with NQ <= 512 / <= 256 with teacher gradients, or AUTO with a frozen teacher,
    d2 <= 64 and NQ >= 32768) -- cfg 3 (Setting 1, NQ = 16384) needs 8 MB, not 143."""
    a256 = lambda n: (n + 255) // 256 * 256
    assert L.streamkl_set_bwd_mode(0) == 0   # AUTO
    assert L.streamkl_bwd_workspace_bytes(1, 32, 65536, 65536, 128, 128, 1) == 32 * 65536 * 16
    assert L.streamkl_bwd_workspace_bytes(1, 32, 16384, 16384, 128, 64, 0) == 32 * 16384 * 16              # cfg 3: 8 MB
    # frozen teacher, d2 <= 64, NQ >= 32768 under AUTO: the one-visit student pass (measured 7-11 % faster), + fp32 dQ2
    assert L.streamkl_bwd_workspace_bytes(1, 8, 32768, 32768, 128, 64, 0) == a256(8 * 32768 * 16) + a256(8 * 32768 * 64 * 4)
    assert L.streamkl_bwd_workspace_bytes(1, 8, 32768, 32768, 128, 48, 0) == a256(8 * 32768 * 16) + a256(8 * 32768 * 64 * 4)   # padded to 64
    assert L.streamkl_bwd_workspace_bytes(1, 8, 32768, 32768, 128, 64, 1) == 8 * 32768 * 16                # teacher gradients: owner kernels
    assert L.streamkl_bwd_workspace_bytes(1, 8, 32768, 32768, 128, 128, 0) == 8 * 32768 * 16               # d2 = 128: owner kernels
    assert L.streamkl_bwd_workspace_bytes(1, 8, 32704, 32768, 128, 64, 0) == 8 * 32704 * 16                # below 32K: owner kernels
    # NQ <= 512 under AUTO: one-visit kernels, + fp32 dQ2 (+ dQ1 with teacher gradients), each region 256-byte aligned
    assert L.streamkl_bwd_workspace_bytes(2, 3, 100, 777, 128, 64, 0) == a256(6 * 128 * 16) + a256(6 * 100 * 64 * 4)
    assert L.streamkl_bwd_workspace_bytes(2, 3, 100, 777, 128, 64, 1) == a256(6 * 128 * 16) + a256(6 * 100 * 64 * 4) + a256(6 * 100 * 128 * 4)
    assert L.streamkl_set_bwd_mode(1) == 0   # SEPARATE: never the accumulators
    assert L.streamkl_bwd_workspace_bytes(2, 3, 100, 777, 128, 64, 0) == 6 * 128 * 16
    assert L.streamkl_bwd_workspace_bytes(2, 3, 100, 777, 128, 64, 1) == 6 * 128 * 16
    assert L.streamkl_set_bwd_mode(2) == 0   # FUSED: always
    assert L.streamkl_bwd_workspace_bytes(1, 32, 16384, 16384, 128, 64, 0) == a256(32 * 16384 * 16) + a256(32 * 16384 * 64 * 4)
    assert L.streamkl_set_bwd_mode(0) == 0
    assert L.streamkl_bwd_workspace_bytes(1, 1, 256, 256, 44, 80, 0) == 0                  # head dim not a multiple of 8: SIMT path, no workspace
    assert L.streamkl_bwd_workspace_bytes(1, 1, 256, 256, 192, 64, 0) == 256 * 16          # head dim > 128: wide owner kernels, statistics only
    assert L.streamkl_bwd_workspace_bytes(1, 1, 256, 256, 264, 64, 0) == 0                 # head dim > 256: SIMT path


def test_splitk_adaptive_split_selection_follows_the_paper_rule(L):
    """W = 1 if P_base >= P_target else min(floor(P_target / P_base), T_K); P_base = bsz * T_Q."""
    f = L.streamkl_fwd_splitk_splits
    assert f(1, 16, 1, 131072, 256) == 16            # P_base = 16 -> floor(256/16)
    assert f(1, 16, 64, 131072, 128) == 8
    assert f(4, 64, 16, 131072, 256) == 1            # P_base = 256 >= P_target: default kernel
    assert f(1, 1, 1, 200, 256) == 2                 # clamped by T_K = ceil(200/128)
    assert f(1, 16, 300, 8192, 256) == 5             # T_Q = ceil(300/128) = 3 -> P_base = 48
    assert f(1, 16, 16, 65536, 0) == 9               # default target: 148 CTAs = one per SM
    assert f(0, 16, 16, 65536, 0) == 1


def test_splitk_workspace_and_argument_checks(L):
    vp = ctypes.c_void_p
    assert L.streamkl_fwd_splitk_workspace_bytes(1, 16, 32, 8) == 16 * 8 * 5 * 32 * 4
    assert L.streamkl_fwd_splitk_workspace_bytes(1, 16, 32, 1) == 0

    def call(ws, ws_bytes, splits=8, d1=128, NK=4096):
        return L.streamkl_fwd_splitk(vp(16), vp(16), vp(16), vp(16), 1, 16, 32, NK, d1, 128, 0.1, 0.1, 0, splits,
                                     vp(16), vp(16), vp(16), vp(ws), ctypes.c_size_t(ws_bytes), vp(0))

    assert call(0, 0) == -5                                   # STREAMKL_ERR_WORKSPACE
    assert call(16, 100) == -5
    assert call(24, 1 << 20) == -3                            # misaligned workspace
    assert call(16, 1 << 20, NK=0) in (-2, -5)                # shape errors are still reported


def test_bwd_mode_selector(L):
    assert L.streamkl_set_bwd_mode(1) == 0 and L.streamkl_set_bwd_mode(2) == 0 and L.streamkl_set_bwd_mode(0) == 0
    assert L.streamkl_set_bwd_mode(7) == -2
    assert all(L.streamkl_set_fwd_plan(v) == 0 for v in (1, 2, 3, 4, 0)) and L.streamkl_set_fwd_plan(5) == -2 and L.streamkl_set_fwd_plan(-1) == -2


def test_no_alloc_splitk_limit_is_checked_on_the_host(L):
    """streamkl_fwd_splitk_noalloc: the capacity is the header's constant, an explicit split count whose partials exceed it is
    refused before the device is touched, and argument errors still come first when it fits."""
    L.streamkl_fwd_splitk_noalloc.restype = ctypes.c_int
    L.streamkl_fwd_splitk_noalloc_capacity.restype = ctypes.c_size_t
    assert L.streamkl_fwd_splitk_noalloc_capacity() == 4 << 20
    assert "#define STREAMKL_NOALLOC_SCRATCH_BYTES (4u << 20)" in open(HEADER).read()
    vp = ctypes.c_void_p

    def call(B, H, NQ, NK, splits, c1=0.125, ptr=16):
        return L.streamkl_fwd_splitk_noalloc(vp(ptr), vp(16), vp(16), vp(16), B, H, NQ, NK, 64, 64, ctypes.c_float(c1),
                                             ctypes.c_float(0.125), 0, splits, vp(16), vp(16), vp(16), vp(0))

    # 32 heads x 256 rows: 160 KiB of partials per chunk, so 25 chunks fit in 4 MiB and 26 do not
    assert call(1, 32, 256, 8192, 26) == -8
    assert L.streamkl_strerror(-8) not in (b"unknown error code", b"workspace missing or too small")
    assert call(1, 32, 256, 8192, 25, c1=float("nan")) == -4          # STREAMKL_ERR_SCALE before any device work
    assert call(1, 32, 256, 8192, 25, ptr=8) == -3                    # STREAMKL_ERR_ALIGN
    assert call(1, 32, 256, 8192, 25) == -6                           # valid arguments, no GPU here: STREAMKL_ERR_CUDA


def test_bwd_refuses_views_whose_gradient_rows_would_overlap(L):
    """Gradients are stored through the input's strides, so a broadcast (stride 0) or self-overlapping view of a tensor that
    receives a gradient is an argument error in the backward (the forward, which only reads, accepts it)."""
    from paper_2606_20005_b200 import StreamKLLayout

    vp = ctypes.c_void_p
    B, H, NQ, NK, d = 2, 4, 8, 16, 64

    def bwd(lay, teacher):
        g1 = vp(16) if teacher else vp(0)
        return L.streamkl_bwd_ex(ctypes.cast(ctypes.pointer(lay), vp), vp(16), vp(16), vp(16), vp(16), B, H, NQ, NK, d, d,
                                 ctypes.c_float(0.125), ctypes.c_float(0.125), 0, vp(16), vp(16), vp(16), vp(16), g1, g1, vp(16), vp(16),
                                 vp(16), ctypes.c_size_t(1 << 30), vp(0))

    def fwd(lay):
        return L.streamkl_fwd_ex(ctypes.cast(ctypes.pointer(lay), vp), vp(16), vp(16), vp(16), vp(16), B, H, NQ, NK, d, d,
                                 ctypes.c_float(0.125), ctypes.c_float(0.125), 0, vp(16), vp(16), vp(16), vp(0))

    def layout(**strides):
        lay = StreamKLLayout()
        lay.dtype = 0
        for name, v in strides.items():
            for i in range(3):
                getattr(lay, name)[i] = v[i]
        return lay

    ok = -6                                                   # valid arguments reach the device check (no GPU here)
    assert bwd(layout(k2_stride=(H * NK * d, NK * d, d)), False) == ok
    assert bwd(layout(k2_stride=(NK * H * d, d, H * d)), False) == ok          # [B][N][H][d]: interleaved, disjoint
    expanded = layout(k2_stride=(H * NK * d, 0, d))           # K2.expand over heads: H owners would store to one dK2 head
    assert fwd(expanded) == ok and bwd(expanded, False) == -2
    assert bwd(layout(q2_stride=(0, NQ * d, d)), False) == -2                  # broadcast batch
    assert bwd(layout(k2_stride=(H * NK * d, d, d)), False) == -2              # heads one row apart: rows of different heads coincide
    assert bwd(layout(q2_stride=(H * NQ * d, NQ * d - 8, d)), False) == -2     # head stride short of a head's rows
    frozen_teacher = layout(k1_stride=(H * NK * d, 0, d))     # a broadcast teacher is fine while it receives no gradient
    assert bwd(frozen_teacher, False) == ok and bwd(frozen_teacher, True) == -2


def test_build_digest_covers_every_source_kind_and_is_location_independent():
    """The stamp that decides whether libstreamkl.so is current hashes every file that reaches the compiler -- the .inc launchers
    included -- under paths relative to the repository, so the same tree gives the same digest wherever it is checked out."""
    from paper_2606_20005_b200 import build

    names = {os.path.basename(f) for f in build._all_inputs()}
    csrc = os.path.join(os.path.dirname(build.__file__), "csrc")
    assert {f for f in os.listdir(csrc) if f.endswith((".cu", ".cuh", ".inc", ".h"))} <= names
    assert "streamkl_bwd_owner.inc" in names and "streamkl.h" in names
    import inspect

    assert "relpath" in inspect.getsource(build._digest)
