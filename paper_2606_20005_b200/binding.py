"""ctypes binding of libstreamkl.so -- same names as include/streamkl.h, argument marshalling only.

Device entry points take torch CUDA tensors (torch supplies device memory and the current stream, nothing
else); `*_host` entry points take numpy arrays (bf16 carried as uint16 bit patterns, or float32).
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

from .build import LIB_PATH

__all__ = [
    "StreamKLError", "lib", "lib_path", "streamkl_fwd", "streamkl_bwd", "streamkl_bwd_workspace_bytes",
    "streamkl_fwd_splitk", "streamkl_fwd_splitk_splits", "streamkl_fwd_splitk_workspace_bytes",
    "streamkl_fwd_splitk_noalloc", "streamkl_fwd_splitk_noalloc_capacity", "STREAMKL_ERR_SCRATCH_LIMIT",
    "streamkl_fwd_host", "streamkl_fwd_bwd_host", "streamkl_host_trim", "streamkl_set_bwd_mode", "streamkl_set_fwd_plan", "STREAMKL_FWD_SINGLE", "STREAMKL_FWD_MULTICAST", "STREAMKL_FWD_PAIR_MMA", "STREAMKL_FWD_PERSISTENT", "STREAMKL_FWD_PER_TILE", "STREAMKL_FWD_AUTO",
    "STREAMKL_BWD_AUTO", "STREAMKL_BWD_SEPARATE", "STREAMKL_BWD_FUSED", "STREAMKL_BF16", "STREAMKL_F16", "STREAMKL_F32", "StreamKLLayout", "streamkl_last_launch_count", "streamkl_strerror",
    "streamkl_profile_enable", "streamkl_profile_collect", "streamkl_kernel_name",
    "streamkl_version",
]

STREAMKL_BF16, STREAMKL_F32, STREAMKL_F16 = 0, 1, 2
STREAMKL_ERR_SCRATCH_LIMIT = -8


class StreamKLLayout(ctypes.Structure):
    """struct streamkl_layout of include/streamkl.h."""

    _fields_ = [("dtype", ctypes.c_int), ("kv_heads", ctypes.c_int), ("q1_stride", ctypes.c_longlong * 3),
                ("k1_stride", ctypes.c_longlong * 3), ("q2_stride", ctypes.c_longlong * 3), ("k2_stride", ctypes.c_longlong * 3),
                ("student_activation", ctypes.c_int)]
STREAMKL_BWD_AUTO, STREAMKL_BWD_SEPARATE, STREAMKL_BWD_FUSED = 0, 1, 2
STREAMKL_FWD_SINGLE, STREAMKL_FWD_MULTICAST, STREAMKL_FWD_PAIR_MMA, STREAMKL_FWD_PERSISTENT, STREAMKL_FWD_PER_TILE = 0, 1, 2, 3, 4
STREAMKL_FWD_AUTO = 0


class StreamKLError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        super().__init__(f"{where}: {streamkl_strerror(code)} (code {code})")


_lib = None


def lib_path() -> str:
    return LIB_PATH


def lib() -> ctypes.CDLL:
    """Load libstreamkl.so (built in-tree by `python -m paper_2606_20005_b200.build`).  Fails loudly if absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            f"{LIB_PATH} is missing: build it with `python -m paper_2606_20005_b200.build` "
            "(there is no CPU fallback for the StreamKL hot path)")
    L = ctypes.CDLL(LIB_PATH)
    vp, ci, cf, sz = ctypes.c_void_p, ctypes.c_int, ctypes.c_float, ctypes.c_size_t
    shape = [ci] * 6 + [cf, cf, ci]  # B,H,NQ,NK,d1,d2,c1,c2,causal
    for name in ("streamkl_fwd", "streamkl_fwd_f32"):
        f = getattr(L, name)
        f.argtypes = [vp] * 4 + shape + [vp] * 3 + [vp]
        f.restype = ci
    for name in ("streamkl_bwd", "streamkl_bwd_f32"):
        f = getattr(L, name)
        f.argtypes = [vp] * 4 + shape + [vp] * 4 + [vp] * 4 + [vp, sz, vp]
        f.restype = ci
    L.streamkl_fwd_ex.argtypes = [vp] + [vp] * 4 + shape + [vp] * 3 + [vp]
    L.streamkl_fwd_ex.restype = ci
    L.streamkl_bwd_ex.argtypes = [vp] + [vp] * 4 + shape + [vp] * 4 + [vp] * 4 + [vp, sz, vp]
    L.streamkl_bwd_ex.restype = ci
    L.streamkl_fwd_splitk.argtypes = [vp] * 4 + shape + [ci] + [vp] * 3 + [vp, sz, vp]
    L.streamkl_fwd_splitk.restype = ci
    L.streamkl_fwd_splitk_ex.argtypes = [vp] + [vp] * 4 + shape + [ci] + [vp] * 3 + [vp, sz, vp]
    L.streamkl_fwd_splitk_ex.restype = ci
    L.streamkl_fwd_splitk_splits.argtypes = [ci] * 5
    L.streamkl_fwd_splitk_splits.restype = ci
    L.streamkl_fwd_splitk_workspace_bytes.argtypes = [ci] * 4
    L.streamkl_fwd_splitk_workspace_bytes.restype = sz
    L.streamkl_fwd_splitk_noalloc.argtypes = [vp] * 4 + shape + [ci] + [vp] * 3 + [vp]
    L.streamkl_fwd_splitk_noalloc.restype = ci
    L.streamkl_fwd_splitk_noalloc_capacity.argtypes = []
    L.streamkl_fwd_splitk_noalloc_capacity.restype = sz
    L.streamkl_bwd_workspace_bytes.argtypes = [ci] * 7
    L.streamkl_bwd_workspace_bytes.restype = sz
    L.streamkl_fwd_host.argtypes = [ci] + [vp] * 4 + shape + [vp] * 3 + [vp]
    L.streamkl_fwd_host.restype = ci
    L.streamkl_fwd_bwd_host.argtypes = [ci] + [vp] * 4 + shape + [vp] + [vp] * 3 + [vp] * 4 + [vp]
    L.streamkl_fwd_bwd_host.restype = ci
    L.streamkl_set_bwd_mode.argtypes = [ci]
    L.streamkl_set_bwd_mode.restype = ci
    L.streamkl_set_fwd_plan.argtypes = [ci]
    L.streamkl_set_fwd_plan.restype = ci
    L.streamkl_host_trim.argtypes = []
    L.streamkl_host_trim.restype = ci
    L.streamkl_last_launch_count.argtypes = []
    L.streamkl_last_launch_count.restype = ci
    L.streamkl_profile_enable.argtypes = [ci]
    L.streamkl_profile_enable.restype = ci
    L.streamkl_profile_collect.argtypes = [ci, vp, vp]
    L.streamkl_profile_collect.restype = ci
    L.streamkl_kernel_name.argtypes = [ci]
    L.streamkl_kernel_name.restype = ctypes.c_char_p
    L.streamkl_strerror.argtypes = [ci]
    L.streamkl_strerror.restype = ctypes.c_char_p
    L.streamkl_version.argtypes = []
    L.streamkl_version.restype = ctypes.c_char_p
    _lib = L
    return L


def streamkl_strerror(code: int) -> str:
    return lib().streamkl_strerror(int(code)).decode()


def streamkl_version() -> str:
    return lib().streamkl_version().decode()


def streamkl_set_fwd_plan(plan: int) -> None:
    """STREAMKL_FWD_AUTO (default: per-tile or persistent by a measured rule) | STREAMKL_FWD_PER_TILE | STREAMKL_FWD_PERSISTENT |
    STREAMKL_FWD_MULTICAST (cluster pairs sharing one multicast K stream) | STREAMKL_FWD_PAIR_MMA (head dims above 128: cluster
    pairs issuing cta_group::2 MMAs).  All plans give bit-identical results."""
    rc = lib().streamkl_set_fwd_plan(int(plan))
    if rc != 0:
        raise StreamKLError(rc, "streamkl_set_fwd_plan")


def streamkl_set_bwd_mode(mode: int) -> None:
    """STREAMKL_BWD_AUTO | STREAMKL_BWD_SEPARATE (deterministic) | STREAMKL_BWD_FUSED (Setting 1, dQ2 by fp32 atomics)."""
    rc = lib().streamkl_set_bwd_mode(int(mode))
    if rc != 0:
        raise StreamKLError(rc, "streamkl_set_bwd_mode")


def streamkl_host_trim() -> None:
    rc = lib().streamkl_host_trim()
    if rc != 0:
        raise StreamKLError(rc, "streamkl_host_trim")


def streamkl_last_launch_count() -> int:
    return int(lib().streamkl_last_launch_count())


def streamkl_profile_enable(on) -> None:
    """on = False/0: off; True/1: on; n > 1: on, with n event pairs created up front (none created inside a timed region)."""
    lib().streamkl_profile_enable(int(on))


def streamkl_profile_collect(max_records: int = 4096):
    """-> list of (kernel_name, ms) for every kernel launched on this thread since profiling was enabled / last collected."""
    ids = (ctypes.c_int * max_records)()
    ms = (ctypes.c_float * max_records)()
    n = lib().streamkl_profile_collect(max_records, ctypes.cast(ids, ctypes.c_void_p), ctypes.cast(ms, ctypes.c_void_p))
    if n < 0:
        raise StreamKLError(n, "streamkl_profile_collect")
    return [(lib().streamkl_kernel_name(ids[i]).decode(), float(ms[i])) for i in range(n)]


def streamkl_kernel_name(kernel_id: int) -> str:
    return lib().streamkl_kernel_name(int(kernel_id)).decode()


def streamkl_bwd_workspace_bytes(B, H, NQ, NK, d1, d2, want_teacher_grads) -> int:
    return int(lib().streamkl_bwd_workspace_bytes(B, H, NQ, NK, d1, d2, int(bool(want_teacher_grads))))


# ------------------------------------------------------------------------------------------ device entry points
def _keep_alive_on(t, stream):
    """A scratch tensor allocated here (on torch's current stream) is used by kernels enqueued on `stream` and dropped when the
    call returns: tell the caching allocator, so that the block is not handed to other work while those kernels still run."""
    if stream is not None:   # a torch.cuda.Stream other than (possibly) the current one
        t.record_stream(stream)


def _check_dev(name, t, dtype=None, strided=False):
    import torch

    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise TypeError(f"{name}: expected a CUDA torch tensor")
    if strided:
        if t.dim() != 4 or (t.shape[-1] > 1 and t.stride(-1) != 1):
            raise TypeError(f"{name}: expected a [B,H,N,d] CUDA tensor whose last dimension is contiguous")
    elif not t.is_contiguous():
        raise TypeError(f"{name}: expected a contiguous CUDA torch tensor")
    if dtype is not None and t.dtype != dtype:
        raise TypeError(f"{name}: expected dtype {dtype}, got {t.dtype}")


def _rows_are_disjoint(t) -> bool:
    """The library's test (rows_are_disjoint in csrc/streamkl.cu) on a [B,H,N,d] tensor: distinct (b,h,n) -> disjoint rows."""
    span = int(t.shape[3])
    for stride, extent in sorted((int(t.stride(i)), int(t.shape[i])) for i in range(3)):
        if extent <= 1:
            continue
        if stride < span:
            return False
        span += stride * (extent - 1)
    return True


def _shape_of(Q1, K1, Q2, K2):
    """-> (B, H, NQ, NK, d1, d2, HK): K tensors may carry HK <= H heads (H % HK == 0; query head h reads K head h // (H // HK))."""
    if Q1.dim() != 4 or K1.dim() != 4 or Q2.dim() != 4 or K2.dim() != 4:
        raise ValueError("Q1,K1,Q2,K2 must be [B,H,N,d]")
    B, H, NQ, d1 = Q1.shape
    HK, NK, d2 = K1.shape[1], K1.shape[2], Q2.shape[3]
    if tuple(K1.shape) != (B, HK, NK, d1) or tuple(Q2.shape) != (B, H, NQ, d2) or tuple(K2.shape) != (B, HK, NK, d2):
        raise ValueError("inconsistent Q1,K1,Q2,K2 shapes")
    if HK < 1 or H % HK != 0:
        raise ValueError("the number of query heads must be a multiple of the number of K heads")
    return B, H, NQ, NK, d1, d2, HK


STREAMKL_ACT_NONE, STREAMKL_ACT_RELU = 0, 1
_ACTS = {None: STREAMKL_ACT_NONE, "none": STREAMKL_ACT_NONE, "relu": STREAMKL_ACT_RELU}


def _layout_of(Q1, K1, Q2, K2, HK, student_activation=None):
    """A StreamKLLayout for 16-bit tensors given as (possibly strided) [B,H,N,d] views, or None when everything is the
    contiguous bf16 / fp32 default that the plain entry points take."""
    import torch

    act = _ACTS[student_activation]
    plain = all(t.is_contiguous() for t in (Q1, K1, Q2, K2)) and HK == Q1.shape[1] and act == STREAMKL_ACT_NONE
    if plain and Q1.dtype in (torch.bfloat16, torch.float32):
        return None
    if Q1.dtype not in (torch.bfloat16, torch.float16):
        raise TypeError("strided tensors / shared K heads / student activations need bfloat16 or float16 inputs")
    L = StreamKLLayout()
    L.student_activation = act
    L.dtype = STREAMKL_BF16 if Q1.dtype == torch.bfloat16 else STREAMKL_F16
    L.kv_heads = int(HK)
    for name, t in (("q1_stride", Q1), ("k1_stride", K1), ("q2_stride", Q2), ("k2_stride", K2)):
        arr = getattr(L, name)
        _, heads, n, d = t.shape
        sb, sh, sn, _ = t.stride()
        # torch leaves the stride of a size-1 axis arbitrary: substitute the packed value (it is never used to move)
        sn = sn if n > 1 else d
        sh = sh if heads > 1 else n * sn
        sb = sb if t.shape[0] > 1 else heads * sh
        arr[0], arr[1], arr[2] = int(sb), int(sh), int(sn)
    return L


def _stream_handle(stream):
    import torch

    if stream is None:
        stream = torch.cuda.current_stream()
    return ctypes.c_void_p(stream.cuda_stream)


def _ptr(t):
    return ctypes.c_void_p(t.data_ptr()) if t is not None else ctypes.c_void_p(0)


def streamkl_fwd(Q1, K1, Q2, K2, c1, c2, causal, kl_rows=None, lse1=None, lse2=None, stream=None, student_activation=None):
    """Forward (Algorithm 1).  Returns (kl_rows, lse1, lse2), each [B,H,NQ] float32.  bf16 / fp16 / fp32 inputs; 16-bit inputs
    may be strided [B,H,N,d] views (last dimension contiguous) and K may have fewer heads than Q (shared K heads)."""
    import torch

    for n, t in (("Q1", Q1), ("K1", K1), ("Q2", Q2), ("K2", K2)):
        _check_dev(n, t, Q1.dtype, strided=True)
    B, H, NQ, NK, d1, d2, HK = _shape_of(Q1, K1, Q2, K2)
    layout = _layout_of(Q1, K1, Q2, K2, HK, student_activation)
    outs = []
    for n, t in (("kl_rows", kl_rows), ("lse1", lse1), ("lse2", lse2)):
        if t is None:
            t = torch.empty((B, H, NQ), dtype=torch.float32, device=Q1.device)
        _check_dev(n, t, torch.float32)
        outs.append(t)
    args = (_ptr(Q1), _ptr(K1), _ptr(Q2), _ptr(K2), B, H, NQ, NK, d1, d2, float(c1), float(c2), int(bool(causal)),
            _ptr(outs[0]), _ptr(outs[1]), _ptr(outs[2]), _stream_handle(stream))
    with torch.cuda.device(Q1.device):
        if layout is not None:
            rc = lib().streamkl_fwd_ex(ctypes.cast(ctypes.pointer(layout), ctypes.c_void_p), *args)
        elif Q1.dtype == torch.bfloat16:
            rc = lib().streamkl_fwd(*args)
        else:
            rc = lib().streamkl_fwd_f32(*args)
    if rc != 0:
        raise StreamKLError(rc, "streamkl_fwd")
    return tuple(outs)


def streamkl_fwd_splitk_splits(B, H, NQ, NK, p_target=0) -> int:
    return int(lib().streamkl_fwd_splitk_splits(B, H, NQ, NK, int(p_target)))


def streamkl_fwd_splitk_workspace_bytes(B, H, NQ, splits) -> int:
    return int(lib().streamkl_fwd_splitk_workspace_bytes(B, H, NQ, int(splits)))


def streamkl_fwd_splitk(Q1, K1, Q2, K2, c1, c2, causal, splits=0, kl_rows=None, lse1=None, lse2=None, workspace=None, stream=None,
                        student_activation=None):
    """Split-K forward for small NQ.  splits <= 0: adaptive.  bf16 / fp16 inputs, possibly strided [B,H,N,d] views, K with fewer heads
    than Q (shared K heads) and the ReLU student go through streamkl_fwd_splitk_ex.  Returns (kl_rows, lse1, lse2)."""
    import torch

    for n, t in (("Q1", Q1), ("K1", K1), ("Q2", Q2), ("K2", K2)):
        _check_dev(n, t, Q1.dtype, strided=True)
    B, H, NQ, NK, d1, d2, HK = _shape_of(Q1, K1, Q2, K2)
    layout = _layout_of(Q1, K1, Q2, K2, HK, student_activation)
    if layout is None and Q1.dtype != torch.bfloat16:
        raise TypeError("streamkl_fwd_splitk: bfloat16 or float16 inputs")
    outs = []
    for n, t in (("kl_rows", kl_rows), ("lse1", lse1), ("lse2", lse2)):
        if t is None:
            t = torch.empty((B, H, NQ), dtype=torch.float32, device=Q1.device)
        _check_dev(n, t, torch.float32)
        outs.append(t)
    w = int(splits) if splits > 0 else streamkl_fwd_splitk_splits(B, H, NQ, NK, 0)
    need = streamkl_fwd_splitk_workspace_bytes(B, H, NQ, w)
    if need > 0 and (workspace is None or workspace.numel() * workspace.element_size() < need):
        workspace = torch.empty(need, dtype=torch.uint8, device=Q1.device)
        _keep_alive_on(workspace, stream)
    ws_bytes = 0 if workspace is None else workspace.numel() * workspace.element_size()
    args = (_ptr(Q1), _ptr(K1), _ptr(Q2), _ptr(K2), B, H, NQ, NK, d1, d2, float(c1), float(c2), int(bool(causal)), w,
            _ptr(outs[0]), _ptr(outs[1]), _ptr(outs[2]), _ptr(workspace), ctypes.c_size_t(ws_bytes), _stream_handle(stream))
    with torch.cuda.device(Q1.device):
        if layout is not None:
            rc = lib().streamkl_fwd_splitk_ex(ctypes.cast(ctypes.pointer(layout), ctypes.c_void_p), *args)
        else:
            rc = lib().streamkl_fwd_splitk(*args)
    if rc != 0:
        raise StreamKLError(rc, "streamkl_fwd_splitk")
    return tuple(outs)


def streamkl_fwd_splitk_noalloc_capacity() -> int:
    """Bytes of split-K scratch built into the loaded library (STREAMKL_NOALLOC_SCRATCH_BYTES, 4 MiB)."""
    return int(lib().streamkl_fwd_splitk_noalloc_capacity())


def streamkl_fwd_splitk_noalloc(Q1, K1, Q2, K2, c1, c2, causal, splits=0, kl_rows=None, lse1=None, lse2=None, stream=None):
    """Split-K forward whose partial statistics live in a fixed 4 MiB array inside the library instead of a workspace tensor,
    for code that must not allocate device memory at the time of the call (a plugin running inside someone else's memory arena,
    a latency-bound decode loop, a process whose HBM share is already spent).  Pass `kl_rows`, `lse1`, `lse2` and this binding
    allocates nothing either; leave them out and it creates the three output tensors for you, as the other bindings do.
    `splits` beyond what fits (B*H*W*5*NQ*4 bytes <= streamkl_fwd_splitk_noalloc_capacity()) raises StreamKLError with code
    STREAMKL_ERR_SCRATCH_LIMIT; splits <= 0 picks a W that fits.  All calls on a GPU share that one array: do not let two of
    them run at the same time (keep them on one stream).  Returns (kl_rows, lse1, lse2)."""
    import torch

    for n, t in (("Q1", Q1), ("K1", K1), ("Q2", Q2), ("K2", K2)):
        _check_dev(n, t, torch.bfloat16)
    B, H, NQ, NK, d1, d2, HK = _shape_of(Q1, K1, Q2, K2)
    if HK != H:
        raise ValueError("streamkl_fwd_splitk_noalloc: shared K heads are not supported")
    outs = []
    for n, t in (("kl_rows", kl_rows), ("lse1", lse1), ("lse2", lse2)):
        if t is None:
            t = torch.empty((B, H, NQ), dtype=torch.float32, device=Q1.device)
        _check_dev(n, t, torch.float32)
        outs.append(t)
    with torch.cuda.device(Q1.device):
        rc = lib().streamkl_fwd_splitk_noalloc(_ptr(Q1), _ptr(K1), _ptr(Q2), _ptr(K2), B, H, NQ, NK, d1, d2, float(c1), float(c2),
                                               int(bool(causal)), int(splits), _ptr(outs[0]), _ptr(outs[1]), _ptr(outs[2]),
                                               _stream_handle(stream))
    if rc != 0:
        raise StreamKLError(rc, "streamkl_fwd_splitk_noalloc")
    return tuple(outs)


def streamkl_bwd(Q1, K1, Q2, K2, c1, c2, causal, kl_rows, lse1, lse2, dkl_rows, teacher=False,
                 dQ1=None, dK1=None, dQ2=None, dK2=None, workspace=None, stream=None, student_activation=None):
    """Backward by recomputation (Alg.2/3 + K-owner transposes).  Returns (dQ1, dK1, dQ2, dK2); dQ1,dK1 None unless teacher."""
    import torch

    for n, t in (("Q1", Q1), ("K1", K1), ("Q2", Q2), ("K2", K2)):
        _check_dev(n, t, Q1.dtype, strided=True)
    for n, t in (("kl_rows", kl_rows), ("lse1", lse1), ("lse2", lse2), ("dkl_rows", dkl_rows)):
        _check_dev(n, t, torch.float32)
    B, H, NQ, NK, d1, d2, HK = _shape_of(Q1, K1, Q2, K2)
    layout = _layout_of(Q1, K1, Q2, K2, HK, student_activation)
    # gradients are stored through their input's strides: an expanded (stride 0) or self-overlapping view would have several
    # CTAs overwrite one another where the true gradient is a sum -- refuse it here, as the library does
    for n, t in (("Q2", Q2), ("K2", K2)) + ((("Q1", Q1), ("K1", K1)) if teacher else ()):
        if not _rows_are_disjoint(t):
            raise ValueError(f"{n}: a tensor that receives a gradient must not be a broadcast or self-overlapping view "
                             "(share K across query heads by giving K fewer heads instead)")
    # every gradient has the shape AND the strides of its input (dQ_t like Q_t, dK_t like K_t)
    like = lambda t: torch.empty_strided(t.shape, t.stride(), dtype=t.dtype, device=t.device)
    if dQ2 is None:
        dQ2 = like(Q2)
    if dK2 is None:
        dK2 = like(K2)
    if teacher:
        if dQ1 is None:
            dQ1 = like(Q1)
        if dK1 is None:
            dK1 = like(K1)
    else:
        dQ1 = dK1 = None
    for n, t, src in (("dQ1", dQ1, Q1), ("dK1", dK1, K1), ("dQ2", dQ2, Q2), ("dK2", dK2, K2)):
        if t is not None:
            _check_dev(n, t, Q1.dtype, strided=True)
            if tuple(t.shape) != tuple(src.shape) or tuple(t.stride()) != tuple(src.stride()):
                raise ValueError(f"{n}: must have the shape and strides of its input")
    need = streamkl_bwd_workspace_bytes(B, H, NQ, NK, d1, d2, teacher)
    if need > 0 and (workspace is None or workspace.numel() * workspace.element_size() < need):
        workspace = torch.empty(need, dtype=torch.uint8, device=Q1.device)
        _keep_alive_on(workspace, stream)
    ws_bytes = 0 if workspace is None else workspace.numel() * workspace.element_size()
    args = (_ptr(Q1), _ptr(K1), _ptr(Q2), _ptr(K2), B, H, NQ, NK, d1, d2, float(c1), float(c2), int(bool(causal)),
            _ptr(kl_rows), _ptr(lse1), _ptr(lse2), _ptr(dkl_rows), _ptr(dQ1), _ptr(dK1), _ptr(dQ2), _ptr(dK2),
            _ptr(workspace), ctypes.c_size_t(ws_bytes), _stream_handle(stream))
    with torch.cuda.device(Q1.device):
        if layout is not None:
            rc = lib().streamkl_bwd_ex(ctypes.cast(ctypes.pointer(layout), ctypes.c_void_p), *args)
        elif Q1.dtype == torch.bfloat16:
            rc = lib().streamkl_bwd(*args)
        else:
            rc = lib().streamkl_bwd_f32(*args)
    if rc != 0:
        raise StreamKLError(rc, "streamkl_bwd")
    return dQ1, dK1, dQ2, dK2


# ------------------------------------------------------------------------------------------ host entry points
def _host_dtype(a: np.ndarray) -> int:
    if a.dtype == np.uint16:
        return STREAMKL_BF16
    if a.dtype == np.float32:
        return STREAMKL_F32
    raise TypeError("host tensors must be uint16 (bf16 bit patterns) or float32")


def _np_ptr(a):
    return ctypes.c_void_p(a.ctypes.data) if a is not None else ctypes.c_void_p(0)


def _host_inputs(Q1, K1, Q2, K2):
    arrs = [np.ascontiguousarray(a) for a in (Q1, K1, Q2, K2)]
    dt = _host_dtype(arrs[0])
    for a in arrs:
        if _host_dtype(a) != dt:
            raise TypeError("Q1,K1,Q2,K2 must share a dtype")
    B, H, NQ, d1 = arrs[0].shape
    NK, d2 = arrs[1].shape[2], arrs[2].shape[3]
    if arrs[1].shape != (B, H, NK, d1) or arrs[2].shape != (B, H, NQ, d2) or arrs[3].shape != (B, H, NK, d2):
        raise ValueError("inconsistent Q1,K1,Q2,K2 shapes")
    return arrs, dt, (B, H, NQ, NK, d1, d2)


def streamkl_fwd_host(Q1, K1, Q2, K2, c1, c2, causal):
    """End-to-end forward with HOST numpy buffers (copies inside the call).  Returns (kl_rows, lse1, lse2) numpy float32."""
    arrs, dt, (B, H, NQ, NK, d1, d2) = _host_inputs(Q1, K1, Q2, K2)
    kl, l1, l2 = (np.empty((B, H, NQ), np.float32) for _ in range(3))
    rc = lib().streamkl_fwd_host(dt, *[_np_ptr(a) for a in arrs], B, H, NQ, NK, d1, d2, float(c1), float(c2),
                                 int(bool(causal)), _np_ptr(kl), _np_ptr(l1), _np_ptr(l2), ctypes.c_void_p(0))
    if rc != 0:
        raise StreamKLError(rc, "streamkl_fwd_host")
    return kl, l1, l2


def streamkl_fwd_bwd_host(Q1, K1, Q2, K2, c1, c2, causal, dkl_rows, teacher=False, out=None):
    """End-to-end forward + backward with HOST numpy buffers.  Returns dict(kl, lse1, lse2, dQ2, dK2[, dQ1, dK1]).

    `out` may carry preallocated (e.g. pinned) result arrays under the same keys."""
    arrs, dt, (B, H, NQ, NK, d1, d2) = _host_inputs(Q1, K1, Q2, K2)
    g = np.ascontiguousarray(dkl_rows, dtype=np.float32)
    if g.shape != (B, H, NQ):
        raise ValueError("dkl_rows must be [B,H,NQ]")
    st = arrs[0].dtype
    out = {} if out is None else out
    spec = {"kl": ((B, H, NQ), np.float32), "lse1": ((B, H, NQ), np.float32), "lse2": ((B, H, NQ), np.float32),
            "dQ2": ((B, H, NQ, d2), st), "dK2": ((B, H, NK, d2), st)}
    if teacher:
        spec["dQ1"] = ((B, H, NQ, d1), st)
        spec["dK1"] = ((B, H, NK, d1), st)
    for k, (shp, dty) in spec.items():
        if k not in out:
            out[k] = np.empty(shp, dty)
        elif out[k].shape != shp or out[k].dtype != dty or not out[k].flags.c_contiguous:
            raise ValueError(f"out[{k!r}] has the wrong shape/dtype/layout")
    rc = lib().streamkl_fwd_bwd_host(dt, *[_np_ptr(a) for a in arrs], B, H, NQ, NK, d1, d2, float(c1), float(c2),
                                     int(bool(causal)), _np_ptr(g), _np_ptr(out["kl"]), _np_ptr(out["lse1"]),
                                     _np_ptr(out["lse2"]), _np_ptr(out.get("dQ1")), _np_ptr(out.get("dK1")),
                                     _np_ptr(out["dQ2"]), _np_ptr(out["dK2"]), ctypes.c_void_p(0))
    if rc != 0:
        raise StreamKLError(rc, "streamkl_fwd_bwd_host")
    return out
