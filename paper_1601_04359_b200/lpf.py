"""Thin ctypes binding over liblpf.so (C ABI: include/lpf.h).  Same names as the C entry points.

Argument marshalling only: every step of the path (bit-pack, trie walk, count, mirror,
objective, swap delta) runs in the CUDA kernels behind the C ABI.  torch is used for device
memory and streams.  There is no CPU fallback: if liblpf.so is missing, loading raises.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_PKG = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_PKG, "liblpf.so")

LPF_OK, LPF_E_INVAL, LPF_E_NOMEM, LPF_E_CUDA, LPF_E_UNSUPPORTED, LPF_E_TOO_LARGE = 0, -1, -2, -3, -4, -5
LPF_STATIC_SCRATCH_BYTES = 256 * 1024
LPF_PRUNE, LPF_NO_TRIE, LPF_S2, LPF_NO_E2 = 1, 2, 4, 8

EXPORTS = (
    "lpf_strerror", "lpf_last_cuda_error", "lpf_build_paths", "lpf_free_paths", "lpf_paths_info",
    "lpf_paths_get", "lpf_paths_program", "lpf_eval", "lpf_eval_both", "lpf_objective",
    "lpf_swap_delta", "lpf_eval_host", "lpf_last_launch_info", "lpf_set_timing", "lpf_last_eval_kernel_ms",
    "lpf_set_tile", "lpf_alu_peak", "lpf_eval_masked", "lpf_anneal", "lpf_reserve", "lpf_eval_sum",
    "lpf_anneal_generate", "lpf_set_teams", "lpf_set_level", "lpf_set_shared_memory",
    "lpf_swap_delta_static", "lpf_set_tmem_stack",
)
LPF_PROPOSE_OPPOSITE, LPF_PROPOSE_INTERFACIAL = 1, 2
LPF_FOR_EVAL, LPF_FOR_EVAL_BOTH, LPF_FOR_MASKED, LPF_FOR_SWAP_DELTA, LPF_FOR_ANNEAL, LPF_FOR_HOST = 1, 2, 4, 8, 16, 32

_lib = None


class LpfError(RuntimeError):
    def __init__(self, code: int, what: str):
        self.code = code
        msg = _lib.lpf_strerror(code).decode() if _lib is not None else str(code)
        if code == LPF_E_CUDA and _lib is not None:
            msg += " (cudaError %d)" % _lib.lpf_last_cuda_error()
        super().__init__("%s: %s" % (what, msg))


def load() -> ctypes.CDLL:
    """dlopen liblpf.so.  Raises if it has not been built (python -m paper_1601_04359_b200.build)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError("liblpf.so is not built (%s): run `python -m paper_1601_04359_b200.build`; "
                           "there is no CPU fallback" % LIB_PATH)
    lib = ctypes.CDLL(LIB_PATH)
    I, I64, U, VP = ctypes.c_int, ctypes.c_int64, ctypes.c_uint, ctypes.c_void_p
    PI64, PI = ctypes.POINTER(ctypes.c_int64), ctypes.POINTER(ctypes.c_int)
    lib.lpf_strerror.argtypes = [I]
    lib.lpf_strerror.restype = ctypes.c_char_p
    lib.lpf_last_cuda_error.argtypes = []
    lib.lpf_last_cuda_error.restype = I
    lib.lpf_build_paths.argtypes = [I, I, ctypes.POINTER(VP)]
    lib.lpf_build_paths.restype = I
    lib.lpf_free_paths.argtypes = [VP]
    lib.lpf_free_paths.restype = None
    lib.lpf_paths_info.argtypes = [VP, PI64, PI64, PI64, PI]
    lib.lpf_paths_info.restype = I
    lib.lpf_paths_get.argtypes = [VP, I, I, VP, I, PI]
    lib.lpf_paths_get.restype = I
    lib.lpf_paths_program.argtypes = [VP, I, I, I, U, VP, I64, PI64, VP, I64, PI64, PI, PI]
    lib.lpf_paths_program.restype = I
    lib.lpf_eval.argtypes = [VP, VP, I, I, I, I, VP, U, VP]
    lib.lpf_eval.restype = I
    lib.lpf_eval_both.argtypes = [VP, VP, I, I, I, VP, U, VP]
    lib.lpf_eval_both.restype = I
    lib.lpf_eval_masked.argtypes = [VP, VP, I, I, I, I, VP, VP, U, VP]
    lib.lpf_eval_masked.restype = I
    lib.lpf_eval_sum.argtypes = [VP, VP, I, I, I, I, VP, U, VP]
    lib.lpf_eval_sum.restype = I
    lib.lpf_reserve.argtypes = [VP, I, I, I, U, U]
    lib.lpf_reserve.restype = I
    lib.lpf_anneal.argtypes = [VP, VP, I, I, I, VP, VP, VP, I64, ctypes.c_double, ctypes.c_double, I64, I64, VP, VP,
                               ctypes.POINTER(ctypes.c_double), VP]
    lib.lpf_anneal.restype = I
    lib.lpf_anneal_generate.argtypes = [VP, VP, I, I, I, VP, I, ctypes.c_uint64, VP, VP, I64, ctypes.c_double,
                                        ctypes.c_double, I64, I64, VP, VP, ctypes.POINTER(ctypes.c_double), VP]
    lib.lpf_anneal_generate.restype = I
    lib.lpf_objective.argtypes = [VP, VP, I, I64, VP, VP]
    lib.lpf_objective.restype = I
    lib.lpf_swap_delta.argtypes = [VP, VP, I, I, I, VP, I64, VP, VP]
    lib.lpf_swap_delta.restype = I
    lib.lpf_swap_delta_static.argtypes = [VP, VP, I, I, I, VP, I64, VP, VP]
    lib.lpf_swap_delta_static.restype = I
    lib.lpf_eval_host.argtypes = [VP, VP, I, I, I, I, VP, U]
    lib.lpf_eval_host.restype = I
    lib.lpf_last_launch_info.argtypes = [VP, PI64]
    lib.lpf_last_launch_info.restype = I
    lib.lpf_set_timing.argtypes = [VP, I]
    lib.lpf_set_timing.restype = I
    lib.lpf_last_eval_kernel_ms.argtypes = [VP, ctypes.POINTER(ctypes.c_float)]
    lib.lpf_last_eval_kernel_ms.restype = I
    lib.lpf_alu_peak.argtypes = [I, ctypes.POINTER(ctypes.c_double)]
    lib.lpf_alu_peak.restype = I
    lib.lpf_set_tile.argtypes = [VP, I, I, I]
    lib.lpf_set_tile.restype = I
    lib.lpf_set_teams.argtypes = [VP, I]
    lib.lpf_set_teams.restype = I
    lib.lpf_set_level.argtypes = [VP, I]
    lib.lpf_set_level.restype = I
    lib.lpf_set_tmem_stack.argtypes = [VP, I]
    lib.lpf_set_tmem_stack.restype = I
    lib.lpf_set_shared_memory.argtypes = [VP, I]
    lib.lpf_set_shared_memory.restype = I
    _lib = lib
    return lib


def _check(rc: int, what: str) -> None:
    if rc != LPF_OK:
        raise LpfError(rc, what)


class Paths:
    """Owner of one `lpf_paths*` (path table + prefix trie + device programs for one m)."""

    def __init__(self, handle: int, m: int, device: int):
        self._h = ctypes.c_void_p(handle)
        self.m = m
        self.device = device

    @property
    def handle(self) -> ctypes.c_void_p:
        if not self._h:
            raise RuntimeError("lpf_paths already freed")
        return self._h

    def close(self) -> None:
        if self._h and _lib is not None:
            _lib.lpf_free_paths(self._h)
        self._h = ctypes.c_void_p(None)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def lpf_build_paths(m: int, device: int = 0) -> Paths:
    """Paper step 1.  device < 0 builds a host-only table (no CUDA call is made)."""
    lib = load()
    h = ctypes.c_void_p(None)
    _check(lib.lpf_build_paths(int(m), int(device), ctypes.byref(h)), "lpf_build_paths")
    return Paths(h.value, int(m), int(device))


def lpf_free_paths(p: Paths) -> None:
    p.close()


def lpf_paths_info(p: Paths) -> dict:
    lib = load()
    a, b, c, d = ctypes.c_int64(), ctypes.c_int64(), ctypes.c_int64(), ctypes.c_int()
    _check(lib.lpf_paths_info(p.handle, ctypes.byref(a), ctypes.byref(b), ctypes.byref(c), ctypes.byref(d)),
           "lpf_paths_info")
    return dict(n_half_vectors=a.value, sum_path_len=b.value, n_trie_nodes=c.value, max_depth=d.value)


def lpf_paths_get(p: Paths, dx: int, dy: int) -> np.ndarray:
    """P_v as int16 [len, 2] (x, y), any v of the template."""
    lib = load()
    cap = max(abs(int(dx)), abs(int(dy))) + 1
    xy = np.zeros((cap, 2), dtype=np.int16)
    n = ctypes.c_int()
    _check(lib.lpf_paths_get(p.handle, int(dx), int(dy), xy.ctypes.data, cap, ctypes.byref(n)), "lpf_paths_get")
    return xy[: n.value]


def lpf_paths_program(p: Paths, H: int, W: int, piece_nodes: int = 0, flags: int = 0):
    """(entries uint64 [n], items int64 [k, 4], n_slots, layout: row strides of the 4 views, the words of one band of
    each view in shared memory, the level K, the number of pattern classes, then 41 ints per class: octant, patterns
    used, pattern of each slot) of the linearised walk program."""
    lib = load()
    ne, ni, ns = ctypes.c_int64(), ctypes.c_int64(), ctypes.c_int()
    strides = (ctypes.c_int * (10 + 41 * 128))()
    _check(lib.lpf_paths_program(p.handle, int(H), int(W), int(piece_nodes), int(flags), None, 0, ctypes.byref(ne),
                                 None, 0, ctypes.byref(ni), ctypes.byref(ns), strides), "lpf_paths_program")
    entries = np.zeros(ne.value, dtype=np.uint64)
    items = np.zeros((ni.value, 4), dtype=np.int64)
    _check(lib.lpf_paths_program(p.handle, int(H), int(W), int(piece_nodes), int(flags), entries.ctypes.data,
                                 ne.value, ctypes.byref(ne), items.ctypes.data, ni.value, ctypes.byref(ni),
                                 ctypes.byref(ns), strides), "lpf_paths_program")
    return entries, items, ns.value, [int(v) for v in strides]


# ---- device entry points (torch tensors in, torch tensors out) -------------------------------

def _torch():
    import torch
    return torch


def _stream_ptr(stream, *tensors) -> int:
    """The launch stream as an integer; tensors handed to the C call are recorded on it, so that a temporary made by
    .contiguous() is not recycled by torch's caching allocator before the enqueued kernels have read it."""
    torch = _torch()
    s = stream if stream is not None else torch.cuda.current_stream()
    for t in tensors:
        if t is not None and t.is_cuda:
            t.record_stream(s)
    return int(s.cuda_stream)


def _on_device(p: "Paths", *tensors) -> None:
    for t in tensors:
        if t is not None and (not t.is_cuda or t.device.index != p.device):
            raise ValueError("tensor on %s, but the lpf_paths table is bound to cuda:%d" % (t.device, p.device))


def _dev_images(images, ndim: int, p: "Paths" = None):
    torch = _torch()
    if not (isinstance(images, torch.Tensor) and images.is_cuda and images.dtype == torch.uint8):
        raise TypeError("images must be a CUDA uint8 tensor")
    if p is not None:
        _on_device(p, images)
    if images.dim() == ndim - 1:
        images = images.unsqueeze(0)
    if images.dim() != ndim:
        raise ValueError("images must be [B, H, W] (or [H, W])")
    return images.contiguous()


def lpf_eval(p: Paths, images, phase: int, flags: int = 0, out=None, stream=None):
    """counts int64 [B, 2m+1, 2m+1] on the device; index [b, dy+m, dx+m]."""
    torch = _torch()
    lib = load()
    images = _dev_images(images, 3, p)
    B, H, W = images.shape
    S = 2 * p.m + 1
    if out is None:
        out = torch.empty((B, S, S), dtype=torch.int64, device=images.device)
    assert out.is_cuda and out.dtype == torch.int64 and out.is_contiguous() and out.numel() == B * S * S
    _on_device(p, out)
    _check(lib.lpf_eval(p.handle, images.data_ptr(), B, H, W, int(phase), out.data_ptr(), int(flags),
                        _stream_ptr(stream, images)), "lpf_eval")
    return out


def lpf_eval_both(p: Paths, images, flags: int = 0, out=None, stream=None):
    """counts int64 [B, 2, 2m+1, 2m+1]; index [b, phase, dy+m, dx+m]."""
    torch = _torch()
    lib = load()
    images = _dev_images(images, 3, p)
    B, H, W = images.shape
    S = 2 * p.m + 1
    if out is None:
        out = torch.empty((B, 2, S, S), dtype=torch.int64, device=images.device)
    assert out.is_cuda and out.dtype == torch.int64 and out.is_contiguous() and out.numel() == B * 2 * S * S
    _on_device(p, out)
    _check(lib.lpf_eval_both(p.handle, images.data_ptr(), B, H, W, out.data_ptr(), int(flags),
                             _stream_ptr(stream, images)), "lpf_eval_both")
    return out


def lpf_eval_masked(p: Paths, images, phase: int, start_mask, flags: int = 0, out=None, stream=None):
    """L2~ counts over the selected start pixels (start_mask uint8 [H, W], non-zero = selected); phase 0 | 1 gives
    int64 [B, 2m+1, 2m+1], phase -1 both phases [B, 2, 2m+1, 2m+1]."""
    torch = _torch()
    lib = load()
    images = _dev_images(images, 3, p)
    B, H, W = images.shape
    assert start_mask.is_cuda and start_mask.dtype == torch.uint8 and tuple(start_mask.shape) == (H, W)
    _on_device(p, start_mask)
    start_mask = start_mask.contiguous()
    S = 2 * p.m + 1
    shape = (B, 2, S, S) if phase < 0 else (B, S, S)
    if out is None:
        out = torch.empty(shape, dtype=torch.int64, device=images.device)
    assert out.is_cuda and out.dtype == torch.int64 and out.is_contiguous() and out.numel() == int(np.prod(shape))
    _on_device(p, out)
    _check(lib.lpf_eval_masked(p.handle, images.data_ptr(), B, H, W, int(phase), start_mask.data_ptr(),
                               out.data_ptr(), int(flags), _stream_ptr(stream, images, start_mask)), "lpf_eval_masked")
    return out


def lpf_eval_sum(p: Paths, images, phase: int, flags: int = 0, out=None, stream=None):
    """Ensemble sum over the B images: int64 [2m+1, 2m+1] (phase 0 | 1) or [2, 2m+1, 2m+1] (phase -1);
    the ensemble average of L2 is out / (B * W * H)."""
    torch = _torch()
    lib = load()
    images = _dev_images(images, 3, p)
    B, H, W = images.shape
    S = 2 * p.m + 1
    shape = (2, S, S) if phase < 0 else (S, S)
    if out is None:
        out = torch.empty(shape, dtype=torch.int64, device=images.device)
    assert out.is_cuda and out.dtype == torch.int64 and out.is_contiguous() and out.numel() == int(np.prod(shape))
    _check(lib.lpf_eval_sum(p.handle, images.data_ptr(), B, H, W, int(phase), out.data_ptr(), int(flags),
                            _stream_ptr(stream, images)), "lpf_eval_sum")
    return out


def lpf_reserve(p: Paths, B: int, H: int, W: int, flags: int = 0, what: int = LPF_FOR_EVAL) -> None:
    """Builds and uploads everything the calls named by `what` (LPF_FOR_*) need for B x H x W images: after it they
    only enqueue work on their stream (no allocation, copy or host synchronisation)."""
    _check(load().lpf_reserve(p.handle, int(B), int(H), int(W), int(flags), int(what)), "lpf_reserve")


def lpf_anneal(p: Paths, image, phase: int, target, pairs, log_u, T_max: float, T_min: float, c_max: int, s_max: int,
               accept_log=None, stream=None):
    """Alg. 3 on the device.  image: CUDA uint8 [H, W], modified in place.  Returns (counts int64 [n_ph, S, S], stats)."""
    torch = _torch()
    lib = load()
    assert image.is_cuda and image.dtype == torch.uint8 and image.dim() == 2 and image.is_contiguous()
    _on_device(p, image, target, pairs, log_u, accept_log)
    H, W = image.shape
    S = 2 * p.m + 1
    n_ph = 2 if phase < 0 else 1
    target = target.contiguous()
    pairs = pairs.contiguous()
    log_u = log_u.contiguous()
    assert target.is_cuda and target.dtype == torch.int64 and target.numel() == n_ph * S * S
    assert pairs.is_cuda and pairs.dtype == torch.int32 and pairs.dim() == 2 and pairs.shape[1] == 4
    assert log_u.is_cuda and log_u.dtype == torch.float64 and log_u.numel() == pairs.shape[0]
    if accept_log is not None:
        assert accept_log.is_cuda and accept_log.dtype == torch.uint8 and accept_log.numel() == pairs.shape[0]
    counts = torch.empty((n_ph, S, S), dtype=torch.int64, device=image.device)
    stats = (ctypes.c_double * 5)()
    _check(lib.lpf_anneal(p.handle, image.data_ptr(), H, W, int(phase), target.data_ptr(), pairs.data_ptr(),
                          log_u.data_ptr(), pairs.shape[0], float(T_max), float(T_min), int(c_max), int(s_max),
                          counts.data_ptr(), accept_log.data_ptr() if accept_log is not None else None, stats,
                          _stream_ptr(stream, target, pairs, log_u)), "lpf_anneal")
    keys = ("steps", "accepted", "levels", "T", "E")
    return counts, dict(zip(keys, [float(v) for v in stats]))


def lpf_anneal_generate(p: Paths, image, phase: int, target, policy: int, seed: int, log_u, T_max: float, T_min: float,
                        c_max: int, s_max: int, accept_log=None, stream=None):
    """Alg. 3 with the modification operator drawing its own pixels (LPF_PROPOSE_OPPOSITE / LPF_PROPOSE_INTERFACIAL).
    Returns (counts int64 [n_ph, S, S], stats, pairs int32 [N, 4]: the proposal decided at every step)."""
    torch = _torch()
    lib = load()
    assert image.is_cuda and image.dtype == torch.uint8 and image.dim() == 2 and image.is_contiguous()
    _on_device(p, image, target, log_u, accept_log)
    H, W = image.shape
    S = 2 * p.m + 1
    n_ph = 2 if phase < 0 else 1
    target = target.contiguous()
    log_u = log_u.contiguous()
    N = log_u.numel()
    assert target.is_cuda and target.dtype == torch.int64 and target.numel() == n_ph * S * S
    assert log_u.is_cuda and log_u.dtype == torch.float64
    if accept_log is not None:
        assert accept_log.is_cuda and accept_log.dtype == torch.uint8 and accept_log.numel() == N
    counts = torch.empty((n_ph, S, S), dtype=torch.int64, device=image.device)
    pairs = torch.zeros((max(N, 1), 4), dtype=torch.int32, device=image.device)
    stats = (ctypes.c_double * 5)()
    _check(lib.lpf_anneal_generate(p.handle, image.data_ptr(), H, W, int(phase), target.data_ptr(), int(policy),
                                   int(seed) & (2 ** 64 - 1), pairs.data_ptr(), log_u.data_ptr(), N, float(T_max),
                                   float(T_min), int(c_max), int(s_max), counts.data_ptr(),
                                   accept_log.data_ptr() if accept_log is not None else None, stats,
                                   _stream_ptr(stream, target, log_u)), "lpf_anneal_generate")
    keys = ("steps", "accepted", "levels", "T", "E")
    return counts, dict(zip(keys, [float(v) for v in stats])), pairs[:N]


def lpf_objective(counts, target, out=None, stream=None):
    """sse[b] = sum_k (counts[b, k] - target[k])^2, exact; returned as an int64 tensor holding the
    uint64 bit pattern (values < 2^63 read directly)."""
    torch = _torch()
    lib = load()
    assert counts.is_cuda and counts.dtype == torch.int64 and target.is_cuda and target.dtype == torch.int64
    counts = counts.contiguous()
    target = target.contiguous()
    K = target.numel()
    assert K > 0 and counts.numel() % K == 0
    B = counts.numel() // K
    if out is None:
        out = torch.empty((B,), dtype=torch.int64, device=counts.device)
    with torch.cuda.device(counts.device):
        _check(lib.lpf_objective(counts.data_ptr(), target.data_ptr(), B, K, out.data_ptr(),
                                 _stream_ptr(stream, counts, target)), "lpf_objective")
    return out


def lpf_swap_delta(p: Paths, image, phase: int, pairs, out=None, stream=None):
    """delta int32 [n, 2m+1, 2m+1] for n independent two-pixel swaps (pairs int32 [n, 4])."""
    torch = _torch()
    lib = load()
    image = _dev_images(image, 3, p)
    if image.shape[0] != 1:
        raise ValueError("lpf_swap_delta takes one base image")
    _, H, W = image.shape
    assert pairs.is_cuda and pairs.dtype == torch.int32 and pairs.dim() == 2 and pairs.shape[1] == 4
    _on_device(p, pairs)
    pairs = pairs.contiguous()
    n = pairs.shape[0]
    S = 2 * p.m + 1
    if out is None:
        out = torch.empty((n, S, S), dtype=torch.int32, device=image.device)
    assert out.is_cuda and out.dtype == torch.int32 and out.is_contiguous() and out.numel() == n * S * S
    _on_device(p, out)
    _check(lib.lpf_swap_delta(p.handle, image.data_ptr(), H, W, int(phase), pairs.data_ptr(), n, out.data_ptr(),
                              _stream_ptr(stream, image, pairs)), "lpf_swap_delta")
    return out


def lpf_swap_delta_static(p: Paths, image, phase: int, pairs, out, stream=None):
    """lpf_swap_delta with its scratch in the library's static device array (at most LPF_STATIC_SCRATCH_BYTES): the call
    allocates nothing, so `out` (int32 [n, 2m+1, 2m+1]) is the caller's.  The trie records must have been uploaded by
    lpf_reserve(..., LPF_FOR_SWAP_DELTA); calls that overlap on one GPU race on the array."""
    torch = _torch()
    lib = load()
    image = _dev_images(image, 3, p)
    if image.shape[0] != 1:
        raise ValueError("lpf_swap_delta_static takes one base image")
    _, H, W = image.shape
    assert pairs.is_cuda and pairs.dtype == torch.int32 and pairs.dim() == 2 and pairs.shape[1] == 4
    assert pairs.is_contiguous()
    _on_device(p, pairs)
    n = pairs.shape[0]
    S = 2 * p.m + 1
    assert out.is_cuda and out.dtype == torch.int32 and out.is_contiguous() and out.numel() == n * S * S
    _on_device(p, out)
    _check(lib.lpf_swap_delta_static(p.handle, image.data_ptr(), H, W, int(phase), pairs.data_ptr(), n,
                                     out.data_ptr(), _stream_ptr(stream, image, pairs)), "lpf_swap_delta_static")
    return out


def lpf_eval_host(p: Paths, images_host, phase: int, counts_host=None, flags: int = 0):
    """End-to-end call with HOST buffers (numpy arrays or CPU tensors, ideally pinned): H2D copy,
    lpf_eval (phase 0/1) or lpf_eval_both (phase < 0), D2H copy, synchronise."""
    lib = load()
    a = images_host.numpy() if hasattr(images_host, "numpy") else np.asarray(images_host)
    if a.dtype != np.uint8 or not a.flags.c_contiguous:
        raise TypeError("images_host must be C-contiguous uint8")
    if a.ndim == 2:
        a = a[None]
    B, H, W = a.shape
    S = 2 * p.m + 1
    shape = (B, 2, S, S) if phase < 0 else (B, S, S)
    if counts_host is None:
        counts_host = np.empty(shape, dtype=np.int64)
    c = counts_host.numpy() if hasattr(counts_host, "numpy") else counts_host
    assert c.dtype == np.int64 and c.flags.c_contiguous and c.size == int(np.prod(shape))
    _check(lib.lpf_eval_host(p.handle, a.ctypes.data, B, H, W, int(phase), c.ctypes.data, int(flags)),
           "lpf_eval_host")
    return counts_host


def lpf_last_launch_info(p: Paths) -> dict:
    lib = load()
    out = (ctypes.c_int64 * 18)()
    _check(lib.lpf_last_launch_info(p.handle, out), "lpf_last_launch_info")
    keys = ("kernels", "work_items", "program_entries", "grid", "block", "smem_bytes", "tile", "G", "level",
            "fused_pairs", "singles", "terminals", "piece_nodes", "teams", "ctas_per_sm", "shallow_vectors",
            "reloads", "classes")
    info = dict(zip(keys, [int(v) for v in out]))
    info["tmem_stack"] = (info["tile"] // 10) % 10          # the mask stack of this launch was in tensor memory
    return info


def lpf_set_timing(p: Paths, enable: bool) -> None:
    _check(load().lpf_set_timing(p.handle, int(bool(enable))), "lpf_set_timing")


def lpf_alu_peak(device: int = 0) -> dict:
    """Measured thread-level integer instruction rates (ops/s) of the device: LOP3, SHF, SHF+SHF+LOP3, POPC."""
    out = (ctypes.c_double * 4)()
    _check(load().lpf_alu_peak(int(device), out), "lpf_alu_peak")
    return dict(zip(("lop3", "shf", "pair", "popc"), [float(v) for v in out]))


def lpf_set_tile(p: Paths, tx: int = 0, ty: int = 0, cta_warps: int = 0) -> None:
    """Tuning hook: thread tile (TX words x TY rows) and warps per CTA of the eval kernel; 0 = automatic."""
    _check(load().lpf_set_tile(p.handle, int(tx), int(ty), int(cta_warps)), "lpf_set_tile")


def lpf_set_level(p: Paths, max_level: int = -1) -> None:
    _check(load().lpf_set_level(p.handle, int(max_level)), "lpf_set_level")


def lpf_set_shared_memory(p: Paths, nbytes: int = 0) -> None:
    """Tuning hook: dynamic shared memory one CTA of the eval kernel may use (>= 16384; 0 = all of the device's)."""
    _check(load().lpf_set_shared_memory(p.handle, int(nbytes)), "lpf_set_shared_memory")


def lpf_set_tmem_stack(p: Paths, enable: bool = True) -> None:
    """Tuning hook: the walker's mask stack in tensor memory (default, big shapes) or always in local memory."""
    _check(load().lpf_set_tmem_stack(p.handle, int(bool(enable))), "lpf_set_tmem_stack")


def lpf_set_teams(p: Paths, n_teams: int = 0) -> None:
    _check(load().lpf_set_teams(p.handle, int(n_teams)), "lpf_set_teams")


def lpf_last_eval_kernel_ms(p: Paths) -> float:
    ms = ctypes.c_float()
    _check(load().lpf_last_eval_kernel_ms(p.handle, ctypes.byref(ms)), "lpf_last_eval_kernel_ms")
    return float(ms.value)


def normalise(counts, H: int, W: int):
    """L2 = count / (W*H): one IEEE double division of exact integers (reading S5)."""
    return np.asarray(counts, dtype=np.float64) / float(int(W) * int(H))
