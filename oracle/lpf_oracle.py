"""ctypes loader for the plain-C oracle in oracle/lpf_oracle.c.

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs.  The product (paper_1601_04359_b200) never imports
this module and this module never imports the product.

Argument marshalling only -- every number comes out of lpf_oracle.c.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lpf_oracle.c")
_LIB = os.path.join(_HERE, "liblpf_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp -shared; rebuilt when the source is newer than the library."""
    stale = force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC)
    if stale:
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-std=c99", "-fopenmp", "-shared", "-fPIC",
                               "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        c_u8p = ctypes.POINTER(ctypes.c_uint8)
        c_i16p = ctypes.POINTER(ctypes.c_int16)
        c_i32p = ctypes.POINTER(ctypes.c_int32)
        c_i64p = ctypes.POINTER(ctypes.c_int64)
        I = ctypes.c_int
        lib.lpf_oracle_in_half.argtypes = [I, I]
        lib.lpf_oracle_in_half.restype = I
        lib.lpf_oracle_path.argtypes = [I, I, c_i16p]
        lib.lpf_oracle_path.restype = I
        lib.lpf_oracle_counts_list.argtypes = [c_u8p, I, I, I, c_i32p, ctypes.c_int64, c_i64p, I]
        lib.lpf_oracle_counts_list.restype = I
        lib.lpf_oracle_counts.argtypes = [c_u8p, I, I, I, I, c_i64p, I, I]
        lib.lpf_oracle_counts.restype = I
        lib.lpf_oracle_counts_sum.argtypes = [c_u8p, I, I, I, I, I, c_i64p, I]
        lib.lpf_oracle_counts_sum.restype = None
        lib.lpf_oracle_sse.argtypes = [c_i64p, c_i64p, ctypes.c_int64]
        lib.lpf_oracle_sse.restype = ctypes.c_uint64
        lib.lpf_oracle_swap_delta_full.argtypes = [c_u8p, I, I, I, I, I, I, I, I, c_i32p, I]
        lib.lpf_oracle_swap_delta_full.restype = I
        lib.lpf_oracle_swap_delta_local.argtypes = [c_u8p, I, I, I, I, I, I, I, I, c_i32p]
        lib.lpf_oracle_swap_delta_local.restype = None
        lib.lpf_oracle_counts_masked.argtypes = [c_u8p, c_u8p, I, I, I, c_i32p, ctypes.c_int64, c_i64p]
        lib.lpf_oracle_counts_masked.restype = None
        lib.lpf_oracle_s2_counts.argtypes = [c_u8p, I, I, I, I, c_i64p]
        lib.lpf_oracle_s2_counts.restype = None
        lib.lpf_oracle_anneal.argtypes = [c_u8p, I, I, I, I, c_i64p, c_i32p, ctypes.POINTER(ctypes.c_double),
                                          ctypes.c_int64, ctypes.c_double, ctypes.c_double, ctypes.c_int64,
                                          ctypes.c_int64, I, c_i64p, ctypes.POINTER(ctypes.c_double), c_u8p]
        lib.lpf_oracle_anneal.restype = None
        lib.lpf_oracle_splitmix64.argtypes = [ctypes.c_uint64, ctypes.c_uint64]
        lib.lpf_oracle_splitmix64.restype = ctypes.c_uint64
        lib.lpf_oracle_propose.argtypes = [c_u8p, I, I, I, ctypes.c_uint64, ctypes.c_int64, c_i32p]
        lib.lpf_oracle_propose.restype = None
        lib.lpf_oracle_anneal_generate.argtypes = [c_u8p, I, I, I, I, c_i64p, I, ctypes.c_uint64, c_i32p,
                                                   ctypes.POINTER(ctypes.c_double), ctypes.c_int64, ctypes.c_double,
                                                   ctypes.c_double, ctypes.c_int64, ctypes.c_int64, I, c_i64p,
                                                   ctypes.POINTER(ctypes.c_double), c_u8p]
        lib.lpf_oracle_anneal_generate.restype = None
        lib.lpf_oracle_max_threads.argtypes = []
        lib.lpf_oracle_max_threads.restype = I
        _lib = lib
    return _lib


def _p(a, ct):
    return a.ctypes.data_as(ctypes.POINTER(ct))


def _img(image):
    a = np.ascontiguousarray(image, dtype=np.uint8)
    if a.ndim != 2:
        raise ValueError("image must be [H, W]")
    return a


def max_threads() -> int:
    return int(_load().lpf_oracle_max_threads())


def in_half(dx: int, dy: int) -> bool:
    return bool(_load().lpf_oracle_in_half(int(dx), int(dy)))


def path(dx: int, dy: int) -> np.ndarray:
    """P_v as int16 [len, 2] (x, y)."""
    n = max(abs(int(dx)), abs(int(dy))) + 1
    xy = np.zeros((n, 2), dtype=np.int16)
    got = _load().lpf_oracle_path(int(dx), int(dy), _p(xy, ctypes.c_int16))
    assert got == n
    return xy


def counts_list(image, phase: int, vecs, threads: int = 0):
    """int64 counts for vecs = [n, 2] (dx, dy); returns (counts, threads_used)."""
    a = _img(image)
    v = np.ascontiguousarray(vecs, dtype=np.int32).reshape(-1, 2)
    out = np.zeros(v.shape[0], dtype=np.int64)
    used = _load().lpf_oracle_counts_list(_p(a, ctypes.c_uint8), a.shape[0], a.shape[1], int(phase),
                                          _p(v, ctypes.c_int32), v.shape[0],
                                          _p(out, ctypes.c_int64), int(threads))
    return out, int(used)


def counts(image, phase: int, m: int, full_template: bool = False, threads: int = 0) -> np.ndarray:
    """int64 [2m+1, 2m+1], index [dy+m, dx+m]."""
    a = _img(image)
    S = 2 * int(m) + 1
    out = np.zeros((S, S), dtype=np.int64)
    _load().lpf_oracle_counts(_p(a, ctypes.c_uint8), a.shape[0], a.shape[1], int(phase), int(m),
                              _p(out, ctypes.c_int64), int(bool(full_template)), int(threads))
    return out


def counts_sum(images, phase: int, m: int, threads: int = 0) -> np.ndarray:
    """Ensemble sum over a stack [B, H, W]: int64 [2m+1, 2m+1]."""
    a = np.ascontiguousarray(images, dtype=np.uint8)
    if a.ndim != 3:
        raise ValueError("images must be [B, H, W]")
    S = 2 * int(m) + 1
    out = np.zeros((S, S), dtype=np.int64)
    _load().lpf_oracle_counts_sum(_p(a, ctypes.c_uint8), a.shape[0], a.shape[1], a.shape[2], int(phase), int(m),
                                  _p(out, ctypes.c_int64), int(threads))
    return out


def counts_masked(image, mask, phase: int, vecs) -> np.ndarray:
    """L2~ counts: hits of each vector over the start pixels with mask != 0."""
    a = _img(image)
    k = np.ascontiguousarray(mask, dtype=np.uint8)
    assert k.shape == a.shape
    v = np.ascontiguousarray(vecs, dtype=np.int32).reshape(-1, 2)
    out = np.zeros(v.shape[0], dtype=np.int64)
    _load().lpf_oracle_counts_masked(_p(a, ctypes.c_uint8), _p(k, ctypes.c_uint8), a.shape[0], a.shape[1], int(phase),
                                     _p(v, ctypes.c_int32), v.shape[0], _p(out, ctypes.c_int64))
    return out


def s2_counts(image, phase: int, m: int) -> np.ndarray:
    """Un-normalised two-point probability of Eq. 6: int64 [2m+1, 2m+1], index [dy+m, dx+m]."""
    a = _img(image)
    S = 2 * int(m) + 1
    out = np.zeros((S, S), dtype=np.int64)
    _load().lpf_oracle_s2_counts(_p(a, ctypes.c_uint8), a.shape[0], a.shape[1], int(phase), int(m),
                                 _p(out, ctypes.c_int64))
    return out


def anneal(image, phase: int, m: int, target, pairs, log_u, T_max: float, T_min: float, c_max: int, s_max: int,
           use_local: bool = False):
    """Alg. 3.  Returns (final image, counts [n_ph, S, S], stats dict, accept log uint8 [N])."""
    a = _img(image).copy()
    S = 2 * int(m) + 1
    n_ph = 2 if phase < 0 else 1
    t = np.ascontiguousarray(target, dtype=np.int64).reshape(n_ph, S, S)
    pr = np.ascontiguousarray(pairs, dtype=np.int32).reshape(-1, 4)
    lu = np.ascontiguousarray(log_u, dtype=np.float64)
    assert lu.shape[0] == pr.shape[0]
    counts_out = np.zeros((n_ph, S, S), dtype=np.int64)
    stats = np.zeros(5, dtype=np.float64)
    log = np.zeros(pr.shape[0], dtype=np.uint8)
    _load().lpf_oracle_anneal(_p(a, ctypes.c_uint8), a.shape[0], a.shape[1], int(phase), int(m), _p(t, ctypes.c_int64),
                              _p(pr, ctypes.c_int32), _p(lu, ctypes.c_double), pr.shape[0], float(T_max), float(T_min),
                              int(c_max), int(s_max), int(bool(use_local)), _p(counts_out, ctypes.c_int64),
                              _p(stats, ctypes.c_double), _p(log, ctypes.c_uint8))
    keys = ("steps", "accepted", "levels", "T", "E")
    return a, counts_out, dict(zip(keys, [float(v) for v in stats])), log


def splitmix64(seed: int, n: int) -> int:
    """n-th output (n = 1, 2, ...) of SplitMix64 seeded with `seed`."""
    return int(_load().lpf_oracle_splitmix64(int(seed) & (2 ** 64 - 1), int(n)))


def propose(image, policy: int, seed: int, k: int) -> np.ndarray:
    """The pair (x_p, y_p, x_q, y_q) the modification operator draws for proposal k from `image` (reading A7)."""
    a = _img(image)
    pair = np.zeros(4, dtype=np.int32)
    _load().lpf_oracle_propose(_p(a, ctypes.c_uint8), a.shape[0], a.shape[1], int(policy), int(seed) & (2 ** 64 - 1),
                               int(k), _p(pair, ctypes.c_int32))
    return pair


def anneal_generate(image, phase: int, m: int, target, policy: int, seed: int, log_u, T_max: float, T_min: float,
                    c_max: int, s_max: int, use_local: bool = False):
    """Alg. 3 with generated proposals.  Returns (final image, counts, stats, accept log, pairs decided int32 [N, 4])."""
    a = _img(image).copy()
    S = 2 * int(m) + 1
    n_ph = 2 if phase < 0 else 1
    t = np.ascontiguousarray(target, dtype=np.int64).reshape(n_ph, S, S)
    lu = np.ascontiguousarray(log_u, dtype=np.float64)
    N = lu.shape[0]
    counts_out = np.zeros((n_ph, S, S), dtype=np.int64)
    stats = np.zeros(5, dtype=np.float64)
    log = np.zeros(N, dtype=np.uint8)
    pairs = np.zeros((N, 4), dtype=np.int32)
    _load().lpf_oracle_anneal_generate(_p(a, ctypes.c_uint8), a.shape[0], a.shape[1], int(phase), int(m),
                                       _p(t, ctypes.c_int64), int(policy), int(seed) & (2 ** 64 - 1),
                                       _p(pairs, ctypes.c_int32), _p(lu, ctypes.c_double), N, float(T_max), float(T_min),
                                       int(c_max), int(s_max), int(bool(use_local)), _p(counts_out, ctypes.c_int64),
                                       _p(stats, ctypes.c_double), _p(log, ctypes.c_uint8))
    keys = ("steps", "accepted", "levels", "T", "E")
    return a, counts_out, dict(zip(keys, [float(v) for v in stats])), log, pairs


def half_sse(c, t, m: int) -> int:
    """Eq. 19 over D (reading A4): sum over the canonical half of (t - c)^2, exact.  The one piece of numpy arithmetic
    in this binding: it is what the tests compare the C file's half_sse_ (inside lpf_oracle_anneal) against."""
    c = np.asarray(c, dtype=np.int64)
    t = np.asarray(t, dtype=np.int64)
    S = 2 * int(m) + 1
    k = np.arange(S * S).reshape(S, S)
    half = k >= (m * S + m)
    d = (t - c)[..., half]
    return int((d * d).sum())


def sse(c, t) -> int:
    c = np.ascontiguousarray(c, dtype=np.int64).ravel()
    t = np.ascontiguousarray(t, dtype=np.int64).ravel()
    assert c.size == t.size
    return int(_load().lpf_oracle_sse(_p(c, ctypes.c_int64), _p(t, ctypes.c_int64), c.size))


def swap_delta_full(image, phase: int, m: int, pair, threads: int = 0) -> np.ndarray:
    a = _img(image)
    S = 2 * int(m) + 1
    out = np.zeros((S, S), dtype=np.int32)
    xp, yp, xq, yq = (int(v) for v in pair)
    _load().lpf_oracle_swap_delta_full(_p(a, ctypes.c_uint8), a.shape[0], a.shape[1], int(phase), int(m),
                                       xp, yp, xq, yq, _p(out, ctypes.c_int32), int(threads))
    return out


def swap_delta_local(image, phase: int, m: int, pair) -> np.ndarray:
    a = _img(image)
    S = 2 * int(m) + 1
    out = np.zeros((S, S), dtype=np.int32)
    xp, yp, xq, yq = (int(v) for v in pair)
    _load().lpf_oracle_swap_delta_local(_p(a, ctypes.c_uint8), a.shape[0], a.shape[1], int(phase), int(m),
                                        xp, yp, xq, yq, _p(out, ctypes.c_int32))
    return out


def normalise(c, H: int, W: int) -> np.ndarray:
    """L2 = count / (W*H): one IEEE double division of exact integers (S5)."""
    return np.asarray(c, dtype=np.float64) / float(int(W) * int(H))
