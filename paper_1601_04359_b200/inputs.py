"""Seeded synthetic inputs shaped like the paper's workloads.

This module holds NONE of the method's arithmetic (no paths, no counting): it only draws
uint8 images and pixel pairs.  It is the one module that both the oracle-side tests and the
CUDA-side tests/bench import, so that both sides see the same bytes.  numpy only.

The paper's own images (chess, 4x4-square suspension, metal foam [22], epithelial cells,
trabecular bone [32]) are not available; these generators stand in
for them with the sizes and statistics BASELINE.json names (recipe in DESIGN.md "Inputs").
"""
from __future__ import annotations

import numpy as np

BASE_SEED = 160104359


def seed_for(config: int, index: int = 0) -> int:
    """config c uses BASE_SEED + 1000*c; image i of a batch adds i."""
    return BASE_SEED + 1000 * int(config) + int(index)


def bernoulli(H: int, W: int, p: float, seed: int) -> np.ndarray:
    """i.i.d. Bernoulli(p) pixels (config 1: 64x64, p = 0.5)."""
    rng = np.random.default_rng(seed)
    return (rng.random((H, W)) < p).astype(np.uint8)


def disks(H: int, W: int, radius: float, fraction: float, seed: int) -> np.ndarray:
    """Periodic Boolean model: disks with uniform real centres are added one at a time
    (pixel in disk iff periodic centre distance^2 <= r^2) until the phase-1 fraction first
    reaches >= fraction.  Configs 2, 4, 5."""
    rng = np.random.default_rng(seed)
    img = np.zeros((H, W), dtype=np.uint8)
    target = int(np.ceil(fraction * H * W))
    r2 = float(radius) ** 2
    ys = np.arange(H, dtype=np.float64)[:, None]
    xs = np.arange(W, dtype=np.float64)[None, :]
    filled = 0
    while filled < target:
        cx = rng.random() * W
        cy = rng.random() * H
        dx = np.abs(xs - cx)
        dx = np.minimum(dx, W - dx)
        dy = np.abs(ys - cy)
        dy = np.minimum(dy, H - dy)
        img[(dx * dx + dy * dy) <= r2] = 1
        filled = int(img.sum())
    return img


def gaussian_field(H: int, W: int, corr_len: float, fraction: float, seed: int) -> np.ndarray:
    """Thresholded periodic Gaussian random field (config 3): white normal noise, periodic
    (FFT) convolution with exp(-r^2 / (2 corr_len^2)), phase 1 = the round(fraction*H*W)
    largest values (rank threshold, so the fraction is exact)."""
    rng = np.random.default_rng(seed)
    noise = rng.standard_normal((H, W))
    yy = np.minimum(np.arange(H), H - np.arange(H)).astype(np.float64)[:, None]
    xx = np.minimum(np.arange(W), W - np.arange(W)).astype(np.float64)[None, :]
    kern = np.exp(-(xx * xx + yy * yy) / (2.0 * corr_len * corr_len))
    field = np.fft.irfft2(np.fft.rfft2(noise) * np.fft.rfft2(kern), s=(H, W))
    k = int(round(fraction * H * W))
    order = np.argsort(field, axis=None, kind="stable")
    img = np.zeros(H * W, dtype=np.uint8)
    if k > 0:
        img[order[-k:]] = 1
    return img.reshape(H, W)


def disk_batch(B: int, H: int, W: int, radius: float, fraction: float, config: int) -> np.ndarray:
    """[B, H, W] stack of independent disk images, image i seeded seed_for(config, i)."""
    return np.stack([disks(H, W, radius, fraction, seed_for(config, i)) for i in range(B)])


def chess(H: int, W: int, square: int) -> np.ndarray:
    """Chess-type morphology with square x square px fields (PAPER.md:312 (i))."""
    y = (np.arange(H) // square)[:, None]
    x = (np.arange(W) // square)[None, :]
    return ((x + y) % 2).astype(np.uint8)


def squares(H: int, W: int, square: int, fraction: float, seed: int) -> np.ndarray:
    """Particulate suspension of equal axis-aligned squares at uniform integer positions,
    overlaps allowed, added until the fraction is reached (PAPER.md:312 (ii), 451)."""
    rng = np.random.default_rng(seed)
    img = np.zeros((H, W), dtype=np.uint8)
    target = int(np.ceil(fraction * H * W))
    while int(img.sum()) < target:
        x0 = int(rng.integers(0, W))
        y0 = int(rng.integers(0, H))
        yy = (y0 + np.arange(square)) % H
        xx = (x0 + np.arange(square)) % W
        img[np.ix_(yy, xx)] = 1
    return img


def stripes(H: int, W: int, period: int, thickness: int, horizontal: bool) -> np.ndarray:
    """Stripes of phase 1: rows (horizontal) or columns with index % period < thickness."""
    if horizontal:
        line = (np.arange(H) % period < thickness).astype(np.uint8)[:, None]
        return np.repeat(line, W, axis=1)
    line = (np.arange(W) % period < thickness).astype(np.uint8)[None, :]
    return np.repeat(line, H, axis=0)


def swap_pairs(image: np.ndarray, n: int, seed: int) -> np.ndarray:
    """int32 [n, 4] = (x_p, y_p, x_q, y_q): p uniform over byte-0 pixels, q uniform over
    byte-1 pixels, independently and with replacement (reading S10)."""
    rng = np.random.default_rng(seed)
    zy, zx = np.nonzero(image == 0)
    oy, ox = np.nonzero(image == 1)
    if zy.size == 0 or oy.size == 0:
        raise ValueError("image needs both phases for a swap")
    ip = rng.integers(0, zy.size, size=n)
    iq = rng.integers(0, oy.size, size=n)
    return np.stack([zx[ip], zy[ip], ox[iq], oy[iq]], axis=1).astype(np.int32)


def anneal_proposals(H: int, W: int, n: int, seed: int):
    """Inputs of the annealing loop (Alg. 3): n proposals of two uniformly drawn pixels, int32 [n, 4] =
    (x_p, y_p, x_q, y_q), and ln(u) of n uniform random numbers u in [0, 1) for the Metropolis rule (float64; -inf for u = 0).
    Both sides receive these arrays; neither draws random numbers itself."""
    rng = np.random.default_rng(seed)
    pairs = np.stack([rng.integers(0, W, n), rng.integers(0, H, n), rng.integers(0, W, n), rng.integers(0, H, n)],
                     axis=1).astype(np.int32)
    with np.errstate(divide="ignore"):
        log_u = np.log(rng.random(n))
    return pairs, log_u


# --- the five BASELINE.json configs -------------------------------------------------

CONFIGS = {
    1: dict(H=64, W=64, m=16, phases=(1,), kind="bernoulli(0.5)"),
    2: dict(H=256, W=256, m=128, phases=(0, 1), kind="disks r=8 phi=0.30"),
    3: dict(H=512, W=512, m=256, phases=(0, 1), kind="gaussian field l=12 phi=0.40"),
    4: dict(H=128, W=128, m=64, phases=(1,), B=1024, kind="disks r=6 phi=0.35, batch + 1 target"),
    5: dict(H=256, W=256, m=64, phases=(1,), n_swaps=100000, kind="disks r=8 phi=0.30, swaps"),
}


def config_image(c: int) -> np.ndarray:
    """The single image of configs 1, 2, 3, 5."""
    if c == 1:
        return bernoulli(64, 64, 0.5, seed_for(1))
    if c == 2:
        return disks(256, 256, 8.0, 0.30, seed_for(2))
    if c == 3:
        return gaussian_field(512, 512, 12.0, 0.40, seed_for(3))
    if c == 5:
        return disks(256, 256, 8.0, 0.30, seed_for(5))
    raise ValueError("config %r has no single image" % (c,))


def config4_batch(B: int = 1024):
    """(images [B,128,128], target image [128,128]); the target is image index B."""
    imgs = disk_batch(B, 128, 128, 6.0, 0.35, 4)
    target = disks(128, 128, 6.0, 0.35, seed_for(4, B))
    return imgs, target


def config5_pairs(image: np.ndarray, n: int = 100000) -> np.ndarray:
    return swap_pairs(image, n, seed_for(5, 1))
