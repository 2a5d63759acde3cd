"""Seeded synthetic inputs shared by the oracle tests, the GPU parity tests, smoke() and bench.py.

Holds NONE of the method's arithmetic (no DCT, DWT, AES, SHA of fragments): only the image recipe of
DESIGN.md section 5 / SURVEY.md 8(d) and the seed -> key/nonce rule. The images stand in for the paper's
bitmap test images, which are not available and are not recreated.

  p(x,y) = 128 + sum_{i=1..8} A_i sin(2 pi (fx_i x/W + fy_i y/H) + phi_i) + N(0, sigma^2)
  A_i ~ U(8,32), fx_i, fy_i ~ U(0,16) cycles/image, phi_i ~ U(0, 2 pi); rounded, clamped to 0..255.

`image(...)` is numpy (CPU); `image_batch_torch(...)` builds the same recipe with torch ops on any device
(used for the 1.6 GB cfg3 batch, generated directly in HBM). The two do not promise identical bytes; a
test that needs the same bytes on both sides generates once and copies.
"""
import hashlib

import numpy as np


def key_nonce(seed: int):
    """key = bytes 0..15, nonce = bytes 16..31 of SHA-256("feds" || decimal seed)."""
    d = hashlib.sha256(b"feds" + str(int(seed)).encode()).digest()
    return d[:16], d[16:]


def batch_nonces(base_nonce: bytes, n: int, priv_bytes: int = 0, stride: int = None) -> np.ndarray:
    """nonce_i = (base + i*stride) mod 2^128, big-endian; uint8[n][16]. stride (in 16-byte counter blocks) defaults to the
    smallest power of two >= max(2^20, ceil(priv_bytes / 16)): the images' counter ranges must not overlap under one key."""
    if stride is None:
        stride = 1 << 20
        while stride * 16 < priv_bytes:
            stride <<= 1
    if stride * 16 < priv_bytes:
        raise ValueError("nonce stride shorter than the private fragment: keystream would be reused")
    base = int.from_bytes(base_nonce, "big")
    out = np.empty((n, 16), dtype=np.uint8)
    for i in range(n):
        out[i] = np.frombuffer(((base + i * stride) % (1 << 128)).to_bytes(16, "big"), dtype=np.uint8)
    return out


def _plane(rng, w, h):
    a = rng.uniform(8.0, 32.0, 8)
    fx = rng.uniform(0.0, 16.0, 8)
    fy = rng.uniform(0.0, 16.0, 8)
    ph = rng.uniform(0.0, 2 * np.pi, 8)
    x = np.arange(w, dtype=np.float64)[None, :] / w
    y = np.arange(h, dtype=np.float64)[:, None] / h
    p = np.full((h, w), 128.0)
    for i in range(8):
        # sin(ax + by + phi) via the angle-sum identity: two outer products instead of h*w sin calls
        ax = 2 * np.pi * fx[i] * x
        by = 2 * np.pi * fy[i] * y + ph[i]
        p += a[i] * (np.sin(ax) * np.cos(by) + np.cos(ax) * np.sin(by))
    return p


def image(w: int, h: int, c: int, seed: int, sigma: float = 8.0, rectangles: int = 0) -> np.ndarray:
    """uint8[H][W][C]; channel ch uses seed 3*seed+ch. `rectangles` flat-colour boxes drawn before the noise."""
    out = np.empty((h, w, c), dtype=np.uint8)
    rrng = np.random.default_rng(1_000_003 * seed + 17)
    rects = []
    for _ in range(rectangles):
        rw = int(rrng.integers(1, max(2, w // 4 + 1)))
        rh = int(rrng.integers(1, max(2, h // 4 + 1)))
        x0 = int(rrng.integers(0, w - rw + 1))
        y0 = int(rrng.integers(0, h - rh + 1))
        rects.append((x0, y0, rw, rh, rrng.integers(0, 256, c)))
    for ch in range(c):
        rng = np.random.default_rng(3 * seed + ch)
        p = _plane(rng, w, h)
        for (x0, y0, rw, rh, col) in rects:
            p[y0:y0 + rh, x0:x0 + rw] = float(col[ch])
        if sigma > 0:
            p += rng.normal(0.0, sigma, (h, w))
        out[:, :, ch] = np.clip(np.rint(p), 0, 255).astype(np.uint8)
    return out


def special(kind: str, w: int, h: int, c: int, seed: int = 0) -> np.ndarray:
    """Correctness-only inputs: zeros, ones (all 255), checker (1-pixel checkerboard), random, impulse."""
    if kind == "zeros":
        return np.zeros((h, w, c), dtype=np.uint8)
    if kind == "ones":
        return np.full((h, w, c), 255, dtype=np.uint8)
    if kind == "checker":
        yy, xx = np.mgrid[0:h, 0:w]
        return np.repeat((((yy + xx) & 1) * 255).astype(np.uint8)[:, :, None], c, axis=2)
    if kind == "random":
        return np.random.default_rng(seed).integers(0, 256, (h, w, c), dtype=np.uint8)
    if kind == "impulse":
        a = np.zeros((h, w, c), dtype=np.uint8)
        a[h // 2, w // 2, :] = 255
        return a
    raise ValueError(kind)


def image_batch_torch(n: int, w: int, h: int, c: int, seed: int, device, sigma: float = 8.0, rectangles: int = 0):
    """The same recipe with torch ops on `device`: uint8[n][H][W][C]. For large batches built directly in HBM."""
    import torch

    gen = torch.Generator(device=device)
    out = torch.empty((n, h, w, c), dtype=torch.uint8, device=device)
    x = torch.arange(w, dtype=torch.float32, device=device)[None, :] / w
    y = torch.arange(h, dtype=torch.float32, device=device)[:, None] / h
    for i in range(n):
        rrng = np.random.default_rng(1_000_003 * (seed + i) + 17)
        rects = []
        for _ in range(rectangles):
            rw = int(rrng.integers(1, max(2, w // 4 + 1)))
            rh = int(rrng.integers(1, max(2, h // 4 + 1)))
            x0 = int(rrng.integers(0, w - rw + 1))
            y0 = int(rrng.integers(0, h - rh + 1))
            rects.append((x0, y0, rw, rh, rrng.integers(0, 256, c)))
        for ch in range(c):
            rng = np.random.default_rng(3 * (seed + i) + ch)
            a = rng.uniform(8.0, 32.0, 8)
            fx = rng.uniform(0.0, 16.0, 8)
            fy = rng.uniform(0.0, 16.0, 8)
            ph = rng.uniform(0.0, 2 * np.pi, 8)
            p = torch.full((h, w), 128.0, dtype=torch.float32, device=device)
            for j in range(8):
                p += float(a[j]) * torch.sin(2 * np.pi * (float(fx[j]) * x + float(fy[j]) * y) + float(ph[j]))
            for (x0, y0, rw, rh, col) in rects:
                p[y0:y0 + rh, x0:x0 + rw] = float(col[ch])
            if sigma > 0:
                gen.manual_seed(int(3 * (seed + i) + ch))
                p += sigma * torch.randn((h, w), generator=gen, dtype=torch.float32, device=device)
            out[i, :, :, ch] = p.round().clamp(0, 255).to(torch.uint8)
    return out
