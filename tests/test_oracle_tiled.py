"""Pins of the oracle's tiled DWT design (oracle/feds_oracle_tiled.c; PAPER.md 6.9.3-6.9.4) against things other
than itself: the storage totals the report prints, the whole-image 5/3 oracle (pinned in test_oracle_transforms.py) on one tile,
the value ranges by adversarial search, hashlib for both keystreams, a Python re-derivation of the bit fields, exact round trips."""
import hashlib

import numpy as np
import pytest

import oracle
import synth

WIDTH = [10] * 12 + [11] * 4 + [10] * 48          # T3: HH2 (indices 12..15) takes 11 bits


def py_fields(data, lo, hi):
    """two's complement fields of coefficients [lo, hi) from a little-endian bit stream (Python integers)"""
    n = int.from_bytes(data, "little")
    out = []
    for i in range(lo, hi):
        b = WIDTH[i]
        f = n & ((1 << b) - 1)
        n >>= b
        out.append(f - (1 << b) if f >> (b - 1) else f)
    return out


def test_storage_totals_are_the_reports():
    """40 bits for level 1, 124 for level 2 (4 x 11 + 8 x 10), 480 public, 644 in all; here byte-aligned per level: 5 + 16 + 60
    bytes per tile = 126.6 % of the input ("about 26% more"), the private part 32.8 % ("at most 32%")."""
    assert sum(WIDTH[0:4]) == 40 and sum(WIDTH[4:16]) == 124 and sum(WIDTH[16:64]) == 480 and sum(WIDTH) == 644
    assert oracle.tiled_private_bytes(512, 512, 1) / 512 ** 2 == 21 / 64 and oracle.tiled_public_bytes(512, 512, 1) / 512 ** 2 == 60 / 64


def test_tile_transform_is_the_two_level_dwt_of_the_tile():
    """T1/T2 against the whole-image oracle run on a single 8x8 image with two levels (same lifting, same extension, same level shift)"""
    rng = np.random.default_rng(3)
    for _ in range(20):
        tile = rng.integers(0, 256, size=(8, 8), dtype=np.uint8)
        plane = oracle.dwt_coefficients(tile[:, :, None], 2)[0]         # 8x8 plane: LL2 top-left, HL right, LH below
        want = np.concatenate([plane[0:2, 0:2].ravel(), plane[0:2, 2:4].ravel(), plane[2:4, 0:2].ravel(), plane[2:4, 2:4].ravel(),
                               plane[0:4, 4:8].ravel(), plane[4:8, 0:4].ravel(), plane[4:8, 4:8].ravel()])
        got = oracle.tiled_forward(tile)
        assert (got == want).all()
        assert (oracle.tiled_inverse(got) == tile).all()


def test_value_ranges_fit_the_fields():
    """first level within 10 bits; second level: one corner needs 11. For every coefficient, the input that drives its
    linear part to the extreme (each pixel at 0 or 255 by the sign of its weight), both signs, plus random search: everything packs."""
    base = oracle.tiled_forward(np.full((8, 8), 128, dtype=np.uint8)).astype(np.float64)
    weights = np.zeros((64, 64))
    for i in range(64):
        t = np.full(64, 128, dtype=np.uint8)
        t[i] = 192
        weights[i] = (oracle.tiled_forward(t.reshape(8, 8)) - base) / 64.0
    lo, hi = np.zeros(64), np.zeros(64)
    for cidx in range(64):
        for sign in (1, -1):
            tile = np.where(sign * weights[:, cidx] > 0, 255, 0).astype(np.uint8).reshape(8, 8)
            coef = oracle.tiled_forward(tile)
            assert oracle.tiled_pack(coef) is not None
            lo, hi = np.minimum(lo, coef), np.maximum(hi, coef)
    rng = np.random.default_rng(1)
    for _ in range(300):
        tile = rng.choice([0, 255], size=(8, 8)).astype(np.uint8)
        coef = oracle.tiled_forward(tile)
        assert oracle.tiled_pack(coef) is not None
        lo, hi = np.minimum(lo, coef), np.maximum(hi, coef)
    assert hi[12:16].max() > 511 or lo[12:16].min() < -512          # HH2 really needs its eleventh bit
    for i in range(64):
        b = WIDTH[i]
        assert -(1 << (b - 1)) <= lo[i] and hi[i] <= (1 << (b - 1)) - 1


@pytest.mark.parametrize("w,h,c", [(8, 8, 1), (64, 32, 3), (72, 24, 4), (136, 8, 1)])
def test_fragment_layout_keystreams_and_round_trip(w, h, c):
    for img in (synth.image(w, h, c, seed=w + h, rectangles=1 if w >= 64 else 0), synth.special("random", w, h, c, seed=5),
                synth.special("checker", w, h, c, seed=6)):
        key, nonce = synth.key_nonce(w)
        priv, pub, dg = oracle.fragment_tiled(img, key, nonce)
        T = (w // 8) * (h // 8) * c
        assert priv.size == 21 * T and pub.size == 60 * T
        sec_a = oracle.aes128_ctr_xor(key, nonce, priv[16 * T:].tobytes())     # T5: level 1 of all tiles is one CTR message, behind level 2
        ntr, ntc = h // 8, w // 8
        for t in sorted({0, T // 2, T - 1}):
            ch, rem = divmod(t, ntr * ntc)
            tr, tc = divmod(rem, ntc)
            coef = oracle.tiled_forward(img[8 * tr:8 * tr + 8, 8 * tc:8 * tc + 8, ch])
            l1 = sec_a[5 * t:5 * t + 5]
            assert py_fields(l1, 0, 4) == list(coef[0:4])
            k2 = hashlib.sha256(l1 + key + nonce).digest()                       # T4
            l2 = bytes(a ^ b_ for a, b_ in zip(priv[16 * t:16 * t + 16].tobytes(), k2[:16]))
            assert py_fields(l2, 4, 16) == list(coef[4:16]) and l2[15] >> 4 == 0
            k3 = hashlib.sha512(l2 + key + nonce).digest()
            l3 = bytes(a ^ b_ for a, b_ in zip(pub[60 * t:60 * t + 60].tobytes(), k3[:60]))
            assert py_fields(l3, 16, 64) == list(coef[16:64])
        assert dg[:32] == oracle.merkle_stream(priv) and dg[32:] == oracle.merkle_stream(pub)   # T6 (merkle_stream is pinned by hashlib)
        rec, fl = oracle.defragment_tiled(priv, pub, w, h, c, key, nonce, expected=dg)
        assert fl == 0 and (rec == img).all()                                                   # no error at all
        p2 = priv.copy(); p2[16 * T + 3] ^= 1
        q2 = pub.copy(); q2[-1] ^= 1
        assert oracle.defragment_tiled(p2, pub, w, h, c, key, nonce, expected=dg)[1] == 1
        assert oracle.defragment_tiled(priv, q2, w, h, c, key, nonce, expected=dg)[1] == 2
