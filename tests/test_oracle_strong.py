"""Pins of the oracle's STRONG level of protection (oracle/feds_oracle_strong.c; PAPER.md 6.3.2) against
things other than itself: FIPS 180-4 SHA-512 through hashlib, the DCT basis through scipy, closed forms, the report's own description
(the public part is the IDCT of the rest of the coefficients), exact round trips. No GPU."""
import hashlib
import struct

import numpy as np
import pytest
import scipy.fft

import oracle
import synth


@pytest.mark.parametrize("n", [0, 1, 3, 24, 55, 56, 64, 111, 112, 119, 120, 127, 128, 129, 239, 240, 256, 1000])
def test_sha512_matches_hashlib(n):
    """FIPS 180-4 6.4 vectors taken from hashlib at test time: every padding boundary of the 128-byte block (111/112: the length
    field just fits / no longer fits), and the sizes the path uses (24 bytes = DC + 5 AC; up to 256 bytes at k = 63)."""
    msg = bytes((7 * i + 3) & 255 for i in range(n))
    assert oracle.sha512(msg) == hashlib.sha512(msg).digest()
    assert oracle.sha512(b"abc") == hashlib.sha512(b"abc").digest()


def test_sha512_million_a():
    msg = b"a" * 1000000
    assert oracle.sha512(msg) == hashlib.sha512(msg).digest()


def test_basis_is_the_orthonormal_dct_basis_in_fixed_point():
    """B[z][p] = rne(4096 b_z(p)): b_z from scipy's orthonormal inverse DCT of a unit coefficient at zigzag position z (an outside
    definition of the basis); DC row = 4096 / 8 exactly; rows orthogonal up to the rounding of the table."""
    B = oracle.strong_basis()
    for z in range(64):
        r, q = oracle.zigzag(z)
        X = np.zeros((8, 8))
        X[r, q] = 1.0
        b = scipy.fft.idctn(X, norm="ortho").reshape(64)
        assert np.abs(B[z] - 4096.0 * b).max() <= 0.5 + 1e-9
    assert (B[0] == 512).all()
    G = B.astype(np.float64) @ B.astype(np.float64).T / 4096.0 ** 2
    assert np.abs(G - np.eye(64)).max() < 2e-3


@pytest.mark.parametrize("k", [0, 2, 5, 9, 31, 63])
def test_remainder_is_the_idct_of_the_rest(k):
    """the public part is "the reverse DCT result of the rest DCT coefficients padded with zero". The oracle's integer
    remainder x - L equals that real-valued image to within one grey level (S1: L is a fixed-point evaluation of the IDCT of
    Part 1, and IDCT(rest) = x - IDCT(Part 1) by linearity); at k = 63 nothing is left and the remainder is 0 or +-1."""
    img = synth.image(64, 48, 3, seed=k + 1, rectangles=3)
    rem = oracle.strong_remainder(img, k).astype(np.float64)
    zz = [oracle.zigzag(z) for z in range(64)]
    worst = 0.0
    for ch in range(3):
        for br in range(6):
            for bc in range(8):
                x = img[8 * br:8 * br + 8, 8 * bc:8 * bc + 8, ch].astype(np.float64)
                X = scipy.fft.dctn(x, norm="ortho")
                for z in range(k + 1):
                    X[zz[z]] = 0.0                      # Part 1 padded with zeros
                rest = scipy.fft.idctn(X, norm="ortho")
                worst = max(worst, np.abs(rem[8 * br:8 * br + 8, 8 * bc:8 * bc + 8, ch] - rest).max())
    assert worst <= 1.0, worst


def test_constant_block_closed_form():
    """A constant block c has DC = 8 c and no AC, q_0 = 64 c, L = (64 c * 512 + 2^14) >> 15 = c exactly, so the remainder is
    zero and the public block IS the SHA-512 digest of Part 1 -- computed here with hashlib and struct, not with the oracle.
    Part 1 is given as the closed form (the double defining sum leaves 1e-14 of noise in the AC terms of a constant block, and a
    hash sees every bit; the all-zero image, whose sums are exactly zero, goes through the whole path as well)."""
    key, nonce = synth.key_nonce(5)
    for c0 in (0, 1, 100, 255):
        img = np.full((8, 16, 1), c0, dtype=np.uint8)
        for k in (0, 5):
            coef = np.array([[8.0 * c0] + [0.0] * k] * 2, dtype=np.float32)
            priv, pub, dg = oracle.fragment_strong_from_priv32(img, coef, k, key, nonce)
            part1 = struct.pack("<%df" % (k + 1), *([8.0 * c0] + [0.0] * k))
            want = hashlib.sha512(part1).digest()
            assert pub[:64].tobytes() == want and pub[64:].tobytes() == want
            # Part 1 itself: AES-CTR of those bytes (two blocks, one CTR message)
            assert oracle.aes128_ctr_xor(key, nonce, priv.tobytes()) == part1 + part1
            if c0 == 0:
                p2, q2, d2 = oracle.fragment_dct_strong(img, k, key, nonce)
                assert (p2 == priv).all() and (q2 == pub).all() and d2 == dg
    # a block whose remainder is not zero: x = L + r with a hand-made Part 1 (DC only, 8 * 100 -> L = 100 everywhere)
    img = np.full((8, 8, 1), 100, dtype=np.uint8)
    img[3, 4, 0] = 97
    img[0, 0, 0] = 230
    priv, pub, _ = oracle.fragment_strong_from_priv32(img, np.array([[800.0]], dtype=np.float32), 0, key, nonce)
    ks = np.frombuffer(hashlib.sha512(struct.pack("<f", 800.0)).digest(), dtype=np.uint8)
    r = (pub ^ ks).reshape(8, 8)
    assert r[3, 4] == 253 and r[0, 0] == 130 and (np.delete(r.reshape(64), [0, 28]) == 0).all()   # -3 and +130 modulo 256


@pytest.mark.parametrize("w,h,c,k", [(8, 8, 1, 0), (16, 8, 1, 5), (64, 32, 3, 5), (72, 24, 4, 2), (40, 16, 3, 63), (136, 8, 1, 31), (32, 32, 3, 26),
                                     (32, 32, 3, 27)])
def test_round_trip_and_sizes(w, h, c, k):
    """fragment -> defragment reproduces every pixel exactly (P:586-595 lossless; S1 makes it exact by construction), the sizes are
    4 (k+1) bytes of Part 1 and 64 bytes of public pixels per block, verification flags follow single-byte corruptions."""
    img = synth.image(w, h, c, seed=w + h + k, rectangles=1 if w >= 32 else 0)
    key, nonce = synth.key_nonce(w + k)
    priv, pub, dg = oracle.fragment_dct_strong(img, k, key, nonce)
    assert priv.size == (w // 8) * (h // 8) * c * (k + 1) * 4 and pub.size == w * h * c
    rec, fl = oracle.defragment_dct_strong(priv, pub, w, h, c, k, key, nonce, expected=dg)
    assert fl == 0 and (rec == img).all()
    # digests: the Merkle layout of DESIGN.md 2.1 over the stored bytes (public leaf = 8 blocks x 64 bytes), by the pinned routine
    assert dg[:32] == oracle.merkle_blocks(priv, c * (h // 8), w // 8, 4 * (k + 1))
    assert dg[32:] == oracle.merkle_blocks(pub, c * (h // 8), w // 8, 64)
    p2 = priv.copy(); p2[0] ^= 1
    q2 = pub.copy(); q2[-1] ^= 0x80
    assert oracle.defragment_dct_strong(p2, pub, w, h, c, k, key, nonce, expected=dg)[1] == 1
    rec2, fl2 = oracle.defragment_dct_strong(priv, q2, w, h, c, k, key, nonce, expected=dg)
    assert fl2 == 2 and (rec2 != img).sum() == 1          # a flipped public bit damages exactly one pixel


def test_keystream_depends_on_part_one_only_and_hides_the_remainder():
    """S2/S3: two blocks with the same Part 1 get the same keystream (the report accepts this); the public bytes of a block
    XOR its keystream give back x - L modulo 256."""
    img = synth.image(32, 16, 1, seed=3, rectangles=1)
    key, nonce = synth.key_nonce(9)
    k = 5
    priv, pub, _ = oracle.fragment_dct_strong(img, k, key, nonce)
    part1 = oracle.aes128_ctr_xor(key, nonce, priv.tobytes())
    rem = oracle.strong_remainder(img, k)
    for b in range(8):
        ks = np.frombuffer(hashlib.sha512(part1[24 * b:24 * b + 24]).digest(), dtype=np.uint8)
        br, bc = divmod(b, 4)
        want = (rem[8 * br:8 * br + 8, 8 * bc:8 * bc + 8, 0].reshape(64) & 255).astype(np.uint8)
        assert ((pub[64 * b:64 * b + 64] ^ ks) == want).all()


def test_from_priv32_equals_whole_path():
    img = synth.image(48, 24, 3, seed=11)
    key, nonce = synth.key_nonce(2)
    k = 5
    priv, pub, dg = oracle.fragment_dct_strong(img, k, key, nonce)
    coef = oracle.dct_coefficients(img).astype(np.float32)[:, :k + 1]
    p2, q2, d2 = oracle.fragment_strong_from_priv32(img, coef, k, key, nonce)
    assert (p2 == priv).all() and (q2 == pub).all() and d2 == dg
