"""Pins of the oracle's packed integer storage (oracle/feds_oracle_packed.c; PAPER.md 6.4.3) against things
other than itself: the storage overheads the report prints, a bit-by-bit re-derivation of the layout in Python, scipy's DCT, hashlib,
exact round trips for both storages. No GPU."""
import hashlib

import numpy as np
import pytest
import scipy.fft

import oracle
import synth


def test_storage_overheads_are_the_reports():
    """11-bit storage = 11 x 6 / 64 / 8 = 12.9 % of the image, 8-bit storage = 5/64 + 11/8/64 = 9.96 % (k = 5, gray)."""
    w = h = 512
    assert oracle.packed_private_bytes(w, h, 1, 5, 11) / (w * h) == pytest.approx(11 * 6 / 64 / 8, abs=1e-12)
    assert oracle.packed_private_bytes(w, h, 1, 5, 8) / (w * h) == pytest.approx(5 / 64 + 11 / 8 / 64, abs=1e-12)
    # a ragged last group of a block row is padded to whole bytes: 9 blocks = 8 + 1 -> 66 + ceil(66 / 8) = 75 bytes per block row
    assert oracle.packed_private_bytes(72, 8, 1, 5, 11) == 66 + 9


def py_pack(q, k, ac_bits):
    """the layout of DESIGN.md 2.4 K2 re-derived with Python integers: one big little-endian number per group"""
    acc, pos = 0, 0
    for blk in q:
        acc |= int(blk[0]) << pos
        pos += 11
        for z in range(1, k + 1):
            v = int(blk[z])
            acc |= ((abs(v) | ((1 << (ac_bits - 1)) if v < 0 else 0)) << pos)
            pos += ac_bits
    return acc.to_bytes((pos + 7) // 8, "little")


@pytest.mark.parametrize("k,ac_bits,nblk", [(5, 11, 8), (5, 8, 8), (0, 11, 8), (63, 11, 8), (63, 8, 3), (2, 8, 1), (9, 11, 5)])
def test_bit_layout(k, ac_bits, nblk):
    rng = np.random.default_rng(k + ac_bits + nblk)
    M = (1 << (ac_bits - 1)) - 1
    q = rng.integers(-M, M + 1, size=(nblk, k + 1)).astype(np.int32)
    q[:, 0] = rng.integers(0, 2048, size=nblk)
    q[0, :] = [2047] + [-M, M][: 0] + [(-M if z % 2 else M) for z in range(1, k + 1)]     # extremes of every field
    data = oracle.pack_group(q, k, ac_bits)
    assert len(data) == (nblk * (11 + k * ac_bits) + 7) // 8
    assert data == py_pack(q, k, ac_bits)
    assert (oracle.unpack_group(data, nblk, k, ac_bits) == q).all()
    if nblk == 8:
        assert len(data) == 11 + k * ac_bits          # eight blocks: exactly b bytes


def test_quantisation_rule():
    """K1: round to nearest even, DC clamped to the 11-bit range that its bound 8 x 255 = 2040 fits, AC to +-(2^(bits-1) - 1)"""
    assert oracle.packed_quantise(2040.0, 1, 11) == 2040 and oracle.packed_quantise(2047.6, 1, 11) == 2047
    assert oracle.packed_quantise(-3.0, 1, 11) == 0
    assert oracle.packed_quantise(0.5, 0, 11) == 0 and oracle.packed_quantise(1.5, 0, 11) == 2 and oracle.packed_quantise(-2.5, 0, 11) == -2
    assert oracle.packed_quantise(1500.0, 0, 11) == 1023 and oracle.packed_quantise(-1500.0, 0, 11) == -1023
    assert oracle.packed_quantise(200.0, 0, 8) == 127 and oracle.packed_quantise(-127.4, 0, 8) == -127
    assert oracle.packed_quantise(float("nan"), 0, 8) == 0


@pytest.mark.parametrize("ac_bits", [11, 8])
@pytest.mark.parametrize("w,h,c,k", [(8, 8, 1, 0), (64, 32, 3, 5), (72, 24, 4, 2), (40, 16, 3, 63), (136, 8, 1, 31)])
def test_round_trip_is_exact_for_both_storages(w, h, c, k, ac_bits):
    """the 11-bit storage is lossless (PSNR infinite). With the remainder taken against the quantised Part 1 (K3) so is
    the 8-bit one -- also on images whose AC coefficients exceed its range (checkerboard: |AC| up to ~1000)."""
    for img in (synth.image(w, h, c, seed=w + k, rectangles=2 if w >= 64 else 0), synth.special("checker", w, h, c, seed=1),
                synth.special("random", w, h, c, seed=2)):
        key, nonce = synth.key_nonce(w + k + ac_bits)
        priv, pub, dg, q = oracle.fragment_dct_packed(img, k, ac_bits, key, nonce)
        assert priv.size == oracle.packed_private_bytes(w, h, c, k, ac_bits) and pub.size == w * h * c
        rec, fl = oracle.defragment_dct_packed(priv, pub, w, h, c, k, ac_bits, key, nonce, expected=dg)
        assert fl == 0 and (rec == img).all()
        p2 = priv.copy(); p2[priv.size // 2] ^= 4
        q2 = pub.copy(); q2[7] ^= 1
        assert oracle.defragment_dct_packed(p2, pub, w, h, c, k, ac_bits, key, nonce, expected=dg)[1] == 1
        assert oracle.defragment_dct_packed(priv, q2, w, h, c, k, ac_bits, key, nonce, expected=dg)[1] == 2


def test_integers_are_the_rounded_dct_and_remainder_is_idct_of_the_rest():
    """q = rne(scipy's orthonormal DCT) wherever that is not within 1e-6 of a tie; the public bytes are, modulo 256, within
    (1 + k/2 ...) grey levels of scipy's IDCT of the rest -- exactly: |(x - L) - IDCT(rest) - IDCT(c - q)| <= 1 with the
    quantisation error of Part 1 carried over to the remainder (that is what makes K3 lossless)."""
    img = synth.image(64, 48, 1, seed=9, rectangles=3)
    k = 5
    key, nonce = synth.key_nonce(1)
    priv, pub, dg, q = oracle.fragment_dct_packed(img, k, 11, key, nonce)
    zz = [oracle.zigzag(z) for z in range(64)]
    for br in range(6):
        for bc in range(8):
            b = br * 8 + bc
            x = img[8 * br:8 * br + 8, 8 * bc:8 * bc + 8, 0].astype(np.float64)
            X = scipy.fft.dctn(x, norm="ortho")
            for z in range(k + 1):
                cz = X[zz[z]]
                if abs(cz - np.floor(cz) - 0.5) > 1e-6:
                    assert q[b, z] == int(np.rint(cz))
            low = np.zeros((8, 8))
            for z in range(k + 1):
                low[zz[z]] = q[b, z]
            want = x - scipy.fft.idctn(low, norm="ortho")                 # the remainder against the quantised Part 1, in reals
            got = pub[64 * b:64 * b + 64].astype(np.float64).reshape(8, 8)
            diff = np.mod(got - want + 128.0, 256.0) - 128.0              # the bytes hold the remainder modulo 256
            assert np.abs(diff).max() <= 1.0


def test_digests_and_ciphertext_by_hand():
    """K4 re-derived with hashlib: private leaves are the groups' bytes, public leaves 8 blocks x 64 bytes, fan-out 16; the private
    stream is one AES-CTR message (oracle.aes128_ctr_xor is pinned by SP 800-38A)."""
    w, h, c, k, bits = 136, 16, 3, 5, 11          # 17 block columns: groups of 8, 8, 1
    img = synth.image(w, h, c, seed=4)
    key, nonce = synth.key_nonce(8)
    priv, pub, dg, q = oracle.fragment_dct_packed(img, k, bits, key, nonce)
    plain = b""
    sizes = []
    for row in range(c * (h // 8)):
        for g0 in (0, 8, 16):
            n = min(8, 17 - g0)
            b0 = row * 17 + g0
            blob = py_pack(q[b0:b0 + n], k, bits)
            plain += blob
            sizes.append(len(blob))
    assert oracle.aes128_ctr_xor(key, nonce, plain) == priv.tobytes()

    def root(leaves):
        d = [hashlib.sha256(x).digest() for x in leaves]
        while len(d) > 1:
            d = [hashlib.sha256(b"".join(d[i:i + 16])).digest() for i in range(0, len(d), 16)]
        return d[0]
    offs = np.concatenate([[0], np.cumsum(sizes)])
    assert dg[:32] == root([priv[offs[i]:offs[i + 1]].tobytes() for i in range(len(sizes))])
    pub_leaves = []
    for row in range(c * (h // 8)):
        for g0 in (0, 8, 16):
            n = min(8, 17 - g0)
            b0 = row * 17 + g0
            pub_leaves.append(pub[64 * b0:64 * (b0 + n)].tobytes())
    assert dg[32:] == root(pub_leaves)


def test_from_q_equals_whole_path():
    img = synth.image(48, 24, 3, seed=11)
    key, nonce = synth.key_nonce(2)
    for bits in (11, 8):
        priv, pub, dg, q = oracle.fragment_dct_packed(img, 5, bits, key, nonce)
        p2, q2, d2 = oracle.fragment_packed_from_q(img, q, 5, bits, key, nonce)
        assert (p2 == priv).all() and (q2 == pub).all() and d2 == dg
