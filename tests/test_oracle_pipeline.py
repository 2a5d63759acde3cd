"""Pins for the oracle's whole fragment / defragment paths (layout, edge cases, round trips). CPU only.

Every expected value here is rebuilt from OUTSIDE libraries (scipy DCT, hashlib, cryptography AES-CTR) or from
plain numpy slicing of the format in DESIGN.md section 2 -- never from the oracle itself or the CUDA path.
"""
import hashlib
import struct

import numpy as np
import pytest
import scipy.fft
from cryptography.hazmat.primitives.ciphers import Cipher, algorithms, modes

import synth

G, F, LEAF = 8, 16, 2048
ZZ = None


def zz(orc):
    global ZZ
    if ZZ is None:
        ZZ = [orc.zigzag(z) for z in range(64)]
    return ZZ


def lib_ctr(key, nonce, data):
    e = Cipher(algorithms.AES(key), modes.CTR(nonce)).encryptor()
    return e.update(data) + e.finalize()


def brute_root(leaves, fan=F):
    if not leaves:
        return hashlib.sha256(b"").digest()
    cur = list(leaves)
    while len(cur) > 1:
        cur = [hashlib.sha256(b"".join(cur[i:i + fan])).digest() for i in range(0, len(cur), fan)]
    return cur[0]


def independent_fragment_dct(orc, img, k, key, nonce):
    """The format of DESIGN.md 2.1 rebuilt with scipy + cryptography + hashlib."""
    h, w, c = img.shape
    nbr, nbc, P, Q = h // 8, w // 8, k + 1, 63 - k
    priv, pub = [], []
    for ch in range(c):
        for br in range(nbr):
            for bc in range(nbc):
                X = scipy.fft.dctn(img[8 * br:8 * br + 8, 8 * bc:8 * bc + 8, ch].astype(np.float64), norm="ortho")
                v = np.array([X[r, q] for (r, q) in zz(orc)]).astype(np.float32)
                priv.append(v[:P].astype("<f4").tobytes())
                pub.append(v[P:].astype("<f4").tobytes())
    ct = lib_ctr(key, nonce, b"".join(priv))
    pubb = b"".join(pub)

    def root(data, per_block):
        if per_block == 0:
            return hashlib.sha256(b"").digest()
        leaves = []
        for r in range(c * nbr):
            for g0 in range(0, nbc, G):
                g1 = min(g0 + G, nbc)
                leaves.append(hashlib.sha256(data[(r * nbc + g0) * per_block:(r * nbc + g1) * per_block]).digest())
        return brute_root(leaves)

    return ct, pubb, root(ct, 4 * P) + root(pubb, 4 * Q)


@pytest.mark.parametrize("w,h,c,k", [(8, 8, 1, 0), (16, 8, 1, 5), (72, 24, 1, 2), (64, 16, 3, 3), (136, 8, 3, 5), (24, 16, 4, 9),
                                     (16, 16, 1, 63), (16, 16, 3, 62)])
def test_fragment_dct_matches_independent_rebuild(orc, w, h, c, k):
    img = synth.image(w, h, c, seed=w + h + c + k)
    key, nonce = synth.key_nonce(w * 1000 + k)
    priv, pub, dg = orc.fragment_dct(img, k, key, nonce)
    ct, pubb, dg2 = independent_fragment_dct(orc, img, k, key, nonce)
    assert priv.size == orc.dct_private_bytes(w, h, c, k) and pub.size == orc.dct_public_bytes(w, h, c, k)
    # float32 rounding of scipy's double vs the oracle's double may differ in the last ulp only where the two doubles
    # straddle a rounding boundary: compare as floats with 1-ulp slack after decrypting, and bit-exact when equal
    pt = np.frombuffer(lib_ctr(key, nonce, priv.tobytes()), dtype="<f4")
    pt2 = np.frombuffer(lib_ctr(key, nonce, ct), dtype="<f4")
    assert np.abs(pt - pt2).max() <= 2.5e-4
    assert np.abs(np.frombuffer(pub.tobytes(), dtype="<f4") - np.frombuffer(pubb, dtype="<f4")).max() <= 2.5e-4 if pub.size else True
    if priv.tobytes() == ct and pub.tobytes() == pubb:
        assert dg == dg2
    # exact layout check independent of rounding: stage-(ii) entry point fed the rebuild's own float32 values
    nb = c * (h // 8) * (w // 8)
    coef32 = np.concatenate([np.frombuffer(lib_ctr(key, nonce, ct), dtype="<f4").reshape(nb, k + 1),
                             np.frombuffer(pubb, dtype="<f4").reshape(nb, 63 - k)], axis=1)
    p2, q2, d2 = orc.fragment_from_coef32(coef32, w, h, c, k, key, nonce)
    assert p2.tobytes() == ct and q2.tobytes() == pubb and d2 == dg2


def test_fragment_sizes_and_paper_storage_arithmetic(orc, paper_pins):
    assert int(paper_pins["private_coeffs_default"]) == 5 + 1                       # k = 5 <-> "DC + 5 AC"
    assert abs(11 * 6 / 64 / 8 * 100 - float(paper_pins["storage_11bit_percent"])) < 0.05
    assert orc.dct_private_bytes(512, 512, 1, 2) == 49152 and orc.dct_public_bytes(512, 512, 1, 2) == 999424
    assert orc.dct_private_bytes(4096, 4096, 3, 5) == 18874368 and orc.dct_public_bytes(4096, 4096, 3, 5) == 182452224
    assert orc.dct_private_bytes(1920, 1080, 3, 3) == 1555200 and orc.dct_public_bytes(1920, 1080, 3, 3) == 23328000
    assert orc.dwt_private_bytes(8192, 8192, 1, 3) == 2097152 and orc.dwt_public_bytes(8192, 8192, 1, 3) == 132120576


@pytest.mark.parametrize("kind", ["zeros", "ones", "checker", "random", "impulse"])
@pytest.mark.parametrize("c,k", [(1, 0), (1, 5), (3, 3), (4, 63)])
def test_dct_round_trip_exact_uint8(orc, kind, c, k):
    img = synth.special(kind, 40, 24, c, seed=k)
    key, nonce = synth.key_nonce(99)
    priv, pub, dg = orc.fragment_dct(img, k, key, nonce)
    rec, flags = orc.defragment_dct(priv, pub, 40, 24, c, k, key, nonce, expected=dg)
    assert flags == 0 and (rec == img).all()            # PSNR infinite = lossless


def test_dct_round_trip_synthetic_and_wrong_key(orc):
    img = synth.image(64, 64, 3, seed=5, rectangles=4)
    key, nonce = synth.key_nonce(5)
    priv, pub, dg = orc.fragment_dct(img, 5, key, nonce)
    rec, flags = orc.defragment_dct(priv, pub, 64, 64, 3, 5, key, nonce, expected=dg)
    assert flags == 0 and (rec == img).all()
    bad, _ = orc.defragment_dct(priv, pub, 64, 64, 3, 5, bytes(16), nonce)
    assert (bad != img).mean() > 0.5                    # without the key the image is not recovered


def test_dct_verify_flags_and_error_confinement(orc):
    img = synth.image(64, 32, 1, seed=6)
    key, nonce = synth.key_nonce(6)
    priv, pub, dg = orc.fragment_dct(img, 3, key, nonce)
    p2 = priv.copy(); p2[99] ^= 0x40     # top (sign/exponent) byte of block 6's DC float
    rec, flags = orc.defragment_dct(p2, pub, 64, 32, 1, 3, key, nonce, expected=dg)
    assert flags == 1
    # CTR: one flipped ciphertext byte damages only the block whose coefficient it belongs to
    blk = 99 // 16                                       # P*4 = 16 bytes per block at k = 3
    diff = (rec != img)[:, :, 0]
    by, bx = divmod(blk, 8)
    mask = np.zeros_like(diff); mask[8 * by:8 * by + 8, 8 * bx:8 * bx + 8] = True
    assert diff[mask].any() and not diff[~mask].any()
    q2 = pub.copy(); q2[-1] ^= 1
    _, flags = orc.defragment_dct(priv, q2, 64, 32, 1, 3, key, nonce, expected=dg)
    assert flags == 2
    _, flags = orc.defragment_dct(p2, q2, 64, 32, 1, 3, key, nonce, expected=dg)
    assert flags == 3
    _, flags = orc.defragment_dct(p2, q2, 64, 32, 1, 3, key, nonce, expected=None)
    assert flags == 0                                    # NULL expected = no verification (A10)


def test_dct_rejects_bad_arguments(orc):
    key, nonce = synth.key_nonce(1)
    for shape, k in [((12, 16, 1), 3), ((16, 12, 1), 3), ((16, 16, 2), 3), ((16, 16, 1), 64), ((16, 16, 1), -1)]:
        with pytest.raises(ValueError):
            orc.fragment_dct(np.zeros(shape, dtype=np.uint8), k, key, nonce)


def test_batch_is_independent_images(orc):
    # A20: each image is its own CTR message and digest pair; nonces = base + i * 2^20
    key, nonce = synth.key_nonce(3)
    nonces = synth.batch_nonces(nonce, 3)
    assert int.from_bytes(nonces[2].tobytes(), "big") == (int.from_bytes(nonce, "big") + 2 * (1 << 20)) % (1 << 128)
    imgs = [synth.image(32, 16, 3, seed=30 + i) for i in range(3)]
    outs = [orc.fragment_dct(im, 3, key, nonces[i].tobytes()) for i, im in enumerate(imgs)]
    assert outs[0][0].tobytes() != outs[1][0].tobytes()


# ---------------------------------------------------------------- DWT path
def independent_fragment_dwt(orc, img, L, key, nonce):
    """DESIGN.md 2.2 rebuilt from the oracle-independent pieces: numpy lifting written here + hashlib + cryptography."""
    h, w, c = img.shape

    def fwd1(x):
        x = x.astype(np.int64)
        n = x.shape[-1]
        ev, od = x[..., 0::2], x[..., 1::2]
        right = np.concatenate([ev[..., 1:], ev[..., -1:]], axis=-1)       # x_ext(N) = x(N-2)
        d = od - np.floor_divide(ev + right, 2)
        left = np.concatenate([d[..., :1], d[..., :-1]], axis=-1)          # d(-1) = d(0)
        s = ev + np.floor_divide(left + d + 2, 4)
        return np.concatenate([s, d], axis=-1)

    priv, pub = [], []
    for ch in range(c):
        p = img[:, :, ch].astype(np.int64) - 128
        bands = []
        for l in range(1, L + 1):
            cw, chh = w >> (l - 1), h >> (l - 1)
            sub = p[:chh, :cw]
            sub = fwd1(sub)                       # rows first
            sub = fwd1(sub.T).T                   # then columns
            p[:chh, :cw] = sub
            bw, bh = cw // 2, chh // 2
            bands.append((sub[:bh, bw:], sub[bh:, :bw], sub[bh:, bw:]))   # HL, LH, HH
        priv.append(p[:h >> L, :w >> L].astype("<i2").tobytes())
        for l in range(L, 0, -1):
            for band in bands[l - 1]:
                pub.append(np.ascontiguousarray(band).astype("<i2").tobytes())
    ct = lib_ctr(key, nonce, b"".join(priv))
    pubb = b"".join(pub)
    root = lambda d: brute_root([hashlib.sha256(d[i:i + LEAF]).digest() for i in range(0, len(d), LEAF)])
    return ct, pubb, root(ct) + root(pubb)


@pytest.mark.parametrize("w,h,c,L", [(2, 2, 1, 1), (16, 8, 1, 1), (64, 32, 1, 2), (48, 80, 3, 3), (64, 64, 4, 4), (128, 64, 1, 6)])
def test_fragment_dwt_matches_independent_rebuild(orc, w, h, c, L):
    img = synth.image(w, h, c, seed=w + L)
    key, nonce = synth.key_nonce(w + h + L)
    priv, pub, dg = orc.fragment_dwt(img, L, key, nonce)
    ct, pubb, dg2 = independent_fragment_dwt(orc, img, L, key, nonce)
    assert priv.tobytes() == ct and pub.tobytes() == pubb and dg == dg2
    rec, flags = orc.defragment_dwt(priv, pub, w, h, c, L, key, nonce, expected=dg)
    assert flags == 0 and (rec == img).all()


@pytest.mark.parametrize("kind", ["zeros", "ones", "checker", "random", "impulse"])
def test_dwt_round_trip_and_flags(orc, kind):
    img = synth.special(kind, 64, 32, 3, seed=4)
    key, nonce = synth.key_nonce(12)
    for L in [1, 2, 3, 4]:
        priv, pub, dg = orc.fragment_dwt(img, L, key, nonce)
        rec, flags = orc.defragment_dwt(priv, pub, 64, 32, 3, L, key, nonce, expected=dg)
        assert flags == 0 and (rec == img).all()
    p2 = priv.copy(); p2[0] ^= 1
    _, flags = orc.defragment_dwt(p2, pub, 64, 32, 3, 4, key, nonce, expected=dg)
    assert flags == 1
    q2 = pub.copy(); q2[7] ^= 0x80
    _, flags = orc.defragment_dwt(priv, q2, 64, 32, 3, 4, key, nonce, expected=dg)
    assert flags == 2


def test_dwt_rejects_bad_arguments(orc):
    key, nonce = synth.key_nonce(1)
    for shape, L in [((12, 16, 1), 3), ((16, 16, 2), 1), ((16, 16, 1), 0), ((16, 16, 1), 7), ((16, 24, 1), 4)]:
        with pytest.raises(ValueError):
            orc.fragment_dwt(np.zeros(shape, dtype=np.uint8), L, key, nonce)


def test_synth_is_seeded_and_shaped():
    a = synth.image(64, 32, 3, seed=1)
    assert a.shape == (32, 64, 3) and a.dtype == np.uint8
    assert (a == synth.image(64, 32, 3, seed=1)).all() and (a != synth.image(64, 32, 3, seed=2)).any()
    k1, n1 = synth.key_nonce(1)
    assert k1 + n1 == hashlib.sha256(b"feds1").digest()
