"""ctypes loader for the CPU oracle (oracle/feds_oracle.c).

TEST INFRASTRUCTURE, NOT PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
`--impl reference` arm import this. Argument marshalling only; all arithmetic is in the C file, which
cites the paper passage each function follows. Format constants (G, F, LEAF) are DESIGN.md section 2's.
"""
import ctypes as C

import numpy as np

from . import build as _build

G_BLOCKS = 8      # blocks per DCT-path leaf
FANOUT = 16       # children per Merkle node
LEAF_BYTES = 2048  # bytes per DWT-path leaf

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
    return _lib


def _u8(a):
    a = np.ascontiguousarray(a, dtype=np.uint8)
    return a, a.ctypes.data_as(C.POINTER(C.c_uint8))


def _key(b):
    b = bytes(b)
    assert len(b) == 16
    return (C.c_uint8 * 16).from_buffer_copy(b)


def sha256(msg) -> bytes:
    a, p = _u8(np.frombuffer(bytes(msg), dtype=np.uint8) if not isinstance(msg, np.ndarray) else msg)
    out = (C.c_uint8 * 32)()
    lib().orc_sha256(p, C.c_uint64(a.size), out)
    return bytes(out)


def merkle_root(digests: bytes, fanout: int = FANOUT) -> bytes:
    a, p = _u8(np.frombuffer(bytes(digests), dtype=np.uint8))
    assert a.size % 32 == 0
    out = (C.c_uint8 * 32)()
    rc = lib().orc_merkle_root(p, C.c_uint64(a.size // 32), C.c_int(fanout), out)
    assert rc == 0, rc
    return bytes(out)


def merkle_stream(data, leaf_bytes: int = LEAF_BYTES, fanout: int = FANOUT) -> bytes:
    a, p = _u8(data if isinstance(data, np.ndarray) else np.frombuffer(bytes(data), dtype=np.uint8))
    out = (C.c_uint8 * 32)()
    rc = lib().orc_merkle_stream(p, C.c_uint64(a.size), C.c_uint64(leaf_bytes), C.c_int(fanout), out)
    assert rc == 0, rc
    return bytes(out)


def merkle_blocks(data, n_rows: int, nbc: int, per_block: int, g: int = G_BLOCKS, fanout: int = FANOUT) -> bytes:
    a, p = _u8(data if isinstance(data, np.ndarray) else np.frombuffer(bytes(data), dtype=np.uint8))
    assert a.size == n_rows * nbc * per_block
    out = (C.c_uint8 * 32)()
    rc = lib().orc_merkle_blocks(p, C.c_uint64(n_rows), C.c_uint64(nbc), C.c_uint64(per_block), C.c_int(g),
                                 C.c_int(fanout), out)
    assert rc == 0, rc
    return bytes(out)


def aes_sbox() -> bytes:
    out = (C.c_uint8 * 256)()
    lib().orc_aes_sbox(out)
    return bytes(out)


def aes128_expand_key(key) -> bytes:
    rk = (C.c_uint8 * 176)()
    lib().orc_aes128_expand_key(_key(key), rk)
    return bytes(rk)


def aes128_encrypt_block(key, block) -> bytes:
    rk = (C.c_uint8 * 176).from_buffer_copy(aes128_expand_key(key))
    out = (C.c_uint8 * 16)()
    lib().orc_aes128_encrypt_block(rk, _key(block), out)
    return bytes(out)


def aes128_ctr_xor(key, nonce, data, first_block: int = 0) -> bytes:
    a = np.array(np.frombuffer(bytes(data), dtype=np.uint8))  # writable copy
    p = a.ctypes.data_as(C.POINTER(C.c_uint8))
    lib().orc_aes128_ctr_xor(_key(key), _key(nonce), C.c_uint64(first_block), p, C.c_uint64(a.size))
    return a.tobytes()


def dct8x8(x) -> np.ndarray:
    x = np.ascontiguousarray(x, dtype=np.float64).reshape(64)
    out = np.empty(64, dtype=np.float64)
    lib().orc_dct8x8(x.ctypes.data_as(C.POINTER(C.c_double)), out.ctypes.data_as(C.POINTER(C.c_double)))
    return out.reshape(8, 8)


def idct8x8(X) -> np.ndarray:
    X = np.ascontiguousarray(X, dtype=np.float64).reshape(64)
    out = np.empty(64, dtype=np.float64)
    lib().orc_idct8x8(X.ctypes.data_as(C.POINTER(C.c_double)), out.ctypes.data_as(C.POINTER(C.c_double)))
    return out.reshape(8, 8)


def zigzag(z: int):
    r, q = C.c_int(), C.c_int()
    rc = lib().orc_zigzag(C.c_int(z), C.byref(r), C.byref(q))
    assert rc == 0
    return r.value, q.value


def _img(image):
    image = np.ascontiguousarray(image, dtype=np.uint8)
    if image.ndim == 2:
        image = image[:, :, None]
    h, w, c = image.shape
    return image, h, w, c


def dct_private_bytes(w, h, c, k):
    return (w // 8) * (h // 8) * c * (k + 1) * 4


def dct_public_bytes(w, h, c, k):
    return (w // 8) * (h // 8) * c * (63 - k) * 4


def dwt_private_bytes(w, h, c, levels):
    return (w >> levels) * (h >> levels) * c * 2


def dwt_public_bytes(w, h, c, levels):
    return (w * h - (w >> levels) * (h >> levels)) * c * 2


def dct_coefficients(image) -> np.ndarray:
    """double coefficients [C*nbr*nbc][64] in zigzag order (fragment block order)."""
    image, h, w, c = _img(image)
    nb = c * (h // 8) * (w // 8)
    out = np.empty((nb, 64), dtype=np.float64)
    rc = lib().orc_dct_coefficients(image.ctypes.data_as(C.POINTER(C.c_uint8)), w, h, c,
                                    out.ctypes.data_as(C.POINTER(C.c_double)))
    assert rc == 0, rc
    return out


def fragment_from_coef32(coef32, w, h, c, k, key, nonce, g=G_BLOCKS, fanout=FANOUT):
    coef32 = np.ascontiguousarray(coef32, dtype=np.float32)
    assert coef32.size == 64 * c * (h // 8) * (w // 8)
    priv = np.empty(dct_private_bytes(w, h, c, k), dtype=np.uint8)
    pub = np.empty(dct_public_bytes(w, h, c, k), dtype=np.uint8)
    dg = (C.c_uint8 * 64)()
    rc = lib().orc_fragment_from_coef32(coef32.ctypes.data_as(C.POINTER(C.c_float)), w, h, c, k, _key(key), _key(nonce),
                                        g, fanout, priv.ctypes.data_as(C.POINTER(C.c_uint8)),
                                        pub.ctypes.data_as(C.POINTER(C.c_uint8)), dg)
    assert rc == 0, rc
    return priv, pub, bytes(dg)


def fragment_dct(image, k, key, nonce, g=G_BLOCKS, fanout=FANOUT):
    image, h, w, c = _img(image)
    priv = np.empty(dct_private_bytes(w, h, c, k), dtype=np.uint8)
    pub = np.empty(dct_public_bytes(w, h, c, k), dtype=np.uint8)
    dg = (C.c_uint8 * 64)()
    rc = lib().orc_fragment_dct(image.ctypes.data_as(C.POINTER(C.c_uint8)), w, h, c, k, _key(key), _key(nonce), g, fanout,
                                priv.ctypes.data_as(C.POINTER(C.c_uint8)), pub.ctypes.data_as(C.POINTER(C.c_uint8)), dg)
    if rc != 0:
        raise ValueError("orc_fragment_dct rc=%d" % rc)
    return priv, pub, bytes(dg)


def defragment_dct(priv, pub, w, h, c, k, key, nonce, expected=None, g=G_BLOCKS, fanout=FANOUT):
    priv, pp = _u8(priv)
    pub, qq = _u8(pub)
    assert priv.size == dct_private_bytes(w, h, c, k) and pub.size == dct_public_bytes(w, h, c, k)
    out = np.empty((h, w, c), dtype=np.uint8)
    flags = C.c_uint32(0)
    exp = (C.c_uint8 * 64).from_buffer_copy(bytes(expected)) if expected is not None else None
    rc = lib().orc_defragment_dct(pp, qq, w, h, c, k, _key(key), _key(nonce), g, fanout, exp,
                                  out.ctypes.data_as(C.POINTER(C.c_uint8)), C.byref(flags))
    if rc != 0:
        raise ValueError("orc_defragment_dct rc=%d" % rc)
    return out, flags.value


def dwt53_fwd_1d(x) -> np.ndarray:
    x = np.ascontiguousarray(x, dtype=np.int32)
    y = np.empty_like(x)
    lib().orc_dwt53_fwd_1d(x.ctypes.data_as(C.POINTER(C.c_int32)), C.c_int(x.size), y.ctypes.data_as(C.POINTER(C.c_int32)))
    return y


def dwt53_inv_1d(y) -> np.ndarray:
    y = np.ascontiguousarray(y, dtype=np.int32)
    x = np.empty_like(y)
    lib().orc_dwt53_inv_1d(y.ctypes.data_as(C.POINTER(C.c_int32)), C.c_int(y.size), x.ctypes.data_as(C.POINTER(C.c_int32)))
    return x


def dwt_coefficients(image, levels) -> np.ndarray:
    """int32 [C][H][W] Mallat-layout planes of the L-level transform of (pixel - 128)."""
    image, h, w, c = _img(image)
    out = np.empty((c, h, w), dtype=np.int32)
    rc = lib().orc_dwt_coefficients(image.ctypes.data_as(C.POINTER(C.c_uint8)), w, h, c, levels,
                                    out.ctypes.data_as(C.POINTER(C.c_int32)))
    if rc != 0:
        raise ValueError("orc_dwt_coefficients rc=%d" % rc)
    return out


def dwt_inverse_plane(plane, levels) -> np.ndarray:
    p = np.array(plane, dtype=np.int32, order="C")
    h, w = p.shape
    rc = lib().orc_dwt53_inv_plane(p.ctypes.data_as(C.POINTER(C.c_int32)), w, h, levels)
    assert rc == 0
    return p


def fragment_dwt(image, levels, key, nonce, leaf_bytes=LEAF_BYTES, fanout=FANOUT):
    image, h, w, c = _img(image)
    if w <= 0 or h <= 0 or levels < 1 or levels > 6 or w % (1 << levels) or h % (1 << levels):
        raise ValueError("bad DWT dims")
    priv = np.empty(dwt_private_bytes(w, h, c, levels), dtype=np.uint8)
    pub = np.empty(dwt_public_bytes(w, h, c, levels), dtype=np.uint8)
    dg = (C.c_uint8 * 64)()
    rc = lib().orc_fragment_dwt(image.ctypes.data_as(C.POINTER(C.c_uint8)), w, h, c, levels, _key(key), _key(nonce),
                                C.c_uint64(leaf_bytes), fanout, priv.ctypes.data_as(C.POINTER(C.c_uint8)),
                                pub.ctypes.data_as(C.POINTER(C.c_uint8)), dg)
    if rc != 0:
        raise ValueError("orc_fragment_dwt rc=%d" % rc)
    return priv, pub, bytes(dg)


def defragment_dwt(priv, pub, w, h, c, levels, key, nonce, expected=None, leaf_bytes=LEAF_BYTES, fanout=FANOUT):
    priv, pp = _u8(priv)
    pub, qq = _u8(pub)
    assert priv.size == dwt_private_bytes(w, h, c, levels) and pub.size == dwt_public_bytes(w, h, c, levels)
    out = np.empty((h, w, c), dtype=np.uint8)
    flags = C.c_uint32(0)
    exp = (C.c_uint8 * 64).from_buffer_copy(bytes(expected)) if expected is not None else None
    rc = lib().orc_defragment_dwt(pp, qq, w, h, c, levels, _key(key), _key(nonce), C.c_uint64(leaf_bytes), fanout, exp,
                                  out.ctypes.data_as(C.POINTER(C.c_uint8)), C.byref(flags))
    if rc != 0:
        raise ValueError("orc_defragment_dwt rc=%d" % rc)
    return out, flags.value


# ------------------------------------------------------------------------------------------ strong level (feds_oracle_strong.c)
def sha512(msg) -> bytes:
    a, p = _u8(np.frombuffer(bytes(msg), dtype=np.uint8))
    out = (C.c_uint8 * 64)()
    lib().orc_sha512(p, C.c_uint64(a.size), out)
    return bytes(out)


def strong_basis() -> np.ndarray:
    """B[z][p] = rne(4096 b_z(p)), int32 [64][64]"""
    out = np.zeros((64, 64), dtype=np.int32)
    lib().orc_strong_basis(out.ctypes.data_as(C.POINTER(C.c_int32)))
    return out


def strong_public_bytes(w, h, c):
    return w * h * c


def fragment_dct_strong(image, k, key, nonce, g=G_BLOCKS, fanout=FANOUT):
    """image -> (private ciphertext, public uint8 [block][64], digests[64]) at the strong level of protection"""
    img, h, w, c = _img(image)
    pi = img.ctypes.data_as(C.POINTER(C.c_uint8))
    priv = np.zeros(dct_private_bytes(w, h, c, k), dtype=np.uint8)
    pub = np.zeros(w * h * c, dtype=np.uint8)
    dg = (C.c_uint8 * 64)()
    rc = lib().orc_fragment_dct_strong(pi, w, h, c, k, _key(key), _key(nonce), g, fanout, priv.ctypes.data_as(C.POINTER(C.c_uint8)),
                                       pub.ctypes.data_as(C.POINTER(C.c_uint8)), dg)
    assert rc == 0, rc
    return priv, pub, bytes(dg)


def fragment_strong_from_priv32(image, priv32, k, key, nonce, g=G_BLOCKS, fanout=FANOUT):
    """stage (ii): everything after the DCT from given float32 private coefficients priv32[b][z <= k]"""
    img, h, w, c = _img(image)
    pi = img.ctypes.data_as(C.POINTER(C.c_uint8))
    p32 = np.ascontiguousarray(priv32, dtype=np.float32)
    assert p32.size == (w // 8) * (h // 8) * c * (k + 1)
    priv = np.zeros(dct_private_bytes(w, h, c, k), dtype=np.uint8)
    pub = np.zeros(w * h * c, dtype=np.uint8)
    dg = (C.c_uint8 * 64)()
    rc = lib().orc_fragment_strong_from_priv32(pi, p32.ctypes.data_as(C.POINTER(C.c_float)), w, h, c, k, _key(key), _key(nonce), g, fanout,
                                               priv.ctypes.data_as(C.POINTER(C.c_uint8)), pub.ctypes.data_as(C.POINTER(C.c_uint8)), dg)
    assert rc == 0, rc
    return priv, pub, bytes(dg)


def defragment_dct_strong(priv, pub, w, h, c, k, key, nonce, expected=None, g=G_BLOCKS, fanout=FANOUT):
    pa, pp = _u8(priv)
    qa, qp = _u8(pub)
    out = np.zeros((h, w, c), dtype=np.uint8)
    fl = C.c_uint32(0)
    exp = (C.c_uint8 * 64).from_buffer_copy(bytes(expected)) if expected is not None else None
    rc = lib().orc_defragment_dct_strong(pp, qp, w, h, c, k, _key(key), _key(nonce), g, fanout, exp,
                                         out.ctypes.data_as(C.POINTER(C.c_uint8)), C.byref(fl))
    assert rc == 0, rc
    return out, int(fl.value)


def strong_remainder(image, k) -> np.ndarray:
    """x - L per pixel (signed, before the reduction modulo 256): int16 [h][w][c]"""
    img, h, w, c = _img(image)
    pi = img.ctypes.data_as(C.POINTER(C.c_uint8))
    out = np.zeros((h, w, c), dtype=np.int16)
    rc = lib().orc_strong_remainder(pi, w, h, c, k, out.ctypes.data_as(C.POINTER(C.c_int16)))
    assert rc == 0, rc
    return out


# ------------------------------------------------------------------------------------------ packed storage (feds_oracle_packed.c)
def packed_private_bytes(w, h, c, k, ac_bits, g=G_BLOCKS):
    lib().orc_packed_private_bytes.restype = C.c_uint64
    return int(lib().orc_packed_private_bytes(w, h, c, k, ac_bits, g))


def packed_quantise(cf, is_dc, ac_bits):
    lib().orc_packed_quantise.argtypes = [C.c_float, C.c_int, C.c_int]
    return int(lib().orc_packed_quantise(C.c_float(cf), int(is_dc), ac_bits))


def pack_group(q, k, ac_bits) -> bytes:
    """q: int32 [nblk][k+1] -> the bytes of one leaf group"""
    q = np.ascontiguousarray(q, dtype=np.int32).reshape(-1, k + 1)
    out = np.zeros((q.shape[0] * (11 + k * ac_bits) + 7) // 8 + 8, dtype=np.uint8)
    lib().orc_pack_group.restype = C.c_uint64
    n = lib().orc_pack_group(q.ctypes.data_as(C.POINTER(C.c_int32)), q.shape[0], k, ac_bits, out.ctypes.data_as(C.POINTER(C.c_uint8)))
    return out[:n].tobytes()


def unpack_group(data, nblk, k, ac_bits) -> np.ndarray:
    a, p = _u8(np.frombuffer(bytes(data), dtype=np.uint8))
    q = np.zeros((nblk, k + 1), dtype=np.int32)
    lib().orc_unpack_group.restype = C.c_uint64
    lib().orc_unpack_group(p, nblk, k, ac_bits, q.ctypes.data_as(C.POINTER(C.c_int32)))
    return q


def fragment_dct_packed(image, k, ac_bits, key, nonce, g=G_BLOCKS, fanout=FANOUT):
    """image -> (private: packed integers under AES-CTR, public: remainder pixels uint8 [block][64], digests[64], q int32 [nb][k+1])"""
    img, h, w, c = _img(image)
    nb = (w // 8) * (h // 8) * c
    priv = np.zeros(packed_private_bytes(w, h, c, k, ac_bits, g), dtype=np.uint8)
    pub = np.zeros(w * h * c, dtype=np.uint8)
    q = np.zeros((nb, k + 1), dtype=np.int32)
    dg = (C.c_uint8 * 64)()
    rc = lib().orc_fragment_dct_packed(img.ctypes.data_as(C.POINTER(C.c_uint8)), w, h, c, k, ac_bits, _key(key), _key(nonce), g, fanout,
                                       priv.ctypes.data_as(C.POINTER(C.c_uint8)), pub.ctypes.data_as(C.POINTER(C.c_uint8)), dg,
                                       q.ctypes.data_as(C.POINTER(C.c_int32)))
    assert rc == 0, rc
    return priv, pub, bytes(dg), q


def fragment_packed_from_q(image, q, k, ac_bits, key, nonce, g=G_BLOCKS, fanout=FANOUT):
    """stage (ii): everything after the quantisation from given integers q[b][z <= k]"""
    img, h, w, c = _img(image)
    q = np.ascontiguousarray(q, dtype=np.int32)
    assert q.size == (w // 8) * (h // 8) * c * (k + 1)
    priv = np.zeros(packed_private_bytes(w, h, c, k, ac_bits, g), dtype=np.uint8)
    pub = np.zeros(w * h * c, dtype=np.uint8)
    dg = (C.c_uint8 * 64)()
    rc = lib().orc_fragment_packed_from_q(img.ctypes.data_as(C.POINTER(C.c_uint8)), q.ctypes.data_as(C.POINTER(C.c_int32)), w, h, c, k, ac_bits,
                                          _key(key), _key(nonce), g, fanout, priv.ctypes.data_as(C.POINTER(C.c_uint8)),
                                          pub.ctypes.data_as(C.POINTER(C.c_uint8)), dg)
    assert rc == 0, rc
    return priv, pub, bytes(dg)


def defragment_dct_packed(priv, pub, w, h, c, k, ac_bits, key, nonce, expected=None, g=G_BLOCKS, fanout=FANOUT):
    pa, pp = _u8(priv)
    qa, qp = _u8(pub)
    out = np.zeros((h, w, c), dtype=np.uint8)
    fl = C.c_uint32(0)
    exp = (C.c_uint8 * 64).from_buffer_copy(bytes(expected)) if expected is not None else None
    rc = lib().orc_defragment_dct_packed(pp, qp, w, h, c, k, ac_bits, _key(key), _key(nonce), g, fanout, exp,
                                         out.ctypes.data_as(C.POINTER(C.c_uint8)), C.byref(fl))
    assert rc == 0, rc
    return out, int(fl.value)


# ------------------------------------------------------------------------------------------ tiled DWT design (feds_oracle_tiled.c)
def tiled_forward(tile) -> np.ndarray:
    """8x8 uint8 tile -> its 64 coefficients in level order (DESIGN.md 2.5 T2)"""
    t, p = _u8(np.ascontiguousarray(tile, dtype=np.uint8).reshape(64))
    out = np.zeros(64, dtype=np.int32)
    lib().orc_tiled_forward(p, out.ctypes.data_as(C.POINTER(C.c_int32)))
    return out


def tiled_inverse(coef) -> np.ndarray:
    cf = np.ascontiguousarray(coef, dtype=np.int32).reshape(64)
    out = np.zeros(64, dtype=np.uint8)
    lib().orc_tiled_inverse(cf.ctypes.data_as(C.POINTER(C.c_int32)), out.ctypes.data_as(C.POINTER(C.c_uint8)))
    return out.reshape(8, 8)


def tiled_pack(coef):
    """-> (level-1 bytes[5], level-2 bytes[16], level-3 bytes[60]) or None when a value does not fit its field"""
    cf = np.ascontiguousarray(coef, dtype=np.int32).reshape(64)
    l1, l2, l3 = (C.c_uint8 * 5)(), (C.c_uint8 * 16)(), (C.c_uint8 * 60)()
    rc = lib().orc_tiled_pack(cf.ctypes.data_as(C.POINTER(C.c_int32)), l1, l2, l3)
    return None if rc else (bytes(l1), bytes(l2), bytes(l3))


def tiled_private_bytes(w, h, c):
    return (w // 8) * (h // 8) * c * 21


def tiled_public_bytes(w, h, c):
    return (w // 8) * (h // 8) * c * 60


def fragment_tiled(image, key, nonce, leaf_bytes=LEAF_BYTES, fanout=FANOUT):
    img, h, w, c = _img(image)
    priv = np.zeros(tiled_private_bytes(w, h, c), dtype=np.uint8)
    pub = np.zeros(tiled_public_bytes(w, h, c), dtype=np.uint8)
    dg = (C.c_uint8 * 64)()
    rc = lib().orc_fragment_tiled(img.ctypes.data_as(C.POINTER(C.c_uint8)), w, h, c, _key(key), _key(nonce), C.c_uint64(leaf_bytes), fanout,
                                  priv.ctypes.data_as(C.POINTER(C.c_uint8)), pub.ctypes.data_as(C.POINTER(C.c_uint8)), dg)
    assert rc == 0, rc
    return priv, pub, bytes(dg)


def defragment_tiled(priv, pub, w, h, c, key, nonce, expected=None, leaf_bytes=LEAF_BYTES, fanout=FANOUT):
    pa, pp = _u8(priv)
    qa, qp = _u8(pub)
    out = np.zeros((h, w, c), dtype=np.uint8)
    fl = C.c_uint32(0)
    exp = (C.c_uint8 * 64).from_buffer_copy(bytes(expected)) if expected is not None else None
    rc = lib().orc_defragment_tiled(pp, qp, w, h, c, _key(key), _key(nonce), C.c_uint64(leaf_bytes), fanout, exp,
                                    out.ctypes.data_as(C.POINTER(C.c_uint8)), C.byref(fl))
    assert rc == 0, rc
    return out, int(fl.value)
