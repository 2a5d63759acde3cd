"""Thin ctypes binding over libfeds.so (include/feds.h): argument marshalling only.

torch supplies device memory and streams; every step of the path runs in the library's CUDA kernels. There is no
CPU fallback: if the library is missing or fails to load, importing this module raises.
"""
import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("FEDS_LIB_PATH") or os.path.join(_HERE, "libfeds.so")

FLAG_NONE = 0
FLAG_NO_DIGEST = 1
FLAG_FORCE_FUSED = 2
FLAG_FORCE_SPLIT = 4
FLAG_DWT_TILED = 8
FLAG_GENERIC_TILES = 16

STATUS = {0: "FEDS_OK", 1: "FEDS_ERR_NULL_POINTER", 2: "FEDS_ERR_BAD_DIMS", 3: "FEDS_ERR_BAD_PARAM",
          4: "FEDS_ERR_WORKSPACE_TOO_SMALL", 5: "FEDS_ERR_CUDA", 6: "FEDS_ERR_MISALIGNED"}

# every symbol include/feds.h and include/feds_debug.h declare
SYMBOLS = [
    "feds_status_string", "feds_last_cuda_error", "feds_merkle_params",
    "feds_dct_private_bytes", "feds_dct_public_bytes", "feds_dwt_private_bytes", "feds_dwt_public_bytes",
    "feds_workspace_bytes",
    "feds_fragment_dct", "feds_defragment_dct", "feds_fragment_dwt", "feds_defragment_dwt",
    "feds_fragment_dct_batch", "feds_defragment_dct_batch", "feds_fragment_dwt_batch", "feds_defragment_dwt_batch",
    "feds_defragment_dwt_batch_2s",
    "feds_fragment_dct_host_scratch_bytes", "feds_fragment_dct_host",
    "feds_defragment_dct_host_scratch_bytes", "feds_defragment_dct_host", "feds_profile_events",
    "feds_aes128_ctr", "feds_sha256_merkle_workspace_bytes", "feds_sha256_merkle", "feds_sha256_merkle_static_max_bytes",
    "feds_sha256_merkle_static", "feds_verify_dct", "feds_verify_dct_batch", "feds_verify_dwt",
    "feds_dct_strong_public_bytes", "feds_fragment_dct_strong", "feds_defragment_dct_strong", "feds_fragment_dct_strong_batch",
    "feds_defragment_dct_strong_batch", "feds_debug_strong_basis_host",
    "feds_dct_packed_private_bytes", "feds_dct_packed_workspace_bytes", "feds_fragment_dct_packed", "feds_defragment_dct_packed",
    "feds_fragment_dct_packed_batch", "feds_defragment_dct_packed_batch",
    "feds_dwt_tiles_private_bytes", "feds_dwt_tiles_public_bytes", "feds_dwt_tiles_workspace_bytes", "feds_fragment_dwt_tiles",
    "feds_defragment_dwt_tiles", "feds_fragment_dwt_tiles_batch", "feds_defragment_dwt_tiles_batch",
    "feds_debug_sha256_host", "feds_debug_aes128_host", "feds_debug_dct8x8_host", "feds_debug_zigzag_host", "feds_debug_launch_count",
]


class FedsError(RuntimeError):
    def __init__(self, code, where):
        self.code = code
        super().__init__("%s returned %s (%d)" % (where, STATUS.get(code, "?"), code))


def _load():
    if not os.path.exists(LIB_PATH):
        raise ImportError("libfeds.so is not built: run `python -m paper_1512_02951_b200.build` (no CPU fallback exists)")
    lib = C.CDLL(LIB_PATH)
    vp, sz, i, u8p = C.c_void_p, C.c_size_t, C.c_int, C.c_char_p
    lib.feds_status_string.restype = C.c_char_p
    lib.feds_status_string.argtypes = [i]
    lib.feds_last_cuda_error.restype = i
    lib.feds_merkle_params.argtypes = [C.POINTER(i)] * 3
    for name in ["feds_dct_private_bytes", "feds_dct_public_bytes", "feds_dwt_private_bytes", "feds_dwt_public_bytes"]:
        getattr(lib, name).restype = sz
        getattr(lib, name).argtypes = [i, i, i, i]
    lib.feds_workspace_bytes.restype = sz
    lib.feds_workspace_bytes.argtypes = [i, i, i, i, i]
    lib.feds_fragment_dct.argtypes = [vp, i, i, i, i, u8p, u8p, vp, vp, vp, vp, sz, vp]
    lib.feds_fragment_dwt.argtypes = lib.feds_fragment_dct.argtypes
    lib.feds_defragment_dct.argtypes = [vp, vp, i, i, i, i, u8p, u8p, vp, vp, vp, vp, sz, vp]
    lib.feds_defragment_dwt.argtypes = lib.feds_defragment_dct.argtypes
    lib.feds_fragment_dct_batch.argtypes = [vp, i, sz, i, i, i, i, u8p, vp, vp, sz, vp, sz, vp, vp, sz, C.c_uint, vp]
    lib.feds_defragment_dct_batch.argtypes = [vp, sz, vp, sz, i, i, i, i, i, u8p, vp, vp, vp, sz, vp, vp, sz, C.c_uint, vp]
    lib.feds_fragment_dwt_batch.argtypes = lib.feds_fragment_dct_batch.argtypes
    lib.feds_fragment_dct_strong.argtypes = lib.feds_fragment_dct.argtypes
    lib.feds_defragment_dct_strong.argtypes = lib.feds_defragment_dct.argtypes
    lib.feds_fragment_dct_strong_batch.argtypes = lib.feds_fragment_dct_batch.argtypes
    lib.feds_defragment_dct_strong_batch.argtypes = lib.feds_defragment_dct_batch.argtypes
    lib.feds_dct_strong_public_bytes.restype = sz
    lib.feds_dct_strong_public_bytes.argtypes = [i, i, i]
    lib.feds_debug_strong_basis_host.argtypes = [vp]
    for name in ["feds_dct_packed_private_bytes", "feds_dct_packed_workspace_bytes"]:
        getattr(lib, name).restype = sz
        getattr(lib, name).argtypes = [i, i, i, i, i]
    for name in ["feds_dwt_tiles_private_bytes", "feds_dwt_tiles_public_bytes", "feds_dwt_tiles_workspace_bytes"]:
        getattr(lib, name).restype = sz
        getattr(lib, name).argtypes = [i, i, i]
    lib.feds_fragment_dwt_tiles.argtypes = [vp, i, i, i, u8p, u8p, vp, vp, vp, vp, sz, vp]
    lib.feds_defragment_dwt_tiles.argtypes = [vp, vp, i, i, i, u8p, u8p, vp, vp, vp, vp, sz, vp]
    lib.feds_fragment_dwt_tiles_batch.argtypes = [vp, i, sz, i, i, i, u8p, vp, vp, sz, vp, sz, vp, vp, sz, vp]
    lib.feds_defragment_dwt_tiles_batch.argtypes = [vp, sz, vp, sz, i, i, i, i, u8p, vp, vp, vp, sz, vp, vp, sz, vp]
    lib.feds_fragment_dct_packed.argtypes = [vp, i, i, i, i, i, u8p, u8p, vp, vp, vp, vp, sz, vp]
    lib.feds_defragment_dct_packed.argtypes = [vp, vp, i, i, i, i, i, u8p, u8p, vp, vp, vp, vp, sz, vp]
    lib.feds_fragment_dct_packed_batch.argtypes = [vp, i, sz, i, i, i, i, i, u8p, vp, vp, sz, vp, sz, vp, vp, sz, vp]
    lib.feds_defragment_dct_packed_batch.argtypes = [vp, sz, vp, sz, i, i, i, i, i, i, u8p, vp, vp, vp, sz, vp, vp, sz, vp]
    lib.feds_defragment_dwt_batch.argtypes = lib.feds_defragment_dct_batch.argtypes
    lib.feds_defragment_dwt_batch_2s.argtypes = list(lib.feds_defragment_dct_batch.argtypes) + [vp, vp, vp]
    lib.feds_defragment_dwt_batch_2s.restype = i
    lib.feds_fragment_dct_host_scratch_bytes.restype = sz
    lib.feds_fragment_dct_host_scratch_bytes.argtypes = [i, i, i, i, i, i]
    lib.feds_fragment_dct_host.argtypes = [vp, i, i, i, i, i, u8p, vp, vp, vp, vp, i, vp, sz, C.POINTER(vp), i, C.c_uint]
    lib.feds_defragment_dct_host_scratch_bytes.restype = sz
    lib.feds_defragment_dct_host_scratch_bytes.argtypes = [i, i, i, i, i, i]
    lib.feds_defragment_dct_host.argtypes = [vp, vp, i, i, i, i, i, u8p, vp, vp, vp, vp, i, vp, sz, C.POINTER(vp), i, C.c_uint]
    lib.feds_verify_dct.argtypes = [vp, vp, i, i, i, i, vp, vp, vp, sz, vp]
    lib.feds_verify_dwt.argtypes = lib.feds_verify_dct.argtypes
    lib.feds_verify_dct_batch.argtypes = [vp, sz, vp, sz, i, i, i, i, i, vp, vp, vp, sz, vp]
    lib.feds_aes128_ctr.argtypes = [vp, vp, sz, u8p, u8p, vp]
    lib.feds_sha256_merkle_workspace_bytes.restype = sz
    lib.feds_sha256_merkle_workspace_bytes.argtypes = [sz]
    lib.feds_sha256_merkle.argtypes = [vp, sz, vp, vp, sz, vp]
    lib.feds_sha256_merkle_static_max_bytes.restype = sz
    lib.feds_sha256_merkle_static_max_bytes.argtypes = []
    lib.feds_sha256_merkle_static.argtypes = [vp, sz, vp, vp]
    lib.feds_sha256_merkle_static.restype = i
    lib.feds_profile_events.argtypes = [vp, vp]
    lib.feds_profile_events.restype = None
    lib.feds_debug_sha256_host.argtypes = [u8p, sz, vp]
    lib.feds_debug_aes128_host.argtypes = [u8p, u8p, vp]
    lib.feds_debug_dct8x8_host.argtypes = [vp, vp, i]
    lib.feds_debug_zigzag_host.argtypes = [vp]
    lib.feds_debug_launch_count.restype = C.c_ulonglong
    lib.feds_debug_launch_count.argtypes = []
    for name in ["feds_fragment_dct", "feds_defragment_dct", "feds_fragment_dwt", "feds_defragment_dwt",
                 "feds_fragment_dct_batch", "feds_defragment_dct_batch", "feds_fragment_dwt_batch", "feds_defragment_dwt_batch",
                 "feds_fragment_dct_host", "feds_defragment_dct_host", "feds_fragment_dct_strong", "feds_defragment_dct_strong",
                 "feds_fragment_dct_strong_batch", "feds_defragment_dct_strong_batch", "feds_fragment_dct_packed", "feds_defragment_dct_packed",
                 "feds_fragment_dct_packed_batch", "feds_defragment_dct_packed_batch", "feds_fragment_dwt_tiles", "feds_defragment_dwt_tiles",
                 "feds_fragment_dwt_tiles_batch", "feds_defragment_dwt_tiles_batch",
                 "feds_aes128_ctr", "feds_sha256_merkle", "feds_verify_dct", "feds_verify_dct_batch", "feds_verify_dwt"]:
        getattr(lib, name).restype = i
    return lib


lib = _load()


def _check(code, where):
    if code != 0:
        raise FedsError(code, where)


def _ptr(t):
    return C.c_void_p(t.data_ptr()) if t is not None else None


def _stream(stream):
    s = stream if stream is not None else torch.cuda.current_stream()
    return C.c_void_p(s.cuda_stream)


def _fork_join_events(owner):
    """the two cudaEvent_t a *_2s call needs, created once per batch object (torch creates the event at its first record)"""
    if not hasattr(owner, "_events"):
        owner._events = [torch.cuda.Event(), torch.cuda.Event()]
        for e in owner._events:
            e.record()
    return tuple(C.c_void_p(e.cuda_event) for e in owner._events)


def _k16(b):
    """key / nonce: exactly 16 bytes (the library reads 16 bytes from the pointer it is given)."""
    b = bytes(b)
    if len(b) != 16:
        raise ValueError("key and nonce must be 16 bytes, got %d" % len(b))
    return b


def _on_stream(stream, *tensors):
    """Tensors allocated here on torch's current stream but used by kernels enqueued on `stream`: tell the caching allocator,
    so that the memory is not handed to other work while those kernels may still run."""
    if stream is not None and stream != torch.cuda.current_stream():
        for t in tensors:
            if t is not None and t.is_cuda:
                t.record_stream(stream)


def launch_count():
    """kernels launched by the library from this thread so far (feds_debug_launch_count)"""
    return int(lib.feds_debug_launch_count())


def merkle_params():
    g, f, l = C.c_int(), C.c_int(), C.c_int()
    lib.feds_merkle_params(C.byref(g), C.byref(f), C.byref(l))
    return g.value, f.value, l.value


def dct_private_bytes(w, h, c, k):
    return lib.feds_dct_private_bytes(w, h, c, k)


def dct_public_bytes(w, h, c, k):
    return lib.feds_dct_public_bytes(w, h, c, k)


def dwt_private_bytes(w, h, c, levels):
    return lib.feds_dwt_private_bytes(w, h, c, levels)


def dwt_public_bytes(w, h, c, levels):
    return lib.feds_dwt_public_bytes(w, h, c, levels)


def workspace_bytes(w, h, c, k_or_levels, is_dwt=False):
    return lib.feds_workspace_bytes(w, h, c, k_or_levels, 1 if is_dwt else 0)


def _u8(n, device):
    return torch.empty(max(int(n), 16), dtype=torch.uint8, device=device)


def _hwc(image):
    assert image.dtype == torch.uint8 and image.is_cuda and image.is_contiguous()
    if image.dim() == 2:
        image = image.unsqueeze(-1)
    h, w, c = image.shape
    return image, int(w), int(h), int(c)


def fragment_dct(image, k, key, nonce, stream=None, workspace=None):
    """feds_fragment_dct: image uint8[H][W][C] (cuda) -> (private, public, digests[64]) device tensors."""
    image, w, h, c = _hwc(image)
    dev = image.device
    priv = _u8(dct_private_bytes(w, h, c, k), dev)
    pub = _u8(dct_public_bytes(w, h, c, k), dev)
    dg = _u8(64, dev)
    ws = workspace if workspace is not None else _u8(workspace_bytes(w, h, c, k), dev)
    _on_stream(stream, priv, pub, dg, ws)
    _check(lib.feds_fragment_dct(_ptr(image), w, h, c, k, _k16(key), _k16(nonce), _ptr(priv), _ptr(pub), _ptr(dg), _ptr(ws),
                                 ws.numel(), _stream(stream)), "feds_fragment_dct")
    return priv[:dct_private_bytes(w, h, c, k)], pub[:dct_public_bytes(w, h, c, k)], dg


def defragment_dct(priv, pub, w, h, c, k, key, nonce, expected=None, stream=None, workspace=None):
    """feds_defragment_dct -> (image uint8[H][W][C], flags int32[1] or None)."""
    dev = priv.device
    out = torch.empty((h, w, c), dtype=torch.uint8, device=dev)
    flags = torch.zeros(1, dtype=torch.int32, device=dev) if expected is not None else None
    ws = workspace if workspace is not None else _u8(workspace_bytes(w, h, c, k), dev)
    _on_stream(stream, out, flags, ws)
    _check(lib.feds_defragment_dct(_ptr(priv), _ptr(pub), w, h, c, k, _k16(key), _k16(nonce), _ptr(expected), _ptr(out),
                                   _ptr(flags), _ptr(ws), ws.numel(), _stream(stream)), "feds_defragment_dct")
    return out, flags


def fragment_dct_strong(image, k, key, nonce, stream=None, workspace=None):
    """feds_fragment_dct_strong: image -> (private ciphertext, public uint8[w*h*c], digests[64]) at the strong level"""
    image, w, h, c = _hwc(image)
    dev = image.device
    priv = _u8(dct_private_bytes(w, h, c, k), dev)
    pub = _u8(lib.feds_dct_strong_public_bytes(w, h, c), dev)
    dg = _u8(64, dev)
    ws = workspace if workspace is not None else _u8(workspace_bytes(w, h, c, k), dev)
    _on_stream(stream, priv, pub, dg, ws)
    _check(lib.feds_fragment_dct_strong(_ptr(image), w, h, c, k, _k16(key), _k16(nonce), _ptr(priv), _ptr(pub), _ptr(dg), _ptr(ws),
                                        ws.numel(), _stream(stream)), "feds_fragment_dct_strong")
    return priv[:dct_private_bytes(w, h, c, k)], pub[:w * h * c], dg


def defragment_dct_strong(priv, pub, w, h, c, k, key, nonce, expected=None, stream=None, workspace=None):
    dev = priv.device
    out = torch.empty((h, w, c), dtype=torch.uint8, device=dev)
    flags = torch.zeros(1, dtype=torch.int32, device=dev) if expected is not None else None
    ws = workspace if workspace is not None else _u8(workspace_bytes(w, h, c, k), dev)
    _on_stream(stream, out, flags, ws)
    _check(lib.feds_defragment_dct_strong(_ptr(priv), _ptr(pub), w, h, c, k, _k16(key), _k16(nonce), _ptr(expected), _ptr(out),
                                          _ptr(flags), _ptr(ws), ws.numel(), _stream(stream)), "feds_defragment_dct_strong")
    return out, flags


def dct_packed_private_bytes(w, h, c, k, ac_bits):
    return lib.feds_dct_packed_private_bytes(w, h, c, k, ac_bits)


def fragment_dct_packed(image, k, ac_bits, key, nonce, stream=None):
    """feds_fragment_dct_packed: image -> (private: packed integers under AES-CTR, public uint8[w*h*c], digests[64])"""
    image, w, h, c = _hwc(image)
    dev = image.device
    pb = dct_packed_private_bytes(w, h, c, k, ac_bits)
    priv, pub, dg = _u8(pb, dev), _u8(w * h * c, dev), _u8(64, dev)
    ws = _u8(lib.feds_dct_packed_workspace_bytes(w, h, c, k, ac_bits), dev)
    _on_stream(stream, priv, pub, dg, ws)
    _check(lib.feds_fragment_dct_packed(_ptr(image), w, h, c, k, ac_bits, _k16(key), _k16(nonce), _ptr(priv), _ptr(pub), _ptr(dg), _ptr(ws),
                                        ws.numel(), _stream(stream)), "feds_fragment_dct_packed")
    return priv[:pb], pub[:w * h * c], dg


def defragment_dct_packed(priv, pub, w, h, c, k, ac_bits, key, nonce, expected=None, stream=None):
    dev = priv.device
    out = torch.empty((h, w, c), dtype=torch.uint8, device=dev)
    flags = torch.zeros(1, dtype=torch.int32, device=dev) if expected is not None else None
    ws = _u8(lib.feds_dct_packed_workspace_bytes(w, h, c, k, ac_bits), dev)
    _on_stream(stream, out, flags, ws)
    _check(lib.feds_defragment_dct_packed(_ptr(priv), _ptr(pub), w, h, c, k, ac_bits, _k16(key), _k16(nonce), _ptr(expected), _ptr(out),
                                          _ptr(flags), _ptr(ws), ws.numel(), _stream(stream)), "feds_defragment_dct_packed")
    return out, flags


class PackedBatch:
    """Pre-allocated buffers for feds_fragment_dct_packed_batch / feds_defragment_dct_packed_batch on n images of one shape."""

    def __init__(self, n, w, h, c, k, ac_bits, device="cuda"):
        self.n, self.w, self.h, self.c, self.k, self.ac_bits = n, w, h, c, k, ac_bits
        self.image_bytes = w * h * c
        self.priv_bytes = dct_packed_private_bytes(w, h, c, k, ac_bits)
        self.pub_bytes = w * h * c
        self.priv_stride = (self.priv_bytes + 15) // 16 * 16
        self.pub_stride = (self.pub_bytes + 15) // 16 * 16
        self.priv = _u8(n * self.priv_stride, device)
        self.pub = _u8(n * self.pub_stride, device)
        self.digests = _u8(n * 64, device)
        self.ws = _u8(n * lib.feds_dct_packed_workspace_bytes(w, h, c, k, ac_bits), device)
        self.flags_out = torch.zeros(n, dtype=torch.int32, device=device)

    def fragment(self, images, key, d_nonces, stream=None):
        _check(lib.feds_fragment_dct_packed_batch(_ptr(images), self.n, self.image_bytes, self.w, self.h, self.c, self.k, self.ac_bits,
                                                  _k16(key), _ptr(d_nonces), _ptr(self.priv), self.priv_stride, _ptr(self.pub),
                                                  self.pub_stride, _ptr(self.digests), _ptr(self.ws), self.ws.numel(), _stream(stream)),
               "feds_fragment_dct_packed_batch")

    def defragment(self, images_out, key, d_nonces, expected=None, stream=None):
        _check(lib.feds_defragment_dct_packed_batch(_ptr(self.priv), self.priv_stride, _ptr(self.pub), self.pub_stride, self.n, self.w,
                                                    self.h, self.c, self.k, self.ac_bits, _k16(key), _ptr(d_nonces), _ptr(expected),
                                                    _ptr(images_out), self.image_bytes, _ptr(self.flags_out), _ptr(self.ws),
                                                    self.ws.numel(), _stream(stream)), "feds_defragment_dct_packed_batch")


def fragment_dwt_tiles(image, key, nonce, stream=None):
    """feds_fragment_dwt_tiles: the report's tiled DWT design -> (private 21 B/tile, public 60 B/tile, digests[64])"""
    image, w, h, c = _hwc(image)
    dev = image.device
    pvb, pbb = lib.feds_dwt_tiles_private_bytes(w, h, c), lib.feds_dwt_tiles_public_bytes(w, h, c)
    priv, pub, dg = _u8(pvb, dev), _u8(pbb, dev), _u8(64, dev)
    ws = _u8(lib.feds_dwt_tiles_workspace_bytes(w, h, c), dev)
    _on_stream(stream, priv, pub, dg, ws)
    _check(lib.feds_fragment_dwt_tiles(_ptr(image), w, h, c, _k16(key), _k16(nonce), _ptr(priv), _ptr(pub), _ptr(dg), _ptr(ws), ws.numel(),
                                       _stream(stream)), "feds_fragment_dwt_tiles")
    return priv[:pvb], pub[:pbb], dg


def defragment_dwt_tiles(priv, pub, w, h, c, key, nonce, expected=None, stream=None):
    dev = priv.device
    out = torch.empty((h, w, c), dtype=torch.uint8, device=dev)
    flags = torch.zeros(1, dtype=torch.int32, device=dev) if expected is not None else None
    ws = _u8(lib.feds_dwt_tiles_workspace_bytes(w, h, c), dev)
    _on_stream(stream, out, flags, ws)
    _check(lib.feds_defragment_dwt_tiles(_ptr(priv), _ptr(pub), w, h, c, _k16(key), _k16(nonce), _ptr(expected), _ptr(out), _ptr(flags),
                                         _ptr(ws), ws.numel(), _stream(stream)), "feds_defragment_dwt_tiles")
    return out, flags


class TilesBatch:
    """Pre-allocated buffers for feds_fragment_dwt_tiles_batch / feds_defragment_dwt_tiles_batch on n images of one shape."""

    def __init__(self, n, w, h, c, device="cuda"):
        self.n, self.w, self.h, self.c = n, w, h, c
        self.image_bytes = w * h * c
        self.priv_bytes = lib.feds_dwt_tiles_private_bytes(w, h, c)
        self.pub_bytes = lib.feds_dwt_tiles_public_bytes(w, h, c)
        self.priv_stride = (self.priv_bytes + 15) // 16 * 16
        self.pub_stride = (self.pub_bytes + 15) // 16 * 16
        self.priv = _u8(n * self.priv_stride, device)
        self.pub = _u8(n * self.pub_stride, device)
        self.digests = _u8(n * 64, device)
        self.ws = _u8(n * lib.feds_dwt_tiles_workspace_bytes(w, h, c), device)
        self.flags_out = torch.zeros(n, dtype=torch.int32, device=device)

    def fragment(self, images, key, d_nonces, stream=None):
        _check(lib.feds_fragment_dwt_tiles_batch(_ptr(images), self.n, self.image_bytes, self.w, self.h, self.c, _k16(key), _ptr(d_nonces),
                                                 _ptr(self.priv), self.priv_stride, _ptr(self.pub), self.pub_stride, _ptr(self.digests),
                                                 _ptr(self.ws), self.ws.numel(), _stream(stream)), "feds_fragment_dwt_tiles_batch")

    def defragment(self, images_out, key, d_nonces, expected=None, stream=None):
        _check(lib.feds_defragment_dwt_tiles_batch(_ptr(self.priv), self.priv_stride, _ptr(self.pub), self.pub_stride, self.n, self.w, self.h,
                                                   self.c, _k16(key), _ptr(d_nonces), _ptr(expected), _ptr(images_out), self.image_bytes,
                                                   _ptr(self.flags_out), _ptr(self.ws), self.ws.numel(), _stream(stream)),
               "feds_defragment_dwt_tiles_batch")


def verify_dct(priv, pub, w, h, c, k, expected, stream=None, workspace=None):
    """feds_verify_dct: integrity of the two fragments against their 64-byte digest pair, no key needed -> flags tensor [1]."""
    dev = priv.device
    flags = torch.zeros(1, dtype=torch.int32, device=dev)
    ws = workspace if workspace is not None else _u8(workspace_bytes(w, h, c, k), dev)
    _on_stream(stream, flags, ws)
    _check(lib.feds_verify_dct(_ptr(priv), _ptr(pub), w, h, c, k, _ptr(expected), _ptr(flags), _ptr(ws), ws.numel(), _stream(stream)),
           "feds_verify_dct")
    return flags


def verify_dwt(priv, pub, w, h, c, levels, expected, stream=None, workspace=None):
    """feds_verify_dwt: integrity of the DWT fragments against their digest pair, no key needed -> flags tensor [1]."""
    dev = priv.device
    flags = torch.zeros(1, dtype=torch.int32, device=dev)
    ws = workspace if workspace is not None else _u8(workspace_bytes(w, h, c, levels, True), dev)
    _on_stream(stream, flags, ws)
    _check(lib.feds_verify_dwt(_ptr(priv), _ptr(pub), w, h, c, levels, _ptr(expected), _ptr(flags), _ptr(ws), ws.numel(), _stream(stream)),
           "feds_verify_dwt")
    return flags


def fragment_dwt(image, levels, key, nonce, stream=None, workspace=None):
    image, w, h, c = _hwc(image)
    dev = image.device
    priv = _u8(dwt_private_bytes(w, h, c, levels), dev)
    pub = _u8(dwt_public_bytes(w, h, c, levels), dev)
    dg = _u8(64, dev)
    ws = workspace if workspace is not None else _u8(workspace_bytes(w, h, c, levels, True), dev)
    _on_stream(stream, priv, pub, dg, ws)
    _check(lib.feds_fragment_dwt(_ptr(image), w, h, c, levels, _k16(key), _k16(nonce), _ptr(priv), _ptr(pub), _ptr(dg), _ptr(ws),
                                 ws.numel(), _stream(stream)), "feds_fragment_dwt")
    return priv[:dwt_private_bytes(w, h, c, levels)], pub[:dwt_public_bytes(w, h, c, levels)], dg


def defragment_dwt(priv, pub, w, h, c, levels, key, nonce, expected=None, stream=None, workspace=None):
    dev = priv.device
    out = torch.empty((h, w, c), dtype=torch.uint8, device=dev)
    flags = torch.zeros(1, dtype=torch.int32, device=dev) if expected is not None else None
    ws = workspace if workspace is not None else _u8(workspace_bytes(w, h, c, levels, True), dev)
    _on_stream(stream, out, flags, ws)
    _check(lib.feds_defragment_dwt(_ptr(priv), _ptr(pub), w, h, c, levels, _k16(key), _k16(nonce), _ptr(expected), _ptr(out),
                                   _ptr(flags), _ptr(ws), ws.numel(), _stream(stream)), "feds_defragment_dwt")
    return out, flags


def aes128_ctr(data, key, nonce, out=None, stream=None):
    """feds_aes128_ctr on a uint8 device tensor; out=None allocates, out=data works in place."""
    data = data.contiguous().view(-1)
    if out is None:
        out = torch.empty_like(data)
    _on_stream(stream, out)
    _check(lib.feds_aes128_ctr(_ptr(data), _ptr(out), data.numel(), _k16(key), _k16(nonce), _stream(stream)), "feds_aes128_ctr")
    return out


def sha256_merkle(data, stream=None, workspace=None):
    """feds_sha256_merkle: 32-byte Merkle root (2048-byte leaves, fan-out 16) of a uint8 device tensor."""
    data = data.contiguous().view(-1)
    root = _u8(32, data.device)
    need = lib.feds_sha256_merkle_workspace_bytes(data.numel())
    ws = workspace if workspace is not None else _u8(max(need, 16), data.device)
    _on_stream(stream, root, ws)
    _check(lib.feds_sha256_merkle(_ptr(data) if data.numel() else None, data.numel(), _ptr(root), _ptr(ws), ws.numel(), _stream(stream)),
           "feds_sha256_merkle")
    return root


def sha256_merkle_static(data, root, stream=None):
    """feds_sha256_merkle_static: the Merkle root of `data` into the caller's 32-byte device tensor `root`; the scratch is the
    library's static device array, nothing is allocated (streams up to feds_sha256_merkle_static_max_bytes())."""
    _check(lib.feds_sha256_merkle_static(_ptr(data) if data.numel() else None, data.numel(), _ptr(root), _stream(stream)),
           "feds_sha256_merkle_static")
    return root


class DctBatch:
    """Pre-allocated buffers for feds_fragment_dct_batch / feds_defragment_dct_batch on n images of one shape."""

    def __init__(self, n, w, h, c, k, device="cuda"):
        self.n, self.w, self.h, self.c, self.k = n, w, h, c, k
        self.image_bytes = w * h * c
        self.priv_bytes = dct_private_bytes(w, h, c, k)
        self.pub_bytes = dct_public_bytes(w, h, c, k)
        self.priv = _u8(n * self.priv_bytes, device)
        self.pub = _u8(n * self.pub_bytes, device)
        self.digests = _u8(n * 64, device)
        self.ws = _u8(n * workspace_bytes(w, h, c, k), device)
        self.flags_out = torch.zeros(n, dtype=torch.int32, device=device)

    def fragment(self, images, key, d_nonces, flags=FLAG_NONE, stream=None):
        assert images.is_cuda and images.dtype == torch.uint8 and images.is_contiguous() and images.numel() == self.n * self.image_bytes
        _check(lib.feds_fragment_dct_batch(_ptr(images), self.n, self.image_bytes, self.w, self.h, self.c, self.k, _k16(key),
                                           _ptr(d_nonces), _ptr(self.priv), self.priv_bytes, _ptr(self.pub), self.pub_bytes,
                                           _ptr(self.digests), _ptr(self.ws), self.ws.numel(), flags, _stream(stream)),
               "feds_fragment_dct_batch")

    def defragment(self, images_out, key, d_nonces, expected=None, flags=FLAG_NONE, stream=None):
        _check(lib.feds_defragment_dct_batch(_ptr(self.priv), self.priv_bytes, _ptr(self.pub), self.pub_bytes, self.n, self.w, self.h,
                                             self.c, self.k, _k16(key), _ptr(d_nonces), _ptr(expected), _ptr(images_out),
                                             self.image_bytes, _ptr(self.flags_out), _ptr(self.ws), self.ws.numel(), flags,
                                             _stream(stream)), "feds_defragment_dct_batch")


    def verify(self, expected=None, stream=None):
        """feds_verify_dct_batch on the batch's own fragments (expected defaults to its own digests) -> flags_out."""
        expected = self.digests if expected is None else expected
        _check(lib.feds_verify_dct_batch(_ptr(self.priv), self.priv_bytes, _ptr(self.pub), self.pub_bytes, self.n, self.w, self.h, self.c,
                                         self.k, _ptr(expected), _ptr(self.flags_out), _ptr(self.ws), self.ws.numel(), _stream(stream)),
               "feds_verify_dct_batch")
        return self.flags_out


class StrongBatch:
    """Pre-allocated buffers for feds_fragment_dct_strong_batch / feds_defragment_dct_strong_batch on n images of one shape."""

    def __init__(self, n, w, h, c, k, device="cuda"):
        self.n, self.w, self.h, self.c, self.k = n, w, h, c, k
        self.image_bytes = w * h * c
        self.priv_bytes = dct_private_bytes(w, h, c, k)
        self.pub_bytes = w * h * c
        self.priv_stride = (self.priv_bytes + 15) // 16 * 16
        self.pub_stride = (self.pub_bytes + 15) // 16 * 16
        self.priv = _u8(n * self.priv_stride, device)
        self.pub = _u8(n * self.pub_stride, device)
        self.digests = _u8(n * 64, device)
        self.ws = _u8(n * workspace_bytes(w, h, c, k), device)
        self.flags_out = torch.zeros(n, dtype=torch.int32, device=device)

    def fragment(self, images, key, d_nonces, flags=FLAG_NONE, stream=None):
        assert images.is_cuda and images.dtype == torch.uint8 and images.is_contiguous() and images.numel() == self.n * self.image_bytes
        _check(lib.feds_fragment_dct_strong_batch(_ptr(images), self.n, self.image_bytes, self.w, self.h, self.c, self.k, _k16(key),
                                                  _ptr(d_nonces), _ptr(self.priv), self.priv_stride, _ptr(self.pub), self.pub_stride,
                                                  _ptr(self.digests), _ptr(self.ws), self.ws.numel(), flags, _stream(stream)),
               "feds_fragment_dct_strong_batch")

    def defragment(self, images_out, key, d_nonces, expected=None, flags=FLAG_NONE, stream=None):
        _check(lib.feds_defragment_dct_strong_batch(_ptr(self.priv), self.priv_stride, _ptr(self.pub), self.pub_stride, self.n, self.w,
                                                    self.h, self.c, self.k, _k16(key), _ptr(d_nonces), _ptr(expected), _ptr(images_out),
                                                    self.image_bytes, _ptr(self.flags_out), _ptr(self.ws), self.ws.numel(), flags,
                                                    _stream(stream)), "feds_defragment_dct_strong_batch")


class DwtBatch:
    """Pre-allocated buffers for feds_fragment_dwt_batch / feds_defragment_dwt_batch on n images of one shape."""

    def __init__(self, n, w, h, c, levels, device="cuda"):
        self.n, self.w, self.h, self.c, self.levels = n, w, h, c, levels
        self.image_bytes = w * h * c
        self.priv_bytes = dwt_private_bytes(w, h, c, levels)
        self.pub_bytes = dwt_public_bytes(w, h, c, levels)
        self.priv_stride = (self.priv_bytes + 15) // 16 * 16
        self.pub_stride = (self.pub_bytes + 15) // 16 * 16
        self.priv = _u8(n * self.priv_stride, device)
        self.pub = _u8(n * self.pub_stride, device)
        self.digests = _u8(n * 64, device)
        self.ws = _u8(n * workspace_bytes(w, h, c, levels, True), device)
        self.flags_out = torch.zeros(n, dtype=torch.int32, device=device)

    def fragment(self, images, key, d_nonces, flags=FLAG_NONE, stream=None):
        assert images.is_cuda and images.dtype == torch.uint8 and images.is_contiguous() and images.numel() == self.n * self.image_bytes
        _check(lib.feds_fragment_dwt_batch(_ptr(images), self.n, self.image_bytes, self.w, self.h, self.c, self.levels, _k16(key),
                                           _ptr(d_nonces), _ptr(self.priv), self.priv_stride, _ptr(self.pub), self.pub_stride,
                                           _ptr(self.digests), _ptr(self.ws), self.ws.numel(), flags, _stream(stream)),
               "feds_fragment_dwt_batch")

    def defragment(self, images_out, key, d_nonces, expected=None, flags=FLAG_NONE, stream=None):
        _check(lib.feds_defragment_dwt_batch(_ptr(self.priv), self.priv_stride, _ptr(self.pub), self.pub_stride, self.n, self.w, self.h,
                                             self.c, self.levels, _k16(key), _ptr(d_nonces), _ptr(expected), _ptr(images_out),
                                             self.image_bytes, _ptr(self.flags_out), _ptr(self.ws), self.ws.numel(), flags,
                                             _stream(stream)), "feds_defragment_dwt_batch")

    def defragment_2s(self, images_out, key, d_nonces, expected, aux_stream, flags=FLAG_NONE, stream=None):
        """feds_defragment_dwt_batch_2s: verification on aux_stream (a torch.cuda.Stream), reconstruction on `stream`"""
        fork, join = _fork_join_events(self)
        _check(lib.feds_defragment_dwt_batch_2s(_ptr(self.priv), self.priv_stride, _ptr(self.pub), self.pub_stride, self.n, self.w, self.h,
                                                self.c, self.levels, _k16(key), _ptr(d_nonces), _ptr(expected), _ptr(images_out),
                                                self.image_bytes, _ptr(self.flags_out), _ptr(self.ws), self.ws.numel(), flags,
                                                _stream(stream), C.c_void_p(aux_stream.cuda_stream), fork, join),
               "feds_defragment_dwt_batch_2s")


def fragment_dct_host(h_images, w, h, c, k, key, h_nonces, h_priv, h_pub, h_digests, images_per_chunk, d_scratch, streams,
                      flags=FLAG_NONE):
    """feds_fragment_dct_host: pinned host tensors in/out, staged over `streams` (torch.cuda.Stream list)."""
    n = h_images.numel() // (w * h * c)
    arr = (C.c_void_p * len(streams))(*[s.cuda_stream for s in streams])
    _check(lib.feds_fragment_dct_host(_ptr(h_images), n, w, h, c, k, _k16(key), _ptr(h_nonces), _ptr(h_priv), _ptr(h_pub),
                                      _ptr(h_digests), images_per_chunk, _ptr(d_scratch), d_scratch.numel(), arr, len(streams), flags),
           "feds_fragment_dct_host")


def host_scratch_bytes(images_per_chunk, n_streams, w, h, c, k):
    return lib.feds_fragment_dct_host_scratch_bytes(images_per_chunk, n_streams, w, h, c, k)


def defragment_dct_host(h_priv, h_pub, n, w, h, c, k, key, h_nonces, h_expected, h_images_out, h_flags, images_per_chunk, d_scratch,
                        streams, flags=FLAG_NONE):
    """feds_defragment_dct_host: pinned host tensors in/out, staged over `streams`."""
    arr = (C.c_void_p * len(streams))(*[s.cuda_stream for s in streams])
    _check(lib.feds_defragment_dct_host(_ptr(h_priv), _ptr(h_pub), n, w, h, c, k, _k16(key), _ptr(h_nonces), _ptr(h_expected),
                                        _ptr(h_images_out), _ptr(h_flags), images_per_chunk, _ptr(d_scratch), d_scratch.numel(), arr,
                                        len(streams), flags), "feds_defragment_dct_host")


def defrag_host_scratch_bytes(images_per_chunk, n_streams, w, h, c, k):
    return lib.feds_defragment_dct_host_scratch_bytes(images_per_chunk, n_streams, w, h, c, k)


def profile_events(ev_start=None, ev_stop=None):
    """Thread-local hook: record the two torch.cuda.Event objects around the fused tile kernel of subsequent DCT calls."""
    for ev in (ev_start, ev_stop):
        if ev is not None and not ev.cuda_event:
            ev.record()  # torch creates the cudaEvent_t lazily; the library re-records it around the kernel
    a = C.c_void_p(ev_start.cuda_event) if ev_start is not None else None
    b_ = C.c_void_p(ev_stop.cuda_event) if ev_stop is not None else None
    lib.feds_profile_events(a, b_)
