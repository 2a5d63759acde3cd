"""CPU-only checks of libfeds.so: it loads, exports every symbol include/feds.h declares, answers the size queries,
rejects bad arguments before touching the device, and its __host__ __device__ arithmetic building blocks (the very
functions the kernels call) agree with outside libraries. No GPU compute is launched here."""
import ctypes as C
import hashlib
import os
import re

import numpy as np
import pytest
import scipy.fft
from cryptography.hazmat.primitives.ciphers import Cipher, algorithms, modes

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def b():
    from paper_1512_02951_b200 import build
    build.build()
    from paper_1512_02951_b200 import binding
    return binding


def test_exports_every_declared_symbol(b):
    header = open(os.path.join(ROOT, "include", "feds.h")).read() + open(os.path.join(ROOT, "include", "feds_debug.h")).read()
    assert "feds_debug_" not in open(os.path.join(ROOT, "include", "feds.h")).read()   # test hooks stay out of the product header
    declared = set(re.findall(r"\b(feds_[a-z0-9_]+)\s*\(", header))
    declared -= {"feds_stream_t"}
    assert declared == set(b.SYMBOLS), declared ^ set(b.SYMBOLS)
    for name in declared:
        assert hasattr(b.lib, name), name


def test_format_constants_match_design(b):
    assert b.merkle_params() == (8, 16, 2048)  # DESIGN.md 2.1 / 2.2


def test_size_queries(b):
    # SURVEY.md 8(a) sizes at the BASELINE configs
    assert b.dct_private_bytes(512, 512, 1, 2) == 49152 and b.dct_public_bytes(512, 512, 1, 2) == 999424
    assert b.dct_private_bytes(4096, 4096, 3, 5) == 18874368 and b.dct_public_bytes(4096, 4096, 3, 5) == 182452224
    assert b.dct_private_bytes(1920, 1080, 3, 3) == 1555200 and b.dct_public_bytes(1920, 1080, 3, 3) == 23328000
    assert b.dwt_private_bytes(8192, 8192, 1, 3) == 2097152 and b.dwt_public_bytes(8192, 8192, 1, 3) == 132120576
    assert b.dct_public_bytes(16, 16, 1, 63) == 0
    for bad in [(12, 16, 1, 3), (16, 16, 2, 3), (16, 16, 1, 64), (0, 16, 1, 3)]:
        assert b.dct_private_bytes(*bad) == 0
    assert b.dwt_private_bytes(16, 24, 1, 4) == 0 and b.dwt_private_bytes(16, 16, 1, 7) == 0
    assert b.workspace_bytes(512, 512, 1, 2) > 0 and b.workspace_bytes(512, 512, 1, 2) % 256 == 0
    assert b.workspace_bytes(8192, 8192, 1, 3, True) >= 2 * (4096 * 4096 + 2048 * 2048 + 1024 * 1024)


def test_argument_errors_are_reported_before_any_launch(b):
    key = bytes(16)
    ok_ptr = C.c_void_p(0x1000)  # never dereferenced: every call below must fail in validation
    f = b.lib.feds_fragment_dct
    assert f(None, 16, 16, 1, 3, key, key, ok_ptr, ok_ptr, ok_ptr, ok_ptr, 1 << 20, None) == 1      # null pointer
    assert f(ok_ptr, 12, 16, 1, 3, key, key, ok_ptr, ok_ptr, ok_ptr, ok_ptr, 1 << 20, None) == 2    # bad dims
    assert f(ok_ptr, 16, 16, 2, 3, key, key, ok_ptr, ok_ptr, ok_ptr, ok_ptr, 1 << 20, None) == 3    # bad channels
    assert f(ok_ptr, 16, 16, 1, 64, key, key, ok_ptr, ok_ptr, ok_ptr, ok_ptr, 1 << 20, None) == 3   # bad k
    assert f(ok_ptr, 64, 64, 1, 3, key, key, ok_ptr, ok_ptr, ok_ptr, ok_ptr, 8, None) == 4          # workspace too small
    assert f(C.c_void_p(0x1001), 16, 16, 1, 3, key, key, ok_ptr, ok_ptr, ok_ptr, ok_ptr, 1 << 20, None) == 6  # misaligned
    g = b.lib.feds_fragment_dwt
    assert g(ok_ptr, 16, 24, 1, 4, key, key, ok_ptr, ok_ptr, ok_ptr, ok_ptr, 1 << 20, None) == 2
    assert g(ok_ptr, 16, 16, 1, 0, key, key, ok_ptr, ok_ptr, ok_ptr, ok_ptr, 1 << 20, None) == 3
    assert g(ok_ptr, 64, 64, 1, 2, key, key, ok_ptr, ok_ptr, ok_ptr, ok_ptr, 8, None) == 4
    assert b.lib.feds_status_string(2) == b"bad dimensions"
    # two-stream verified defragment: needs digests, flags, a second stream (not the call's own) and both events
    t = b.lib.feds_defragment_dwt_batch_2s
    args = [ok_ptr, 4096, ok_ptr, 4096, 1, 64, 64, 1, 2, key, ok_ptr, ok_ptr, ok_ptr, 4096, ok_ptr, ok_ptr, 1 << 20, 0]
    assert t(*args, ok_ptr, None, ok_ptr, ok_ptr) == 1                      # no aux stream
    assert t(*args, ok_ptr, C.c_void_p(0x2000), None, ok_ptr) == 1           # no fork event
    assert t(*args, ok_ptr, ok_ptr, ok_ptr, ok_ptr) == 3                     # aux stream == stream
    no_digests = list(args); no_digests[11] = None
    assert t(*no_digests, ok_ptr, C.c_void_p(0x2000), ok_ptr, ok_ptr) == 1   # nothing to verify: use feds_defragment_dwt_batch
    bad = list(args); bad[5] = 62
    assert t(*bad, ok_ptr, C.c_void_p(0x2000), ok_ptr, ok_ptr) == 2          # bad dims come first


def test_binding_has_no_cpu_fallback():
    src = open(os.path.join(ROOT, "paper_1512_02951_b200", "binding.py")).read()
    assert "oracle" not in src.replace("no CPU fallback", "")
    for f in os.listdir(os.path.join(ROOT, "paper_1512_02951_b200", "csrc")):
        assert "oracle" not in open(os.path.join(ROOT, "paper_1512_02951_b200", "csrc", f)).read().replace("oracle/", "")


# ---------------------------------------------------------------- device arithmetic, run on the host
@pytest.mark.parametrize("n", [0, 1, 3, 55, 56, 63, 64, 65, 119, 120, 128, 1000, 2048])
def test_device_sha256_compress(b, n):
    msg = np.random.default_rng(n).integers(0, 256, n, dtype=np.uint8).tobytes()
    out = (C.c_uint8 * 32)()
    b.lib.feds_debug_sha256_host(msg, n, out)
    assert bytes(out) == hashlib.sha256(msg).digest()


def test_device_aes_ttables(b, kat):
    out = (C.c_uint8 * 16)()
    b.lib.feds_debug_aes128_host(bytes.fromhex(kat["fips197_B_key"]), bytes.fromhex(kat["fips197_B_in"]), out)
    assert bytes(out).hex() == kat["fips197_B_out"]
    b.lib.feds_debug_aes128_host(bytes.fromhex(kat["fips197_C1_key"]), bytes.fromhex(kat["fips197_C1_in"]), out)
    assert bytes(out).hex() == kat["fips197_C1_out"]
    rng = np.random.default_rng(1)
    for _ in range(200):
        key = rng.integers(0, 256, 16, dtype=np.uint8).tobytes()
        blk = rng.integers(0, 256, 16, dtype=np.uint8).tobytes()
        e = Cipher(algorithms.AES(key), modes.ECB()).encryptor()
        b.lib.feds_debug_aes128_host(key, blk, out)
        assert bytes(out) == e.update(blk) + e.finalize()


def test_device_dct_factorisation(b):
    rng = np.random.default_rng(2)
    worst = 0.0
    blocks = [rng.integers(0, 256, (8, 8)) for _ in range(300)]
    blocks += [np.full((8, 8), 255), np.zeros((8, 8)), (np.indices((8, 8)).sum(0) % 2) * 255, rng.integers(0, 2, (8, 8)) * 255]
    for x in blocks:
        xin = np.ascontiguousarray(x, dtype=np.float32)
        out = np.empty(64, dtype=np.float32)
        b.lib.feds_debug_dct8x8_host(xin.ctypes.data, out.ctypes.data, 0)
        ref = scipy.fft.dctn(x.astype(np.float64), norm="ortho")
        worst = max(worst, np.abs(out.reshape(8, 8) - ref).max())
        back = np.empty(64, dtype=np.float32)
        b.lib.feds_debug_dct8x8_host(out.ctypes.data, back.ctypes.data, 1)
        assert (np.rint(back.reshape(8, 8)) == x).all()       # exact uint8 round trip
    assert worst < 1e-3, worst                                # BASELINE tolerance (host float32 ~ device float32 up to FMA contraction)


def test_device_zigzag_table(b, paper_pins):
    out = (C.c_int * 64)()
    b.lib.feds_debug_zigzag_host(out)
    zz = [(v // 8, v % 8) for v in out]
    want = [tuple(int(t) for t in p.split(",")) for p in paper_pins["zigzag_first6"].split()]
    assert zz[:6] == want
    assert sorted(out) == list(range(64))
    for a, c in zip(zz, zz[1:]):
        assert max(abs(a[0] - c[0]), abs(a[1] - c[1])) == 1


def test_header_is_plain_c(tmp_path):
    """include/feds.h is a C ABI: it must compile as C99 with nothing but the standard headers (no CUDA, no C++)."""
    import shutil
    import subprocess
    gcc = shutil.which("gcc")
    if gcc is None:
        pytest.skip("no gcc")
    src = tmp_path / "use_feds.c"
    src.write_text('#include "feds.h"\nint main(void) { feds_stream_t s = 0; (void)s; return (int)feds_dct_private_bytes(8, 8, 1, 0) == 4 ? 0 : 1; }\n')
    res = subprocess.run([gcc, "-std=c99", "-Wall", "-Wextra", "-Werror", "-fsyntax-only", "-I", os.path.join(ROOT, "include"), str(src)],
                         capture_output=True, text=True)
    assert res.returncode == 0, res.stderr


def test_strong_level_basis_table_equals_the_oracles():
    """The strong level's fixed-point DCT basis B[z][p] = rne(4096 b_z(p)) decides stored bytes, so the library's
    table (built at compile time from a Taylor series) and the oracle's (libm) must agree in all 4096 entries."""
    import ctypes as C
    import numpy as np
    import oracle
    from paper_1512_02951_b200 import binding
    out = np.zeros(4096, dtype=np.int32)
    binding.lib.feds_debug_strong_basis_host(out.ctypes.data)
    assert (out.reshape(64, 64) == oracle.strong_basis()).all()


def test_sizes_and_argument_errors_of_the_widened_entry_points(b):
    """strong level, packed storage, tiled DWT design: sizes as the formats of DESIGN.md 2.3-2.5 define them, and
    argument errors reported before anything is enqueued (no GPU needed: every call below must fail in validation)."""
    L = b.lib
    key = bytes(16)
    ok = C.c_void_p(0x1000)
    assert L.feds_dct_strong_public_bytes(1920, 1080, 3) == 1920 * 1080 * 3 and L.feds_dct_strong_public_bytes(12, 16, 1) == 0
    # 66 bytes per 8 blocks (11-bit), 51 (8-bit) at k = 5; a ragged group rounds up to whole bytes
    assert L.feds_dct_packed_private_bytes(512, 512, 1, 5, 11) == 512 * 512 * 66 // 512
    assert L.feds_dct_packed_private_bytes(512, 512, 1, 5, 8) == 512 * 512 * 51 // 512
    assert L.feds_dct_packed_private_bytes(72, 8, 1, 5, 11) == 66 + 9 and L.feds_dct_packed_private_bytes(64, 8, 1, 5, 9) == 0
    assert L.feds_dct_packed_workspace_bytes(64, 8, 1, 5, 11) >= L.feds_workspace_bytes(64, 8, 1, 5, 0) + 66
    assert L.feds_dwt_tiles_private_bytes(512, 512, 1) == 4096 * 21 and L.feds_dwt_tiles_public_bytes(512, 512, 1) == 4096 * 60
    assert L.feds_dwt_tiles_private_bytes(12, 8, 1) == 0 and L.feds_dwt_tiles_workspace_bytes(512, 512, 1) % 256 == 0
    f = L.feds_fragment_dct_strong
    assert f(None, 16, 16, 1, 3, key, key, ok, ok, ok, ok, 1 << 20, None) == 1
    assert f(ok, 12, 16, 1, 3, key, key, ok, ok, ok, ok, 1 << 20, None) == 2
    assert f(ok, 16, 16, 1, 64, key, key, ok, ok, ok, ok, 1 << 20, None) == 3
    assert f(ok, 64, 64, 1, 3, key, key, ok, ok, ok, ok, 8, None) == 4
    assert f(ok, 16, 16, 1, 3, key, key, C.c_void_p(0x1004), ok, ok, ok, 1 << 20, None) == 6
    g = L.feds_fragment_dct_packed
    assert g(ok, 16, 16, 1, 3, 11, key, key, None, ok, ok, ok, 1 << 20, None) == 1
    assert g(ok, 16, 20, 1, 3, 11, key, key, ok, ok, ok, ok, 1 << 20, None) == 2
    assert g(ok, 16, 16, 1, 3, 10, key, key, ok, ok, ok, ok, 1 << 20, None) == 3            # ac_bits must be 11 or 8
    assert g(ok, 64, 64, 1, 3, 8, key, key, ok, ok, ok, ok, 8, None) == 4
    h = L.feds_defragment_dct_packed
    assert h(ok, ok, 16, 16, 1, 3, 11, key, key, ok, ok, None, ok, 1 << 20, None) == 1      # expected digests without a flag word
    t = L.feds_fragment_dwt_tiles
    assert t(ok, 16, 12, 1, key, key, ok, ok, ok, ok, 1 << 20, None) == 2
    assert t(ok, 16, 16, 2, key, key, ok, ok, ok, ok, 1 << 20, None) == 3
    assert t(ok, 16, 16, 1, key, None, ok, ok, ok, ok, 1 << 20, None) == 1
    assert t(ok, 64, 64, 1, key, key, ok, ok, ok, ok, 8, None) == 4
    assert t(ok, 16, 16, 1, key, key, ok, C.c_void_p(0x1008), ok, ok, 1 << 20, None) == 6
