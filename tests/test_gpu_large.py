"""GPU parity at the large end of BASELINE configs[4] (the sweep): square images 8192^2 and 16384^2, DCT k in {0, 2, 5, 9} and
DWT levels in {1, 2, 3, 4} -- SURVEY.md 8(d) row 5: "on larger sizes digests only". At these sizes a fragment is 0.8-4.2 GB, i.e.
byte offsets pass 2^31 (RGB) and 2^32 (four channels, 16384 x 17408, k = 0): exactly where a 32-bit index in a kernel would wrap.

DCT, per (size, k), in the launch configuration bench.py's sweep times (feds_fragment_dct / feds_defragment_dct, one image):
  * both digests: the oracle's Merkle root (orc_merkle_blocks) of the fragment bytes the GPU stored, bit-exact;
  * stage (i) on sampled 64x64 crops, among them the first and the very last blocks of the image (largest block index, largest
    CTR counter): private words are decrypted with the ORACLE's keystream at that counter offset and all 64 coefficients compared
    with the oracle's double DCT (<= 1e-3) -- a wrong counter, a wrapped offset or a misplaced run fails here;
  * exact uint8 round trip through the verifying defragment, flags 0.
DWT: everything is integer, so the whole of orc_fragment_dwt's output is compared (fragments and digests bit-exact), plus the round trip.
The oracle calls of one size run on a few host threads (ctypes releases the GIL); nothing else is shared between the cases.
"""
from concurrent.futures import ThreadPoolExecutor

import numpy as np
import pytest
import torch

import synth

pytestmark = pytest.mark.gpu
TOL = 1e-3


@pytest.fixture(scope="module")
def b():
    from paper_1512_02951_b200 import binding
    assert torch.cuda.is_available()
    return binding


def _image(w, h, c, seed):
    """The sweep's recipe generated in HBM (numpy would take minutes at 16384^2); the same bytes go to both sides."""
    d = synth.image_batch_torch(1, w, h, c, seed=seed, device="cuda")[0].contiguous()
    return d, d.cpu().numpy()


def _check_crops(orc, img, priv, pub, k, key, nonce, crops):
    """stage (i) on 64x64 crops given as (block row, block col): decrypt the private runs with the oracle's keystream."""
    h, w, c = img.shape
    nbr, nbc, P, Q = h // 8, w // 8, k + 1, 63 - k
    for by, bx in crops:
        ref = orc.dct_coefficients(np.ascontiguousarray(img[8 * by:8 * by + 64, 8 * bx:8 * bx + 64, :])).reshape(c, 8, 8, 64)
        for ch in range(c):
            for r in range(8):
                b0 = (ch * nbr + by + r) * nbc + bx                       # 8 consecutive blocks of one block row
                lo, hi = 4 * P * b0, 4 * P * (b0 + 8)
                first = lo // 16                                          # counter block holding byte `lo`
                ct = priv[16 * first:min(priv.size, (hi + 15) // 16 * 16)].tobytes()
                pt = orc.aes128_ctr_xor(key, nonce, ct, first_block=first)[lo - 16 * first:hi - 16 * first]
                got = np.concatenate([np.frombuffer(pt, dtype="<f4").reshape(8, P),
                                      np.frombuffer(pub[4 * Q * b0:4 * Q * (b0 + 8)].tobytes(), dtype="<f4").reshape(8, Q)], axis=1)
                assert np.abs(got - ref[ch, r]).max() <= TOL, (by, bx, ch, r)


def _dct_size(orc, b, size, c, ks, seed, h=None):
    w, h = size, (h or size)
    d_img, img = _image(w, h, c, seed)
    nbr, nbc = h // 8, w // 8
    rng = np.random.default_rng(size + c)
    crops = [(0, 0), (nbr - 8, nbc - 8)] + [(int(rng.integers(0, nbr - 8)), int(rng.integers(0, nbc - 8))) for _ in range(2)]
    jobs = []
    with ThreadPoolExecutor(max_workers=4) as ex:
        for k in ks:
            key, nonce = synth.key_nonce(size + k)
            priv, pub, dg = b.fragment_dct(d_img, k, key, nonce)
            rec, flags = b.defragment_dct(priv, pub, w, h, c, k, key, nonce, expected=dg)
            torch.cuda.synchronize()
            assert int(flags.item()) == 0 and torch.equal(rec, d_img), k      # stage (iii): exact uint8 round trip
            assert priv.numel() == orc.dct_private_bytes(w, h, c, k) and pub.numel() == orc.dct_public_bytes(w, h, c, k)
            pv, pb, dgb = priv.cpu().numpy(), pub.cpu().numpy(), dg.cpu().numpy().tobytes()
            del priv, pub, rec
            torch.cuda.empty_cache()
            P, Q = k + 1, 63 - k
            jobs.append((k, "private", dgb[:32], ex.submit(orc.merkle_blocks, pv, c * nbr, nbc, 4 * P)))
            jobs.append((k, "public", dgb[32:], ex.submit(orc.merkle_blocks, pb, c * nbr, nbc, 4 * Q)))
            jobs.append((k, "coefficients", None, ex.submit(_check_crops, orc, img, pv, pb, k, key, nonce, crops)))
        for k, what, want, fut in jobs:
            got = fut.result()
            if want is not None:
                assert got == want, "%s digest differs at size %d, k = %d" % (what, size, k)


@pytest.mark.parametrize("size", [8192, 16384])
def test_sweep_large_dct(orc, b, size):
    _dct_size(orc, b, size, 3, [0, 2, 5, 9], seed=5000 + size)


def test_fragment_offsets_beyond_2_pow_32(orc, b):
    """16384 x 17408 x 4 channels, k = 0: the public fragment is 4.49 GB, so byte offsets cross 2^31 and 2^32 inside one fragment
    (and the private one, 71 MB, has 4.5 M counter blocks)."""
    assert orc.dct_public_bytes(16384, 17408, 4, 0) > 1 << 32
    _dct_size(orc, b, 16384, 4, [0], seed=77, h=17408)


@pytest.mark.parametrize("size", [8192, 16384])
def test_sweep_large_dwt(orc, b, size):
    w = h = size
    c = 3
    d_img, img = _image(size, size, c, seed=6000 + size)
    with ThreadPoolExecutor(max_workers=4) as ex:
        futs = {}
        for L in [1, 2, 3, 4]:
            key, nonce = synth.key_nonce(size + 10 * L)
            futs[L] = ex.submit(orc.fragment_dwt, img, L, key, nonce)         # the oracle works while the GPU does
        for L in [1, 2, 3, 4]:
            key, nonce = synth.key_nonce(size + 10 * L)
            priv, pub, dg = b.fragment_dwt(d_img, L, key, nonce)
            rec, flags = b.defragment_dwt(priv, pub, w, h, c, L, key, nonce, expected=dg)
            torch.cuda.synchronize()
            assert int(flags.item()) == 0 and torch.equal(rec, d_img), L
            pv, pb, dgb = priv.cpu().numpy(), pub.cpu().numpy(), dg.cpu().numpy().tobytes()
            del priv, pub, rec
            torch.cuda.empty_cache()
            op, oq, odg = futs.pop(L).result()
            assert dgb == odg, "digests differ at size %d, L = %d" % (size, L)
            assert (pv == op).all() and (pb == oq).all(), "fragments differ at size %d, L = %d" % (size, L)
