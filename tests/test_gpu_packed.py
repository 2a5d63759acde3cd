"""GPU parity of the packed integer storage (feds_fragment_dct_packed / feds_defragment_dct_packed; PAPER.md 6.4.3, P:562-599;
DESIGN.md 2.4) through the C ABI against the oracle (oracle/feds_oracle_packed.c).

The stored integers are roundings of float32 DCT output, so where a coefficient lies within the float32 error of a rounding tie two
integers are correct. Parity is again the two-stage protocol:
  (i)   the integers the GPU stored (private fragment decrypted with the oracle's AES-CTR and unpacked with the oracle's bit reader,
        whose layout is pinned against a Python re-derivation) against the oracle's double DCT: |q - clamp(c)| <= 0.5 + 1e-3;
  (ii)  the oracle fed those integers: packed ciphertext, all public bytes and both Merkle digests bit-exact;
  (iii) exact uint8 round trips GPU(GPU), oracle(GPU), GPU(oracle), for both storages.
"""
import numpy as np
import pytest
import torch

import synth

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def b():
    from paper_1512_02951_b200 import binding
    assert torch.cuda.is_available()
    return binding


def gpu_integers(orc, priv, w, h, c, k, bits, key, nonce):
    plain = np.frombuffer(orc.aes128_ctr_xor(key, nonce, priv.tobytes()), dtype=np.uint8)
    nbc, rows = w // 8, c * (h // 8)
    q = np.zeros((rows * nbc, k + 1), dtype=np.int32)
    off = 0
    for r in range(rows):
        for g0 in range(0, nbc, 8):
            n = min(8, nbc - g0)
            nbytes = (n * (11 + k * bits) + 7) // 8
            q[r * nbc + g0:r * nbc + g0 + n] = orc.unpack_group(plain[off:off + nbytes].tobytes(), n, k, bits)
            off += nbytes
    assert off == plain.size
    return q


def check(orc, b, img, k, bits, seed):
    h, w, c = img.shape
    key, nonce = synth.key_nonce(seed)
    d_img = torch.from_numpy(img).cuda()
    priv, pub, dg = b.fragment_dct_packed(d_img, k, bits, key, nonce)
    torch.cuda.synchronize()
    pv, pb, dgb = priv.cpu().numpy(), pub.cpu().numpy(), dg.cpu().numpy().tobytes()
    assert pv.size == orc.packed_private_bytes(w, h, c, k, bits) and pb.size == w * h * c
    q = gpu_integers(orc, pv, w, h, c, k, bits, key, nonce)
    ref = orc.dct_coefficients(img)[:, :k + 1].copy()                                      # (i)
    M = (1 << (bits - 1)) - 1
    ref[:, 0] = np.clip(ref[:, 0], 0, 2047)
    ref[:, 1:] = np.clip(ref[:, 1:], -M, M)
    assert np.abs(q - ref).max() <= 0.5 + 1e-3
    p2, q2, d2 = orc.fragment_packed_from_q(img, q, k, bits, key, nonce)                    # (ii)
    assert (p2 == pv).all(), "private (packed ciphertext) differs"
    assert (q2 == pb).all(), "public bytes differ"
    assert d2 == dgb, "digests differ"
    rec, flags = b.defragment_dct_packed(priv, pub, w, h, c, k, bits, key, nonce, expected=dg)   # (iii)
    torch.cuda.synchronize()
    assert int(flags.item()) == 0 and torch.equal(rec, d_img)
    rec2, _ = b.defragment_dct_packed(priv, pub, w, h, c, k, bits, key, nonce)
    assert torch.equal(rec2, d_img)
    orec, ofl = orc.defragment_dct_packed(pv, pb, w, h, c, k, bits, key, nonce, expected=dgb)
    assert ofl == 0 and (orec == img).all()
    op, oq, odg, _ = orc.fragment_dct_packed(img, k, bits, key, nonce)
    rec3, fl3 = b.defragment_dct_packed(torch.from_numpy(op).cuda(), torch.from_numpy(oq).cuda(), w, h, c, k, bits, key, nonce,
                                        expected=torch.frombuffer(bytearray(odg), dtype=torch.uint8).cuda())
    torch.cuda.synchronize()
    assert int(fl3.item()) == 0 and torch.equal(rec3, d_img)
    return d_img, priv, pub, dg, key, nonce


@pytest.mark.parametrize("bits", [11, 8])
@pytest.mark.parametrize("w,h,c,k", [(8, 8, 1, 0), (8, 8, 1, 5), (16, 16, 4, 63), (64, 8, 1, 3), (72, 24, 1, 5), (1080, 16, 3, 5), (136, 40, 4, 9),
                                     (512, 512, 1, 5), (256, 264, 3, 5), (520, 24, 3, 26), (64, 64, 1, 32), (40, 8, 3, 4), (1920, 136, 3, 5),
                                     # w % 64 == 0 and a tile per block row: the bulk-copy tile kernels, all three PMAX forms, ragged last tiles
                                     (256, 40, 4, 9), (320, 24, 3, 3), (512, 16, 1, 15), (256, 16, 3, 0), (576, 72, 4, 2), (1024, 24, 1, 7),
                                     (512, 8, 1, 16), (1920, 8, 3, 12)])
def test_packed_parity_and_round_trips(orc, b, w, h, c, k, bits):
    check(orc, b, synth.image(w, h, c, seed=w + 3 * h + c + k, rectangles=2 if w >= 64 and h >= 16 else 0), k, bits, seed=w * 3 + k + bits)


@pytest.mark.parametrize("bits", [11, 8])
@pytest.mark.parametrize("kind", ["zeros", "ones", "checker", "random", "impulse"])
def test_packed_special_images(orc, b, kind, bits):
    """checkerboard and random bytes push AC coefficients past the 8-bit field (clamped, K1); the round trip stays exact (K3)"""
    for c in (1, 3, 4):
        check(orc, b, synth.special(kind, 96, 32, c, seed=c), 9, bits, seed=17)


def test_packed_verify_flags(orc, b):
    img = synth.image(264, 64, 3, seed=23, rectangles=2)
    d_img, priv, pub, dg, key, nonce = check(orc, b, img, 5, 11, seed=23)
    q2 = pub.clone(); q2[999] ^= 0x10
    rec, fl = b.defragment_dct_packed(priv, q2, 264, 64, 3, 5, 11, key, nonce, expected=dg)
    assert int(fl.item()) == 2 and int((rec != d_img).sum().item()) == 1
    p2 = priv.clone(); p2[70] ^= 0x01
    rec, fl = b.defragment_dct_packed(p2, pub, 264, 64, 3, 5, 11, key, nonce, expected=dg)
    assert int(fl.item()) == 1 and not torch.equal(rec, d_img)


@pytest.mark.parametrize("w,h,k,bits", [(264, 40, 5, 11), (320, 40, 3, 8)])   # thread-per-group kernels; tile kernels
def test_packed_batch_equals_singles(orc, b, w, h, k, bits):
    n, c = 4, 3
    key, nonce = synth.key_nonce(37)
    batch = b.PackedBatch(n, w, h, c, k, bits)
    nonces = synth.batch_nonces(nonce, n, priv_bytes=batch.priv_bytes)
    imgs = np.stack([synth.image(w, h, c, seed=500 + i, rectangles=1) for i in range(n)])
    d_imgs, d_non = torch.from_numpy(imgs).cuda(), torch.from_numpy(nonces).cuda()
    batch.fragment(d_imgs, key, d_non)
    torch.cuda.synchronize()
    for i in range(n):
        priv, pub, dg = b.fragment_dct_packed(d_imgs[i].contiguous(), k, bits, key, nonces[i].tobytes())
        assert torch.equal(batch.priv[i * batch.priv_stride:i * batch.priv_stride + batch.priv_bytes], priv)
        assert torch.equal(batch.pub[i * batch.pub_stride:i * batch.pub_stride + batch.pub_bytes], pub)
        assert torch.equal(batch.digests[64 * i:64 * i + 64], dg)
    out = torch.zeros_like(d_imgs)
    batch.defragment(out, key, d_non, expected=batch.digests)
    assert torch.equal(out, d_imgs) and int(batch.flags_out.abs().sum().item()) == 0
    batch.priv[1 * batch.priv_stride + 3] ^= 2
    batch.defragment(out, key, d_non, expected=batch.digests)
    assert batch.flags_out.cpu().tolist() == [0, 1, 0, 0]


def test_packed_full_hd_image_and_overheads(orc, b):
    """one 1920x1080 RGB image, k = 5: private = 12.9 % (11-bit) / 9.96 % (8-bit) of the image, stage (ii) on the whole image"""
    img = synth.image(1920, 1080, 3, seed=8, rectangles=8)
    for bits, frac in ((11, 11 * 6 / 64 / 8), (8, 5 / 64 + 11 / 8 / 64)):
        d_img, priv, pub, dg, key, nonce = check(orc, b, img, 5, bits, seed=8)
        assert priv.numel() / img.size == pytest.approx(frac, abs=1e-9)


def test_packed_config3_batch_full_size(orc, b):
    """BASELINE config 3 (256 x 1920x1080 RGB, k = 3) through the packed 11-bit storage, in the launch configuration bench.py
    times (feds_*_dct_packed_batch, tile kernels with 148 persistent CTAs): every image comes back exactly with no flag raised;
    a sample of images -- first, last and six in between -- goes through stages (i) and (ii) against the oracle on host threads."""
    from concurrent.futures import ThreadPoolExecutor
    n, w, h, c, k, bits = 256, 1920, 1080, 3, 3, 11
    key, nonce = synth.key_nonce(33)
    batch = b.PackedBatch(n, w, h, c, k, bits)
    nonces = synth.batch_nonces(nonce, n, priv_bytes=batch.priv_bytes)
    d_non = torch.from_numpy(nonces).cuda()
    d_imgs = synth.image_batch_torch(n, w, h, c, seed=3300, device="cuda", rectangles=8)
    batch.fragment(d_imgs, key, d_non)
    out = torch.zeros_like(d_imgs)
    batch.defragment(out, key, d_non, expected=batch.digests)
    torch.cuda.synchronize()
    assert torch.equal(out, d_imgs) and int(batch.flags_out.abs().sum().item()) == 0
    M = (1 << (bits - 1)) - 1

    def one(i):
        img = d_imgs[i].cpu().numpy()
        pv = batch.priv[i * batch.priv_stride:i * batch.priv_stride + batch.priv_bytes].cpu().numpy()
        pb = batch.pub[i * batch.pub_stride:i * batch.pub_stride + batch.pub_bytes].cpu().numpy()
        q = gpu_integers(orc, pv, w, h, c, k, bits, key, nonces[i].tobytes())
        ref = orc.dct_coefficients(img)[:, :k + 1].copy()
        ref[:, 0] = np.clip(ref[:, 0], 0, 2047)
        ref[:, 1:] = np.clip(ref[:, 1:], -M, M)
        assert np.abs(q - ref).max() <= 0.5 + 1e-3, i
        p2, q2, d2 = orc.fragment_packed_from_q(img, q, k, bits, key, nonces[i].tobytes())
        assert (p2 == pv).all() and (q2 == pb).all() and d2 == batch.digests[64 * i:64 * i + 64].cpu().numpy().tobytes(), i
        return i

    sample = [0, 37, 74, 111, 148, 185, 222, 255]
    with ThreadPoolExecutor(8) as ex:
        assert sorted(ex.map(one, sample)) == sample
    batch.pub[200 * batch.pub_stride + 77] ^= 1
    batch.defragment(out, key, d_non, expected=batch.digests)
    want = [0] * n
    want[200] = 2
    assert batch.flags_out.cpu().tolist() == want
