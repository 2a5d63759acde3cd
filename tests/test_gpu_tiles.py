"""GPU parity of the report's tiled DWT design (feds_fragment_dwt_tiles / feds_defragment_dwt_tiles; PAPER.md 6.9.3-6.9.4, P:788-822;
DESIGN.md 2.5) through the C ABI against the oracle (oracle/feds_oracle_tiled.c). Everything is integer arithmetic, AES, SHA-256 and
SHA-512: one correct result, compared bit for bit in one stage -- private fragment, public fragment, digests, reconstruction."""
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


def run_case(orc, b, img, seed):
    h, w, c = img.shape
    key, nonce = synth.key_nonce(seed)
    d_img = torch.from_numpy(img).cuda()
    priv, pub, dg = b.fragment_dwt_tiles(d_img, key, nonce)
    torch.cuda.synchronize()
    op, oq, odg = orc.fragment_tiled(img, key, nonce)
    assert priv.numel() == orc.tiled_private_bytes(w, h, c) and pub.numel() == orc.tiled_public_bytes(w, h, c)
    T = (w // 8) * (h // 8) * c
    pv = priv.cpu().numpy()
    assert (pv[:16 * T] == op[:16 * T]).all(), "level 2 (SHA-256 keystream) differs"
    assert (pv[16 * T:] == op[16 * T:]).all(), "level 1 (AES-CTR) differs"
    assert (pub.cpu().numpy() == oq).all(), "level 3 (SHA-512 keystream) differs"
    assert dg.cpu().numpy().tobytes() == odg, "digests differ"
    rec, flags = b.defragment_dwt_tiles(priv, pub, w, h, c, key, nonce, expected=dg)
    torch.cuda.synchronize()
    assert int(flags.item()) == 0 and torch.equal(rec, d_img)          # recovered "without any error"
    rec2, _ = b.defragment_dwt_tiles(priv, pub, w, h, c, key, nonce)
    assert torch.equal(rec2, d_img)
    return d_img, priv, pub, dg, key, nonce


@pytest.mark.parametrize("w,h,c", [(8, 8, 1), (16, 8, 1), (64, 32, 1), (48, 80, 3), (272, 144, 1), (136, 72, 3), (512, 512, 1), (1024, 320, 3),
                                   (128, 64, 4), (2056, 8, 1), (1920, 1080, 3)])
def test_tiles_parity_and_round_trip(orc, b, w, h, c):
    run_case(orc, b, synth.image(w, h, c, seed=w + h, rectangles=2 if min(w, h) >= 32 else 0), seed=w + c)


@pytest.mark.parametrize("kind", ["zeros", "ones", "checker", "random", "impulse"])
def test_tiles_special_images(orc, b, kind):
    """checkerboards and random bytes ("any kind of data ... every byte as a pixel") drive the coefficients to the ends of their
    10/11-bit fields"""
    for c in (1, 3, 4):
        run_case(orc, b, synth.special(kind, 160, 96, c, seed=c), seed=5)


def test_tiles_extreme_tiles_fit_their_fields(orc, b):
    """an image made of the adversarial tiles of the range search (every pixel 0 or 255): bit-exact, exact round trip"""
    rng = np.random.default_rng(7)
    img = rng.choice([0, 255], size=(64, 512, 1)).astype(np.uint8)
    run_case(orc, b, img, seed=11)


def test_tiles_verify_flags_and_nonce_carry(orc, b):
    img = synth.image(256, 128, 3, seed=9)
    d_img, priv, pub, dg, key, nonce = run_case(orc, b, img, seed=9)
    T = 32 * 16 * 3
    p2 = priv.clone(); p2[16 * T + 7] ^= 1          # a level-1 byte: AES section
    _, fl = b.defragment_dwt_tiles(p2, pub, 256, 128, 3, key, nonce, expected=dg)
    assert int(fl.item()) == 1
    q2 = pub.clone(); q2[-2] ^= 0x10
    rec, fl = b.defragment_dwt_tiles(priv, q2, 256, 128, 3, key, nonce, expected=dg)
    assert int(fl.item()) == 2
    bad = (rec != d_img).any(dim=2).cpu().numpy()
    assert bad.any() and not bad[:120, :].any() and not bad[:, :248].any()       # confined to the last tile
    # a nonce whose low 64 bits are about to wrap: the 128-bit counter carries, the IV of the keystream hashes is the same 16 bytes
    d2 = torch.from_numpy(img).cuda()
    nonce2 = bytes([1] * 8 + [0xFF] * 8)
    pr, pb_, dg2 = b.fragment_dwt_tiles(d2, key, nonce2)
    op, oq, odg = orc.fragment_tiled(img, key, nonce2)
    assert (pr.cpu().numpy() == op).all() and (pb_.cpu().numpy() == oq).all() and dg2.cpu().numpy().tobytes() == odg


def test_tiles_batch_equals_oracle_per_image(orc, b):
    n, w, h, c = 3, 272, 48, 3
    key, nonce = synth.key_nonce(41)
    batch = b.TilesBatch(n, w, h, c)
    nonces = synth.batch_nonces(nonce, n, priv_bytes=batch.priv_bytes)
    imgs = np.stack([synth.image(w, h, c, seed=700 + i, rectangles=1) for i in range(n)])
    d_imgs, d_non = torch.from_numpy(imgs).cuda(), torch.from_numpy(nonces).cuda()
    batch.fragment(d_imgs, key, d_non)
    torch.cuda.synchronize()
    for i in range(n):
        op, oq, odg = orc.fragment_tiled(imgs[i], key, nonces[i].tobytes())
        assert (batch.priv[i * batch.priv_stride:i * batch.priv_stride + batch.priv_bytes].cpu().numpy() == op).all(), i
        assert (batch.pub[i * batch.pub_stride:i * batch.pub_stride + batch.pub_bytes].cpu().numpy() == oq).all(), i
        assert batch.digests[64 * i:64 * i + 64].cpu().numpy().tobytes() == odg, i
    out = torch.zeros_like(d_imgs)
    batch.defragment(out, key, d_non, expected=batch.digests)
    assert torch.equal(out, d_imgs) and int(batch.flags_out.abs().sum().item()) == 0
    batch.pub[1 * batch.pub_stride + 9] ^= 4
    batch.defragment(out, key, d_non, expected=batch.digests)
    assert batch.flags_out.cpu().tolist() == [0, 2, 0]


def test_tiles_config4_full_size(orc, b):
    """8192 x 8192 gray (BASELINE config 4) through the batch entry points bench.py times for this design: both fragments and the
    digests are the oracle's, bit for bit; the image comes back exactly; a flipped bit in either fragment raises its flag."""
    w = h = 8192
    img = synth.image(w, h, 1, seed=44)
    key, nonce = synth.key_nonce(44)
    batch = b.TilesBatch(1, w, h, 1)
    d_img = torch.from_numpy(img).cuda()
    d_non = torch.frombuffer(bytearray(nonce), dtype=torch.uint8).cuda().view(1, 16)
    batch.fragment(d_img, key, d_non)
    torch.cuda.synchronize()
    op, oq, odg = orc.fragment_tiled(img, key, nonce)
    assert (batch.priv[:batch.priv_bytes].cpu().numpy() == op).all() and (batch.pub[:batch.pub_bytes].cpu().numpy() == oq).all()
    assert batch.digests.cpu().numpy().tobytes() == odg
    out = torch.zeros_like(d_img)
    batch.defragment(out, key, d_non, expected=batch.digests)
    torch.cuda.synchronize()
    assert torch.equal(out, d_img) and batch.flags_out.cpu().tolist() == [0]
    batch.pub[batch.pub_bytes - 1] ^= 0x80
    batch.priv[0] ^= 1
    batch.defragment(out, key, d_non, expected=batch.digests)
    assert batch.flags_out.cpu().tolist() == [3]
