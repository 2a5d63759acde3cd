"""GPU parity tests for the DWT path through the C ABI. Everything is integer: coefficients, ciphertext, digests and the
reconstruction are bit-exact against the oracle in one stage."""
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


def run_case(orc, b, img, L, seed):
    h, w, c = img.shape
    key, nonce = synth.key_nonce(seed)
    d_img = torch.from_numpy(img).cuda()
    priv, pub, dg = b.fragment_dwt(d_img, L, key, nonce)
    torch.cuda.synchronize()
    op, oq, odg = orc.fragment_dwt(img, L, key, nonce)
    assert (priv.cpu().numpy() == op).all(), "private (LL ciphertext) differs"
    assert (pub.cpu().numpy() == oq).all(), "public subbands differ"
    assert dg.cpu().numpy().tobytes() == odg, "digests differ"
    rec, flags = b.defragment_dwt(priv, pub, w, h, c, L, key, nonce, expected=dg)
    torch.cuda.synchronize()
    assert int(flags.item()) == 0 and torch.equal(rec, d_img)      # recovered "without any error"
    rec2, _ = b.defragment_dwt(priv, pub, w, h, c, L, key, nonce)
    assert torch.equal(rec2, d_img)
    return d_img, priv, pub, dg, key, nonce


@pytest.mark.parametrize("w,h,c,L", [(2, 2, 1, 1), (16, 8, 1, 1), (64, 32, 1, 2), (48, 80, 3, 3), (272, 144, 1, 3), (136, 72, 3, 2),
                                     (512, 512, 1, 3), (1024, 320, 3, 4), (128, 64, 4, 6), (2048, 64, 1, 1), (64, 2048, 1, 5),
                                     (1032, 520, 1, 3)])
def test_dwt_parity_and_round_trip(orc, b, w, h, c, L):
    run_case(orc, b, synth.image(w, h, c, seed=w + h + L, rectangles=2 if min(w, h) >= 32 else 0), L, seed=w + L)


@pytest.mark.parametrize("kind", ["zeros", "ones", "checker", "random", "impulse"])
def test_dwt_special_images(orc, b, kind):
    for L in [1, 2, 3, 4]:
        run_case(orc, b, synth.special(kind, 160, 96, 3, seed=L), L, seed=5)


def test_dwt_verify_flags(orc, b):
    img = synth.image(256, 128, 3, seed=9)
    d_img, priv, pub, dg, key, nonce = run_case(orc, b, img, 3, seed=9)
    p2 = priv.clone(); p2[0] ^= 1
    _, flags = b.defragment_dwt(p2, pub, 256, 128, 3, 3, key, nonce, expected=dg)
    assert int(flags.item()) == 1
    q2 = pub.clone(); q2[-2] ^= 0x10
    _, flags = b.defragment_dwt(priv, q2, 256, 128, 3, 3, key, nonce, expected=dg)
    assert int(flags.item()) == 2
    # the same check without the key (feds_verify_dwt)
    assert int(b.verify_dwt(priv, pub, 256, 128, 3, 3, dg).item()) == 0
    assert int(b.verify_dwt(p2, pub, 256, 128, 3, 3, dg).item()) == 1
    assert int(b.verify_dwt(priv, q2, 256, 128, 3, 3, dg).item()) == 2
    assert int(b.verify_dwt(p2, q2, 256, 128, 3, 3, dg).item()) == 3


def test_config4_full_size(orc, b):
    """8192x8192 grayscale, 3 levels (BASELINE config 4): bit-exact on everything."""
    run_case(orc, b, synth.image(8192, 8192, 1, seed=4), 3, seed=4)


@pytest.mark.parametrize("w,h,c,L", [(1024, 320, 3, 4), (2048, 64, 1, 1), (7696, 96, 1, 2), (496, 80, 3, 1)])
def test_streaming_and_tiled_level_kernels_agree(orc, b, w, h, c, L, monkeypatch):
    """The register-streaming level kernels (several column strips, halo lanes, row tiles) and the tiled shared-memory
    kernels they replace on aligned sizes compute identical fragments; the oracle decides which is right."""
    img = synth.image(w, h, c, seed=w + L)
    key, nonce = synth.key_nonce(w)
    d_img = torch.from_numpy(img).cuda()
    fast = b.fragment_dwt(d_img, L, key, nonce)
    monkeypatch.setenv("FEDS_DWT_TILED", "1")
    tiled = b.fragment_dwt(d_img, L, key, nonce)
    rec_tiled, _ = b.defragment_dwt(fast[0], fast[1], w, h, c, L, key, nonce)
    monkeypatch.delenv("FEDS_DWT_TILED")
    rec_fast, _ = b.defragment_dwt(tiled[0], tiled[1], w, h, c, L, key, nonce)
    torch.cuda.synchronize()
    for x, y in zip(fast, tiled):
        assert torch.equal(x, y)
    op, oq, odg = orc.fragment_dwt(img, L, key, nonce)
    assert (fast[0].cpu().numpy() == op).all() and (fast[1].cpu().numpy() == oq).all() and fast[2].cpu().numpy().tobytes() == odg
    assert torch.equal(rec_tiled, d_img) and torch.equal(rec_fast, d_img)
