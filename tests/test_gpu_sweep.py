"""GPU parity over BASELINE configs[4] (the sweep): square RGB images, DCT k in {0, 2, 5, 9}, DWT levels in {1, 2, 3, 4}.
Sizes up to 2048^2: full parity for every (k | L); 4096^2: fragments and digests through the oracle's byte-level stages
(SURVEY.md 8(d), table row 5). The larger sweep sizes differ from these only in the number of leaf groups per warp."""
import numpy as np
import pytest
import torch

import synth

pytestmark = pytest.mark.gpu
TOL = 1e-3   # BASELINE north_star: max abs coefficient error, FP32 kernel against the double oracle


@pytest.fixture(scope="module")
def b():
    from paper_1512_02951_b200 import binding
    assert torch.cuda.is_available()
    return binding


def _coef(orc, priv, pub, nb, k, key, nonce):
    pt = np.frombuffer(orc.aes128_ctr_xor(key, nonce, priv.tobytes()), dtype="<f4").reshape(nb, k + 1)
    return np.concatenate([pt, np.frombuffer(pub.tobytes(), dtype="<f4").reshape(nb, 63 - k)], axis=1)


@pytest.mark.parametrize("size", [256, 512, 1024, 2048, 4096])
@pytest.mark.parametrize("k", [0, 2, 5, 9])
def test_sweep_dct(orc, b, size, k):
    w = h = size
    c = 3
    img = synth.image(w, h, c, seed=size + k)
    key, nonce = synth.key_nonce(size + k)
    d_img = torch.from_numpy(img).cuda()
    priv, pub, dg = b.fragment_dct(d_img, k, key, nonce)
    rec, flags = b.defragment_dct(priv, pub, w, h, c, k, key, nonce, expected=dg)
    torch.cuda.synchronize()
    assert int(flags.item()) == 0 and torch.equal(rec, d_img)                      # stage (iii): exact uint8 round trip
    nb = c * (h // 8) * (w // 8)
    pv, pb = priv.cpu().numpy(), pub.cpu().numpy()
    coef = _coef(orc, pv, pb, nb, k, key, nonce)
    p2, q2, d2 = orc.fragment_from_coef32(coef, w, h, c, k, key, nonce)            # stage (ii): bytes and digests bit-exact
    assert (p2 == pv).all() and (q2 == pb).all() and d2 == dg.cpu().numpy().tobytes()
    # stage (i): coefficients against the double oracle -- whole image up to 1024^2, three 64x64 crops above
    if size <= 1024:
        assert np.abs(coef - orc.dct_coefficients(img)).max() <= TOL
    else:
        c4 = coef.reshape(c, h // 8, w // 8, 64)
        rng = np.random.default_rng(size)
        for _ in range(3):
            by, bx = int(rng.integers(0, h // 8 - 8)), int(rng.integers(0, w // 8 - 8))
            ref = orc.dct_coefficients(np.ascontiguousarray(img[8 * by:8 * by + 64, 8 * bx:8 * bx + 64, :])).reshape(c, 8, 8, 64)
            assert np.abs(c4[:, by:by + 8, bx:bx + 8, :] - ref).max() <= TOL
    if size <= 1024:   # cross round trip: the oracle reconstructs from the GPU's fragments
        rec2, fl2 = orc.defragment_dct(pv, pb, w, h, c, k, key, nonce, expected=dg.cpu().numpy().tobytes())
        assert fl2 == 0 and (rec2 == img).all()


@pytest.mark.parametrize("size", [256, 512, 1024, 2048, 4096])
@pytest.mark.parametrize("levels", [1, 2, 3, 4])
def test_sweep_dwt(orc, b, size, levels):
    w = h = size
    c = 3
    img = synth.image(w, h, c, seed=size + levels)
    key, nonce = synth.key_nonce(size + 10 * levels)
    d_img = torch.from_numpy(img).cuda()
    priv, pub, dg = b.fragment_dwt(d_img, levels, key, nonce)
    rec, flags = b.defragment_dwt(priv, pub, w, h, c, levels, key, nonce, expected=dg)
    torch.cuda.synchronize()
    assert int(flags.item()) == 0 and torch.equal(rec, d_img)
    op, oq, odg = orc.fragment_dwt(img, levels, key, nonce)                        # all-integer path: one stage, bit-exact
    assert (priv.cpu().numpy() == op).all() and (pub.cpu().numpy() == oq).all() and dg.cpu().numpy().tobytes() == odg
