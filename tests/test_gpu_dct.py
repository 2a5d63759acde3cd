"""GPU parity tests for the DCT path, through the C ABI (paper_1512_02951_b200.binding), against the CPU oracle.

Two-stage protocol:
  (i)   GPU coefficients (private part decrypted with the known key) vs the oracle's DOUBLE coefficients: max abs <= 1e-3
        (BASELINE.json north_star tolerance: FP32 against the double oracle, 8-bit inputs);
  (ii)  the oracle's pack + AES-CTR + SHA-256/Merkle fed the GPU's own float32 coefficient bytes: private ciphertext, public
        bytes and both digests bit-exact;
  (iii) reconstructions bit-exact uint8: GPU(GPU), oracle(GPU fragments), GPU(oracle fragments).
"""
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


def gpu_coefficients(orc, priv, pub, nb, k, key, nonce):
    """float32 [nb][64] zigzag-ordered coefficients recovered from the GPU fragments."""
    pt = np.frombuffer(orc.aes128_ctr_xor(key, nonce, priv.tobytes()), dtype="<f4").reshape(nb, k + 1)
    pu = np.frombuffer(pub.tobytes(), dtype="<f4").reshape(nb, 63 - k)
    return np.concatenate([pt, pu], axis=1)


def check_fragment_parity(orc, b, img, k, seed, check_coefficients=True):
    h, w, c = img.shape
    key, nonce = synth.key_nonce(seed)
    d_img = torch.from_numpy(img).cuda()
    priv, pub, dg = b.fragment_dct(d_img, k, key, nonce)
    torch.cuda.synchronize()
    priv, pub, dg = priv.cpu().numpy(), pub.cpu().numpy(), dg.cpu().numpy().tobytes()
    nb = c * (h // 8) * (w // 8)
    assert priv.size == orc.dct_private_bytes(w, h, c, k) and pub.size == orc.dct_public_bytes(w, h, c, k)
    coef32 = gpu_coefficients(orc, priv, pub, nb, k, key, nonce)
    if check_coefficients:                                                  # stage (i)
        ref = orc.dct_coefficients(img)
        err = np.abs(coef32.astype(np.float64) - ref).max()
        assert err <= TOL, err
    p2, q2, d2 = orc.fragment_from_coef32(coef32, w, h, c, k, key, nonce)   # stage (ii)
    assert (p2 == priv).all(), "private ciphertext differs"
    assert (q2 == pub).all(), "public bytes differ"
    assert d2[:32] == dg[:32], "private digest differs"
    assert d2[32:] == dg[32:], "public digest differs"
    return d_img, priv, pub, dg, key, nonce


CASES = [
    (8, 8, 1, 0), (8, 8, 1, 63), (16, 16, 4, 63), (64, 8, 1, 3), (72, 24, 1, 5), (1080, 16, 3, 3), (136, 40, 4, 9),
    (512, 512, 1, 2),      # BASELINE config 1
    (256, 264, 3, 5), (1032, 8, 1, 2), (520, 24, 3, 31), (64, 64, 1, 32), (128, 16, 3, 62), (40, 8, 3, 4), (2056, 8, 1, 1),
]


@pytest.mark.parametrize("w,h,c,k", CASES)
def test_fragment_parity_and_round_trips(orc, b, w, h, c, k):
    img = synth.image(w, h, c, seed=w + 3 * h + c + k, rectangles=2 if w >= 64 and h >= 16 else 0)
    d_img, priv, pub, dg, key, nonce = check_fragment_parity(orc, b, img, k, seed=w * 7 + k)
    d_priv, d_pub = torch.from_numpy(priv).cuda(), torch.from_numpy(pub).cuda()
    if pub.size == 0:
        d_pub = torch.zeros(16, dtype=torch.uint8, device="cuda")
    d_dg = torch.frombuffer(bytearray(dg), dtype=torch.uint8).cuda()
    # (iii) GPU defragment of GPU fragments, with verification
    rec, flags = b.defragment_dct(d_priv, d_pub, w, h, c, k, key, nonce, expected=d_dg)
    torch.cuda.synchronize()
    assert int(flags.item()) == 0
    assert torch.equal(rec, d_img)
    # without verification
    rec2, _ = b.defragment_dct(d_priv, d_pub, w, h, c, k, key, nonce)
    assert torch.equal(rec2, d_img)
    # oracle defragment of GPU fragments
    orec, oflags = orc.defragment_dct(priv, pub, w, h, c, k, key, nonce, expected=dg)
    assert oflags == 0 and (orec == img).all()
    # GPU defragment of ORACLE fragments (whose coefficient bytes come from the double DCT)
    op, oq, odg = orc.fragment_dct(img, k, key, nonce)
    d_op = torch.from_numpy(op).cuda()
    d_oq = torch.from_numpy(oq).cuda() if oq.size else torch.zeros(16, dtype=torch.uint8, device="cuda")
    d_odg = torch.frombuffer(bytearray(odg), dtype=torch.uint8).cuda()
    rec3, flags3 = b.defragment_dct(d_op, d_oq, w, h, c, k, key, nonce, expected=d_odg)
    torch.cuda.synchronize()
    assert int(flags3.item()) == 0 and torch.equal(rec3, d_img)


@pytest.mark.parametrize("kind", ["zeros", "ones", "checker", "random", "impulse"])
@pytest.mark.parametrize("c", [1, 3, 4])
def test_special_images(orc, b, kind, c):
    img = synth.special(kind, 96, 32, c, seed=c)
    d_img, priv, pub, dg, key, nonce = check_fragment_parity(orc, b, img, 5, seed=11)
    rec, flags = b.defragment_dct(torch.from_numpy(priv).cuda(), torch.from_numpy(pub).cuda(), 96, 32, c, 5, key, nonce,
                                  expected=torch.frombuffer(bytearray(dg), dtype=torch.uint8).cuda())
    torch.cuda.synchronize()
    assert int(flags.item()) == 0 and torch.equal(rec, d_img)   # T6: lossless


def test_dc_bound_on_device(orc, b):
    img = np.full((8, 64, 1), 255, dtype=np.uint8)
    key, nonce = synth.key_nonce(1)
    priv, pub, _ = b.fragment_dct(torch.from_numpy(img).cuda(), 0, key, nonce)
    dc = np.frombuffer(orc.aes128_ctr_xor(key, nonce, priv.cpu().numpy().tobytes()), dtype="<f4")
    assert np.abs(dc - 2040.0).max() < 1e-3
    assert np.abs(np.frombuffer(pub.cpu().numpy().tobytes(), dtype="<f4")).max() < 1e-3


def test_verify_flags_and_error_confinement(orc, b):
    w, h, c, k = 128, 32, 1, 3
    img = synth.image(w, h, c, seed=6)
    key, nonce = synth.key_nonce(6)
    d_img = torch.from_numpy(img).cuda()
    priv, pub, dg = b.fragment_dct(d_img, k, key, nonce)
    p2 = priv.clone(); p2[99] ^= 0x40          # top byte of block 6's DC
    rec, flags = b.defragment_dct(p2, pub, w, h, c, k, key, nonce, expected=dg)
    assert int(flags.item()) == 1
    diff = (rec != d_img)[:, :, 0].cpu().numpy()
    mask = np.zeros_like(diff); mask[0:8, 48:56] = True
    assert diff[mask].any() and not diff[~mask].any()            # CTR: damage confined to one 8x8 block
    q2 = pub.clone(); q2[-1] ^= 1
    _, flags = b.defragment_dct(priv, q2, w, h, c, k, key, nonce, expected=dg)
    assert int(flags.item()) == 2
    _, flags = b.defragment_dct(p2, q2, w, h, c, k, key, nonce, expected=dg)
    assert int(flags.item()) == 3
    bad, _ = b.defragment_dct(priv, pub, w, h, c, k, bytes(16), nonce)
    assert (bad != d_img).float().mean().item() > 0.5            # wrong key does not reconstruct


@pytest.mark.parametrize("w,h,c,k", [(264, 48, 3, 3), (72, 8, 1, 0), (1032, 16, 1, 5), (136, 24, 4, 63), (2048, 16, 3, 9)])
def test_verify_without_key(orc, b, w, h, c, k):
    """feds_verify_dct: a fragment holder checks integrity against the digest pair with no key (A8); every single
    flipped byte of either fragment is confined to its own flag bit."""
    img = synth.image(w, h, c, seed=w + k)
    key, nonce = synth.key_nonce(w + 1)
    priv, pub, dg = b.fragment_dct(torch.from_numpy(img).cuda(), k, key, nonce)
    # the digests are the oracle's for these stored bytes
    assert dg.cpu().numpy().tobytes() == orc.fragment_from_coef32(
        gpu_coefficients(orc, priv.cpu().numpy(), pub.cpu().numpy(), c * (h // 8) * (w // 8), k, key, nonce), w, h, c, k, key, nonce)[2]
    assert int(b.verify_dct(priv, pub, w, h, c, k, dg).item()) == 0
    rng = np.random.default_rng(w)
    for _ in range(4):
        p2 = priv.clone()
        p2[int(rng.integers(0, priv.numel()))] ^= 1 << int(rng.integers(0, 8))
        assert int(b.verify_dct(p2, pub, w, h, c, k, dg).item()) == 1
        if pub.numel() > 16 and k < 63:
            q2 = pub.clone()
            q2[int(rng.integers(0, b.dct_public_bytes(w, h, c, k)))] ^= 1 << int(rng.integers(0, 8))
            assert int(b.verify_dct(priv, q2, w, h, c, k, dg).item()) == 2
    d2 = dg.clone(); d2[40] ^= 4
    assert int(b.verify_dct(priv, pub, w, h, c, k, d2).item()) == 2


def test_counter_carry_on_device(orc, b):
    # nonce just below the 32-bit and 64-bit carry boundaries (A6)
    img = synth.image(64, 32, 1, seed=8)
    key, _ = synth.key_nonce(8)
    for nonce in [bytes.fromhex("000000000000000000000000fffffffe"), bytes.fromhex("0000000000000000fffffffffffffffe"),
                  bytes.fromhex("fffffffffffffffffffffffffffffffd")]:
        priv, pub, dg = b.fragment_dct(torch.from_numpy(img).cuda(), 3, key, nonce)
        coef = gpu_coefficients(orc, priv.cpu().numpy(), pub.cpu().numpy(), 32, 3, key, nonce)
        p2, q2, d2 = orc.fragment_from_coef32(coef, 64, 32, 1, 3, key, nonce)
        assert (p2 == priv.cpu().numpy()).all() and d2 == dg.cpu().numpy().tobytes()
        assert np.abs(coef - orc.dct_coefficients(img)).max() <= TOL


def test_batch_equals_singles(orc, b):
    n, w, h, c, k = 5, 136, 24, 3, 3
    key, nonce = synth.key_nonce(21)
    nonces = synth.batch_nonces(nonce, n)
    imgs = np.stack([synth.image(w, h, c, seed=100 + i, rectangles=1) for i in range(n)])
    d_imgs = torch.from_numpy(imgs).cuda()
    batch = b.DctBatch(n, w, h, c, k)
    d_nonces = torch.from_numpy(nonces).cuda()
    batch.fragment(d_imgs, key, d_nonces)
    torch.cuda.synchronize()
    for i in range(n):
        pv, pb, dg = b.fragment_dct(d_imgs[i].contiguous(), k, key, nonces[i].tobytes())
        assert torch.equal(pv, batch.priv[i * batch.priv_bytes:(i + 1) * batch.priv_bytes])
        assert torch.equal(pb, batch.pub[i * batch.pub_bytes:(i + 1) * batch.pub_bytes])
        assert torch.equal(dg, batch.digests[64 * i:64 * i + 64])
    out = torch.empty_like(d_imgs)
    batch.defragment(out, key, d_nonces, expected=batch.digests)
    torch.cuda.synchronize()
    assert torch.equal(out, d_imgs) and int(batch.flags_out.abs().sum().item()) == 0
    batch.pub[batch.pub_bytes * 3 + 5] ^= 0x80
    batch.defragment(out, key, d_nonces, expected=batch.digests)
    assert batch.flags_out.cpu().tolist() == [0, 0, 0, 2, 0]
    batch.flags_out.zero_()
    assert batch.verify().cpu().tolist() == [0, 0, 0, 2, 0]
    # no-digest flag: same fragment bytes, digests untouched
    batch2 = b.DctBatch(n, w, h, c, k)
    batch2.digests.fill_(7)
    batch2.fragment(d_imgs, key, d_nonces, flags=b.FLAG_NO_DIGEST)
    torch.cuda.synchronize()
    batch.pub[batch.pub_bytes * 3 + 5] ^= 0x80
    assert torch.equal(batch2.priv, batch.priv) and torch.equal(batch2.pub, batch.pub) and bool((batch2.digests == 7).all())


def test_host_staged_entry_point(orc, b):
    n, w, h, c, k = 7, 64, 32, 3, 3
    key, nonce = synth.key_nonce(31)
    nonces = synth.batch_nonces(nonce, n)
    imgs = np.stack([synth.image(w, h, c, seed=200 + i) for i in range(n)])
    h_imgs = torch.from_numpy(imgs).pin_memory()
    h_non = torch.from_numpy(nonces).pin_memory()
    pb_, qb_ = b.dct_private_bytes(w, h, c, k), b.dct_public_bytes(w, h, c, k)
    h_priv = torch.empty(n * pb_, dtype=torch.uint8).pin_memory()
    h_pub = torch.empty(n * qb_, dtype=torch.uint8).pin_memory()
    h_dg = torch.empty(n * 64, dtype=torch.uint8).pin_memory()
    streams = [torch.cuda.Stream() for _ in range(3)]
    scratch = torch.empty(b.host_scratch_bytes(2, 3, w, h, c, k), dtype=torch.uint8, device="cuda")
    b.fragment_dct_host(h_imgs, w, h, c, k, key, h_non, h_priv, h_pub, h_dg, 2, scratch, streams)
    for s in streams:
        s.synchronize()
    for i in range(n):
        pv, pu, dg = b.fragment_dct(torch.from_numpy(imgs[i]).cuda(), k, key, nonces[i].tobytes())
        assert (pv.cpu() == h_priv[i * pb_:(i + 1) * pb_]).all() and (pu.cpu() == h_pub[i * qb_:(i + 1) * qb_]).all()
        assert (dg.cpu() == h_dg[64 * i:64 * i + 64]).all()


def test_host_staged_calls_interleaved_without_sync(orc, b):
    """fragment and verified defragment of sub-batches alternately on the same streams and the same scratch, no
    synchronisation until the end (bench.py's e2e pattern): both calls must see the same scratch slot per stream."""
    n, w, h, c, k = 26, 264, 48, 3, 3
    ipc, ns = 2, 3
    key, nonce = synth.key_nonce(41)
    nonces = synth.batch_nonces(nonce, n)
    imgs = np.stack([synth.image(w, h, c, seed=300 + i) for i in range(n)])
    ib, pb_, qb_ = w * h * c, b.dct_private_bytes(w, h, c, k), b.dct_public_bytes(w, h, c, k)
    h_imgs = torch.from_numpy(imgs).view(-1).pin_memory()
    h_non = torch.from_numpy(nonces).pin_memory()
    h_priv = torch.zeros(n * pb_, dtype=torch.uint8).pin_memory()
    h_pub = torch.zeros(n * qb_, dtype=torch.uint8).pin_memory()
    h_dg = torch.zeros(n * 64, dtype=torch.uint8).pin_memory()
    h_out = torch.zeros(n * ib, dtype=torch.uint8).pin_memory()
    h_fl = torch.full((n,), 7, dtype=torch.int32).pin_memory()
    assert b.host_scratch_bytes(ipc, ns, w, h, c, k) == b.defrag_host_scratch_bytes(ipc, ns, w, h, c, k)
    scratch = torch.empty(b.host_scratch_bytes(ipc, ns, w, h, c, k), dtype=torch.uint8, device="cuda")
    streams = [torch.cuda.Stream() for _ in range(ns)]
    sub = ipc * ns
    for a in range(0, n, sub):
        m = min(sub, n - a)
        b.fragment_dct_host(h_imgs[a * ib:(a + m) * ib], w, h, c, k, key, h_non[a:a + m], h_priv[a * pb_:(a + m) * pb_],
                            h_pub[a * qb_:(a + m) * qb_], h_dg[64 * a:64 * (a + m)], ipc, scratch, streams)
        b.defragment_dct_host(h_priv[a * pb_:(a + m) * pb_], h_pub[a * qb_:(a + m) * qb_], m, w, h, c, k, key, h_non[a:a + m],
                              h_dg[64 * a:64 * (a + m)], h_out[a * ib:(a + m) * ib], h_fl[a:a + m], ipc, scratch, streams)
    for s in streams:
        s.synchronize()
    assert torch.equal(h_out, h_imgs) and int(h_fl.abs().sum().item()) == 0
    # fragments on the host are the ones the device-resident call produces
    for i in [0, 5, 13, 25]:
        pv, pu, dg = b.fragment_dct(torch.from_numpy(imgs[i]).cuda(), k, key, nonces[i].tobytes())
        assert (pv.cpu() == h_priv[i * pb_:(i + 1) * pb_]).all() and (pu.cpu() == h_pub[i * qb_:(i + 1) * qb_]).all()
        assert (dg.cpu() == h_dg[64 * i:64 * i + 64]).all()


# ---------------------------------------------------------------- full BASELINE sizes, in the configuration bench.py times
def test_config2_full_size(orc, b):
    """4096x4096 RGB, k=5: whole-image stage (ii) + round trip; coefficients on sampled crops (the double DCT is slow)."""
    w = h = 4096; c = 3; k = 5
    img = synth.image(w, h, c, seed=2)
    d_img, priv, pub, dg, key, nonce = check_fragment_parity(orc, b, img, k, seed=2, check_coefficients=False)
    nb = c * (h // 8) * (w // 8)
    coef = gpu_coefficients(orc, priv, pub, nb, k, key, nonce).reshape(c, h // 8, w // 8, 64)
    rng = np.random.default_rng(0)
    for _ in range(6):
        by, bx = int(rng.integers(0, h // 8 - 8)), int(rng.integers(0, w // 8 - 8))
        crop = np.ascontiguousarray(img[8 * by:8 * by + 64, 8 * bx:8 * bx + 64, :])
        ref = orc.dct_coefficients(crop).reshape(c, 8, 8, 64)
        assert np.abs(coef[:, by:by + 8, bx:bx + 8, :] - ref).max() <= TOL
    rec, flags = b.defragment_dct(torch.from_numpy(priv).cuda(), torch.from_numpy(pub).cuda(), w, h, c, k, key, nonce,
                                  expected=torch.frombuffer(bytearray(dg), dtype=torch.uint8).cuda())
    torch.cuda.synchronize()
    assert int(flags.item()) == 0 and torch.equal(rec, d_img)


def test_config3_batch_full_size(orc, b):
    """256 x 1920x1080 RGB, k=3, batched as bench.py launches it. Stage (ii) -- ciphertext, public bytes and both digests through
    the oracle's pack + AES-CTR + SHA-256 -- on ALL 256 images, the oracle calls spread over host threads
    (ctypes releases the GIL); stage (i) on a crop of every 8th image; then the exact round trip of the whole batch."""
    from concurrent.futures import ThreadPoolExecutor
    n, w, h, c, k = 256, 1920, 1080, 3, 3
    key, nonce = synth.key_nonce(3)
    nonces = synth.batch_nonces(nonce, n)
    d_imgs = synth.image_batch_torch(n, w, h, c, seed=3000, device="cuda", rectangles=16)
    d_nonces = torch.from_numpy(nonces).cuda()
    batch = b.DctBatch(n, w, h, c, k)
    batch.fragment(d_imgs, key, d_nonces)
    torch.cuda.synchronize()
    nb = c * (h // 8) * (w // 8)
    dgs = batch.digests.cpu().numpy().reshape(n, 64)

    def one(i, priv, pub, img):
        nz = nonces[i].tobytes()
        coef = gpu_coefficients(orc, priv, pub, nb, k, key, nz)
        p2, q2, d2 = orc.fragment_from_coef32(coef, w, h, c, k, key, nz)
        assert (p2 == priv).all() and (q2 == pub).all() and d2 == dgs[i].tobytes(), i
        if img is not None:
            crop = np.ascontiguousarray(img[512:576, 960:1024, :])
            ref = orc.dct_coefficients(crop).reshape(c, 8, 8, 64)
            assert np.abs(coef.reshape(c, h // 8, w // 8, 64)[:, 64:72, 120:128, :] - ref).max() <= TOL, i
        return i

    with ThreadPoolExecutor(max_workers=16) as ex:
        futs = []
        for i in range(n):
            priv = batch.priv[i * batch.priv_bytes:(i + 1) * batch.priv_bytes].cpu().numpy()
            pub = batch.pub[i * batch.pub_bytes:(i + 1) * batch.pub_bytes].cpu().numpy()
            img = d_imgs[i].cpu().numpy() if i % 8 == 0 or i == n - 1 else None
            futs.append(ex.submit(one, i, priv, pub, img))
            if len(futs) >= 32:                      # bound the host copies in flight
                futs.pop(0).result()
        for f in futs:
            f.result()
    out = torch.empty_like(d_imgs)
    batch.defragment(out, key, d_nonces, expected=batch.digests)
    torch.cuda.synchronize()
    assert torch.equal(out, d_imgs) and int(batch.flags_out.abs().sum().item()) == 0
    # every image's digests are distinct (independent CTR messages, A20)
    assert len({bytes(r[:32]) for r in dgs}) == n


# the digest-free path runs different kernels (persistent tile kernels, feds_dct_tile.cuh): same arithmetic, other data movement
@pytest.mark.parametrize("n,w,h,c,k", [(1, 8, 8, 1, 0), (1, 8, 8, 1, 63), (2, 264, 16, 3, 3), (1, 1032, 24, 1, 5), (3, 1920, 16, 3, 3),
                                       (1, 4104, 8, 1, 2), (2, 520, 40, 4, 7), (1, 776, 8, 3, 0), (1, 256, 64, 3, 9), (1, 512, 8, 4, 62),
                                       (1, 2048, 8, 3, 31), (1, 2048, 8, 3, 32)])
def test_digest_free_tile_kernels(orc, b, n, w, h, c, k):
    key, nonce = synth.key_nonce(w + k)
    nonces = synth.batch_nonces(nonce, n)
    imgs = np.stack([synth.image(w, h, c, seed=7 * w + i + k, rectangles=1 if w >= 64 and h >= 16 else 0) for i in range(n)])
    d_imgs = torch.from_numpy(imgs).cuda()
    d_nonces = torch.from_numpy(nonces).cuda()
    full, plain = b.DctBatch(n, w, h, c, k), b.DctBatch(n, w, h, c, k)
    for t in (full.priv, full.pub, plain.priv, plain.pub):
        t.fill_(0xA5)   # torch.empty may hand back a buffer that already holds the right bytes
    full.fragment(d_imgs, key, d_nonces)
    plain.fragment(d_imgs, key, d_nonces, flags=b.FLAG_NO_DIGEST)
    torch.cuda.synchronize()
    assert torch.equal(plain.priv, full.priv), "private fragments differ"
    assert torch.equal(plain.pub, full.pub), "public fragments differ"
    # stage (i)/(ii) against the oracle on the tile kernels' own output, image 0
    pv = plain.priv[:plain.priv_bytes].cpu().numpy()
    pb = plain.pub[:plain.pub_bytes].cpu().numpy()
    coef = gpu_coefficients(orc, pv, pb, w * h * c // 64, k, key, nonces[0].tobytes())
    assert np.abs(coef - orc.dct_coefficients(imgs[0])).max() <= TOL
    p2, q2, _ = orc.fragment_from_coef32(coef, w, h, c, k, key, nonces[0].tobytes())
    assert (p2 == pv).all() and (q2 == pb).all()
    # inverse without verification: tile kernel; with verification: fused kernel; both exact
    out = torch.zeros_like(d_imgs)
    plain.defragment(out, key, d_nonces)
    assert torch.equal(out, d_imgs)
    out.zero_()
    full.defragment(out, key, d_nonces, expected=full.digests)
    assert torch.equal(out, d_imgs) and int(full.flags_out.abs().sum().item()) == 0


# The digest-free path has two sets of tile kernels: the bulk-copy (TMA) ones (feds_dct_tma.cuh: w % 32 == 0, tiles of 32 / 64 blocks
# in linear block order that may wrap into the next block row) and the generic ones (any w; FEDS_FLAG_GENERIC_TILES forces them).
# Same arithmetic, other data movement: identical bytes both ways, the oracle's for these coefficient bytes, exact round trips
# of either kernel's fragments through either inverse kernel.
TMA_CASES = [(1, 512, 8, 1, 3), (1, 512, 512, 1, 2), (2, 576, 40, 1, 0), (1, 256, 8, 3, 3), (2, 288, 24, 3, 3), (3, 1920, 16, 3, 3),
             (1, 1920, 1080, 3, 3), (2, 288, 40, 3, 4), (1, 320, 24, 3, 5), (1, 288, 24, 3, 62), (1, 256, 16, 3, 63), (2, 352, 24, 4, 7),
             (1, 256, 8, 4, 0), (1, 800, 56, 4, 2), (1, 2048, 8, 3, 31), (5, 640, 72, 1, 9)]


@pytest.mark.parametrize("n,w,h,c,k", TMA_CASES)
def test_bulk_copy_and_generic_tile_kernels_agree(orc, b, n, w, h, c, k):
    key, nonce = synth.key_nonce(w + 2 * k + c)
    nonces = synth.batch_nonces(nonce, n)
    imgs = np.stack([synth.image(w, h, c, seed=13 * w + i + k, rectangles=1) for i in range(n)])
    d_imgs = torch.from_numpy(imgs).cuda()
    d_nonces = torch.from_numpy(nonces).cuda()
    tma, gen = b.DctBatch(n, w, h, c, k), b.DctBatch(n, w, h, c, k)
    for t in (tma.priv, tma.pub, gen.priv, gen.pub):
        t.fill_(0x3C)
    tma.fragment(d_imgs, key, d_nonces, flags=b.FLAG_NO_DIGEST)
    gen.fragment(d_imgs, key, d_nonces, flags=b.FLAG_NO_DIGEST | b.FLAG_GENERIC_TILES)
    torch.cuda.synchronize()
    assert torch.equal(tma.priv, gen.priv), "private fragments differ"
    assert torch.equal(tma.pub, gen.pub), "public fragments differ"
    for i in sorted({0, n - 1}):
        pv = tma.priv[i * tma.priv_bytes:(i + 1) * tma.priv_bytes].cpu().numpy()
        pb = tma.pub[i * tma.pub_bytes:(i + 1) * tma.pub_bytes].cpu().numpy()
        coef = gpu_coefficients(orc, pv, pb, w * h * c // 64, k, key, nonces[i].tobytes())
        if w * h <= 1 << 19:
            assert np.abs(coef - orc.dct_coefficients(imgs[i])).max() <= TOL
        p2, q2, _ = orc.fragment_from_coef32(coef, w, h, c, k, key, nonces[i].tobytes())
        assert (p2 == pv).all() and (q2 == pb).all()
    for flags in (b.FLAG_NO_DIGEST, b.FLAG_NO_DIGEST | b.FLAG_GENERIC_TILES):
        out = torch.full_like(d_imgs, 0x77)
        tma.defragment(out, key, d_nonces, flags=flags)
        assert torch.equal(out, d_imgs)


# Steps 1-5 (and 6-8 with verification) run either as the digest-free tile kernel and the leaf-hash kernel one after the other (the
# default: measured faster) or in ONE warp-specialised kernel (feds_dct_fused.cuh: bulk-copy tile groups + hash warps; needs
# w % 64 == 0 and at least one tile per block row). FEDS_FLAG_FORCE_FUSED / FEDS_FLAG_FORCE_SPLIT pick the route. Both routes must
# produce the same bytes, digests, images and flags at any size and any k.
WS_CASES = [(1, 512, 8, 1, 3), (2, 256, 16, 3, 3), (1, 1024, 24, 1, 5), (3, 1920, 16, 3, 7), (2, 512, 40, 4, 1), (1, 2048, 8, 1, 9),
            (1, 256, 64, 3, 31), (1, 512, 8, 4, 61), (1, 2048, 8, 3, 63), (7, 1920, 136, 3, 3), (1, 4096, 264, 3, 5), (3, 2048, 72, 4, 3),
            (2, 8192, 24, 1, 3), (40, 256, 64, 3, 3), (2, 320, 24, 3, 4), (1, 576, 16, 1, 0), (2, 1920, 1080, 3, 2)]


@pytest.mark.parametrize("n,w,h,c,k", WS_CASES)
def test_fused_and_split_routes_agree(orc, b, n, w, h, c, k):
    key, nonce = synth.key_nonce(w + k)
    nonces = synth.batch_nonces(nonce, n)
    imgs = np.stack([synth.image(w, h, c, seed=11 * w + i + k) for i in range(n)])
    d_imgs = torch.from_numpy(imgs).cuda()
    d_nonces = torch.from_numpy(nonces).cuda()
    fused, split = b.DctBatch(n, w, h, c, k), b.DctBatch(n, w, h, c, k)
    for t in (fused.priv, fused.pub, fused.digests, split.priv, split.pub, split.digests):
        t.fill_(0x5A)
    fused.fragment(d_imgs, key, d_nonces, flags=b.FLAG_FORCE_FUSED)
    split.fragment(d_imgs, key, d_nonces, flags=b.FLAG_FORCE_SPLIT)
    torch.cuda.synchronize()
    assert torch.equal(fused.priv, split.priv) and torch.equal(fused.pub, split.pub) and torch.equal(fused.digests, split.digests)
    # and they are the oracle's for these coefficient bytes (first and last image)
    for i in sorted({0, n - 1}):
        pv = fused.priv[i * fused.priv_bytes:(i + 1) * fused.priv_bytes].cpu().numpy()
        pb = fused.pub[i * fused.pub_bytes:(i + 1) * fused.pub_bytes].cpu().numpy()
        coef = gpu_coefficients(orc, pv, pb, w * h * c // 64, k, key, nonces[i].tobytes())
        if w * h <= 1 << 19:
            assert np.abs(coef - orc.dct_coefficients(imgs[i])).max() <= TOL
        p2, q2, d2 = orc.fragment_from_coef32(coef, w, h, c, k, key, nonces[i].tobytes())
        assert (p2 == pv).all() and (q2 == pb).all() and d2 == fused.digests[64 * i:64 * i + 64].cpu().numpy().tobytes()
    # verified defragment on both routes: exact image, flags 0; then one flipped byte per fragment in chosen images
    for flag in (b.FLAG_FORCE_FUSED, b.FLAG_FORCE_SPLIT):
        out = torch.zeros_like(d_imgs)
        fused.flags_out.fill_(9)
        fused.defragment(out, key, d_nonces, expected=split.digests, flags=flag)
        assert torch.equal(out, d_imgs) and int(fused.flags_out.abs().sum().item()) == 0
    if k < 63:
        split.pub[(n - 1) * split.pub_bytes + split.pub_bytes - 1] ^= 0x01
    split.priv[5] ^= 0x80
    want = [0] * n
    want[0] |= 1
    if k < 63:
        want[n - 1] |= 2
    outs = []
    for flag in (b.FLAG_FORCE_FUSED, b.FLAG_FORCE_SPLIT):
        out = torch.zeros_like(d_imgs)
        split.defragment(out, key, d_nonces, expected=fused.digests, flags=flag)
        assert split.flags_out.cpu().tolist() == want
        outs.append(out)
    assert torch.equal(outs[0], outs[1])      # the image is written regardless (A10), identically on both routes


def test_forced_route_that_cannot_run_is_refused(b):
    """FEDS_FLAG_FORCE_FUSED on a shape the fused kernels do not support (ragged last leaf: (w/8) % 8 != 0; narrower than a tile) returns
    FEDS_ERR_BAD_PARAM before anything is enqueued; both force flags together likewise."""
    key, nonce = synth.key_nonce(1)
    for (w, h, c, k) in [(520, 16, 3, 3), (224, 16, 3, 3), (288, 16, 1, 3)]:
        img = torch.zeros((1, h, w, c), dtype=torch.uint8, device="cuda")
        non = torch.zeros((1, 16), dtype=torch.uint8, device="cuda")
        batch = b.DctBatch(1, w, h, c, k)
        with pytest.raises(b.FedsError) as e:
            batch.fragment(img, key, non, flags=b.FLAG_FORCE_FUSED)
        assert e.value.code == 3
        batch.fragment(img, key, non, flags=b.FLAG_FORCE_SPLIT)
        with pytest.raises(b.FedsError) as e:
            batch.defragment(img.clone(), key, non, expected=batch.digests, flags=b.FLAG_FORCE_FUSED)
        assert e.value.code == 3
    batch = b.DctBatch(1, 64, 8, 1, 3)
    with pytest.raises(b.FedsError):
        batch.fragment(torch.zeros((1, 8, 64, 1), dtype=torch.uint8, device="cuda"), key, torch.zeros((1, 16), dtype=torch.uint8, device="cuda"),
                       flags=b.FLAG_FORCE_FUSED | b.FLAG_FORCE_SPLIT)


def test_device_dct_bits_equal_the_host_build(orc, b):
    """The 8x8 transform is written with explicitly rounded mul / add / fma, so the kernels and the host build of the same
    function (feds_debug_dct8x8_host, gcc) agree bit for bit: fragments do not depend on compiler contraction choices."""
    import ctypes as C
    w, h, c, k = 256, 64, 1, 63
    img = synth.image(w, h, c, seed=5, rectangles=3)
    key = bytes(16)
    priv, _, _ = b.fragment_dct(torch.from_numpy(img).cuda(), k, key, bytes(16))
    ks = np.frombuffer(orc.aes128_ctr_xor(key, bytes(16), bytes(priv.numel())), dtype=np.uint8)
    coef = np.frombuffer((priv.cpu().numpy() ^ ks).tobytes(), dtype="<f4").reshape(h // 8, w // 8, 64)
    zz = (C.c_int * 64)()
    b.lib.feds_debug_zigzag_host(zz)
    zz = np.array(list(zz))
    for (br, bc) in [(0, 0), (3, 17), (7, 31), (5, 2)]:
        x = np.ascontiguousarray(img[8 * br:8 * br + 8, 8 * bc:8 * bc + 8, 0], dtype=np.float32)
        out = np.empty(64, dtype=np.float32)
        b.lib.feds_debug_dct8x8_host(x.ctypes.data, out.ctypes.data, 0)
        assert (out[zz].view(np.uint32) == coef[br, bc].view(np.uint32)).all()


def test_cuda_graph_capture_and_replay(orc, b):
    """The library allocates nothing, keeps no state and never synchronises (include/feds.h), so a fragment + verified defragment
    pair -- DCT and DWT -- can be captured into a CUDA graph once and replayed on new pixels: the replays' fragments and digests are
    the ones a direct call produces, bit for bit (and the direct call's are the oracle's, as every other test here checks)."""
    n, w, h, c, k, L = 2, 512, 64, 3, 3, 2
    key, nonce = synth.key_nonce(77)
    nonces = synth.batch_nonces(nonce, n)
    d_non = torch.from_numpy(nonces).cuda()
    imgs = [torch.from_numpy(np.stack([synth.image(w, h, c, seed=900 + 10 * r + i) for i in range(n)])).cuda() for r in range(3)]
    d_in = imgs[0].clone()
    d_out, d_out2 = torch.zeros_like(d_in), torch.zeros_like(d_in)
    dct, dwt = b.DctBatch(n, w, h, c, k), b.DwtBatch(n, w, h, c, L)

    def work():
        dct.fragment(d_in, key, d_non)
        dct.defragment(d_out, key, d_non, expected=dct.digests)
        dwt.fragment(d_in, key, d_non)
        dwt.defragment(d_out2, key, d_non, expected=dwt.digests)

    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        work()                                   # first calls set kernel attributes: keep them out of the capture
    torch.cuda.current_stream().wait_stream(side)
    torch.cuda.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=side):
        work()
    ref_dct, ref_dwt = b.DctBatch(n, w, h, c, k), b.DwtBatch(n, w, h, c, L)
    for r in (1, 2, 0):
        d_in.copy_(imgs[r])
        for t in (dct.priv, dct.pub, dct.digests, dwt.priv, dwt.pub, dwt.digests, d_out, d_out2):
            t.zero_()
        dct.flags_out.fill_(7); dwt.flags_out.fill_(7)
        graph.replay()
        torch.cuda.synchronize()
        ref_dct.fragment(imgs[r], key, d_non)
        ref_dwt.fragment(imgs[r], key, d_non)
        torch.cuda.synchronize()
        assert torch.equal(dct.priv, ref_dct.priv) and torch.equal(dct.pub, ref_dct.pub) and torch.equal(dct.digests, ref_dct.digests)
        assert torch.equal(dwt.priv, ref_dwt.priv) and torch.equal(dwt.pub, ref_dwt.pub) and torch.equal(dwt.digests, ref_dwt.digests)
        assert torch.equal(d_out, imgs[r]) and torch.equal(d_out2, imgs[r])
        assert int(dct.flags_out.abs().sum().item()) == 0 and int(dwt.flags_out.abs().sum().item()) == 0
    # the replayed fragments are the oracle's for image 0 of the last round
    pv = dct.priv[:dct.priv_bytes].cpu().numpy()
    pb = dct.pub[:dct.pub_bytes].cpu().numpy()
    coef = gpu_coefficients(orc, pv, pb, w * h * c // 64, k, key, nonces[0].tobytes())
    p2, q2, d2 = orc.fragment_from_coef32(coef, w, h, c, k, key, nonces[0].tobytes())
    assert (p2 == pv).all() and (q2 == pb).all() and d2 == dct.digests[:64].cpu().numpy().tobytes()
    op, oq, odg = orc.fragment_dwt(imgs[0][0].cpu().numpy(), L, key, nonces[0].tobytes())
    assert (dwt.priv[:dwt.priv_bytes].cpu().numpy() == op).all() and dwt.digests[:64].cpu().numpy().tobytes() == odg

