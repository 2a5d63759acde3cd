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
    """8192x8192 grayscale, 3 levels (BASELINE config 4): bit-exact on everything -- and once more through the calls and in the
    launch configuration bench.py times (batch entry points, the verified defragment on two streams): fragments and digests are
    the oracle's, the image comes back exactly, a flipped bit in either fragment raises its flag."""
    img = synth.image(8192, 8192, 1, seed=4)
    run_case(orc, b, img, 3, seed=4)
    key, nonce = synth.key_nonce(4)
    batch = b.DwtBatch(1, 8192, 8192, 1, 3)
    d_img = torch.from_numpy(img).cuda()
    d_non = torch.frombuffer(bytearray(nonce), dtype=torch.uint8).cuda().view(1, 16)
    batch.fragment(d_img, key, d_non)
    op, oq, odg = orc.fragment_dwt(img, 3, key, nonce)
    assert (batch.priv[:batch.priv_bytes].cpu().numpy() == op).all() and (batch.pub[:batch.pub_bytes].cpu().numpy() == oq).all()
    assert batch.digests.cpu().numpy().tobytes() == odg
    aux, rec = torch.cuda.Stream(), torch.zeros_like(d_img)
    batch.flags_out.fill_(9)
    batch.defragment_2s(rec, key, d_non, batch.digests, aux)
    torch.cuda.synchronize()
    assert torch.equal(rec, d_img) and batch.flags_out.cpu().tolist() == [0]
    batch.pub[batch.pub_bytes - 1] ^= 0x80
    batch.priv[0] ^= 1
    batch.defragment_2s(rec, key, d_non, batch.digests, aux)
    torch.cuda.synchronize()
    assert batch.flags_out.cpu().tolist() == [3]


@pytest.mark.parametrize("w,h,c,L", [(1024, 320, 3, 4), (2048, 64, 1, 1), (7696, 96, 1, 2), (496, 80, 3, 1)])
def test_streaming_and_tiled_level_kernels_agree(orc, b, w, h, c, L):
    """The register-streaming level kernels (several column strips, halo lanes, row tiles) and the tiled shared-memory
    kernels they replace on aligned sizes (FEDS_FLAG_DWT_TILED) compute identical fragments; the oracle decides which is right."""
    img = synth.image(w, h, c, seed=w + L)
    key, nonce = synth.key_nonce(w)
    d_img = torch.from_numpy(img).cuda().unsqueeze(0).contiguous()
    d_non = torch.frombuffer(bytearray(nonce), dtype=torch.uint8).cuda().view(1, 16)
    fast, tiled = b.DwtBatch(1, w, h, c, L), b.DwtBatch(1, w, h, c, L)
    fast.fragment(d_img, key, d_non)
    tiled.fragment(d_img, key, d_non, flags=b.FLAG_DWT_TILED)
    rec_tiled, rec_fast = torch.zeros_like(d_img), torch.zeros_like(d_img)
    fast.defragment(rec_tiled, key, d_non, flags=b.FLAG_DWT_TILED)     # tiled inverse of the streaming kernels' fragments
    tiled.defragment(rec_fast, key, d_non)                             # and the other way round
    torch.cuda.synchronize()
    assert torch.equal(fast.priv, tiled.priv) and torch.equal(fast.pub, tiled.pub) and torch.equal(fast.digests, tiled.digests)
    op, oq, odg = orc.fragment_dwt(img, L, key, nonce)
    assert (fast.priv[:fast.priv_bytes].cpu().numpy() == op).all() and (fast.pub[:fast.pub_bytes].cpu().numpy() == oq).all()
    assert fast.digests.cpu().numpy().tobytes() == odg
    assert torch.equal(rec_tiled, d_img) and torch.equal(rec_fast, d_img)


@pytest.mark.parametrize("n,w,h,c,L", [(3, 64, 32, 1, 2), (4, 272, 144, 3, 3), (2, 1024, 320, 3, 4), (5, 16, 8, 1, 1), (3, 48, 80, 4, 2),
                                       (2, 2048, 512, 1, 3),
                                       # public trees of 1,536 / 2,304 leaves: the spread-out tree top with four and six trees in flight
                                       (2, 2048, 1024, 1, 1), (3, 1024, 1024, 3, 2)])
def test_dwt_batch_equals_oracle_per_image(orc, b, n, w, h, c, L):
    """feds_fragment_dwt_batch / feds_defragment_dwt_batch: every image is an independent CTR message with its own nonce and digest
    pair (A20); each image's fragments and digests are the oracle's, bit for bit; verification flags are per image."""
    key, nonce = synth.key_nonce(w + n)
    imgs = np.stack([synth.image(w, h, c, seed=50 * w + i, rectangles=1 if min(w, h) >= 32 else 0) for i in range(n)])
    batch = b.DwtBatch(n, w, h, c, L)
    nonces = synth.batch_nonces(nonce, n, priv_bytes=batch.priv_bytes)
    d_imgs, d_non = torch.from_numpy(imgs).cuda(), torch.from_numpy(nonces).cuda()
    batch.fragment(d_imgs, key, d_non)
    torch.cuda.synchronize()
    for i in range(n):
        op, oq, odg = orc.fragment_dwt(imgs[i], L, key, nonces[i].tobytes())
        assert (batch.priv[i * batch.priv_stride:i * batch.priv_stride + batch.priv_bytes].cpu().numpy() == op).all(), i
        assert (batch.pub[i * batch.pub_stride:i * batch.pub_stride + batch.pub_bytes].cpu().numpy() == oq).all(), i
        assert batch.digests[64 * i:64 * i + 64].cpu().numpy().tobytes() == odg, i
    out = torch.zeros_like(d_imgs)
    batch.defragment(out, key, d_non, expected=batch.digests)
    torch.cuda.synchronize()
    assert torch.equal(out, d_imgs) and int(batch.flags_out.abs().sum().item()) == 0
    victim = n - 1
    batch.pub[victim * batch.pub_stride + 3] ^= 0x20
    batch.priv[0] ^= 1
    batch.defragment(out, key, d_non, expected=batch.digests)
    want = [0] * n
    want[victim] |= 2
    want[0] |= 1
    assert batch.flags_out.cpu().tolist() == want


@pytest.mark.gpu
@pytest.mark.parametrize("n,w,h,c,L", [(1, 1024, 512, 1, 3), (3, 256, 128, 3, 2)])
def test_two_stream_defragment_equals_single_stream(orc, b, n, w, h, c, L):
    """feds_defragment_dwt_batch_2s (verification on a second stream, joined at the end): the image and the flags are those of the
    single-stream call, which the tests above pin to the oracle -- also after tampering, also when the pair of streams is captured
    into one CUDA graph and replayed."""
    key, nonce = synth.key_nonce(5 * w + n)
    imgs = np.stack([synth.image(w, h, c, seed=70 * w + i, rectangles=2) for i in range(n)])
    batch = b.DwtBatch(n, w, h, c, L)
    nonces = synth.batch_nonces(nonce, n, priv_bytes=batch.priv_bytes)
    d_imgs, d_non = torch.from_numpy(imgs).cuda(), torch.from_numpy(nonces).cuda()
    batch.fragment(d_imgs, key, d_non)
    aux = torch.cuda.Stream()
    out = torch.zeros_like(d_imgs)
    batch.flags_out.fill_(9)
    batch.defragment_2s(out, key, d_non, batch.digests, aux)
    torch.cuda.synchronize()
    assert torch.equal(out, d_imgs) and batch.flags_out.cpu().tolist() == [0] * n
    # capture both streams into one graph (the first call above set the kernel attributes), replay on tampered fragments
    main = torch.cuda.Stream()
    main.wait_stream(torch.cuda.current_stream())
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=main):
        batch.defragment_2s(out, key, d_non, batch.digests, aux, stream=main)
    batch.pub[(n - 1) * batch.pub_stride + 11] ^= 0x40
    batch.priv[5] ^= 1
    want = [0] * n
    want[n - 1] |= 2
    want[0] |= 1
    ref_out = torch.zeros_like(d_imgs)
    batch.defragment(ref_out, key, d_non, expected=batch.digests)
    torch.cuda.synchronize()
    assert batch.flags_out.cpu().tolist() == want
    for _ in range(3):
        out.zero_(); batch.flags_out.fill_(9)
        graph.replay()
        torch.cuda.synchronize()
        assert torch.equal(out, ref_out) and batch.flags_out.cpu().tolist() == want
