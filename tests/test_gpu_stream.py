"""GPU parity tests for the stream primitives of the C ABI (feds_aes128_ctr, feds_sha256_merkle): bit-exact against the
oracle's FIPS-197 / SP 800-38A CTR and its Merkle-of-SHA-256 over 2048-byte leaves (A6, A9).
feds_aes128_ctr on the image bytes is the report's "AES over the whole image" baseline."""
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


def _bytes(n, seed):
    return np.random.default_rng(seed).integers(0, 256, size=n, dtype=np.uint8)


# sizes: empty, sub-block, one block, ragged tails, several CTAs of the 4 KB-table kernel, and past the 4 MiB switch to the
# conflict-free 128 KB-table kernel (with a ragged tail there too)
@pytest.mark.parametrize("n", [0, 1, 15, 16, 17, 4096, 65536 + 5, 1 << 20, (4 << 20) - 16, (4 << 20) + 16 * 3 + 7, 12_000_003])
def test_aes_ctr_matches_oracle(orc, b, n):
    key, nonce = synth.key_nonce(n % 97)
    data = _bytes(n, n)
    d = torch.from_numpy(data).cuda()
    ct = b.aes128_ctr(d, key, nonce)
    torch.cuda.synchronize()
    want = np.frombuffer(orc.aes128_ctr_xor(key, nonce, data.tobytes()), dtype=np.uint8)
    assert (ct.cpu().numpy() == want).all()
    # CTR is its own inverse; in place
    b.aes128_ctr(ct, key, nonce, out=ct)
    assert torch.equal(ct, d)


def test_aes_ctr_counter_carry(orc, b):
    # nonce whose low 64 bits are about to wrap: the carry must run through all 128 bits (SP 800-38A B.1, A6)
    key, _ = synth.key_nonce(3)
    nonce = bytes([0x12] * 7) + b"\xff" * 8 + b"\xfe"   # + 2 wraps the low 72 bits
    data = _bytes(16 * 64, 5)
    ct = b.aes128_ctr(torch.from_numpy(data).cuda(), key, nonce)
    want = np.frombuffer(orc.aes128_ctr_xor(key, nonce, data.tobytes()), dtype=np.uint8)
    assert (ct.cpu().numpy() == want).all()


def test_aes_ctr_sp800_38a_f51(orc, b, kat):
    # SP 800-38A F.5.1 CTR-AES128.Encrypt, first block (tests/golden/standards_kat.txt)
    key = bytes.fromhex(kat["sp80038a_key"])
    ctr = bytes.fromhex(kat["sp80038a_ctr"])
    pt = bytes.fromhex(kat["sp80038a_pt"])
    ct = b.aes128_ctr(torch.frombuffer(bytearray(pt), dtype=torch.uint8).cuda(), key, ctr)
    assert ct.cpu().numpy().tobytes().hex() == kat["sp80038a_ct"]


# leaves: none, one short, exactly one, one + 1 byte, 16 leaves (one node), 17, 4096 (tail kernel limit), 4097 (a wide level), big ragged
# the last four: tree tops of 65 / 65 / 128 / 252 first-level nodes, ragged at every level (the spread-out top kernel's counters)
@pytest.mark.parametrize("n", [0, 5, 2048, 2049, 16 * 2048, 17 * 2048 - 3, 4096 * 2048, 4097 * 2048 + 11, 30_000_001,
                               1024 * 2048 + 1, 1030 * 2048 + 5, 2047 * 2048 + 1, 4032 * 2048 - 7])
def test_sha256_merkle_matches_oracle(orc, b, n):
    data = _bytes(n, n + 1)
    root = b.sha256_merkle(torch.from_numpy(data).cuda())
    torch.cuda.synchronize()
    assert root.cpu().numpy().tobytes() == orc.merkle_stream(data.tobytes())


def test_full_image_aes_baseline_round_trip(orc, b):
    # NEXT-1: encrypt every byte of an image, decrypt, compare; ciphertext sampled against the oracle block by block
    img = synth.image(1024, 768, 3, seed=11)
    key, nonce = synth.key_nonce(11)
    d = torch.from_numpy(img).cuda().view(-1)
    ct = b.aes128_ctr(d, key, nonce)
    pt = b.aes128_ctr(ct, key, nonce)
    assert torch.equal(pt, d)
    raw = img.tobytes()
    for blk in [0, 1, 4095, 4096, 65535, len(raw) // 16 - 1]:
        want = orc.aes128_ctr_xor(key, nonce, raw[16 * blk:16 * blk + 16], first_block=blk)
        assert ct[16 * blk:16 * blk + 16].cpu().numpy().tobytes() == want
