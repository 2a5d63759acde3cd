"""N > 1 host logic on CPU: two gloo ranks split a batch by image (paper_1512_02951_b200.sharding), each fragments its
shard (with the CPU oracle standing in for the device here -- test infrastructure only), and the gathered digests equal the
single-process result bit for bit: the fragments of image i do not depend on the number of ranks."""
import os
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
N, W, H, C, K = 5, 32, 16, 3, 3


def _all_digests(first, count):
    import oracle
    import synth
    from paper_1512_02951_b200 import sharding
    key, nonce = synth.key_nonce(77)
    nonces = sharding.nonces_for(nonce, first, count)
    out = np.zeros((count, 64), dtype=np.uint8)
    for j in range(count):
        img = synth.image(W, H, C, seed=500 + first + j)
        _, _, dg = oracle.fragment_dct(img, K, key, nonces[j].tobytes())
        out[j] = np.frombuffer(dg, dtype=np.uint8)
    return out


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_1512_02951_b200 import sharding
    first, count = sharding.shard_range(N, world, rank)
    local = torch.from_numpy(_all_digests(first, count))
    padded = torch.zeros((N, 64), dtype=torch.uint8)          # all_gather needs equal shapes: pad to N rows
    padded[:count] = local
    bufs = [torch.zeros_like(padded) for _ in range(world)]
    dist.all_gather(bufs, padded)
    t = sharding.max_over_ranks(10.0 + rank)
    if rank == 0:
        rows = []
        for r in range(world):
            f, cnt = sharding.shard_range(N, world, r)
            rows.append(bufs[r][:cnt])
        q.put((torch.cat(rows).numpy(), t))
    dist.destroy_process_group()


def test_shard_range_covers_batch_exactly():
    from paper_1512_02951_b200 import sharding
    for n in [0, 1, 5, 256, 257]:
        for world in [1, 2, 3, 8]:
            spans = [sharding.shard_range(n, world, r) for r in range(world)]
            assert spans[0][0] == 0 and sum(c for _, c in spans) == n
            for (f0, c0), (f1, _) in zip(spans, spans[1:]):
                assert f1 == f0 + c0
            assert max(c for _, c in spans) - min(c for _, c in spans) <= 1
    with pytest.raises(ValueError):
        sharding.shard_range(4, 2, 2)


def test_nonces_depend_on_global_index_only():
    import synth
    from paper_1512_02951_b200 import sharding
    _, nonce = synth.key_nonce(1)
    whole = sharding.nonces_for(nonce, 0, 7)
    assert (whole == synth.batch_nonces(nonce, 7)).all()
    assert (sharding.nonces_for(nonce, 3, 4) == whole[3:]).all()
    top = bytes([0xff] * 16)
    assert sharding.nonces_for(top, 1, 1)[0].tobytes() == ((1 << 20) - 1).to_bytes(16, "big")   # wraps mod 2^128


def test_nonce_stride_covers_the_private_fragment():
    """with one key, the counter ranges of consecutive images must not overlap whatever the fragment size. A private
    fragment above 16 MiB (2^20 blocks) must widen the stride; a stride that is too short is refused."""
    import synth
    from paper_1512_02951_b200 import sharding
    _, nonce = synth.key_nonce(2)
    priv = 4096 * 4096 * 3 // 64 * 6 * 4                   # BASELINE configs[1]: 18.9 MB private fragment per image
    assert priv > (1 << 20) * 16
    stride = sharding.nonce_stride(priv)
    assert stride * 16 >= priv and stride & (stride - 1) == 0
    a = sharding.nonces_for(nonce, 0, 3, priv_bytes=priv)
    vals = [int.from_bytes(r.tobytes(), "big") for r in a]
    blocks = (priv + 15) // 16
    for x, y in zip(vals, vals[1:]):
        assert (y - x) % (1 << 128) >= blocks                # image i's last counter < image i+1's first
    assert (a == synth.batch_nonces(nonce, 3, priv_bytes=priv)).all()
    with pytest.raises(ValueError):
        sharding.nonces_for(nonce, 0, 2, priv_bytes=priv, stride=1 << 20)
    with pytest.raises(ValueError):
        synth.batch_nonces(nonce, 2, priv_bytes=priv, stride=1 << 20)
    assert sharding.nonce_stride(1555200) == 1 << 20         # cfg3 keeps the round-1 stride: stored digests do not move


def test_two_gloo_ranks_equal_single_process():
    world, port = 2, 29500 + (os.getpid() % 2000)
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    got, tmax = q.get(timeout=180)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert tmax == 11.0                                   # MAX over ranks of (10 + rank)
    assert (got == _all_digests(0, N)).all()
