"""feds_sha256_merkle_static: the entry point that allocates nothing (its scratch is a static device array inside the library).

Collected last on purpose (the suite runs with pytest -x). Its root must be the one feds_sha256_merkle computes with a caller's
workspace -- bit for bit, the tolerance of every digest test here -- on two calls in a row that share the static array (the second
on a shorter, different stream, so that stale leaf digests and tree levels of the first would show), and the oracle's.
"""
import ctypes as C

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


@pytest.fixture(scope="module")
def orc():
    import oracle
    return oracle


def _stream(n, seed):
    return torch.from_numpy(np.random.default_rng(seed).integers(0, 256, n, dtype=np.uint8)).cuda()


def test_static_scratch_root_equals_workspace_path_on_consecutive_calls(orc, b):
    # 20 MiB + ragged tail: 10,241 leaves -> the wide level kernel and the spread-out tree top (its counters live in the scratch);
    # then 3 MiB - 5: a tree that fits the single-CTA top; then one leaf, then the empty stream; then the long one again
    sizes = [(20 << 20) + 77, (3 << 20) - 5, 1500, 0, (20 << 20) + 77]
    root = torch.zeros(32, dtype=torch.uint8, device="cuda")
    for i, n in enumerate(sizes):
        data = _stream(n, seed=100 + i)
        want = b.sha256_merkle(data)                       # existing path: workspace from the caller
        torch.cuda.synchronize()
        before = torch.cuda.memory_allocated()
        root.fill_(0xEE)
        b.sha256_merkle_static(data, root)
        b.sha256_merkle_static(data, root)                 # twice in a row on the same stream: same scratch, same answer
        torch.cuda.synchronize()
        assert torch.cuda.memory_allocated() <= before     # the binding marshals arguments only (the count may drop: garbage of earlier tests)
        assert torch.equal(root, want), (i, n)
        if n <= (3 << 20):
            assert root.cpu().numpy().tobytes() == orc.merkle_stream(data.cpu().numpy().tobytes()), (i, n)


def test_static_scratch_limits_and_errors(b):
    limit = b.lib.feds_sha256_merkle_static_max_bytes()
    assert limit == 64 << 20
    ok_ptr = C.c_void_p(0x1000)   # never dereferenced: the calls below fail in validation, nothing is enqueued
    f = b.lib.feds_sha256_merkle_static
    assert f(ok_ptr, limit + 1, ok_ptr, None) == 3          # FEDS_ERR_BAD_PARAM: beyond the static scratch
    assert f(None, 16, ok_ptr, None) == 1 and f(ok_ptr, 16, None, None) == 1
    assert f(C.c_void_p(0x1001), 16, ok_ptr, None) == 6     # misaligned, as feds_sha256_merkle
    # the largest stream it accepts, against the workspace path
    data = _stream(limit, seed=7)
    root = torch.zeros(32, dtype=torch.uint8, device="cuda")
    b.sha256_merkle_static(data, root)
    assert torch.equal(root, b.sha256_merkle(data))
