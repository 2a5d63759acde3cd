"""Host-side batch sharding for N > 1 ranks (one process per GPU). The path shards by image: every image is an
independent CTR message with its own nonce and digest pair (A20), so ranks exchange nothing on the data
path -- "replicas / batch split only, no collective". The only collective is the MAX of the timed
region in bench.py. Nonces are a function of the GLOBAL image index, so the fragments of image i do not depend on how
many ranks the batch was split over.
"""
import numpy as np


def shard_range(n_total: int, world: int, rank: int):
    """Contiguous split of n_total images over `world` ranks: (first_global_index, count) for `rank`."""
    if world < 1 or not (0 <= rank < world) or n_total < 0:
        raise ValueError("bad shard arguments")
    base, extra = divmod(n_total, world)
    count = base + (1 if rank < extra else 0)
    first = rank * base + min(rank, extra)
    return first, count


def nonce_stride(priv_bytes: int, min_stride: int = 1 << 20) -> int:
    """Counter blocks between the nonces of consecutive images: a power of two >= ceil(priv_bytes / 16), so that the CTR counter
    ranges [nonce_i, nonce_i + ceil(priv_bytes / 16)) of the images never overlap under the one key (include/feds.h, batch entry
    points; overlapping ranges would reuse keystream)."""
    need = max(1, (int(priv_bytes) + 15) // 16)
    stride = max(1, int(min_stride))
    while stride < need:
        stride <<= 1
    return stride


def nonces_for(base_nonce: bytes, first_global_index: int, count: int, priv_bytes: int = 0, stride: int = None) -> np.ndarray:
    """uint8[count][16]: nonce of global image i = (base + i * stride) mod 2^128, big-endian (one IV per image).
    `priv_bytes` = size of one image's private fragment; the stride is chosen (or, when given, checked) so that the images'
    counter ranges cannot overlap."""
    if stride is None:
        stride = nonce_stride(priv_bytes)
    if stride * 16 < priv_bytes:
        raise ValueError("nonce stride %d blocks is shorter than the private fragment (%d bytes): keystream would be reused" % (stride, priv_bytes))
    base = int.from_bytes(base_nonce, "big")
    out = np.empty((count, 16), dtype=np.uint8)
    for j in range(count):
        v = (base + (first_global_index + j) * stride) % (1 << 128)
        out[j] = np.frombuffer(v.to_bytes(16, "big"), dtype=np.uint8)
    return out


def max_over_ranks(value: float, device=None) -> float:
    """MAX-reduce a per-rank timing; identity when torch.distributed is not initialised."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
