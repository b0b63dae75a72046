"""Plumbing of a particle-sharded run: which particles a rank owns, how the ranks agree on an NCCL
communicator for libshd, and -- for callers that drive the split calls themselves -- the all-gather of the shards'
partial sums in rank order.  No arithmetic of the method lives here: the partial sums are opaque bytes, added by the
library's kernel (k_finish1) in the fixed rank order in which this module lays them out.
"""
from __future__ import annotations

import numpy as np


def shard_range(N: int, rank: int, world: int):
    """[begin, end) of the particles of `rank`: contiguous ranges, the first N % world ranks hold one more."""
    if not (0 <= rank < world) or N < world:
        raise ValueError("bad rank / world / N")
    base, extra = divmod(int(N), int(world))
    begin = rank * base + min(rank, extra)
    return begin, begin + base + (1 if rank < extra else 0)


def local_positions(hi: np.ndarray, lo: np.ndarray, d: int, N: int, rank: int, world: int):
    """axis-major (x[a*N + j]) global arrays -> this rank's axis-major arrays"""
    a, b = shard_range(N, rank, world)
    cut = lambda x: np.ascontiguousarray(np.asarray(x).reshape(d, N)[:, a:b]).reshape(-1)
    return cut(hi), cut(lo)


def broadcast_bytes(payload: bytes | None, nbytes: int, src: int = 0, device="cpu") -> bytes:
    """`payload` of rank `src` to every rank of the default torch.distributed group (any backend)."""
    import torch
    import torch.distributed as dist
    t = torch.zeros(nbytes, dtype=torch.uint8, device=device)
    if dist.get_rank() == src:
        t.copy_(torch.frombuffer(bytearray(payload), dtype=torch.uint8))
    dist.broadcast(t, src=src)
    return bytes(t.cpu().numpy().tobytes())


def init_comm(h, device="cuda"):
    """Give the sharded handle `h` (shd_set_shard already called) a library-owned NCCL communicator: rank 0 draws the
    unique id, torch.distributed carries its 128 bytes to the others, every rank calls shd_comm_init (collective)."""
    import torch.distributed as dist
    from . import shd
    uid = shd.comm_unique_id() if dist.get_rank() == 0 else None
    h.comm_init(broadcast_bytes(uid, 128, 0, device))


def gather_partials(mine):
    """all-gather of one uint8 tensor per rank into one tensor, rank 0 first (what shd_rho_finish expects)."""
    import torch
    import torch.distributed as dist
    world = dist.get_world_size()
    out = torch.empty(world * mine.numel(), dtype=torch.uint8, device=mine.device)
    dist.all_gather_into_tensor(out, mine.contiguous())
    return out
