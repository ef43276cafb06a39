"""Multi-GPU sharding of one integration (the paper farms blocks of samples over GPUs by MPI).

Samples are independent and addressed by their Philox counter, so rank r integrates the contiguous sample range
shard_range(n, r, world) with no data-path collective; the only exchange is one all_gather of the 80-byte fg_result
per rank, after which every rank merges the shards exactly (double-double sums add) in rank order.
"""
import ctypes as C

import numpy as np


def shard_range(n_samples, rank, world):
    """Contiguous split of [0, n) into `world` ranges whose sizes differ by at most one: returns (first, count)."""
    base, rem = divmod(int(n_samples), int(world))
    first = rank * base + min(rank, rem)
    return first, base + (1 if rank < rem else 0)


def gather_and_merge(local_result, group=None, device=None):
    """all_gather of raw fg_result structs (as bytes) and exact merge in rank order.  Works on gloo (CPU tensors) and
    nccl (pass device=torch.device('cuda', i)).  Returns the merged raw fg_result."""
    import torch
    import torch.distributed as dist
    from . import fg
    nbytes = C.sizeof(fg.fg_result)
    buf = np.frombuffer(bytes(local_result), dtype=np.uint8).copy()
    t = torch.from_numpy(buf)
    if device is not None:
        t = t.to(device)
    world = dist.get_world_size(group)
    outs = [torch.empty_like(t) for _ in range(world)]
    dist.all_gather(outs, t, group=group)
    merged = None
    for o in outs:
        r = fg.fg_result.from_buffer_copy(o.cpu().numpy().tobytes()[:nbytes])
        merged = r if merged is None else fg.result_merge(merged, r)
    return merged


def integrate_sharded(plan, n_samples, seed, rank, world, group=None, device=None, stream=None, first_sample=0):
    """Each rank integrates its own sample range on its own GPU; results are merged on every rank."""
    first, cnt = shard_range(n_samples, rank, world)
    from . import fg
    if cnt > 0:
        local = plan.integrate_range(first_sample + first, cnt, seed, stream=stream, raw=True)
    else:
        local = fg.fg_result()
    return gather_and_merge(local, group=group, device=device)
