"""Multi-GPU sharding of one integration (the paper farms blocks of samples over GPUs by MPI).

Samples are independent and addressed by their Philox counter, so rank r integrates the contiguous sample range
shard_range(n, r, world) with no data-path collective; the only exchange is one all_gather of the fg_result struct
(88 bytes) per rank, after which every rank merges the shards exactly (double-double sums add) in rank order.

Two forms:
  integrate_sharded        blocking: every rank returns the merged result (host struct);
  integrate_sharded_async  the shard result stays on the device (no host synchronisation); gather_device() exchanges a whole
                           table of such results with ONE all_gather and merge_gathered() folds it on the host afterwards
                           (bench.py times this form).
"""
import ctypes as C

import numpy as np

RESULT_DOUBLES = 11          # sizeof(fg_result) / 8


def shard_range(n_samples, rank, world):
    """Contiguous split of [0, n) into `world` ranges whose sizes differ by at most one: returns (first, count)."""
    base, rem = divmod(int(n_samples), int(world))
    first = rank * base + min(rank, rem)
    return first, base + (1 if rank < rem else 0)


def merge_results(results):
    """Exact merge (fg_result_merge) of raw fg_result structs in list order."""
    from . import fg
    merged = None
    for r in results:
        merged = r if merged is None else fg.result_merge(merged, r)
    return merged


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
    return merge_results([fg.fg_result.from_buffer_copy(o.cpu().numpy().tobytes()[:nbytes]) for o in outs])


def integrate_sharded(plan, n_samples, seed, rank, world, group=None, device=None, stream=None, first_sample=0):
    """Each rank integrates its own sample range on its own GPU; results are merged on every rank."""
    first, cnt = shard_range(n_samples, rank, world)
    from . import fg
    if cnt > 0:
        local = plan.integrate_range(first_sample + first, cnt, seed, stream=stream, raw=True)
    else:
        local = fg.fg_result()
    if world == 1:
        return local
    return gather_and_merge(local, group=group, device=device)


def integrate_shards_on_one_device(plan, n_samples, seed, world, stream=None, first_sample=0):
    """The same split and the same merge with the `world` shards run one after another on this device (tests; a
    single-GPU box): bit for bit what `world` ranks would return."""
    from . import fg
    parts = []
    for rank in range(world):
        first, cnt = shard_range(n_samples, rank, world)
        parts.append(plan.integrate_range(first_sample + first, cnt, seed, stream=stream, raw=True) if cnt > 0 else fg.fg_result())
    return merge_results(parts)


def integrate_sharded_async(plan, n_samples, seed, rank, world, out_dev_ptr, stream=None, first_sample=0):
    """Enqueues this rank's shard; its fg_result is left at device address out_dev_ptr (RESULT_DOUBLES doubles)."""
    first, cnt = shard_range(n_samples, rank, world)
    if cnt > 0:
        plan.integrate_async(first_sample + first, cnt, seed, out_dev_ptr, stream=stream)
    return cnt


def gather_device(table, world, group=None):
    """table: float64 device tensor [k, RESULT_DOUBLES] of shard results (bit patterns of fg_result).  One all_gather;
    returns a [world, k, RESULT_DOUBLES] device tensor on every rank (the table itself when world == 1)."""
    if world == 1:
        return table.unsqueeze(0)
    import torch
    import torch.distributed as dist
    out = torch.empty((world,) + tuple(table.shape), dtype=table.dtype, device=table.device)
    dist.all_gather_into_tensor(out, table.contiguous(), group=group)
    return out


def merge_gathered(gathered):
    """Host: [world, k, RESULT_DOUBLES] tensor -> list of k merged raw fg_result structs (rank order)."""
    from . import fg
    arr = gathered.detach().cpu().numpy()
    world, k = arr.shape[0], arr.shape[1]
    nbytes = C.sizeof(fg.fg_result)
    out = []
    for j in range(k):
        parts = [fg.fg_result.from_buffer_copy(arr[r, j].tobytes()[:nbytes]) for r in range(world)]
        out.append(merge_results([p for p in parts if p.n_samples > 0] or parts[:1]))
    return out


def run_batch_rounds(batch, n_rounds, block_samples, sched_seed, rank, world, integrate, group=None, device=None):
    """One block schedule (paper_1909_08015_b200.sched.Batch) run by `world` ranks: in every round each rank
    draws the same `world` blocks (same batch state, same Philox uniform), integrates the one with its own index --
    integrate(graph, first_sample, n) -> (raw fg_result, seconds) -- and after one all_gather of the block results every rank
    folds all of them in block order, so the states stay identical.  Returns the list of (graph, first_sample) drawn."""
    import torch
    import torch.distributed as dist
    from . import fg
    nbytes = C.sizeof(fg.fg_result)
    log = []
    for _ in range(n_rounds):
        blocks = [batch.next(sched_seed, block_samples) for _ in range(world)]
        log.extend(blocks)
        j, first = blocks[rank]
        res, seconds = integrate(j, first, block_samples)
        if world == 1:
            batch.fold(j, res, seconds)
            continue
        buf = np.zeros(nbytes + 8, dtype=np.uint8)
        buf[:nbytes] = np.frombuffer(bytes(res), dtype=np.uint8); buf[nbytes:] = np.frombuffer(np.float64(seconds).tobytes(), dtype=np.uint8)
        t = torch.from_numpy(buf)
        if device is not None:
            t = t.to(device)
        outs = [torch.empty_like(t) for _ in range(world)]
        dist.all_gather(outs, t, group=group)
        for r, o in enumerate(outs):
            raw = o.cpu().numpy().tobytes()
            batch.fold(blocks[r][0], fg.fg_result.from_buffer_copy(raw[:nbytes]), float(np.frombuffer(raw[nbytes:nbytes + 8], dtype=np.float64)[0]))
    return log
