"""Multi-GPU sharding of the event loop.

Events are independent and every stage is a stateless function of the global event index
(the Philox counter is the global index), so the path shards with NO data-path
collective: rank r of W evaluates a contiguous range of global event indices on its own GPU.  The
only exchange is the final reduction of three batch sums (sum ME, sum ME^2, sum of event weights),
one all-reduce of three doubles (NCCL over NVLink on GPUs, gloo in the CPU tests).
"""
import torch
import torch.distributed as dist


def event_range(rank, world, n_total, first_event=0):
    """Contiguous, disjoint, exhaustive split of [first_event, first_event + n_total): (first, count)."""
    if not (0 <= rank < world) or n_total < 0:
        raise ValueError("bad rank/world/n_total")
    base, rem = divmod(n_total, world)
    count = base + (1 if rank < rem else 0)
    first = first_event + rank * base + min(rank, rem)
    return first, count


def reduce_sums(local_sums, group=None):
    """All-reduce (sum) of a small float64 tensor of batch sums; identity when not distributed."""
    t = local_sums.to(torch.float64)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
    return t


def sharded_sums(compute, n_total, first_event=0, rank=None, world=None, device="cpu", group=None):
    """Runs `compute(first, count) -> (sum_me, sum_me2, sum_w)` on this rank's event range and
    returns the global (mean ME, standard error of the mean, mean event weight, n_total)."""
    if rank is None:
        rank = dist.get_rank(group) if dist.is_initialized() else 0
    if world is None:
        world = dist.get_world_size(group) if dist.is_initialized() else 1
    first, count = event_range(rank, world, n_total, first_event)
    s = compute(first, count) if count > 0 else (0.0, 0.0, 0.0)
    t = reduce_sums(torch.tensor([float(s[0]), float(s[1]), float(s[2])], dtype=torch.float64, device=device), group)
    mean = t[0].item() / n_total
    var = max(t[1].item() / n_total - mean * mean, 0.0)
    return mean, (var / n_total) ** 0.5, t[2].item() / n_total, n_total


def gpu_compute(process, seed=7):
    """compute() for sharded_sums: the CUDA path on this rank's device for a Process handle: events generated and
    evaluated by mg_sigmakin_fused, batch sums by mg_weight_sums_async (everything stays on the device until the one
    9-double copy at the end)."""
    def compute(first, count):
        dev, dt = process.device, process.dtype
        me = torch.empty(count, dtype=dt, device=dev)
        w = torch.empty(count, dtype=dt, device=dev)
        ew = torch.empty(count, dtype=dt, device=dev)
        process.sigmakin_fused(seed, first, count, me, w, ew)
        s_me = process.weight_sums_async(me, count)
        s_ew = process.weight_sums_async(ew, count)
        v = torch.cat([s_me, s_ew]).cpu()
        return v[0].item(), v[1].item(), v[3].item()
    return compute
