"""Multi-GPU plumbing of the path: patch groups are independent, so
hydro_solve shards over ranks with no data-path collective; the only exchange is one scalar -- the
hydro_dt maximum -- so that every shard of an AMR level advances with the same dt.  One process per GPU;
torch.distributed supplies the transport (NCCL on GPUs, gloo in the CPU tests).  No method arithmetic here."""
import torch
import torch.distributed as dist


def shard_range(Ng, rank, world):
    """Contiguous, balanced partition of Ng groups: ranks < Ng % world get one extra group."""
    if Ng < 0 or world < 1 or not 0 <= rank < world:
        raise ValueError("shard_range: need Ng >= 0 and 0 <= rank < world")
    base, extra = divmod(Ng, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def global_max(speed):
    """In-place MAX all-reduce of the hydro_dt scalar (tensor on the rank's device).  NaN (a bad cell on any
    rank) must win, as it does inside hydro_dt: collectives do not promise NaN propagation, so it travels as +inf and is
    turned back into NaN afterwards (hydro_solve would read +inf as dt = 0 and silently do an identity update)."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return speed
    flag = torch.isnan(speed)
    speed.copy_(torch.where(flag, torch.full_like(speed, float("inf")), speed))
    dist.all_reduce(speed, op=dist.ReduceOp.MAX)
    speed.copy_(torch.where(torch.isinf(speed), torch.full_like(speed, float("nan")), speed))
    return speed
