"""Walker sharding across ranks - host logic only.

Walkers are independent ("vectorizes the computation over an array of sources"; the paper's
2-GPU mode splits that array), so the path shards by rows of params[B, 11] with the data
stream replicated on every GPU.  There is no data-path collective: each rank evaluates its own rows and
the only exchange is the concatenation of the logL slices (8 B per walker).
"""
import torch
import torch.distributed as dist


def shard_rows(B, world, rank):
    """Contiguous balanced row range [start, stop) of rank `rank`; the first B % world ranks get one extra row."""
    if world < 1 or not (0 <= rank < world) or B < 0:
        raise ValueError("bad shard arguments")
    base, extra = divmod(B, world)
    start = rank * base + min(rank, extra)
    return start, start + base + (1 if rank < extra else 0)


def sharded_loglike(evaluate, params, group=None):
    """logL[B] for params[B, 11] with the rows split across the ranks of `group`.

    evaluate(rows) -> 1-D float64 tensor of len(rows) on the rows' device (e.g. lambda p: mbhl_loglike(ctx, p)).
    Every rank passes the same params and receives the full logL vector, rows in the original order.
    Without an initialised process group this is evaluate(params).
    """
    if not (dist.is_available() and dist.is_initialized()):
        return evaluate(params)
    world, rank = dist.get_world_size(group), dist.get_rank(group)
    B = int(params.shape[0])
    start, stop = shard_rows(B, world, rank)
    mine = evaluate(params[start:stop])
    if mine.shape != (stop - start,) or mine.dtype != torch.float64:
        raise ValueError("evaluate must return a float64 vector with one entry per row")
    # all_gather needs equal sizes: pad every slice to the largest one
    width = -(-B // world) if B else 0
    padded = torch.zeros(width, dtype=torch.float64, device=mine.device)
    padded[: stop - start] = mine
    parts = [torch.empty_like(padded) for _ in range(world)]
    dist.all_gather(parts, padded, group=group)
    out = torch.empty(B, dtype=torch.float64, device=mine.device)
    for r in range(world):
        a, b = shard_rows(B, world, r)
        out[a:b] = parts[r][: b - a]
    return out
