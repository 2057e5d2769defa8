"""Multi-GPU layout of the inversion: contiguous pixel ranges, one process per GPU, no data-path collective.

Pixels are independent (the paper suggests one GPU per MPI rank over scanlines), and the GA's
random streams are keyed by GLOBAL pixel id (reading G0), so rank r inverting pixels [start, start + count) with
`pixel_id_base = start` reproduces the single-GPU result bit for bit.  The only communication is the optional gather of
the 40 B/pixel results at the end (`gather_results`), which works on any torch.distributed backend (nccl on the GPU
box, gloo in the CPU tests).  This module holds host logic only: the compute is `binding.ga_invert`.
"""


def pixel_shard(n_pixels, rank, world):
    """Balanced contiguous range of rank `rank`: returns (start, count). The first n_pixels % world ranks get one more."""
    if world < 1 or not (0 <= rank < world) or n_pixels < 0:
        raise ValueError("bad shard request: n_pixels=%r rank=%r world=%r" % (n_pixels, rank, world))
    q, r = divmod(int(n_pixels), int(world))
    start = rank * q + min(rank, r)
    return start, q + (1 if rank < r else 0)


def shard_counts(n_pixels, world):
    return [pixel_shard(n_pixels, r, world)[1] for r in range(world)]


def invert_shard(engine, obs_local, start, **kw):
    """Runs `engine` (binding.ga_invert, or any callable with its signature) on this rank's pixels, keyed globally."""
    return engine(obs_local, pixel_id_base=start, **kw)


def gather_results(params_local, chi2_local, n_pixels, group=None):
    """All-gathers the per-rank results into full [n_pixels, M] / [n_pixels] tensors on every rank.

    Shards may differ by one pixel, so each rank pads to the largest shard before the (equal-size) all_gather.
    """
    import torch
    import torch.distributed as dist
    world, rank = dist.get_world_size(group), dist.get_rank(group)
    counts = shard_counts(n_pixels, world)
    if params_local.shape[0] != counts[rank] or chi2_local.shape[0] != counts[rank]:
        raise ValueError("rank %d holds %d pixels, its shard has %d" % (rank, params_local.shape[0], counts[rank]))
    cmax, M = max(counts), params_local.shape[1]
    buf = torch.zeros((cmax, M + 1), dtype=params_local.dtype, device=params_local.device)
    buf[:counts[rank], :M] = params_local
    buf[:counts[rank], M] = chi2_local
    parts = [torch.empty_like(buf) for _ in range(world)]
    dist.all_gather(parts, buf, group=group)
    full = torch.cat([p[:c] for p, c in zip(parts, counts)], dim=0)
    return full[:, :M].contiguous(), full[:, M].contiguous()
