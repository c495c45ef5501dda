"""Multiple-walker metadynamics with the walkers spread over ranks, one process per GPU.

The per-step path shards by replica with no collective.  The one exchange multiple-walker metadynamics needs is at a deposit
event (every `stride` steps): every rank must append the hills of ALL walkers, in global replica order, so that the hill
lists stay identical.  That is an all-gather of R_local x (n_cv + 1) binary32 numbers per rank (config 1: 6 KB every 500
steps) -- latency-bound, so it is NCCL's all-gather through torch.distributed, not a kernel of ours.  Marshalling only: the
heights and the append are the library's kernels (psg_hill_heights, psg_append_hills).
"""


def deposit_hill_all_ranks(ctx, d_xi, d_mask=None, group=None):
    """One synchronous deposit event of the walkers of every rank.  ``d_xi`` [R_local][n_cv] float32 and ``d_mask`` [R_local]
    uint8 (optional) are this rank's; R_local is the same on every rank.  Afterwards every rank's hill list equals the list
    a single context holding all walkers (rank 0's first) would have built with ``deposit_hill``.  Returns the number of
    (centre, height) pairs appended, zero heights of masked-out walkers included (the library skips them)."""
    import torch
    import torch.distributed as dist

    R = int(d_xi.shape[0])
    d_h = torch.empty(R, dtype=torch.float32, device=d_xi.device)
    ctx.hill_heights(d_xi, d_mask, d_h)
    world = dist.get_world_size(group) if dist.is_available() and dist.is_initialized() else 1
    if world == 1:
        ctx.append_hills(d_xi, d_h)
        return R
    xs = [torch.empty_like(d_xi) for _ in range(world)]
    hs = [torch.empty_like(d_h) for _ in range(world)]
    dist.all_gather(xs, d_xi.contiguous(), group=group)      # rank order = global replica order
    dist.all_gather(hs, d_h, group=group)
    ctx.append_hills(torch.cat(xs).contiguous(), torch.cat(hs).contiguous())
    return world * R
