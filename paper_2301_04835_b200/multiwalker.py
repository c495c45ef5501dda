"""Shared-state methods with the walkers spread over ranks, one process per GPU.

The per-step path shards by replica.  Two methods share state between walkers and need ONE exchange each:

* multiple-walker metadynamics, at a deposit event (every `stride` steps): every rank must append the hills of ALL walkers,
  in global replica order, so that the hill lists stay identical -- an all-gather of R_local x (n_cv + 1) binary32 numbers
  per rank (config 1: 6 KB every 500 steps);
* shared-grid ABF, every step: the histogram and force-sum contributions of all ranks' replicas must be in the grid before
  anyone reads a mean force (reading R-ABF-2) -- an all-reduce of n_bins x (1 + n_cv) numbers (config 2: 48 KB).

Both are latency-bound, so they are NCCL's collectives through torch.distributed, not kernels of ours.  Marshalling only:
heights, appends, binning, grid update and forces are the library's kernels.  The collectives run on torch's CURRENT
stream; the helpers order it against the ctx stream in both directions when the two differ.
"""


def _world(group):
    import torch.distributed as dist
    return dist.get_world_size(group) if dist.is_available() and dist.is_initialized() else 1


class _Ordered:
    """with _Ordered(ctx, tensor): the collectives issued inside wait for the ctx stream's earlier work, and the ctx stream's
    later work waits for them (no-op for CPU tensors, or when the ctx enqueues on torch's current stream)"""

    def __init__(self, ctx, t):
        self.ext = self.cur = None
        h = getattr(ctx, "stream_handle", None)
        if h is not None and t.is_cuda:
            import torch
            cur = torch.cuda.current_stream(t.device)
            if int(h) != int(cur.cuda_stream):
                self.cur, self.ext = cur, torch.cuda.ExternalStream(int(h), device=t.device)

    def __enter__(self):
        if self.ext is not None:
            self.cur.wait_stream(self.ext)
        return self

    def __exit__(self, *exc):
        if self.ext is not None:
            self.ext.wait_stream(self.cur)
        return False


def deposit_hill_all_ranks(ctx, d_xi, d_mask=None, group=None):
    """One synchronous deposit event of the walkers of every rank.  ``d_xi`` [R_local][n_cv] float32 and ``d_mask`` [R_local]
    uint8 (optional) are this rank's; R_local is the same on every rank.  Afterwards every rank holds the IDENTICAL hill
    list: the centres a single context holding all walkers (rank 0's first) would have appended with ``deposit_hill``, with
    heights equal to that context's up to the binary32 rounding of V_old (the hill sum's chunking depends on the number of
    walkers per context).  Walkers masked out are dropped by their zero height; a well-tempered height that underflows to
    0.0f is dropped likewise (it would add nothing to the bias).  Returns the number of (centre, height) pairs gathered."""
    import torch
    import torch.distributed as dist

    R = int(d_xi.shape[0])
    d_h = torch.empty(R, dtype=torch.float32, device=d_xi.device)
    ctx.hill_heights(d_xi, d_mask, d_h)
    world = _world(group)
    if world == 1:
        ctx.append_hills(d_xi, d_h)
        return R
    with _Ordered(ctx, d_h):
        xs = [torch.empty_like(d_xi) for _ in range(world)]
        hs = [torch.empty_like(d_h) for _ in range(world)]
        dist.all_gather(xs, d_xi.contiguous(), group=group)      # rank order = global replica order
        dist.all_gather(hs, d_h, group=group)
        cx, ch = torch.cat(xs).contiguous(), torch.cat(hs).contiguous()
    ctx.append_hills(cx, ch)
    return world * R


def abf_step_all_ranks(ctx, d_pos, d_force, d_fsample, group=None):
    """One ABF step of the replicas of every rank on ONE shared grid (every rank keeps an identical copy):
    ``abf_accumulate_delta`` (this rank's histogram / force-sum contributions of the step) -> all-reduce (sum) over ranks ->
    ``abf_apply_grid_delta`` (grid += total, mean force from the updated grid, force scatter).  The int32 histogram is the one
    a single context holding all replicas builds, bit for bit; the binary32 force sums agree up to the order of additions.
    The two delta buffers live on the ctx object and are reused."""
    import torch
    import torch.distributed as dist

    buf = getattr(ctx, "_abf_delta", None)
    if buf is None or buf[0].device != d_pos.device:
        nb = ctx.abf_n_bins()
        buf = (torch.empty(nb, dtype=torch.int32, device=d_pos.device),
               torch.empty(nb * ctx.n_cv, dtype=torch.float32, device=d_pos.device))
        ctx._abf_delta = buf
    d_h, d_f = buf
    ctx.abf_accumulate_delta(d_pos, d_fsample, d_h, d_f)
    if _world(group) > 1:
        with _Ordered(ctx, d_h):
            dist.all_reduce(d_h, op=dist.ReduceOp.SUM, group=group)
            dist.all_reduce(d_f, op=dist.ReduceOp.SUM, group=group)
    ctx.abf_apply_grid_delta(d_h, d_f, d_pos, d_force)
