"""Channel-sharded evaluation across GPUs (the strong-scaling split of the path).

The channels of Eq. (5) are independent up to the final sums: positions are replicated, rank g
evaluates the channels a with a mod G == g (its own plan with those exponents -- one batched
transform over its channels), and ONE exchange step follows the gather:

    F   = sum over ranks of the rank's force contribution      all-reduce, N x 3
    E   = sum over ranks of the rank's channel energies         all-reduce, 1 double
    phi = per channel, owned by the rank that evaluated it      (optionally all-gathered)

One process per GPU, ``torch.distributed`` for the plumbing (NCCL on GPUs; the same code runs under
gloo on CPU tensors, which is how tests/test_multi_rank.py covers it with oracle evaluations).  No
arithmetic of the path lives here: the evaluation is a callable -- on a GPU box the C library.
"""
import torch
import torch.distributed as dist


def channel_partition(n_channels, world, rank):
    """Indices of the channels rank `rank` owns: a = rank, rank + world, ... (round robin, so that
    repeated exponents -- config 3 lists every exponent twice -- spread over the ranks)."""
    if not (0 <= rank < world):
        raise ValueError("rank outside the world")
    return list(range(rank, n_channels, world))


def reduce_results(E_local, F_local, group=None):
    """The exchange step: sums E (float64 tensor of 1) and F (N x 3) over the ranks, in place.
    Ranks that own no channel pass zeros.  Returns (E, F)."""
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(F_local, op=dist.ReduceOp.SUM, group=group)
        dist.all_reduce(E_local, op=dist.ReduceOp.SUM, group=group)
    return E_local, F_local


def gather_potentials(phi_local, n_channels, world, rank, group=None):
    """phi[C][N] on every rank from the per-rank blocks (channel a sits on rank a mod world).  Optional:
    an MD step needs only F and E."""
    N = phi_local.shape[1]
    per = (n_channels + world - 1) // world
    pad = torch.zeros((per, N), dtype=phi_local.dtype, device=phi_local.device)
    pad[: phi_local.shape[0]] = phi_local
    if dist.is_available() and dist.is_initialized() and world > 1:
        blocks = [torch.empty_like(pad) for _ in range(world)]
        dist.all_gather(blocks, pad, group=group)
    else:
        blocks = [pad]
    phi = torch.empty((n_channels, N), dtype=phi_local.dtype, device=phi_local.device)
    for r in range(world):
        own = channel_partition(n_channels, world, r)
        if own:
            phi[own] = blocks[r][: len(own)]
    return phi


class ChannelShardedPlan:
    """pswf_lr plan over this rank's channels + the exchange step.  `box` as in binding.Plan."""

    def __init__(self, box, grid, w, c, exponents, rank=None, world=None, group=None, **plan_kw):
        from . import binding
        self.group = group
        self.world = world if world is not None else (dist.get_world_size(group) if dist.is_initialized() else 1)
        self.rank = rank if rank is not None else (dist.get_rank(group) if dist.is_initialized() else 0)
        self.n_channels = len(exponents)
        self.own = channel_partition(self.n_channels, self.world, self.rank)
        self.plan = None
        if self.own:
            self.plan = binding.Plan(box, grid, w, c, [exponents[a] for a in self.own], **plan_kw)
        self.dtype = torch.float64 if plan_kw.get("precision", "f32") == "f64" else torch.float32

    def execute(self, pos, q, want_phi=False):
        """pos [N,3], q [C,N] device tensors replicated on every rank.  Returns (E, F[, phi]) identical on
        every rank; E is a float64 tensor of 1."""
        dev = pos.device
        n = pos.shape[0]
        E = torch.zeros(1, dtype=torch.float64, device=dev)
        F = torch.zeros((n, 3), dtype=self.dtype, device=dev)
        phi_l = torch.zeros((len(self.own), n), dtype=self.dtype, device=dev)
        if self.plan is not None:
            q_l = q[self.own].contiguous()
            st = torch.cuda.current_stream(dev).cuda_stream
            self.plan.execute(n, pos, q_l, E, phi_l if want_phi else None, F, st)
        reduce_results(E, F, self.group)
        if want_phi:
            return E, F, gather_potentials(phi_l, self.n_channels, self.world, self.rank, self.group)
        return E, F

    def destroy(self):
        if self.plan is not None:
            self.plan.destroy()
            self.plan = None
