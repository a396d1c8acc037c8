"""torch.autograd entry point of the PSWF-LR reciprocal-space energy.

The paper obtains forces and dE/dq by automatic differentiation of the LR operator so that an
upstream MLIP can back-propagate through it.  Here the forward pass is ONE
``pswf_lr_execute`` call that returns the energy together with phi = dE/dq and F = -dE/dr (the
analytic gather of §8(a) row a5); backward only scales those by the incoming gradient.  Argument
marshalling and chain-rule glue only: all arithmetic of the path runs in the CUDA library.
"""
import torch

from . import binding


class _LongRangeEnergy(torch.autograd.Function):
    @staticmethod
    def forward(ctx, pos, q, plan, full):
        dt = torch.float64 if plan.precision == binding.PSWF_LR_F64 else torch.float32
        if not (pos.is_cuda and q.is_cuda):
            raise RuntimeError("pswf_lr: tensors must live on a CUDA device (there is no CPU fallback)")
        pos_c = pos.detach().to(dt).contiguous()
        q_c = q.detach().to(dt).contiguous()
        n = pos_c.shape[0]
        C = plan.n_channels
        if q_c.shape != (C, n) or pos_c.shape != (n, 3):
            raise ValueError("pos must be [N,3] and q [n_channels,N]")
        E = torch.empty(1, dtype=torch.float64, device=pos.device)
        phi = torch.empty((C, n), dtype=dt, device=pos.device)
        F = torch.empty((n, 3), dtype=dt, device=pos.device)
        st = torch.cuda.current_stream(pos.device).cuda_stream
        plan.execute(n, pos_c, q_c, E, phi, F, st)
        if full:   # + real-space complement - self term: the complete inverse-power energy (S65)
            plan.execute_real(n, pos_c, q_c, E, phi, F, accumulate=True, stream=st)
        ctx.save_for_backward(phi, F)
        ctx.in_dtypes = (pos.dtype, q.dtype)
        return E[0]

    @staticmethod
    def backward(ctx, gE):
        phi, F = ctx.saved_tensors
        g = gE.to(phi.dtype)
        gpos = (-g) * F if ctx.needs_input_grad[0] else None      # dE/dr = -F
        gq = g * phi if ctx.needs_input_grad[1] else None         # dE/dq = phi
        if gpos is not None:
            gpos = gpos.to(ctx.in_dtypes[0])
        if gq is not None:
            gq = gq.to(ctx.in_dtypes[1])
        return gpos, gq, None, None


def long_range_energy(plan, pos, q, full=False):
    """E_lr(pos, q) as a differentiable 0-dim float64 tensor.  ``plan`` is a ``binding.Plan``;
    ``pos`` [N,3] and ``q`` [n_channels,N] are CUDA tensors.  d/dpos = -F, d/dq = phi.
    ``full=False``: the reciprocal-space part (the hot path); ``full=True``: reciprocal + real-space
    complement - self term, i.e. the complete periodic inverse-power energy (S65)."""
    return _LongRangeEnergy.apply(pos, q, plan, bool(full))
