"""Helpers for the -m gpu tests: run the CUDA path through the C ABI and fetch numpy results."""
import numpy as np
import torch

from paper_2606_06617_b200 import binding


def rel(a, b):
    a, b = np.ravel(np.asarray(a, dtype=np.float64)), np.ravel(np.asarray(b, dtype=np.float64))
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def make_plan(wl, **kw):
    args = dict(box=wl["box"], grid=wl["grid"], w=wl["w"], c=wl["c"], exponents=wl["exponents"],
                precision=wl["precision"])
    args.update(kw)
    return binding.Plan(**args)


def run_gpu(wl, plan=None, want=("E", "phi", "F"), pos=None, q=None, **kw):
    """One execute on cuda:0.  Returns dict(E, E_channels, phi, F, info) as float64 numpy."""
    own = plan is None
    if own:
        plan = make_plan(wl, **kw)
    dt = torch.float64 if plan.precision == binding.PSWF_LR_F64 else torch.float32
    dev = torch.device("cuda:0")
    pos_h = wl["pos"] if pos is None else pos
    q_h = wl["q"] if q is None else q
    n = len(pos_h)
    C = plan.n_channels
    pos_d = torch.as_tensor(np.ascontiguousarray(pos_h), dtype=dt, device=dev).contiguous()
    q_d = torch.as_tensor(np.ascontiguousarray(q_h), dtype=dt, device=dev).contiguous()
    E = torch.full((1,), float("nan"), dtype=torch.float64, device=dev) if "E" in want else None
    phi = torch.full((C, n), float("nan"), dtype=dt, device=dev) if "phi" in want else None
    F = torch.full((n, 3), float("nan"), dtype=dt, device=dev) if "F" in want else None
    Ech = torch.zeros(C, dtype=torch.float64, device=dev)
    stream = torch.cuda.current_stream().cuda_stream
    plan.execute(n, pos_d, q_d, E, phi, F, stream)
    plan.channel_energies(Ech, stream)
    torch.cuda.synchronize()
    out = dict(E=None if E is None else float(E.item()), E_channels=Ech.cpu().numpy(),
               phi=None if phi is None else phi.double().cpu().numpy(),
               F=None if F is None else F.double().cpu().numpy(), info=plan.info())
    if own:
        plan.destroy()
    return out
