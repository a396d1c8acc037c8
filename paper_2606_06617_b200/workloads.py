"""Seeded synthetic inputs shaped like BASELINE.json's five configurations.

This module holds NONE of the method's arithmetic: it only draws positions and latent
charges (numpy, seeded) and names the plan parameters of each configuration.  It serves the
tests, ``bench.py`` and ``__graft_entry__.smoke()``; the oracle and the CUDA path both receive
the arrays it returns.  Recipes are stated in DESIGN.md §4.  The paper's own benchmark cells
(NaCl / SWM4-NDP / LiPF6 base cells, Pt-water, ByteFF electrolyte) are not
available; these inputs stand in for them.
"""
import numpy as np

C_MOLLIFIER = 12.024   # the paper's accuracy-benchmark bandwidth


def _water_like(rng, n_mol, L):
    """n_mol rigid 3-site molecules: O uniform in the box, H at 0.96 A, HOH = 104.5 deg,
    uniformly random orientation.  Returns pos (3 n_mol, 3) ordered O,H,H per molecule."""
    O = rng.uniform(0.0, L, size=(n_mol, 3))
    # random orthonormal pair (e1, e2) per molecule
    a = rng.normal(size=(n_mol, 3))
    a /= np.linalg.norm(a, axis=1, keepdims=True)
    b = rng.normal(size=(n_mol, 3))
    b -= (b * a).sum(1, keepdims=True) * a
    b /= np.linalg.norm(b, axis=1, keepdims=True)
    half = np.deg2rad(104.5) / 2.0
    d = 0.96
    H1 = O + d * (np.cos(half) * a + np.sin(half) * b)
    H2 = O + d * (np.cos(half) * a - np.sin(half) * b)
    pos = np.stack([O, H1, H2], axis=1).reshape(-1, 3)
    return np.mod(pos, L)


def _neutral_normal(rng, n, std=0.5):
    q = rng.normal(0.0, std, size=n)
    return q - q.mean()


def make(cfg, n_atoms=None, seed=None):
    """Return a dict: pos (N,3), q (C,N), exponents, box, grid, w, c, precision ('f32'|'f64'),
    name.  ``n_atoms`` shrinks/grows the system at FIXED box and grid (used by tests that need
    smaller instances of the same shape).  Arrays are float64; fp32 configs are rounded to
    float32 and back so that the oracle and the GPU see identical numbers."""
    cfg = int(cfg)
    rng = np.random.default_rng(cfg if seed is None else seed)
    if cfg == 1:
        N = 64 if n_atoms is None else n_atoms
        L = 10.0
        pos = rng.uniform(0.0, L, size=(N, 3))
        q = np.where(np.arange(N) % 2 == 0, 1.0, -1.0)[None, :]
        out = dict(name="cfg1-tiny-point-charges", box=[L] * 3, grid=[16] * 3, w=6,
                   exponents=[1], precision="f64")
    elif cfg == 2:
        n_mol = 1000 if n_atoms is None else n_atoms // 3
        L = 31.0
        pos = _water_like(rng, n_mol, L)
        N = len(pos)
        q1 = np.tile([-0.834, 0.417, 0.417], n_mol)
        q6 = rng.lognormal(0.0, 0.3, size=N)
        q = np.stack([q1, q6])
        out = dict(name="cfg2-water-like", box=[L] * 3, grid=[32] * 3, w=6,
                   exponents=[1, 6], precision="f32")
    elif cfg == 3:
        nx, ny, nz = 20, 30, 40                     # rock-salt sites, spacing a/2 = 2.82 A
        a2 = 5.64 / 2.0
        ii, jj, kk = np.meshgrid(np.arange(nx), np.arange(ny), np.arange(nz), indexing="ij")
        pos = np.stack([ii, jj, kk], -1).reshape(-1, 3) * a2
        box = [nx * a2, ny * a2, nz * a2]
        pos = pos + rng.normal(0.0, 0.3, size=pos.shape)
        if n_atoms is not None:
            pos = pos[rng.permutation(len(pos))[:n_atoms]]
        pos = np.mod(pos, box)
        N = len(pos)
        q = np.stack([_neutral_normal(rng, N) for _ in range(8)])
        out = dict(name="cfg3-ionic-melt", box=box, grid=[64] * 3, w=8,
                   exponents=[1, 1, 2, 2, 3, 3, 6, 6], precision="f32")
    elif cfg == 4:
        Ntot = 1_000_000 if n_atoms is None else n_atoms
        n_mol = Ntot // 3
        L = 215.0
        pos = _water_like(rng, n_mol, L)
        pad = Ntot - 3 * n_mol                      # zero-charge padding atoms
        if pad:
            pos = np.concatenate([pos, rng.uniform(0.0, L, size=(pad, 3))])
        N = len(pos)
        live = np.arange(N) < 3 * n_mol
        q1 = np.concatenate([np.tile([-0.834, 0.417, 0.417], n_mol), np.zeros(pad)])
        q1b = np.where(live, rng.normal(0.0, 0.5, size=N), 0.0)
        q1b[live] -= q1b[live].mean()
        q3 = np.where(live, rng.normal(0.0, 0.5, size=N), 0.0)
        q3[live] -= q3[live].mean()
        q6 = np.where(live, rng.lognormal(0.0, 0.3, size=N), 0.0)
        q = np.stack([q1, q1b, q3, q6])
        out = dict(name="cfg4-production-md-box", box=[L] * 3, grid=[128] * 3, w=8,
                   exponents=[1, 1, 3, 6], precision="f32")
    elif cfg == 5:
        N = 200_000 if n_atoms is None else n_atoms
        box = [60.0, 60.0, 300.0]
        pos = np.stack([rng.uniform(0, 60.0, N), rng.uniform(0, 60.0, N),
                        rng.uniform(100.0, 200.0, N)], axis=1)
        q = np.stack([_neutral_normal(rng, N) for _ in range(3)])
        out = dict(name="cfg5-interface-slab", box=box, grid=[64, 64, 320], w=8,
                   exponents=[1, 2, 6], precision="f32")
    else:
        raise ValueError("cfg must be 1..5")
    out["c"] = C_MOLLIFIER
    if out["precision"] == "f32":
        pos = pos.astype(np.float32).astype(np.float64)
        q = q.astype(np.float32).astype(np.float64)
        pos = np.where(pos >= np.asarray(out["box"]), 0.0, pos)  # float32 rounding up to L
    out["pos"] = np.ascontiguousarray(pos)
    out["q"] = np.ascontiguousarray(q)
    return out


def md_displacements(cfg_seed, n_steps, n_atoms, sigma=0.01):
    """Seeded per-step displacements N(0, sigma^2) per coordinate (config 4's stepping loop)."""
    rng = np.random.default_rng(10_000 + cfg_seed)
    for _ in range(n_steps):
        yield rng.normal(0.0, sigma, size=(n_atoms, 3))
