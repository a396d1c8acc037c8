"""Validation scaffold: the pieces of (S65) that are NOT on the hot path (float64).

TEST INFRASTRUCTURE ONLY (see oracle/__init__.py).  Never timed.  `real_space_parts` is the
parity target of the library's real-space row (pswf_lr_execute_real).
It exists so the oracle's reciprocal part can be pinned to physics the paper fixes: the total

    E^(p) = E_real + (1/2V) sum_{k!=0} Phi^ |rho|^2 + E_0 - E_self        (S65)

must equal the plain periodic inverse-power energy, independently of (c, r_c).
"""
import itertools
import numpy as np
from scipy.special import erfc
from .kernels import Mollifier
from .direct import direct_sums, cell_matrix


def image_range(cell, r):
    """Per lattice direction, the largest |n_d| whose image can come within r: ceil(r / width_d) with
    width_d = V / |a_e x a_f| the distance between the cell faces spanned by the other two vectors."""
    V = abs(np.linalg.det(cell))
    width = np.array([V / np.linalg.norm(np.cross(cell[(d + 1) % 3], cell[(d + 2) % 3])) for d in range(3)])
    return np.ceil(r / width).astype(int)


def real_space_complement(pos, q, p, box, moll):
    """E_real = 1/2 sum_n sum_{i,j}' q_i q_j L_{p,r_c}(|r_ij + n.L|)   (S64)-(S65).
    L_{p,r_c} vanishes beyond r_c, so only images within r_c are visited."""
    pos = np.asarray(pos, dtype=np.float64)
    q = np.asarray(q, dtype=np.float64)
    cell = cell_matrix(box)
    nmax = image_range(cell, moll.r_c)
    E = 0.0
    d0 = pos[:, None, :] - pos[None, :, :]
    qq = q[:, None] * q[None, :]
    for n in itertools.product(*[range(-k, k + 1) for k in nmax]):
        d = d0 + np.asarray(n, dtype=np.float64) @ cell
        r = np.sqrt((d ** 2).sum(-1))
        mask = (r > 0) & (r < moll.r_c)
        if n == (0, 0, 0):
            mask &= ~np.eye(len(pos), dtype=bool)
        E += 0.5 * np.sum(qq[mask] * moll.L_phys(p, r[mask]))
    return float(E)


def real_space_parts(pos, q, exponents, box, c, r_c, fd=1e-6, subset=None):
    """Real-space complement minus self term for several channels: returns (E, phi[C][N], F[N][3]) with
        E   = sum_a [ 1/2 sum_n sum_{i,j}' q_i^a q_j^a L_{p_a,r_c}(|r_ij + n.L|) - E_self^a ]   (S64)-(S66)
        phi = dE/dq_i^a = sum_j q_j^a L(r_ij) - S_p(0) q_i^a / r_c^p
        F_i = -dE/dr_i, with dL/dr by central differences of L (step fd): the scaffold has no
              closed-form derivative of its own, and none is needed at 1e-8 relative accuracy.
    With `subset` (atom indices) only those atoms' phi and F are computed (rows of the pair sum against
    ALL atoms) and E is None: the sampled check of large systems.
    The image loops cover ceil(r_c / width) cells around positions INSIDE the cell: wrap them first."""
    pos = np.asarray(pos, dtype=np.float64)
    q = np.atleast_2d(np.asarray(q, dtype=np.float64))
    cell = cell_matrix(box)
    moll = Mollifier(c, r_c)
    N = len(pos)
    phi = np.zeros_like(q)
    F = np.zeros((N, 3))
    nmax = image_range(cell, r_c)
    rows = np.arange(N) if subset is None else np.asarray(subset)
    d0 = pos[None, :, :] - pos[rows, None, :]       # d0[i, j] = r_j - r_rows[i]
    for n in itertools.product(*[range(-k, k + 1) for k in nmax]):
        d = d0 + np.asarray(n, dtype=np.float64) @ cell
        r = np.sqrt((d ** 2).sum(-1))
        mask = (r > 0) & (r < r_c)
        if not mask.any():
            continue
        ii, jj = np.nonzero(mask)
        rr = r[ii, jj]
        ri = rows[ii]
        for a, p in enumerate(exponents):
            L = moll.L_phys(p, rr)
            dL = (moll.L_phys(p, np.minimum(rr + fd, r_c * (1 - 1e-15))) - moll.L_phys(p, rr - fd)) / \
                 (np.minimum(rr + fd, r_c * (1 - 1e-15)) - (rr - fd))
            np.add.at(phi[a], ri, q[a, jj] * L)
            f = (q[a, ri] * q[a, jj] * dL / rr)[:, None] * d[ii, jj]      # F_i = + qq L'(r) (r_j - r_i)/r
            np.add.at(F, ri, f)
    for a, p in enumerate(exponents):
        phi[a] -= moll.S_zero(p) * q[a] / r_c ** p
    if subset is not None:
        return None, phi[:, rows], F[rows]
    E = 0.5 * float(np.sum(q * phi))
    return E, phi, F


def self_energy(q, p, moll):
    """E_self = S_p(0) Q_self / (2 r_c^p)      (S66)."""
    q = np.asarray(q, dtype=np.float64)
    return float(moll.S_zero(p) * np.sum(q ** 2) / (2 * moll.r_c ** p))


def total_energy(pos, q, p, box, c, r_c):
    """Full decomposition (S65) for one channel; reciprocal part = oracle A without a grid."""
    moll = Mollifier(c, r_c)
    E_rec, _, _, _ = direct_sums(pos, q[None, :], [p], box, c, r_c, grid=None)
    return real_space_complement(pos, q, p, box, moll) + E_rec - self_energy(q, p, moll)


def ewald_erfc_energy(pos, q, box, alpha, r_cut, kmax):
    """Classical Coulomb Ewald sum (Eq. (12) with p = 1: G = erfc(alpha r)), tinfoil
    boundary, neutralising background for net charge.  Independent of every PSWF routine."""
    pos = np.asarray(pos, dtype=np.float64)
    q = np.asarray(q, dtype=np.float64)
    box = np.asarray(box, dtype=np.float64)
    V = float(np.prod(box))
    nmax = np.ceil(r_cut / box).astype(int)
    E = 0.0
    d0 = pos[:, None, :] - pos[None, :, :]
    qq = q[:, None] * q[None, :]
    for n in itertools.product(*[range(-k, k + 1) for k in nmax]):
        d = d0 + np.asarray(n) * box
        r = np.sqrt((d ** 2).sum(-1))
        mask = (r > 0) & (r < r_cut)
        E += 0.5 * np.sum(qq[mask] * erfc(alpha * r[mask]) / r[mask])
    ax = [np.arange(-kmax, kmax + 1)] * 3
    m = np.stack(np.meshgrid(*ax, indexing="ij"), -1).reshape(-1, 3)
    m = m[np.any(m != 0, axis=1)]
    k = 2 * np.pi * m / box
    k2 = (k ** 2).sum(1)
    rho = (q[None, :] * np.exp(1j * k @ pos.T)).sum(1)
    E += (2 * np.pi / V) * np.sum(np.exp(-k2 / (4 * alpha ** 2)) / k2 * np.abs(rho) ** 2)
    E -= alpha / np.sqrt(np.pi) * np.sum(q ** 2)
    E -= np.pi * q.sum() ** 2 / (2 * V * alpha ** 2)
    return float(E)


def brute_force_image_sum(pos, q, p, box, nmax):
    """1/2 sum_{|n_d|<=nmax} sum_{i,j}' q_i q_j / |r_ij + n.L|^p  (absolutely convergent for p > 3)."""
    pos = np.asarray(pos, dtype=np.float64)
    q = np.asarray(q, dtype=np.float64)
    cell = cell_matrix(box)
    d0 = pos[:, None, :] - pos[None, :, :]
    qq = q[:, None] * q[None, :]
    E = 0.0
    rng = range(-nmax, nmax + 1)
    for n in itertools.product(rng, rng, rng):
        d = d0 + np.asarray(n, dtype=np.float64) @ cell
        r2 = (d ** 2).sum(-1)
        mask = r2 > 0
        E += 0.5 * np.sum(qq[mask] * r2[mask] ** (-p / 2.0))
    return float(E)
