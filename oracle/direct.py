"""Oracle A: direct non-uniform Fourier sums, O(N*K), no grid (float64).

TEST INFRASTRUCTURE ONLY (see oracle/__init__.py).

Definition (Eq. (5)-(6)), per channel a with exponent p:

    rho_a(k) = sum_j q_j^a e^{i k.r_j},                    k = 2 pi (m_x/L_x, m_y/L_y, m_z/L_z)
               (general cell, "cell tensor Omega": rows a_1, a_2, a_3 of the 3x3 matrix h are the
                lattice vectors, r = s h with fractional s, and k_m = 2 pi m h^-T so that k_m . r = 2 pi m . s;
                V = |det h|.  `box` may be three edge lengths or such a 3x3 matrix everywhere below.)
    E        = 1/(2V) sum_a [ sum_{k in K} Phi^_p(k) |rho_a(k)|^2 + Phi0_p (Q_net^a)^2 ]
    phi_i^a  = dE/dq_i^a = (1/V) [ sum_K Phi^_p(k) Re(e^{-i k.r_i} rho_a(k)) + Phi0_p Q_net^a ]
    F_i      = -dE/dr_i (q fixed)
             = -(1/V) sum_a q_i^a sum_K Phi^_p(k) k Im(e^{-i k.r_i} rho_a(k))
               (d|rho|^2/dr_i = 2 Re(conj(rho) i k q_i e^{ik.r_i}) = 2 q_i k Im(e^{-ik.r_i} rho))

Mode set K (reading R-modes): all m != 0 with |k| r_c < c (Phi^_p == 0 beyond,
PAPER.md:836) and, when a grid is given, |m_d| < M_d/2 (modes the grid can carry).
No self term and no real-space term: this is the reciprocal part of (S65) only.
"""
import ctypes
import os
import subprocess
import numpy as np
from .kernels import Mollifier


def cell_matrix(box):
    """3x3 cell matrix (rows = lattice vectors) from three edge lengths or a 3x3 array."""
    box = np.asarray(box, dtype=np.float64)
    return np.diag(box) if box.ndim == 1 else box.reshape(3, 3)


def recip_vectors(box, m):
    """k_m = 2 pi m h^-T (rows), Cartesian."""
    return 2 * np.pi * np.asarray(m, dtype=np.float64) @ np.linalg.inv(cell_matrix(box)).T


def mode_set(box, c, r_c, grid=None, half=False):
    """Integer mode vectors m (K,3) of the set K above.  half=True keeps one of each
    +-m pair (the first non-zero component positive)."""
    cell = cell_matrix(box)
    kc = c / r_c
    # |m_d| = |a_d . k| / 2 pi <= |a_d| |k| / 2 pi
    mmax = np.floor(kc * np.linalg.norm(cell, axis=1) / (2 * np.pi)).astype(int) + 1
    if grid is not None:
        # |m_d| < M_d/2  (strict: Nyquist planes excluded, reading R11)
        lim = (np.asarray(grid) - 1) // 2
        mmax = np.minimum(mmax, lim)
    ax = [np.arange(-mm, mm + 1) for mm in mmax]
    m = np.stack(np.meshgrid(*ax, indexing="ij"), axis=-1).reshape(-1, 3)
    k = recip_vectors(cell, m)
    kn = np.sqrt((k ** 2).sum(1))
    keep = (kn * r_c < c) & np.any(m != 0, axis=1)
    m = m[keep]
    if half:
        pos = (m[:, 0] > 0) | ((m[:, 0] == 0) & (m[:, 1] > 0)) | \
              ((m[:, 0] == 0) & (m[:, 1] == 0) & (m[:, 2] > 0))
        m = m[pos]
    return m


def direct_sums(pos, q, exponents, box, c, r_c, grid=None, subset=None, zero_mode=True,
                chunk=2048):
    """E (float), E_channels (C,), phi (C,n_sub), F (n_sub,3) by the sums above (numpy).

    pos (N,3), q (C,N), exponents (C,), box (3,).  subset: indices of the atoms whose
    phi/F are wanted (default all).  The sum runs over the FULL mode set (both +-k).
    """
    pos = np.asarray(pos, dtype=np.float64)
    q = np.atleast_2d(np.asarray(q, dtype=np.float64))
    cell = cell_matrix(box)
    C, N = q.shape
    V = float(abs(np.linalg.det(cell)))
    moll = Mollifier(c, r_c)
    m = mode_set(cell, c, r_c, grid, half=False)
    k = recip_vectors(cell, m)                    # (K,3)
    kn = np.sqrt((k ** 2).sum(1))
    kn_u, inv = np.unique(kn, return_inverse=True)   # Phi^ depends on |k| only
    idx = np.arange(N) if subset is None else np.asarray(subset)
    # structure factors rho_a(k), Eq. (6)
    rho = np.zeros((C, len(k)), dtype=np.complex128)
    for s in range(0, N, chunk):
        ph = np.exp(1j * pos[s:s + chunk] @ k.T)  # (n,K)
        rho += q[:, s:s + chunk] @ ph
    E_ch = np.zeros(C)
    phi = np.zeros((C, len(idx)))
    F = np.zeros((len(idx), 3))
    for a, p in enumerate(exponents):
        Ph = moll.Phi_hat(int(p), kn_u)[inv]      # (K,)
        Qnet = q[a].sum()
        E_ch[a] = (Ph * np.abs(rho[a]) ** 2).sum() / (2 * V)
        if zero_mode:
            E_ch[a] += moll.Phi0(int(p)) * Qnet ** 2 / (2 * V)
        for s in range(0, len(idx), chunk):
            ii = idx[s:s + chunk]
            t = np.exp(-1j * pos[ii] @ k.T) * rho[a]          # e^{-ik.r_i} rho_a(k)
            phi[a, s:s + chunk] = (t.real * Ph).sum(1) / V
            F[s:s + chunk] -= q[a, ii, None] * ((t.imag * Ph) @ k) / V
        if zero_mode:
            phi[a] += moll.Phi0(int(p)) * Qnet / V
    return float(E_ch.sum()), E_ch, phi, F


# ---------------------------------------------------------------------------------
# The same sums in plain C (oracle/direct_sum.c) for the large configurations.
# ---------------------------------------------------------------------------------
_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB = None


def build_c(force=False):
    """Compile oracle/direct_sum.c -> oracle/liboracle_direct.so (gcc -O2 -fopenmp)."""
    src = os.path.join(_HERE, "direct_sum.c")
    out = os.path.join(_HERE, "liboracle_direct.so")
    if force or not os.path.exists(out) or os.path.getmtime(out) < os.path.getmtime(src):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-std=c11",
                               "-o", out, src, "-lm"])
    return out


def _lib():
    global _LIB
    if _LIB is None:
        _LIB = ctypes.CDLL(build_c())
        _LIB.oracle_direct_sums.restype = ctypes.c_int
        _LIB.oracle_threads.restype = ctypes.c_int
    return _LIB


def c_threads():
    return int(_lib().oracle_threads())


def direct_sums_c(pos, q, exponents, box, c, r_c, grid=None, subset=None, zero_mode=True):
    """Same contract as direct_sums(), evaluated by oracle/direct_sum.c over the half mode
    set (x2; rho(-k) = conj rho(k) and Phi^ is even, so the +-k terms of Eq. (5) are equal).
    The mollifier values Phi^_p(|k|) per mode are computed here with kernels.py and passed in.
    """
    pos = np.ascontiguousarray(pos, dtype=np.float64)
    q = np.ascontiguousarray(np.atleast_2d(q), dtype=np.float64)
    cell = cell_matrix(box)
    C, N = q.shape
    moll = Mollifier(c, r_c)
    m = np.ascontiguousarray(mode_set(cell, c, r_c, grid, half=True), dtype=np.int32)
    K = len(m)
    kn = np.sqrt((recip_vectors(cell, m) ** 2).sum(1))
    # the C routine takes fractional coordinates s = r h^-1 (k_m . r = 2 pi m . s), the reciprocal
    # basis 2 pi h^-T (row d = the k vector of m = e_d) for the force, and the cell volume
    frac = np.ascontiguousarray(pos @ np.linalg.inv(cell))
    recip = np.ascontiguousarray(2 * np.pi * np.linalg.inv(cell).T)
    V = float(abs(np.linalg.det(cell)))
    kn_u, inv = np.unique(kn, return_inverse=True)   # Phi^ depends on |k| only
    Ph = np.empty((C, K))
    cache = {}
    for a, p in enumerate(exponents):
        if int(p) not in cache:
            cache[int(p)] = moll.Phi_hat(int(p), kn_u)[inv]
        Ph[a] = cache[int(p)]
    Phi0 = np.array([moll.Phi0(int(p)) if zero_mode else 0.0 for p in exponents])
    idx = np.ascontiguousarray(np.arange(N) if subset is None else subset, dtype=np.int64)
    E_ch = np.zeros(C)
    phi = np.zeros((C, len(idx)))
    F = np.zeros((len(idx), 3))
    dp = ctypes.POINTER(ctypes.c_double)

    def P(a, t=dp):
        return a.ctypes.data_as(t)
    rc = _lib().oracle_direct_sums(
        ctypes.c_long(N), P(frac), ctypes.c_int(C), P(q), P(recip), ctypes.c_double(V),
        ctypes.c_long(K), P(m, ctypes.POINTER(ctypes.c_int32)), P(Ph), P(Phi0),
        ctypes.c_long(len(idx)), P(idx, ctypes.POINTER(ctypes.c_int64)),
        P(E_ch), P(phi), P(F))
    if rc != 0:
        raise RuntimeError("oracle_direct_sums failed: %d" % rc)
    return float(E_ch.sum()), E_ch, phi, F


# ---------------------------------------------------------------------------------
# Virial of the reciprocal sum ("forces and virials").
# ---------------------------------------------------------------------------------
def virial_direct(pos, q, exponents, box, c, r_c, grid=None, zero_mode=True):
    """W_ab = -dE/d(eps_ab) of Eq. (5) under a homogeneous strain r -> (1 + eps) r of atoms and cell at
    fixed q and fixed r_c:  k -> (1 - eps) k, V -> V (1 + tr eps), rho(k) unchanged, hence

        W_ab = (1/2V) sum_{k in K} |rho(k)|^2 [ Phi^(k) delta_ab + Phi^'(k) k_a k_b / |k| ]
               + delta_ab Phi0 Q_net^2 / (2V).

    Phi^' is taken by central differences of Mollifier.Phi_hat (the oracle has no closed form of
    its own for it).  Returns the symmetric 3x3 tensor, summed over channels."""
    pos = np.asarray(pos, dtype=np.float64)
    q = np.atleast_2d(np.asarray(q, dtype=np.float64))
    cell = cell_matrix(box)
    V = float(abs(np.linalg.det(cell)))
    moll = Mollifier(c, r_c)
    m = mode_set(cell, c, r_c, grid, half=False)
    k = recip_vectors(cell, m)
    kn = np.sqrt((k ** 2).sum(1))
    rho = q @ np.exp(1j * pos @ k.T)               # (C, K)
    W = np.zeros((3, 3))
    kc = c / r_c
    for a, p in enumerate(exponents):
        h = 1e-6 * kn
        up = np.minimum(kn + h, kc * (1 - 1e-14))
        Ph = moll.Phi_hat(int(p), kn)
        dPh = (moll.Phi_hat(int(p), up) - moll.Phi_hat(int(p), kn - h)) / (up - (kn - h))
        r2 = np.abs(rho[a]) ** 2
        W += np.eye(3) * (Ph * r2).sum() / (2 * V)
        W += np.einsum("k,ka,kb->ab", dPh * r2 / kn, k, k) / (2 * V)
        if zero_mode:
            W += np.eye(3) * moll.Phi0(int(p)) * q[a].sum() ** 2 / (2 * V)
    return W
