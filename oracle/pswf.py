"""Order-zero prolate spheroidal wave function psi_0^c (oracle, float64).

TEST INFRASTRUCTURE ONLY (see oracle/__init__.py).

The paper defines psi_0^c as the eigenfunction of the truncated Fourier
operator F_c[phi](x) = int_{-1}^{1} phi(t) e^{icxt} dt with the largest
|eigenvalue| (Eq. (7)-(8); SI (S37)-(S38)),
normalised by psi_0^c(0) = 1.  It does not say how to
compute it (it cites Osipov-Rokhlin-Xiao).  DESIGN.md reading R-psi:
the textbook construction -- F_c commutes with the prolate differential operator
L = -d/dx (1-x^2) d/dx + c^2 x^2, whose lowest eigenfunction is psi_0^c; expand in
the even normalised Legendre polynomials Pbar_k = sqrt(k+1/2) P_k, in which L is
symmetric tridiagonal:

    A[k,k]   = k(k+1) + c^2 (2k(k+1)-1) / ((2k+3)(2k-1))
    A[k,k+2] = c^2 (k+1)(k+2) / ((2k+3) sqrt((2k+1)(2k+5))),   k = 0, 2, 4, ...

(from (1-x^2)P_k'' - 2xP_k' = -k(k+1)P_k and the three-term recurrence for x^2 P_k).
The eigen-relation (S38) itself is NOT used here; tests/test_oracle_pswf.py checks
it by quadrature, which pins this construction to the paper's definition.
"""
import numpy as np
from numpy.polynomial import legendre as npleg


class PSWF0:
    """psi_0^c on [-1,1] with psi(0)=1, as a Legendre series."""

    def __init__(self, c, nterms=None):
        c = float(c)
        if not (c > 0):
            raise ValueError("c must be positive")
        self.c = c
        n = int(nterms) if nterms else int(2 * c) + 40  # number of even terms
        k = 2.0 * np.arange(n)  # k = 0, 2, 4, ...
        diag = k * (k + 1) + c * c * (2 * k * (k + 1) - 1) / ((2 * k + 3) * (2 * k - 1))
        off = c * c * (k[:-1] + 1) * (k[:-1] + 2) / (
            (2 * k[:-1] + 3) * np.sqrt((2 * k[:-1] + 1) * (2 * k[:-1] + 5)))
        A = np.diag(diag) + np.diag(off, 1) + np.diag(off, -1)
        evals, evecs = np.linalg.eigh(A)
        beta = evecs[:, 0]  # lowest eigenvalue of L  <->  psi_0
        self.chi0 = float(evals[0])
        # Legendre-series coefficients in the un-normalised P_k basis (all degrees).
        leg = np.zeros(2 * n - 1)
        leg[0::2] = beta * np.sqrt(k + 0.5)
        leg /= npleg.legval(0.0, leg)  # psi(0) = 1
        self.leg = leg
        # lambda_0 = int_{-1}^{1} psi / psi(0)                       (S41)
        self.lambda0 = float(self.integral(-1.0, 1.0))
        # C_0 = int_0^1 psi_0^c(x) dx                              Eq. (3)
        self.C0 = float(self.integral(0.0, 1.0))

    # -- pointwise -------------------------------------------------------------
    def __call__(self, x):
        """psi_0^c(x) for |x| <= 1 (no zero-extension here)."""
        return npleg.legval(np.asarray(x, dtype=np.float64), self.leg)

    def deriv(self, x, m=1):
        """m-th derivative of psi_0^c at x, |x| <= 1."""
        return npleg.legval(np.asarray(x, dtype=np.float64), npleg.legder(self.leg, m))

    def window(self, x):
        """Zero-extended window: psi(x) for |x|<=1, 0 outside.  Eq. (21)."""
        x = np.asarray(x, dtype=np.float64)
        return np.where(np.abs(x) <= 1.0, npleg.legval(np.clip(x, -1, 1), self.leg), 0.0)

    # -- integrals -------------------------------------------------------------
    def integral(self, a, b):
        """int_a^b psi_0^c(t) dt (exact antiderivative of the series)."""
        F = npleg.legint(self.leg)
        return npleg.legval(np.asarray(b, dtype=np.float64), F) - \
            npleg.legval(np.asarray(a, dtype=np.float64), F)


_GL_NODES, _GL_WEIGHTS = np.polynomial.legendre.leggauss(160)


def quad(f, a, b):
    """Gauss-Legendre (160 nodes) of f over [a,b]; a,b may be arrays (broadcast)."""
    a = np.asarray(a, dtype=np.float64)[..., None]
    b = np.asarray(b, dtype=np.float64)[..., None]
    t = 0.5 * (b - a) * _GL_NODES + 0.5 * (b + a)
    return np.sum(f(t) * _GL_WEIGHTS, axis=-1) * 0.5 * (b - a)[..., 0]
