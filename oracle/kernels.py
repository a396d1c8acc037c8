"""PSWF-mollified inverse-power kernels, p = 1..6 and p = 8, 10 (oracle, float64).

TEST INFRASTRUCTURE ONLY (see oracle/__init__.py).

Notation follows the SI: phi(x) = psi_0^c(x)/psi_0^c(0) (S42),
C_0 = int_0^1 phi (S43), kappa = k r_c, x = kappa/c.
Truncation convention: phi^(k) == 0 for |k| > c, so S^_p(kappa) = 0
for kappa >= c.
"""
import numpy as np
from .pswf import PSWF0, quad

PI = np.pi


class Mollifier:
    """All p = 1..6 kernels for one (c, r_c)."""

    def __init__(self, c, r_c=1.0):
        self.c = float(c)
        self.r_c = float(r_c)
        self.psi = PSWF0(c)
        self.C0 = self.psi.C0

    # ---- ingredients of Theorem 1 -------------------------------------------
    def _A(self, x):
        """(1/C_0) int_0^x phi      (appears in (S48), (S50), (S52))."""
        return self.psi.integral(0.0, x) / self.C0

    def _J(self, n, x):
        """int_x^1 t^n phi(t) dt    (appears in (S50)-(S52))."""
        return quad(lambda t: t ** n * self.psi(t), x, np.ones_like(x))

    def _Llog(self, x):
        """int_x^1 (phi(t) - 1)/t dt  (appears in (S49), (S51), (S77))."""
        def f(t):
            # (phi(t)-1)/t is smooth: phi(0) = 1.  Guard t = 0 (never a GL node).
            return (self.psi(t) - 1.0) / t
        return quad(f, x, np.ones_like(x))

    # ---- Fourier-side splittings, Theorem 1 (S47)-(S52), PAPER.md:852-864 -----
    def S_hat(self, p, kappa):
        """S^_p(kappa), kappa = k r_c > 0 (dimensionless).  Zero for kappa >= c."""
        kappa = np.asarray(kappa, dtype=np.float64)
        c, C0 = self.c, self.C0
        inside = kappa < c
        kap = np.where(inside, kappa, 0.5 * c)  # dummy argument outside the band
        x = kap / c
        if p == 1:   # (S47)
            val = 4 * PI * self.psi(x) / kap ** 2
        elif p == 2:  # (S48)
            val = 2 * PI ** 2 / kap - 2 * PI ** 2 / (C0 * kap) * self.psi.integral(0.0, x)
        elif p == 3:  # (S49)
            val = -4 * PI * np.log(x) + 4 * PI * self._Llog(x)
        elif p == 4:  # (S50)
            val = -PI ** 2 * (kap - kap * self._A(x) - (c / C0) * self._J(1, x))
        elif p == 5:  # (S51)   int (1-phi)/t = -Llog
            val = (2 * PI / 3) * (kap ** 2 * np.log(x) - kap ** 2 * self._Llog(x)
                                  + c ** 2 * self._J(1, x))
        elif p == 6:  # (S52)
            val = (PI ** 2 / 12) * (kap ** 3 - kap ** 3 * self._A(x)
                                    - 3 * c * kap ** 2 / (2 * C0) * self._J(1, x)
                                    + c ** 3 / (2 * C0) * self._J(3, x))
        elif p == 8:
            # (S56), applied to (S52): S^_8(k) = (1/6) int_k^c s S^_6(s) ds  ("The Fourier-space
            # transforms S^_8 and S^_10 follow from (S56) applied to S^_6 in (S52) and S^_8", PAPER.md:905;
            # the upper limit is c by the truncation convention).  With J_n(x) = int_x^1 t^n phi,
            # 1 - A = J_0 / C_0 and int_x^1 y^m J_n(y) dy = (J_{m+n+1}(x) - x^{m+1} J_n(x)) / (m+1):
            #   S^_6 = pi^2 c^3/(12 C_0) [x^3 J_0 - (3/2) x^2 J_1 + (1/2) J_3]
            #   S^_8 = pi^2 c^5/(72 C_0) [-x^5 J_0/5 + (3/8) x^4 J_1 - x^2 J_3/4 + (3/40) J_5]
            val = (PI ** 2 * c ** 5 / (72 * C0)) * (-x ** 5 * self._J(0, x) / 5 + 0.375 * x ** 4 * self._J(1, x)
                                                     - 0.25 * x ** 2 * self._J(3, x) + 0.075 * self._J(5, x))
        elif p == 10:
            # (S56) once more: S^_10(k) = (1/8) int_k^c s S^_8(s) ds
            #   = pi^2 c^7/(576 C_0) [x^7 J_0/35 - x^6 J_1/16 + x^4 J_3/16 - (3/80) x^2 J_5 + J_7/112]
            val = (PI ** 2 * c ** 7 / (576 * C0)) * (x ** 7 * self._J(0, x) / 35 - x ** 6 * self._J(1, x) / 16
                                                      + x ** 4 * self._J(3, x) / 16 - 0.0375 * x ** 2 * self._J(5, x)
                                                      + self._J(7, x) / 112)
        else:
            raise ValueError("p must be in 1..6, 8 or 10")
        return np.where(inside, val, 0.0)

    def Phi_hat(self, p, k):
        """Phi^_p(k) = r_c^(3-p) S^_p(k r_c).   (S60)."""
        k = np.asarray(k, dtype=np.float64)
        return self.r_c ** (3 - p) * self.S_hat(p, k * self.r_c)

    # ---- k = 0 constants: E_0 = Phi0 * Q_net^2 / (2V) -------------------------
    def Phi0(self, p):
        """Zero-mode constant Phi^_p^(0) with E_0^(p) = Phi0 Q_net^2/(2V).

        p=1: (S72)-(S73) PAPER.md:995-1004 with E_IB := 0 (reading R7);
             the SI form is used, not main-text Eq. (18) (reading R6).
        p=2: (S74)-(S75) PAPER.md:1011-1016.
        p=3: finite-part convention (S77)-(S78) PAPER.md:1024-1028 (= Eq. (19)).
        p>3: Phi^_p(0) (S79) PAPER.md:1034 (= Eq. (17)).
        """
        c, C0, rc = self.c, self.C0, self.r_c
        zero = np.zeros(())
        one = np.ones(())
        if p == 1:
            return float(-(2 * PI * rc ** 2 / C0) * quad(lambda u: u ** 2 * self.psi(u), zero, one))
        if p == 2:
            return float(-4 * PI * rc * C0)
        if p == 3:
            return float(4 * PI * (np.log(c / rc) + self._Llog(zero)))
        if p == 4:   # limit kappa -> 0 of (S50)
            return float(rc ** (3 - 4) * PI ** 2 * (c / C0) * self._J(1, zero))
        if p == 5:   # limit of (S51): kappa^2 ln x -> 0
            return float(rc ** (3 - 5) * (2 * PI / 3) * c ** 2 * self._J(1, zero))
        if p == 6:   # limit of (S52)
            return float(rc ** (3 - 6) * (PI ** 2 / 12) * c ** 3 / (2 * C0) * self._J(3, zero))
        if p == 8:   # (S79) with the k -> 0 limit of S^_8 above
            return float(rc ** (3 - 8) * (PI ** 2 * c ** 5 / (72 * C0)) * 0.075 * self._J(5, zero))
        if p == 10:
            return float(rc ** (3 - 10) * (PI ** 2 * c ** 7 / (576 * C0)) * self._J(7, zero) / 112)
        raise ValueError("p must be in 1..6, 8 or 10")

    # ---- real-space long-range kernels (validation scaffold) ------------------
    def S_zero(self, p):
        """S_p(0) from table (S67); even derivatives of phi at 0 from
        the moment formula (S40)."""
        c, C0 = self.c, self.C0

        def d0(two_n):
            n = two_n // 2
            mom = 2 * quad(lambda t: t ** two_n * self.psi(t), np.zeros(()), np.ones(()))
            return float((-1) ** n * c ** two_n * mom / self.psi.lambda0)
        if p == 8:     # (S59)
            return d0(8) / 40320
        if p == 10:
            return -d0(10) / 3628800
        return {1: 1 / C0, 2: -d0(2) / 2, 3: -d0(2) / (3 * C0), 4: d0(4) / 24,
                5: d0(4) / (45 * C0), 6: -d0(6) / 720}[p]

    def S_real(self, p, r):
        """Dimensionless long-range part S_p(r): Props. 2-7, (S17),(S18),(S19),(S24),
        (S29),(S33); S_p(r) = r^-p for r >= 1 (phi truncated at 1)."""
        r = np.asarray(r, dtype=np.float64)
        C0 = self.C0
        inner = r < 1.0
        rr = np.where(inner & (r > 0), r, 0.5)
        phi = self.psi(rr)
        Phi = self.psi.integral(0.0, rr)
        d1 = self.psi.deriv(rr, 1)
        d2 = self.psi.deriv(rr, 2)
        if p == 1:
            val = Phi / (C0 * rr)
        elif p == 2:
            val = (1 - phi) / rr ** 2
        elif p == 3:
            val = (Phi - rr * phi) / (C0 * rr ** 3)
        elif p == 4:
            val = (1 - phi + 0.5 * rr * d1) / rr ** 4
        elif p == 5:
            val = (Phi - rr * phi + rr ** 2 * d1 / 3) / (C0 * rr ** 5)
        elif p == 6:
            val = (1 - phi + 0.625 * rr * d1 - 0.125 * rr ** 2 * d2) / rr ** 6
        elif p == 8:    # Corollary 1 (S57)
            d3 = self.psi.deriv(rr, 3)
            val = (1 - phi + (11 / 16) * rr * d1 - (3 / 16) * rr ** 2 * d2 + rr ** 3 * d3 / 48) / rr ** 8
        elif p == 10:   # (S58)
            d3 = self.psi.deriv(rr, 3)
            d4 = self.psi.deriv(rr, 4)
            val = (1 - phi + (93 / 128) * rr * d1 - (29 / 128) * rr ** 2 * d2 + (7 / 192) * rr ** 3 * d3
                   - rr ** 4 * d4 / 384) / rr ** 10
        else:
            raise ValueError("p must be in 1..6, 8 or 10")
        with np.errstate(divide="ignore"):
            out = np.where(inner, val, np.where(r > 0, r, 1.0) ** (-float(p)))
        return np.where(r == 0, self.S_zero(p), out)

    def S_phys(self, p, r):
        """S_{p,r_c}(r) = r_c^-p S_p(r/r_c).   (S64)."""
        return self.r_c ** (-p) * self.S_real(p, np.asarray(r) / self.r_c)

    def L_phys(self, p, r):
        """Real-space complement L_{p,r_c}(r) = r^-p - S_{p,r_c}(r); zero for r >= r_c."""
        r = np.asarray(r, dtype=np.float64)
        return np.where(r < self.r_c, r ** (-float(p)) - self.S_phys(p, r), 0.0)
