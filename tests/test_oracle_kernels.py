"""Pins for oracle/kernels.py: Theorem 1 (S47)-(S52), the real-space splittings (S17)-(S33),
S_p(0) (S67) and the k = 0 constants, against relations the paper states independently of the
formulas the oracle types in (radial Fourier transform (S2), recurrences (S53)-(S56), limits)."""
import numpy as np
import pytest

from oracle.kernels import Mollifier
from oracle.pswf import quad

PI = np.pi


@pytest.fixture(scope="module")
def m30():
    return Mollifier(30.0, 1.0)


@pytest.fixture(scope="module")
def m12():
    return Mollifier(12.024, 1.0)


def _ft_compact(f, k, n_panels=64):
    """(4 pi / k) int_0^1 r f(r) sin(k r) dr   -- radial transform (S2), of a
    function supported in the unit ball, by composite Gauss-Legendre."""
    edges = np.linspace(0.0, 1.0, n_panels + 1)
    tot = 0.0
    for a, b in zip(edges[:-1], edges[1:]):
        tot += quad(lambda r: r * f(r) * np.sin(k * r), a, b)
    return 4 * PI / k * tot


@pytest.mark.parametrize("p,bare", [(1, lambda k: 4 * PI / k ** 2), (2, lambda k: 2 * PI ** 2 / k)])
def test_S_hat_p12_by_radial_transform(m30, p, bare):
    """S^_p = FT(1/r^p) - FT(L_p), with FT(1/r^p) from Lemma 1 (S5),(S6), and
    FT(L_p) by direct quadrature of (S2) on the compactly supported complement of (S17)/(S18).
    Ties the Fourier-side formulas (S47),(S48) to the REAL-space splittings."""
    for kappa in (0.7, 3.1, 11.0, 23.0):
        # L_p(r) = r^-p - S_p(r), r < 1.  r * L_1 = 1 - Phi/C0 ; r * L_2 = phi / r  (integrable).
        ft_L = _ft_compact(lambda r: r ** (-float(p)) - m30.S_real(p, r), kappa)
        want = bare(kappa) - ft_L
        got = float(m30.S_hat(p, kappa))
        assert abs(got - want) < 2e-9 * bare(kappa), (p, kappa, got, want)


@pytest.mark.parametrize("p", [1, 2, 3, 4, 6, 8])
@pytest.mark.parametrize("c", [12.024, 30.0])
def test_fourier_recurrence_S56(p, c):
    """d/dk S^_{p+2}(k) = -(k/p) S^_p(k)    (S56), PAPER.md:884 (central differences)."""
    m = Mollifier(c, 1.0)
    k = np.array([0.31, 1.7, 0.37 * c, 0.8 * c, 0.97 * c])
    hk = 1e-4
    d = (m.S_hat(p + 2, k + hk) - m.S_hat(p + 2, k - hk)) / (2 * hk)
    want = -(k / p) * m.S_hat(p, k)
    assert np.max(np.abs(d - want)) < 2e-7 * np.max(np.abs(want))


@pytest.mark.parametrize("p", [6, 8])
def test_S_hat_8_10_are_the_integral_S56(m12, p):
    """S^_{p+2}(k) = (1/p) int_k^c s S^_p(s) ds   (S56), PAPER.md:884 with the truncation convention
    (PAPER.md:836), by composite Gauss-Legendre of the oracle's S^_p: pins the closed forms typed for
    p = 8, 10 (and their normalisation, which the derivative form of (S56) leaves free)."""
    c = m12.c
    for kappa in (0.4, 2.9, 0.55 * c, 0.9 * c):
        edges = np.linspace(kappa, c, 9)
        I = sum(quad(lambda s: s * m12.S_hat(p, s), a, b) for a, b in zip(edges[:-1], edges[1:]))
        got = float(m12.S_hat(p + 2, kappa))
        assert abs(got - I / p) < 1e-11 * abs(float(m12.S_hat(p + 2, 0.01))), (p, kappa, got, I / p)


@pytest.mark.parametrize("p", [2, 3, 4, 5, 6, 8, 10])
def test_S_hat_vanishes_at_band_edge(m12, p):
    """S^_p(c) = 0, PAPER.md:866 (fixes the integration constant the recurrence leaves free)."""
    scale = abs(float(m12.S_hat(p, 0.3 * m12.c)))
    assert abs(float(m12.S_hat(p, m12.c * (1 - 1e-12)))) < 1e-9 * scale
    assert float(m12.S_hat(p, m12.c)) == 0.0
    assert float(m12.S_hat(p, 1.5 * m12.c)) == 0.0


def test_S_hat_1_band_edge_is_phi1(m12):
    """For p = 1 the edge value is 4 pi phi(1)/c^2, small but not zero (reading R8)."""
    v = float(m12.S_hat(1, m12.c * (1 - 1e-13)))
    assert abs(v - 4 * PI * m12.psi(1.0) / m12.c ** 2) < 1e-12
    assert 0 < v < 1e-5


@pytest.mark.parametrize("p", [1, 2])
def test_small_k_limits_singular(m12, p):
    """k -> 0: S^_1 -> 4 pi/k^2, S^_2 -> 2 pi^2/k (the windowed kernels keep the bare singularity,
    PAPER.md:866 'unwindowed transform plus a smooth correction')."""
    k = 1e-4
    bare = 4 * PI / k ** 2 if p == 1 else 2 * PI ** 2 / k
    assert abs(float(m12.S_hat(p, k)) / bare - 1) < 1e-3


@pytest.mark.parametrize("p", [4, 5, 6, 8, 10])
def test_Phi0_is_small_k_limit(p):
    """(S79)/(17): for p > 3 the zero-mode constant is the k -> 0 limit of Phi^_p."""
    m = Mollifier(12.024, 2.3)
    lim = float(m.Phi_hat(p, 1e-7))
    assert abs(m.Phi0(p) - lim) < 1e-5 * abs(lim)


def test_Phi0_p3_finite_part():
    """(S77): FP_{k->0} Phi^_3 = lim [Phi^_3(k) + 4 pi ln k]."""
    m = Mollifier(12.024, 2.3)
    k = 1e-6
    assert abs(m.Phi0(3) - (float(m.Phi_hat(3, k)) + 4 * PI * np.log(k))) < 1e-8


def test_Phi0_p12_are_minus_integral_of_complement():
    """(S69)-(S71): E_bg = -(Q^2/2V) I_p, I_p = 4 pi int r^2 L_{p,r_c}(r) dr; so Phi0_p = -I_p."""
    m = Mollifier(12.024, 1.9)
    for p in (1, 2):
        I = 4 * PI * sum(quad(lambda r: r ** 2 * m.L_phys(p, r), a, b)
                         for a, b in zip(np.linspace(0, 1.9, 33)[:-1], np.linspace(0, 1.9, 33)[1:]))
        assert abs(m.Phi0(p) + I) < 1e-10 * I


def test_scaling_S60():
    """Phi^_p(k; r_c) = r_c^(3-p) S^_p(k r_c)    (S60)."""
    a, b = Mollifier(12.024, 1.0), Mollifier(12.024, 3.7)
    k = np.array([0.2, 1.0, 2.5])
    for p in (1, 2, 3, 4, 5, 6, 8, 10):
        assert np.allclose(b.Phi_hat(p, k), 3.7 ** (3 - p) * a.S_hat(p, k * 3.7), rtol=1e-14)


def test_main_text_Eq14_p6_equals_SI(m12):
    """Eq. (14), typed from the main text (lambda_0 psi(x/c), C^_0 = 2 c C_0^2 (S45))
    equals the SI form (S52) the oracle uses."""
    c, C0, lam = m12.c, m12.C0, m12.psi.lambda0
    Chat0 = quad(lambda x: lam * m12.psi(x / c), 0.0, c)
    assert abs(Chat0 - 2 * c * C0 ** 2) < 1e-13        # (S45)
    f = lambda x: lam * m12.psi(x / c)
    for k in (0.9, 4.4, 10.0):
        rc = 1.0
        val = PI ** 2 / (12 * Chat0) * (Chat0 * k ** 3 - k ** 3 * quad(f, 0.0, k * rc)
                                        - 3 * k ** 2 / (2 * rc) * quad(lambda x: x * f(x), k * rc, c)
                                        + 1 / (2 * rc ** 3) * quad(lambda x: x ** 3 * f(x), k * rc, c))
        # the four terms cancel towards the band edge: tolerance relative to S^_6(0)
        assert abs(val - float(m12.S_hat(6, k))) < 1e-12 * m12.Phi0(6)


# ---- real-space side (validation scaffold) ----------------------------------------------

@pytest.mark.parametrize("p", range(1, 7))
def test_S_real_small_r_limit_is_S67(m12, p):
    """lim_{r->0} S_p(r) = table (S67), PAPER.md:958-967 (derivatives at 0 via (S40))."""
    r = 2e-2
    # S_p is even and smooth: S_p(r) = S_p(0) + O(r^2)
    assert abs(float(m12.S_real(p, r)) / m12.S_zero(p) - 1) < 3e-2
    r2 = 1e-2
    extrap = (4 * float(m12.S_real(p, r2)) - float(m12.S_real(p, r))) / 3   # Richardson in r^2
    tol = {1: 1e-6, 2: 1e-6, 3: 1e-5, 4: 1e-4, 5: 1e-3, 6: 5e-2}[p]        # O(r^4) remainder; cancellation grows with p
    assert abs(extrap / m12.S_zero(p) - 1) < tol


@pytest.mark.parametrize("p", [8, 10])
def test_S_real_8_10_small_r_limit_is_S59(p):
    """(S59): S_8(0) = phi^(8)(0)/8!, S_10(0) = -phi^(10)(0)/10! (derivatives at 0 from the
    moments (S40)).  A narrow-band window (c = 4) keeps c r small where r^-p is still representable."""
    m = Mollifier(4.0, 1.0)
    r, r2 = 0.16, 0.08
    extrap = (4 * float(m.S_real(p, r2)) - float(m.S_real(p, r))) / 3   # Richardson in r^2
    assert abs(extrap / m.S_zero(p) - 1) < {8: 2e-3, 10: 2e-2}[p]
    assert m.S_zero(p) > 0


@pytest.mark.parametrize("p", [1, 2, 3, 4, 5, 6, 8, 10])
def test_S_real_matches_bare_kernel_outside(m30, p):
    """S_p(r) = 1/r^p for r >= 1 and is continuous there up to O(phi(1))."""
    assert float(m30.S_real(p, 1.3)) == pytest.approx(1.3 ** -p, rel=1e-15)
    # the jump at r = 1 is O(c^n phi(1)) with n the highest derivative of phi in the numerator
    assert abs(float(m30.S_real(p, 1 - 1e-9)) - 1.0) < {8: 1e-5, 10: 1e-3}.get(p, 1e-7)


@pytest.mark.parametrize("p", [1, 2, 3, 4, 6, 8])
def test_real_space_recurrence_S55(m12, p):
    """S_{p+2}(r) = -(1/(p r)) dS_p/dr    (S53)-(S55)."""
    # (numerator / r^p loses digits at small r: the higher exponents are checked further out)
    r = np.array([0.15, 0.4, 0.77]) if p < 6 else np.array([0.3, 0.5, 0.77])
    hr = 1e-5
    d = (m12.S_real(p, r + hr) - m12.S_real(p, r - hr)) / (2 * hr)
    want = m12.S_real(p + 2, r)
    assert np.max(np.abs(-d / (p * r) - want) / np.abs(want)) < 1e-6


def test_G1_and_G6_main_text(m12):
    """Eq. (3)-(4): G_p(r) = (r/r_c)^p S_p(r/r_c)  ((S60)-(S61))."""
    r = np.array([0.2, 0.5, 0.9])
    G1 = m12.psi.integral(0.0, r) / m12.C0
    assert np.allclose(r * m12.S_real(1, r), G1, rtol=1e-13)
    G6 = 1 - m12.psi(r) + 5 * r / 8 * m12.psi.deriv(r, 1) - r ** 2 / 8 * m12.psi.deriv(r, 2)
    assert np.allclose(r ** 6 * m12.S_real(6, r), G6, rtol=1e-12)
