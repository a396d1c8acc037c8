"""Pins for oracle/pswf.py against the paper's DEFINITION of psi_0^c (not the construction
the oracle uses) and against an independent library routine."""
import numpy as np
import pytest
from scipy.special import pro_ang1

from oracle.pswf import PSWF0, quad

CS = [4.0, 12.024, 13.75, 30.0]


@pytest.mark.parametrize("c", CS)
def test_eigen_relation_S38(c):
    """lambda_0 psi(x) = int_{-1}^{1} psi(t) e^{icxt} dt   (S38).
    The oracle builds psi from the prolate ODE; this checks the integral-operator definition."""
    psi = PSWF0(c)
    x = np.linspace(-1, 1, 21)
    lhs = psi.lambda0 * psi(x)
    rhs = np.array([quad(lambda t: psi(t) * np.cos(c * xi * t), -1.0, 1.0) for xi in x])
    assert np.max(np.abs(lhs - rhs)) < 5e-14 * psi.lambda0
    # imaginary part vanishes (psi even)
    im = np.array([quad(lambda t: psi(t) * np.sin(c * xi * t), -1.0, 1.0) for xi in x])
    assert np.max(np.abs(im)) < 1e-14


@pytest.mark.parametrize("c", CS)
def test_largest_eigenvalue_and_shape(c):
    """psi_0 belongs to the LARGEST |lambda|: psi_n has n zeros in (-1,1), so the
    order-zero function is the one without a sign change; it is even,
    psi(0) = 1 and decreases on [0,1] (Def. 1)."""
    psi = PSWF0(c)
    x = np.linspace(0, 1, 400)
    v = psi(x)
    assert abs(v[0] - 1.0) < 1e-15
    assert np.all(v > 0)
    assert np.all(np.diff(v) < 0)
    assert np.max(np.abs(psi(-x) - v)) < 1e-15


@pytest.mark.parametrize("c", CS)
def test_lambda0_is_integral_S41(c):
    """lambda_0 psi(0) = int psi  (S41), PAPER.md:828  =>  lambda_0 = 2 C_0 (psi even)."""
    psi = PSWF0(c)
    assert abs(psi.lambda0 - 2 * psi.C0) < 1e-15
    assert abs(psi.lambda0 - quad(lambda t: psi(t), -1.0, 1.0)) < 1e-14


@pytest.mark.parametrize("c", [4.0, 12.024, 13.75])
def test_against_scipy_pro_ang1(c):
    """Library special case: angular prolate function S_00(c, x); ratio to its value at 0."""
    psi = PSWF0(c)
    x = np.linspace(0, 0.99, 34)
    ref = np.array([pro_ang1(0, 0, c, xi)[0] for xi in x]) / pro_ang1(0, 0, c, 0.0)[0]
    assert np.max(np.abs(psi(x) - ref)) < 1e-12


def test_large_c_asymptote():
    """lambda_0 -> sqrt(2 pi / c) and psi(x) -> exp(-c x^2 / 2) as c grows (classical asymptotics)."""
    psi = PSWF0(30.0)
    assert abs(psi.lambda0 / np.sqrt(2 * np.pi / 30.0) - 1) < 1e-6
    x = np.linspace(0, 0.3, 7)
    assert np.max(np.abs(psi(x) - np.exp(-30.0 * x ** 2 / 2))) < 0.02


@pytest.mark.parametrize("c", CS)
def test_moment_formula_S40(c):
    """lambda_0 psi^(2n)(0) = (-1)^n c^(2n) int t^(2n) psi   (S40)."""
    psi = PSWF0(c)
    for n in (1, 2, 3):
        lhs = psi.lambda0 * psi.deriv(0.0, 2 * n)
        rhs = (-1) ** n * c ** (2 * n) * quad(lambda t: t ** (2 * n) * psi(t), -1.0, 1.0)
        assert abs(lhs - rhs) < 1e-9 * abs(rhs)


def test_series_truncation_converged():
    a, b = PSWF0(13.75), PSWF0(13.75, nterms=120)
    x = np.linspace(-1, 1, 101)
    assert np.max(np.abs(a(x) - b(x))) < 1e-14
    assert abs(a.lambda0 - b.lambda0) < 1e-15


def test_window_zero_extension():
    psi = PSWF0(16.65)
    assert psi.window(1.0000001) == 0.0 and psi.window(-1.5) == 0.0
    assert psi.window(0.25) == psi(0.25)
