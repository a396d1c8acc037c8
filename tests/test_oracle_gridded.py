"""Pins for oracle B (oracle/gridded.py): it must converge spectrally to oracle A (the definition)
as the window widens, and be the exact gradient of its own discrete energy."""
import numpy as np
import pytest

from oracle import gridded as G
from oracle.direct import direct_sums
from oracle.pswf import PSWF0
from paper_2606_06617_b200 import workloads


def _rel(a, b):
    return np.linalg.norm(np.ravel(a) - np.ravel(b)) / np.linalg.norm(np.ravel(b))


@pytest.fixture(scope="module")
def cfg1():
    w = workloads.make(1)
    w["r_c"] = G.default_r_c(w["box"], w["grid"], w["c"])
    return w


@pytest.fixture(scope="module")
def cfg1_A(cfg1):
    w = cfg1
    return direct_sums(w["pos"], w["q"], w["exponents"], w["box"], w["c"], w["r_c"], grid=w["grid"])


@pytest.mark.parametrize("width,tolE,tolF", [(6, 3e-6, 1e-4), (8, 2e-7, 5e-6), (12, 1e-10, 3e-9),
                                             (16, 2e-13, 5e-12)])
def test_B_converges_to_A(cfg1, cfg1_A, width, tolE, tolF):
    """Spectral convergence in the window width, config-1 system (eta = 0.5).
    Levels follow SURVEY.md §8(c)'s probe table (w=6: 3e-7/2.3e-5 ... w=16: 7e-16/1.5e-14)."""
    w = cfg1
    E, Ech, phi, F = G.gridded(w["pos"], w["q"], w["exponents"], w["box"], w["grid"], width,
                               w["c"], w["r_c"], G.default_c_w(width))
    EA, _, phiA, FA = cfg1_A
    assert abs(E - EA) / abs(EA) < tolE
    assert _rel(F, FA) < tolF
    assert _rel(phi, phiA) < tolF


def test_fp32_gates_reachable_at_spec_width(cfg1, cfg1_A):
    """DESIGN.md reading R1(iii): at the specified w = 6, |B - A| is inside the fp32 gates
    (1e-5 in E, 1e-4 in F), so the discretisation leaves room for fp32 rounding."""
    w = cfg1
    E, _, _, F = G.gridded(w["pos"], w["q"], w["exponents"], w["box"], w["grid"], w["w"],
                           w["c"], w["r_c"], G.default_c_w(w["w"]))
    assert abs(E - cfg1_A[0]) / abs(cfg1_A[0]) < 1e-5
    assert _rel(F, cfg1_A[3]) < 1e-4


def test_spectral_energy_equals_half_q_phi(cfg1):
    """Reading R10: with D = (h^3/M_tot) Phi^/W^^2 and unnormalised DFTs, Eq. (26)'s Fourier-space
    reduction equals 1/2 sum q phi to rounding."""
    w = cfg1
    E, Ech, phi, F, im = G.gridded(w["pos"], w["q"], w["exponents"], w["box"], w["grid"], 8,
                                   w["c"], w["r_c"], G.default_c_w(8), intermediates=True)
    assert np.allclose(im["E_spec"], Ech, rtol=1e-13)


def test_multichannel_all_exponents_vs_A():
    """All six exponents, non-cubic box, anisotropic h, charged channels (zero modes on the grid)."""
    rng = np.random.default_rng(12)
    box = np.array([11.0, 12.5, 10.0])
    grid = [18, 20, 16]
    N = 30
    pos = rng.uniform(0, 1, (N, 3)) * box
    q = rng.normal(0, 0.5, (6, N))
    ex = [1, 2, 3, 4, 5, 6]
    c = 12.024
    r_c = G.default_r_c(box, grid, c)
    EA, EchA, phiA, FA = direct_sums(pos, q, ex, box, c, r_c, grid=grid)
    E, Ech, phi, F = G.gridded(pos, q, ex, box, grid, 12, c, r_c, G.default_c_w(12))
    assert np.max(np.abs(Ech - EchA) / np.abs(EchA)) < 1e-9
    assert _rel(F, FA) < 1e-8
    for a in range(6):
        assert _rel(phi[a], phiA[a]) < 1e-8


def test_B_forces_are_exact_gradient_of_B_energy(cfg1):
    """Gather with derivative weights = exact gradient of the discrete energy."""
    w = cfg1
    args = (w["q"], w["exponents"], w["box"], w["grid"], w["w"], w["c"], w["r_c"], G.default_c_w(w["w"]))
    E, _, phi, F = G.gridded(w["pos"], *args)
    h = 1e-5
    for i, d in ((0, 0), (5, 1), (63, 2)):
        pp, pm = w["pos"].copy(), w["pos"].copy()
        pp[i, d] += h
        pm[i, d] -= h
        fd = -(G.gridded(pp, *args)[0] - G.gridded(pm, *args)[0]) / (2 * h)
        assert abs(fd - F[i, d]) < 2e-8 * np.abs(F).max()


def test_B_net_force_and_translation_at_aliasing_level(cfg1):
    """Reading R12: for the gridded scheme sum F = 0 and translation invariance hold only to the
    aliasing level, not to rounding (contrast with oracle A's exact invariants)."""
    w = cfg1
    args = (w["q"], w["exponents"], w["box"], w["grid"], 8, w["c"], w["r_c"], G.default_c_w(8))
    E, _, _, F = G.gridded(w["pos"], *args)
    frms = np.sqrt((F ** 2).mean())
    assert np.abs(F.sum(0)).max() < 1e-3 * frms * np.sqrt(len(F))
    E2 = G.gridded(w["pos"] + np.array([0.211, 0.377, -0.119]), *args)[0]
    assert abs(E2 - E) / abs(E) < 1e-6


def test_window_transform_Eq22():
    """W^(k) = omega lambda_0 psi(omega k / c_w)  (Eq. (22)) against direct quadrature
    of the zero-extended window (Eq. (21)) -- i.e. the band relation (S39) in physical units."""
    from oracle.pswf import quad
    c_w, wd, h, L, M = 16.65, 6, 0.625, 10.0, 16
    psi = PSWF0(c_w)
    m, Wh = G.window_hat_1d(psi, wd, M)        # the factor lambda_0 psi(pi w m / (M c_w)); omega is applied by multiplier()
    omega = wd * h / 2
    for mi in (0, 1, 3, 5, -4):
        k = 2 * np.pi * mi / L
        direct = quad(lambda x: psi(x / omega) * np.cos(k * x), -omega, omega)
        assert abs(direct - omega * Wh[list(m).index(mi)]) < 1e-13


def test_stencil_rule_R4():
    box, grid, w = [10.0] * 3, [16] * 3, 6
    pos = np.array([[0.0, 0.3, 9.99], [5.0, 0.625 * 3, 0.625 * 3 + 1e-9]])
    i0, z = G.stencil(pos, box, grid, w)
    assert i0.tolist() == [[-3, -2, 13], [5, 0, 1]]
    assert np.all(z >= -1.0) and np.all(z < 1.0)
    assert np.allclose(np.diff(z, axis=-1), 2.0 / w)


def test_spread_conserves_charge_to_aliasing_level():
    """sum_g rho_g h^3 = Q W^(0) up to aliasing (Poisson summation of the window)."""
    rng = np.random.default_rng(0)
    box, grid, w, c_w = [10.0] * 3, [16] * 3, 8, G.default_c_w(8)
    pos = rng.uniform(0, 10, (10, 3))
    q = rng.uniform(0.5, 1.5, (1, 10))
    rho = G.spread(pos, q, box, grid, w, c_w)
    psi = PSWF0(c_w)
    W0 = (w * 0.625 / 2 * psi.lambda0) ** 3
    assert abs(rho.sum() * 0.625 ** 3 / (q.sum() * W0) - 1) < 1e-6


# ---- general (triclinic) cells ------------------------------------------------------------------

def _tri_system():
    rng = np.random.default_rng(31)
    cell = np.array([[9.0, 0.0, 0.0], [2.0, 8.5, 0.0], [-1.5, 1.2, 10.0]])
    pos = rng.uniform(0, 1, (20, 3)) @ cell
    q = rng.normal(0, 0.6, (2, 20))
    return pos, q, cell, [1, 6]


@pytest.mark.parametrize("w,tol", [(8, 2e-5), (16, 1e-9)])
def test_B_converges_to_A_in_a_triclinic_cell(w, tol):
    """Oracle B with the grid in fractional coordinates against the direct k-sum in the same triclinic
    cell: aliasing-level agreement at w = 8, 1e-9 at w = 16 (the same gates as the orthorhombic case)."""
    from oracle.direct import direct_sums
    pos, q, cell, ex = _tri_system()
    grid = [18, 20, 22]
    c = 12.024
    r_c = G.default_r_c(cell, grid, c)
    E, Ech, phi, F = G.gridded(pos, q, ex, cell, grid, w, c, r_c, G.default_c_w(w))
    Ea, Echa, phia, Fa = direct_sums(pos, q, ex, cell, c, r_c, grid=grid)
    assert abs(E - Ea) < tol * abs(Ea)
    assert np.linalg.norm(F - Fa) < 10 * tol * np.linalg.norm(Fa)
    assert np.linalg.norm(phi - phia) < 10 * tol * np.linalg.norm(phia)


def test_B_triclinic_forces_are_gradient_of_its_own_energy():
    pos, q, cell, ex = _tri_system()
    grid, w, c = [18, 20, 22], 8, 12.024
    r_c = G.default_r_c(cell, grid, c)
    args = (q, ex, cell, grid, w, c, r_c, G.default_c_w(w))
    E, _, phi, F = G.gridded(pos, *args)
    h = 1e-5
    for i, d in ((1, 0), (7, 1), (12, 2)):
        pp, pm = pos.copy(), pos.copy()
        pp[i, d] += h
        pm[i, d] -= h
        fd = -(G.gridded(pp, *args)[0] - G.gridded(pm, *args)[0]) / (2 * h)
        assert abs(fd - F[i, d]) < 2e-6 * np.abs(F).max()


def test_B_orthorhombic_cell_matrix_equals_box_vector():
    """A diagonal 3x3 cell reproduces the box-vector results bit for bit in the stencil and to rounding in
    the energies (the code path is the general one in both cases)."""
    rng = np.random.default_rng(32)
    box, grid, w, c = [9.0, 10.0, 8.0], [16, 18, 16], 6, 12.024
    pos = rng.uniform(0, 1, (15, 3)) * box
    q = rng.normal(0, 1, (1, 15))
    r_c = G.default_r_c(box, grid, c)
    i0a, za = G.stencil(pos, box, grid, w)
    i0b, zb = G.stencil(pos, np.diag(box), grid, w)
    assert np.array_equal(i0a, i0b) and np.array_equal(za, zb)
    a = G.gridded(pos, q, [1], box, grid, w, c, r_c, G.default_c_w(w))
    b = G.gridded(pos, q, [1], np.diag(box), grid, w, c, r_c, G.default_c_w(w))
    assert abs(a[0] - b[0]) < 1e-14 * abs(a[0]) and np.allclose(a[3], b[3], rtol=1e-13, atol=0)


def test_C_loops_equal_numpy_loops():
    """oracle/gridded_sum.c (used for the million-atom configuration) is the numpy oracle B to rounding,
    in an orthorhombic and in a triclinic cell."""
    rng = np.random.default_rng(33)
    for box in ([9.0, 10.0, 8.0], np.array([[9.0, 0, 0], [2.0, 8.5, 0], [-1.5, 1.2, 10.0]])):
        grid, w, c = [16, 18, 20], 6, 12.024
        cell = np.diag(box) if np.ndim(box) == 1 else box
        pos = rng.uniform(-0.2, 1.2, (25, 3)) @ cell
        q = rng.normal(0, 1, (3, 25))
        r_c = G.default_r_c(box, grid, c)
        a = G.gridded(pos, q, [1, 3, 6], box, grid, w, c, r_c, G.default_c_w(w))
        b = G.gridded_c(pos, q, [1, 3, 6], box, grid, w, c, r_c, G.default_c_w(w))
        assert abs(a[0] - b[0]) < 1e-13 * abs(a[0])
        assert np.allclose(a[2], b[2], rtol=0, atol=1e-13 * np.abs(a[2]).max())
        assert np.allclose(a[3], b[3], rtol=0, atol=1e-13 * np.abs(a[3]).max())


@pytest.mark.parametrize("width", [6, 8])
def test_window_bandwidth_optimum(cfg1, cfg1_A, width):
    """DESIGN.md reading R3: the default window bandwidth c_w = w (3.55 - 1.55 eta) (2.775 w at eta = 0.5) sits
    at the minimum of the force error of the gridded scheme against the direct k-sum: a scan of c_w / w over
    2.2 .. 3.4 has its best value within 0.15 of the default, and the default beats both ends by 3x or more."""
    w = cfg1
    FA = cfg1_A[3]
    ratios = np.array([2.2, 2.5, 2.65, 2.775, 2.9, 3.05, 3.4])
    err = []
    for r in ratios:
        F = G.gridded(w["pos"], w["q"], w["exponents"], w["box"], w["grid"], width, w["c"], w["r_c"], r * width)[3]
        err.append(_rel(F, FA))
    err = np.array(err)
    assert abs(ratios[np.argmin(err)] - G.default_c_w(width) / width) <= 0.15, (ratios, err)
    assert err[3] * 3 < err[0] and err[3] * 3 < err[-1], err
