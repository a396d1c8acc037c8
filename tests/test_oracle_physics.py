"""Physics pins for oracle A (oracle/direct.py, oracle/direct_sum.c): the reciprocal sum, completed
by the validation scaffold to the full decomposition (S65), must reproduce lattice energies the
mathematics fixes, for every exponent, independently of (c, r_c)."""
import itertools
import numpy as np
import pytest

from oracle import scaffold
from oracle.direct import direct_sums, direct_sums_c, mode_set
from oracle.kernels import Mollifier


def _rock_salt():
    pos, q = [], []
    for i, j, k in itertools.product(range(2), repeat=3):
        pos.append([i, j, k])
        q.append((-1.0) ** (i + j + k))
    return np.array(pos, float), np.array(q), [2.0, 2.0, 2.0]


@pytest.mark.parametrize("c,r_c", [(30.0, 1.3), (24.0, 1.7)])
def test_madelung_nacl(golden, c, r_c):
    """north_star pin: NaCl Madelung constant 1.747565 (p = 1), via (S65) with tinfoil E_IB = 0."""
    pos, q, box = _rock_salt()
    E = scaffold.total_energy(pos, q, 1, box, c, r_c)
    M = -E / 4.0          # 8 ions, nearest-neighbour distance 1: E = -(8/2) M
    assert abs(M - golden["madelung_nacl_northstar"]) < 5e-7
    assert abs(M - golden["madelung_nacl"]) < 2e-9


def _sc_sum_brute(p, R=24):
    """sum_{0<|n|<=R} |n|^-p + 4 pi int_R^inf r^(2-p) dr, shell-corrected (independent of the oracle)."""
    ax = np.arange(-R, R + 1)
    n2 = (ax[:, None, None] ** 2 + ax[None, :, None] ** 2 + ax[None, None, :] ** 2).astype(float)
    mask = (n2 > 0) & (n2 <= R * R)
    tail = 4 * np.pi * R ** (3.0 - p) / (p - 3.0)
    return float(np.sum(n2[mask] ** (-p / 2.0)) + tail)


@pytest.mark.parametrize("p", [4, 5, 6])
def test_simple_cubic_lattice_sums(golden, p):
    """One unit 'charge' in a unit cube: 2E = sum_{n != 0} |n|^-p.  Exercises the non-neutral zero
    mode (S79) and the self term (S66)-(S67)."""
    ref = golden["sc_lattice_sum_p%d" % p]
    # the golden value itself is checked by brute force (tolerance = its truncation error)
    assert abs(_sc_sum_brute(p) - ref) < {4: 2e-2, 5: 3e-4, 6: 1e-5}[p]
    E = scaffold.total_energy(np.zeros((1, 3)), np.ones(1), p, [1.0, 1.0, 1.0], 30.0, 0.9)
    assert abs(2 * E - ref) < {4: 2e-9, 5: 1e-7, 6: 2e-9}[p] * ref   # p = 5 golden has 9 digits


@pytest.mark.parametrize("p", [8, 10])
def test_simple_cubic_lattice_sums_p8_p10(p):
    """The same pin for the exponents of SI Section 6 (Corollary 1, (S56)-(S59)): one unit weight in a unit
    cube, 2E = sum_{n != 0} |n|^-p.  The reference is the brute-force sum itself (it converges like R^(3-p):
    remainder below 1e-7 at R = 24), no stored value."""
    ref = _sc_sum_brute(p)
    assert 6.0 < ref < 7.0
    E = scaffold.total_energy(np.zeros((1, 3)), np.ones(1), p, [1.0, 1.0, 1.0], 30.0, 0.9)
    assert abs(2 * E - ref) < 2e-7 * ref, (2 * E, ref)


@pytest.mark.parametrize("p,nmax,tol", [(10, 5, 2e-7), (8, 8, 2e-7), (6, 6, 2e-6), (5, 8, 2e-4), (4, 10, 2e-3)])
def test_brute_force_image_sums_random_box(p, nmax, tol):
    """Random 6-atom non-neutral box, orthorhombic: (S65) vs 1/2 sum_n sum' q_i q_j / r^p (p > 3
    converges absolutely; the remainder is bounded by the integral tail and corrected with it)."""
    rng = np.random.default_rng(42 + p)
    box = np.array([3.1, 2.7, 3.6])
    pos = rng.uniform(0, 1, (6, 3)) * box
    q = rng.normal(0, 1, 6)
    # (the self term grows like c^p / p!: p = 8, 10 need a wider band for the same absolute accuracy)
    E = scaffold.total_energy(pos, q, p, box, 24.0 if p <= 6 else 32.0, 1.2)
    brute = scaffold.brute_force_image_sum(pos, q, p, box, nmax)
    # tail of the image sum beyond the summed block, continuum estimate
    R = (nmax + 0.5) * box.min()
    tail = 0.5 * q.sum() ** 2 * 4 * np.pi * R ** (3.0 - p) / ((p - 3.0) * np.prod(box))
    assert abs(E - brute) < max(tol * abs(E), 3 * abs(tail)), (E, brute, tail)


def test_p3_neutral_vs_brute_force():
    """p = 3, neutral random box: spherical image sum converges like 1/R^2; Richardson-extrapolated
    brute force against (S65).  (A charged p = 3 channel is pinned by invariance below.)"""
    rng = np.random.default_rng(7)
    box = np.array([2.0, 2.0, 2.0])
    pos = rng.uniform(0, 2, (4, 3))
    q = rng.normal(0, 1, 4)
    q -= q.mean()
    E = scaffold.total_energy(pos, q, 3, box, 24.0, 0.9)
    b = [scaffold.brute_force_image_sum(pos, q, 3, box, n) for n in (6, 12)]
    # cubic-block truncation of a neutral 1/r^3 sum: error ~ 1/n^2
    extrap = (4 * b[1] - b[0]) / 3
    assert abs(E - extrap) < 3e-4 * max(1.0, abs(E)), (E, b, extrap)


@pytest.mark.parametrize("p", [1, 2, 3, 4, 5, 6, 8, 10])
@pytest.mark.parametrize("neutral", [True, False])
def test_total_energy_independent_of_c_and_rc(p, neutral):
    """'SR+LR split' pin for every exponent: (S65) must not depend on (c, r_c), including the
    zero-mode conventions (S73), (S75), (S78) for charged channels."""
    rng = np.random.default_rng(100 + p)
    box = np.array([3.0, 3.4, 2.8])
    pos = rng.uniform(0, 1, (5, 3)) * box
    q = rng.normal(0, 1, 5)
    if neutral:
        q -= q.mean()
    # band-limit error of the window ~ exp(-c) times the size of the cancelling parts, which grow like
    # c^p / p!: the two highest exponents are compared at wider bands
    c1, c2, tol = (30.0, 26.0, 2e-9) if p <= 6 else (38.0, 34.0, 2e-8)
    E1 = scaffold.total_energy(pos, q, p, box, c1, 1.1)
    E2 = scaffold.total_energy(pos, q, p, box, c2, 1.35)
    assert abs(E1 - E2) < tol * max(1.0, abs(E1)), (E1, E2)


@pytest.mark.parametrize("neutral", [True, False])
def test_p1_matches_classical_erfc_ewald(neutral):
    """'short-range-plus-long-range split matches full Ewald' (north_star): p = 1 PSWF total vs the
    classical erfc Ewald sum (Eq. (12) special case) on the same box."""
    rng = np.random.default_rng(3)
    box = np.array([3.0, 3.3, 2.9])
    pos = rng.uniform(0, 1, (6, 3)) * box
    q = rng.normal(0, 1, 6)
    if neutral:
        q -= q.mean()
    E_pswf = scaffold.total_energy(pos, q, 1, box, 30.0, 1.2)
    E_ewald = scaffold.ewald_erfc_energy(pos, q, box, alpha=2.6, r_cut=2.9, kmax=16)
    assert abs(E_pswf - E_ewald) < 1e-8 * max(1.0, abs(E_ewald)), (E_pswf, E_ewald)


# ---- derivatives and invariants of oracle A itself ------------------------------------------

def _small_system(seed=5, N=9, C=3):
    rng = np.random.default_rng(seed)
    box = np.array([9.0, 10.0, 8.5])
    pos = rng.uniform(0, 1, (N, 3)) * box
    q = rng.normal(0, 0.7, (C, N))
    q[0] -= q[0].mean()
    return pos, q, box, [1, 3, 6]


def test_forces_are_minus_gradient_fd():
    pos, q, box, ex = _small_system()
    c, r_c = 12.024, 3.0
    E, _, phi, F = direct_sums(pos, q, ex, box, c, r_c)
    h = 1e-5
    for i in (0, 4):
        for d in range(3):
            pp, pm = pos.copy(), pos.copy()
            pp[i, d] += h
            pm[i, d] -= h
            fd = -(direct_sums(pp, q, ex, box, c, r_c)[0] - direct_sums(pm, q, ex, box, c, r_c)[0]) / (2 * h)
            assert abs(fd - F[i, d]) < 1e-7 * np.abs(F).max()


def test_phi_is_dE_dq_fd():
    pos, q, box, ex = _small_system()
    c, r_c = 12.024, 3.0
    E, _, phi, F = direct_sums(pos, q, ex, box, c, r_c)
    h = 1e-6
    for a, i in ((0, 1), (1, 3), (2, 8)):
        qp, qm = q.copy(), q.copy()
        qp[a, i] += h
        qm[a, i] -= h
        fd = (direct_sums(pos, qp, ex, box, c, r_c)[0] - direct_sums(pos, qm, ex, box, c, r_c)[0]) / (2 * h)
        assert abs(fd - phi[a, i]) < 1e-8 * np.abs(phi).max()
    assert abs(E - 0.5 * np.sum(q * phi)) < 1e-13 * abs(E)


def test_net_force_zero_and_translation_invariance():
    pos, q, box, ex = _small_system()
    c, r_c = 12.024, 3.0
    E, Ech, phi, F = direct_sums(pos, q, ex, box, c, r_c)
    assert np.abs(F.sum(0)).max() < 1e-13 * np.abs(F).max()
    shift = np.array([0.37, -1.21, 4.4])
    E2, _, phi2, F2 = direct_sums(pos + shift, q, ex, box, c, r_c)
    assert abs(E - E2) < 1e-13 * abs(E)
    assert np.abs(F - F2).max() < 1e-12 * np.abs(F).max()
    assert np.abs(phi - phi2).max() < 1e-12 * np.abs(phi).max()
    # periodic images: moving one atom by a lattice vector changes nothing
    pos3 = pos.copy()
    pos3[2] += box * np.array([1, -2, 3])
    assert abs(direct_sums(pos3, q, ex, box, c, r_c)[0] - E) < 1e-12 * abs(E)


def test_c_oracle_equals_numpy_oracle_and_half_equals_full():
    pos, q, box, ex = _small_system(seed=11, N=40, C=3)
    c, r_c = 12.024, 2.5
    grid = [16, 18, 14]
    a = direct_sums(pos, q, ex, box, c, r_c, grid=grid)
    b = direct_sums_c(pos, q, ex, box, c, r_c, grid=grid)
    assert abs(a[0] - b[0]) < 1e-13 * abs(a[0])
    assert np.allclose(a[1], b[1], rtol=1e-12)
    assert np.allclose(a[2], b[2], rtol=0, atol=1e-13 * np.abs(a[2]).max())
    assert np.allclose(a[3], b[3], rtol=0, atol=1e-13 * np.abs(a[3]).max())
    sub = np.array([3, 17, 39])
    bs = direct_sums_c(pos, q, ex, box, c, r_c, grid=grid, subset=sub)
    assert np.allclose(bs[2], a[2][:, sub], rtol=0, atol=1e-13 * np.abs(a[2]).max())
    assert np.allclose(bs[3], a[3][sub], rtol=0, atol=1e-13 * np.abs(a[3]).max())
    full, half = mode_set(box, c, r_c, grid), mode_set(box, c, r_c, grid, half=True)
    assert len(full) == 2 * len(half)
    assert {tuple(v) for v in full} == {tuple(v) for v in half} | {tuple(-v) for v in half}


def test_mode_set_limits():
    box = np.array([10.0, 10.0, 10.0])
    c, r_c = 12.024, 4.78
    m = mode_set(box, c, r_c, grid=[16, 16, 16])
    k = 2 * np.pi * m / box
    assert np.all(np.sqrt((k ** 2).sum(1)) * r_c < c)
    assert np.abs(m).max() <= 7
    assert not np.any(np.all(m == 0, axis=1))
    # |m| < c L / (2 pi r_c) = 4.0035: lattice points with 0 < |m|^2 <= 16 (Gauss sphere count
    # 1+6+12+8+6+24+24+0+12+30+24+24+8+24+48+0+6 = 257 including the origin)
    assert len(m) == 256


def test_real_space_parts_energy_forces_potentials():
    """scaffold.real_space_parts (parity target of pswf_lr_execute_real): its energy equals the pinned
    real_space_complement - self_energy, F = -dE/dr and phi = dE/dq by central differences of E."""
    from oracle.scaffold import real_space_parts, real_space_complement, self_energy
    from oracle.kernels import Mollifier
    rng = np.random.default_rng(11)
    box = np.array([9.0, 10.0, 11.0])
    N = 14
    pos = rng.uniform(0, 1, (N, 3)) * box
    q = rng.normal(0, 1, (3, N))
    ex = [1, 4, 6]
    c, r_c = 12.024, 4.2
    E, phi, F = real_space_parts(pos, q, ex, box, c, r_c)
    moll = Mollifier(c, r_c)
    E_ref = sum(real_space_complement(pos, q[a], ex[a], box, moll) - self_energy(q[a], ex[a], moll)
                for a in range(3))
    assert abs(E - E_ref) < 1e-12 * abs(E_ref)
    h = 1e-5
    for i, d in [(0, 0), (5, 2), (9, 1)]:
        pp, pm = pos.copy(), pos.copy()
        pp[i, d] += h
        pm[i, d] -= h
        fd = -(real_space_parts(pp, q, ex, box, c, r_c)[0] - real_space_parts(pm, q, ex, box, c, r_c)[0]) / (2 * h)
        assert abs(fd - F[i, d]) < 1e-6 * np.abs(F).max()
    for a, i in [(0, 3), (2, 7)]:
        qp, qm = q.copy(), q.copy()
        qp[a, i] += h
        qm[a, i] -= h
        fd = (real_space_parts(pos, qp, ex, box, c, r_c)[0] - real_space_parts(pos, qm, ex, box, c, r_c)[0]) / (2 * h)
        assert abs(fd - phi[a, i]) < 1e-8 * np.abs(phi).max()


def test_virial_direct_matches_strain_derivative_of_energy():
    """oracle.direct.virial_direct: the diagonal equals -dE/d(eps_aa) by central differences of the
    direct k-sum under a homogeneous strain of atoms and cell (mode integers fixed), charged and
    neutral channels, p = 1, 3, 6; the tensor is symmetric and its off-diagonal part changes sign
    under the mirror x -> -x (so a swapped or dropped index cannot hide)."""
    from oracle.direct import virial_direct, mode_set
    from oracle.kernels import Mollifier
    rng = np.random.default_rng(3)
    box = np.array([9.0, 10.0, 11.5])
    N = 20
    pos = rng.uniform(0, 1, (N, 3)) * box
    q = rng.normal(0, 1, (3, N))
    q[0] -= q[0].mean()
    ex = [1, 3, 6]
    c, r_c = 12.024, 3.4
    W = virial_direct(pos, q, ex, box, c, r_c)
    assert np.allclose(W, W.T, rtol=0, atol=1e-13 * np.abs(W).max())
    m = mode_set(box, c, r_c, None, half=False)

    def energy(bx, ps):           # Eq. (5) on the FIXED integer mode set
        V = np.prod(bx)
        k = 2 * np.pi * m / bx
        kn = np.sqrt((k ** 2).sum(1))
        rho = q @ np.exp(1j * ps @ k.T)
        moll = Mollifier(c, r_c)
        E = 0.0
        for a, p in enumerate(ex):
            ph = np.where(kn * r_c < c, moll.Phi_hat(p, np.minimum(kn, c / r_c * (1 - 1e-14))), 0.0)
            E += (ph * np.abs(rho[a]) ** 2).sum() / (2 * V) + moll.Phi0(p) * q[a].sum() ** 2 / (2 * V)
        return E

    for d in range(3):
        e = 1e-6
        sp, sm = np.ones(3), np.ones(3)
        sp[d] += e
        sm[d] -= e
        fd = -(energy(box * sp, pos * sp) - energy(box * sm, pos * sm)) / (2 * e)
        assert abs(fd - W[d, d]) < 2e-7 * np.abs(W).max(), (d, fd, W[d, d])
    pm = pos.copy()
    pm[:, 0] = box[0] - pm[:, 0]
    Wm = virial_direct(pm, q, ex, box, c, r_c)
    assert np.allclose(Wm[0, 1], -W[0, 1], atol=1e-10 * np.abs(W).max())
    assert np.allclose(Wm[0, 2], -W[0, 2], atol=1e-10 * np.abs(W).max())
    assert np.allclose(Wm[1, 2], W[1, 2], atol=1e-10 * np.abs(W).max())
    assert np.allclose(np.diag(Wm), np.diag(W), atol=1e-10 * np.abs(W).max())


# ---- general (triclinic) cells: "cell tensor Omega", PAPER.md:76 ------------------------------

_SHEAR = np.array([[1, 0, 0], [1, 1, 0], [0, -1, 1]])     # unimodular: T h spans the same lattice as h


def test_madelung_nacl_in_sheared_and_primitive_cells(golden):
    """The rock-salt Madelung constant from (S65) does not depend on how the lattice is described: the
    conventional cube re-described by sheared lattice vectors (same lattice, same 8 ions), and the
    two-ion primitive fcc cell with 60-degree angles."""
    pos, q, box = _rock_salt()
    cell = _SHEAR @ np.diag(box)
    E = scaffold.total_energy(pos, q, 1, cell, 30.0, 1.3)
    assert abs(-E / 4.0 - golden["madelung_nacl"]) < 2e-9
    prim = np.array([[1.0, 1.0, 0.0], [0.0, 1.0, 1.0], [1.0, 0.0, 1.0]])
    E2 = scaffold.total_energy(np.array([[0.0, 0, 0], [1.0, 0, 0]]), np.array([1.0, -1.0]), 1, prim, 30.0, 0.9)
    assert abs(-E2 - golden["madelung_nacl"]) < 2e-9         # one ion pair: E = -M


@pytest.mark.parametrize("p", [1, 3, 6, 8])
def test_oracle_A_is_invariant_under_relabelling_the_lattice(p):
    """Oracle A alone: E, phi and F of a random charged system are the same for the box diag(L) and for
    the sheared description T diag(L) of the same lattice (the mode SET is the same reciprocal lattice,
    only its integer labels change)."""
    rng = np.random.default_rng(300 + p)
    box = np.array([6.0, 7.0, 6.5])
    pos = rng.uniform(0, 1, (7, 3)) * box
    q = rng.normal(0, 1, (1, 7))
    a = direct_sums(pos, q, [p], box, 12.024, 2.0)
    b = direct_sums(pos, q, [p], _SHEAR @ np.diag(box), 12.024, 2.0)
    assert abs(a[0] - b[0]) < 1e-12 * abs(a[0])
    assert np.allclose(a[2], b[2], rtol=0, atol=1e-12 * np.abs(a[2]).max())
    assert np.allclose(a[3], b[3], rtol=0, atol=1e-12 * np.abs(a[3]).max())


def _triclinic_system(seed=11, N=8):
    rng = np.random.default_rng(seed)
    cell = np.array([[8.0, 0.0, 0.0], [2.1, 7.5, 0.0], [-1.3, 1.7, 9.0]])
    pos = rng.uniform(0, 1, (N, 3)) @ cell
    q = rng.normal(0, 0.7, (3, N))
    q[0] -= q[0].mean()
    return pos, q, cell, [1, 4, 6]


def test_triclinic_forces_potentials_and_c_oracle():
    """Triclinic cell: F = -dE/dr and phi = dE/dq by central differences of E; the C routine equals the
    numpy sums; a lattice translation of one atom changes nothing."""
    pos, q, cell, ex = _triclinic_system()
    c, r_c = 12.024, 2.6
    E, Ech, phi, F = direct_sums(pos, q, ex, cell, c, r_c)
    h = 1e-5
    for i, d in ((0, 0), (3, 1), (5, 2)):
        pp, pm = pos.copy(), pos.copy()
        pp[i, d] += h
        pm[i, d] -= h
        fd = -(direct_sums(pp, q, ex, cell, c, r_c)[0] - direct_sums(pm, q, ex, cell, c, r_c)[0]) / (2 * h)
        assert abs(fd - F[i, d]) < 1e-7 * np.abs(F).max()
    qp, qm = q.copy(), q.copy()
    qp[1, 2] += h
    qm[1, 2] -= h
    fdq = (direct_sums(pos, qp, ex, cell, c, r_c)[0] - direct_sums(pos, qm, ex, cell, c, r_c)[0]) / (2 * h)
    assert abs(fdq - phi[1, 2]) < 1e-7 * np.abs(phi).max()
    Ec, Echc, phic, Fc = direct_sums_c(pos, q, ex, cell, c, r_c)
    assert abs(E - Ec) < 1e-13 * abs(E) and np.allclose(F, Fc, atol=1e-13 * np.abs(F).max(), rtol=0)
    assert np.allclose(phi, phic, atol=1e-13 * np.abs(phi).max(), rtol=0)
    moved = pos.copy()
    moved[2] += cell[1] - cell[2]
    assert abs(direct_sums(moved, q, ex, cell, c, r_c)[0] - E) < 1e-12 * abs(E)
    assert np.abs(F.sum(0)).max() < 1e-12 * np.abs(F).max()


def test_triclinic_total_energy_vs_brute_force_and_invariance():
    """(S65) in a triclinic cell: p = 6 against the plain image sum, and (c, r_c)-invariance for a charged
    p = 1 channel (background convention (S73) with V = |det h|)."""
    pos, q, cell, _ = _triclinic_system(seed=12, N=6)
    E = scaffold.total_energy(pos, q[1], 6, cell, 24.0, 1.2)
    nmax = 6
    brute = scaffold.brute_force_image_sum(pos, q[1], 6, cell, nmax)
    R = (nmax + 0.5) * 7.0
    tail = 0.5 * q[1].sum() ** 2 * 4 * np.pi * R ** -3.0 / (3.0 * abs(np.linalg.det(cell)))
    assert abs(E - brute) < max(2e-6 * abs(E), 3 * abs(tail)), (E, brute, tail)
    E1 = scaffold.total_energy(pos, q[2], 1, cell, 30.0, 1.1)
    E2 = scaffold.total_energy(pos, q[2], 1, cell, 26.0, 1.35)
    assert abs(E1 - E2) < 2e-9 * max(1.0, abs(E1))


def test_triclinic_virial_is_the_strain_derivative():
    """All six components of W_ab = -dE/d(eps_ab) in a triclinic cell by central differences of E under
    r -> (1 + eps) r, h -> h (1 + eps)^T (symmetric eps)."""
    from oracle.direct import virial_direct
    pos, q, cell, ex = _triclinic_system(seed=13, N=6)
    c, r_c = 12.024, 2.6
    W = virial_direct(pos, q, ex, cell, c, r_c)
    assert np.allclose(W, W.T, atol=1e-13)
    e = 1e-6
    for a, b in ((0, 0), (1, 1), (2, 2), (0, 1), (0, 2), (1, 2)):
        eps = np.zeros((3, 3))
        eps[a, b] += 0.5
        eps[b, a] += 0.5
        Ep = direct_sums(pos @ (np.eye(3) + e * eps).T, q, ex, cell @ (np.eye(3) + e * eps).T, c, r_c)[0]
        Em = direct_sums(pos @ (np.eye(3) - e * eps).T, q, ex, cell @ (np.eye(3) - e * eps).T, c, r_c)[0]
        assert abs(-(Ep - Em) / (2 * e) - W[a, b]) < 2e-6 * np.abs(W).max(), (a, b)
