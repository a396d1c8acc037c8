"""Oracle B: the gridded evaluation (spread / FFT / scale / inverse FFT / gather) in float64.

TEST INFRASTRUCTURE ONLY (see oracle/__init__.py).

Follows PAPER.md:274-307 step by step (Eq. (20)-(26)) with the inverse-FFT + gather ending
that BASELINE.json's north_star asks for (it is the derivative of Eq. (26) w.r.t. q and r,
PAPER.md:76, 1099).  The window is evaluated from the Legendre series of psi_0^{c_w}
(oracle/pswf.py), never from fitted polynomials.  Readings used:

  R3  the window bandwidth c_w is a parameter separate from the mollifier's c;
  R4  u = r_d/h_d with r wrapped into [0,L); i0 = ceil(u - w/2); the atom touches grid points
      i0 .. i0+w-1 (mod M_d); window argument z_t = (i0 + t - u)/(w/2) in [-1, 1) (the order of the
      float64 operations that decide i0 is fixed in stencil());
  R10 D_p(m) = (h_x h_y h_z / M_tot) Phi^_p(|k_m|) / W^(k_m)^2 with unnormalised forward and
      inverse DFTs, so that 1/2 sum_m D |rho^|^2 = 1/2 sum_i q_i phi_i;
  R11 multiplier zero on Nyquist planes and for |k| r_c >= c; the m = 0 entry carries the
      zero-mode constant Phi0_p of (S73)/(S75)/(S78)/(S79).
"""
import numpy as np
from .pswf import PSWF0
from .kernels import Mollifier
from .direct import cell_matrix, recip_vectors


def inverse_cell(box):
    """h^-1 for fractional coordinates s = r h^-1 (rows of h = lattice vectors).  An orthorhombic box gets
    exactly diag(1/L), so that s = x * (1/L) as reading R4 states."""
    cell = cell_matrix(box)
    if np.count_nonzero(cell - np.diag(np.diag(cell))) == 0:
        return np.diag(1.0 / np.diag(cell))
    return np.linalg.inv(cell)


def stencil(pos, box, grid, w):
    """(i0 (N,3) int, z (N,3,w) float): first grid index and window arguments (reading R4).

    R4 fixes the arithmetic that decides the integer i0 (so that the oracle and the kernel take
    the same decision for atoms sitting exactly on a grid point): s = x * (1/L); s -= floor(s);
    u' = s * M - w/2;  i0 = ceil(u');  delta = i0 - u';  z_t = (t + delta) / (w/2) - 1, each
    operation rounded to float64 separately."""
    pos = np.asarray(pos, dtype=np.float64)
    grid = np.asarray(grid)
    Hi = inverse_cell(box)
    # general cell ("cell tensor Omega"): the grid lives in fractional coordinates,
    # s_d = (r_0 Hi[0][d] + r_1 Hi[1][d]) + r_2 Hi[2][d], products and sums rounded separately in this
    # order; for an orthorhombic box the two zero terms leave s = x * (1/L) bit for bit
    s = (pos[:, 0:1] * Hi[0][None, :] + pos[:, 1:2] * Hi[1][None, :]) + pos[:, 2:3] * Hi[2][None, :]
    s = s - np.floor(s)                           # wrap into [0, 1)
    s = np.where(s >= 1.0, 0.0, s)                # guard the rounding case s == 1
    u = s * grid.astype(np.float64) - w / 2.0
    cu = np.ceil(u)
    i0 = cu.astype(np.int64)
    delta = cu - u                                # in [0, 1)
    t = np.arange(w)
    z = (t[None, None, :] + delta[:, :, None]) / (w / 2.0) - 1.0
    return i0, z


def window_hat_1d(psi_w, w, M):
    """One factor of W^_pswf, Eq. (22), at the M signed DFT indices m of one dimension:
    lambda_0 psi_0^{c_w}(omega k_d / c_w) with omega k_d = (w h / 2)(2 pi m / L) = pi w m / M -- a function
    of the index only, in any cell; the lengths omega_d = w h_d / 2 are collected in multiplier()."""
    m = np.fft.fftfreq(M, d=1.0 / M)              # 0,1,..,-1 signed integers
    arg = np.pi * w * m / (M * psi_w.c)
    val = psi_w.lambda0 * psi_w(np.clip(arg, -1, 1))
    return m, np.where(np.abs(arg) <= 1.0, val, np.nan)


def multiplier(p, box, grid, w, c, r_c, c_w, zero_mode=True):
    """D_p(m) on the full (Mx,My,Mz) DFT grid (readings R10, R11).  Eq. (25)."""
    cell = cell_matrix(box)
    grid = np.asarray(grid)
    V = float(abs(np.linalg.det(cell)))
    hvol = V / np.prod(grid)                      # volume of a grid cell (h_x h_y h_z when orthorhombic)
    psi_w = PSWF0(c_w)
    moll = Mollifier(c, r_c)
    ms, Wh = zip(*[window_hat_1d(psi_w, w, grid[d]) for d in range(3)])
    MX, MY, MZ = np.meshgrid(*ms, indexing="ij")
    kvec = recip_vectors(cell, np.stack([MX, MY, MZ], axis=-1).reshape(-1, 3))
    kn = np.sqrt((kvec ** 2).sum(1)).reshape(tuple(grid))
    # W^ = prod_d omega_d lambda_0 psi(.), prod_d omega_d = (w/2)^3 x (grid-cell volume): the window is a
    # tensor product in fractional coordinates, its transform carries the Jacobian |det h|
    What = (w / 2.0) ** 3 * hvol * Wh[0][:, None, None] * Wh[1][None, :, None] * Wh[2][None, None, :]
    nyq = np.zeros(tuple(grid), dtype=bool)
    for d in range(3):
        if grid[d] % 2 == 0:
            sl = [slice(None)] * 3
            sl[d] = grid[d] // 2
            nyq[tuple(sl)] = True
    inside = (kn * r_c < c) & ~nyq
    inside[0, 0, 0] = False
    Ph = np.zeros(tuple(grid))
    kn_u, inv = np.unique(kn[inside], return_inverse=True)    # Phi^ depends on |k| only
    Ph[inside] = moll.Phi_hat(p, kn_u)[inv]
    with np.errstate(invalid="ignore"):
        D = np.where(inside, Ph / What ** 2, 0.0)
    if np.isnan(D).any():
        raise ValueError("window transform used outside its band (grid too coarse for c_w)")
    if zero_mode:
        D[0, 0, 0] = moll.Phi0(p) / What[0, 0, 0] ** 2
    return D * hvol / np.prod(grid)


def spread(pos, q, box, grid, w, c_w):
    """rho_grid^a = sum_j q_j^a [W(r - r_j)]_*   Eq. (20)-(21),(24)."""
    q = np.atleast_2d(np.asarray(q, dtype=np.float64))
    grid = np.asarray(grid)
    psi_w = PSWF0(c_w)
    i0, z = stencil(pos, box, grid, w)
    Wd = psi_w(z)                                              # (N,3,w)
    rho = np.zeros((q.shape[0],) + tuple(grid))
    t = np.arange(w)
    for j in range(len(i0)):
        ix = (i0[j, 0] + t) % grid[0]
        iy = (i0[j, 1] + t) % grid[1]
        iz = (i0[j, 2] + t) % grid[2]
        W3 = Wd[j, 0][:, None, None] * Wd[j, 1][None, :, None] * Wd[j, 2][None, None, :]
        for a in range(q.shape[0]):
            # distinct (ix,iy,iz) triples as long as w <= M_d, so fancy += is safe
            rho[a][np.ix_(ix, iy, iz)] += q[a, j] * W3
    return rho


def gather(phig, pos, box, grid, w, c_w):
    """phi_i^a = sum_g W(x_g - r_i) phi_g^a and its gradient w.r.t. r_i (window derivative)."""
    grid = np.asarray(grid)
    Hi = inverse_cell(box)
    psi_w = PSWF0(c_w)
    i0, z = stencil(pos, box, grid, w)
    Wd = psi_w(z)
    # derivative along the fractional coordinate s_d: z = 2 (t + i0 - s_d M_d + w/2)/w - 1, dz/ds_d = -2 M_d/w
    # (orthorhombic: d/dr = (1/L) d/ds = -psi'(z)/omega, omega = w h/2); Cartesian gradient below
    dWd = -psi_w.deriv(z, 1) * (2.0 * grid[None, :, None] / w)
    C = phig.shape[0]
    N = len(i0)
    phi = np.zeros((C, N))
    grad = np.zeros((C, N, 3))
    t = np.arange(w)
    for j in range(N):
        ix = (i0[j, 0] + t) % grid[0]
        iy = (i0[j, 1] + t) % grid[1]
        iz = (i0[j, 2] + t) % grid[2]
        wx, wy, wz = Wd[j]
        dx, dy, dz = dWd[j]
        for a in range(C):
            blk = phig[a][np.ix_(ix, iy, iz)]
            phi[a, j] = np.einsum("i,j,k,ijk->", wx, wy, wz, blk)
            grad[a, j, 0] = np.einsum("i,j,k,ijk->", dx, wy, wz, blk)
            grad[a, j, 1] = np.einsum("i,j,k,ijk->", wx, dy, wz, blk)
            grad[a, j, 2] = np.einsum("i,j,k,ijk->", wx, wy, dz, blk)
    # d/dr_e = sum_d (ds_d/dr_e) d/ds_d = sum_d Hi[e][d] d/ds_d
    grad = np.einsum("ed,and->ane", Hi, grad)
    return phi, grad


def gridded(pos, q, exponents, box, grid, w, c, r_c, c_w, zero_mode=True, intermediates=False):
    """Steps (i)-(iv) + inverse FFT + gather.  Returns E, E_channels, phi (C,N), F (N,3)
    (and, optionally, the real grid after spreading and the scaled spectrum)."""
    q = np.atleast_2d(np.asarray(q, dtype=np.float64))
    C, N = q.shape
    rho = spread(pos, q, box, grid, w, c_w)                    # (i)
    rho_hat = np.fft.fftn(rho, axes=(1, 2, 3))                 # (ii), unnormalised
    phig = np.empty_like(rho)
    E_spec = np.zeros(C)
    Dcache = {}
    scaled = np.empty_like(rho_hat)
    for a, p in enumerate(exponents):
        if int(p) not in Dcache:
            Dcache[int(p)] = multiplier(int(p), box, grid, w, c, r_c, c_w, zero_mode)
        D = Dcache[int(p)]
        scaled[a] = D * rho_hat[a]                             # (iii)
        E_spec[a] = 0.5 * np.sum(D * np.abs(rho_hat[a]) ** 2)  # (iv), Eq. (26)
        phig[a] = np.fft.ifftn(scaled[a]).real * np.prod(grid)  # unnormalised inverse
    phi, grad = gather(phig, pos, box, grid, w, c_w)
    F = -np.einsum("an,and->nd", q, grad)
    E_ch = 0.5 * np.einsum("an,an->a", q, phi)
    out = (float(E_ch.sum()), E_ch, phi, F)
    if intermediates:
        out = out + (dict(rho=rho, scaled=scaled, phig=phig, E_spec=E_spec),)
    return out


def default_r_c(box, grid, c, eta=0.5):
    """Reading R2: r_c such that max_d h_d = eta pi r_c / c  (Eq. (29))."""
    h = np.linalg.norm(cell_matrix(box), axis=1) / np.asarray(grid)    # |a_d| / M_d
    return float(c * h.max() / (eta * np.pi))


def default_c_w(w, eta=0.5):
    """Reading R3: window bandwidth c_w = w (3.55 - 1.55 eta)."""
    return float(w * (3.55 - 1.55 * eta))


# ---------------------------------------------------------------------------------
# The same evaluation with the two atom loops in plain C (oracle/gridded_sum.c), for the large
# configurations; stencil, window values, multiplier and FFTs are the numpy code above.
# ---------------------------------------------------------------------------------
_LIBG = None


def build_c(force=False):
    """Compile oracle/gridded_sum.c -> oracle/liboracle_gridded.so (gcc -O2 -fopenmp)."""
    import os
    import subprocess
    here = os.path.dirname(os.path.abspath(__file__))
    src, out = os.path.join(here, "gridded_sum.c"), os.path.join(here, "liboracle_gridded.so")
    if force or not os.path.exists(out) or os.path.getmtime(out) < os.path.getmtime(src):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-std=c11", "-o", out, src])
    return out


def _libg():
    global _LIBG
    if _LIBG is None:
        import ctypes
        _LIBG = ctypes.CDLL(build_c())
        _LIBG.oracle_gridded_threads.restype = ctypes.c_int
    return _LIBG


def c_threads():
    return int(_libg().oracle_gridded_threads())


def gridded_c(pos, q, exponents, box, grid, w, c, r_c, c_w, zero_mode=True, timings=None, multipliers=None):
    """gridded() with spread() and gather() replaced by their plain-C transcriptions.  Same returns
    (E, E_channels, phi, F).  `timings`, if a dict, receives the seconds spent per step.  `multipliers`
    may carry {p: D_p} from an earlier call with the same cell and parameters (they depend on neither
    positions nor charges: the plan-time part of the method) and is filled in otherwise."""
    import ctypes
    import time
    t0 = time.perf_counter()
    q = np.ascontiguousarray(np.atleast_2d(np.asarray(q, dtype=np.float64)))
    C, N = q.shape
    grid_a = np.ascontiguousarray(grid, dtype=np.int64)
    Hi = inverse_cell(box)
    psi_w = PSWF0(c_w)
    i0, z = stencil(pos, box, grid_a, w)
    i0 = np.ascontiguousarray(i0, dtype=np.int64)
    Wd = np.ascontiguousarray(psi_w(z))                                   # (N,3,w)
    dWd = np.ascontiguousarray(-psi_w.deriv(z, 1) * (2.0 * grid_a[None, :, None] / w))
    t1 = time.perf_counter()
    P = lambda a, t=ctypes.POINTER(ctypes.c_double): a.ctypes.data_as(t)
    PI = ctypes.POINTER(ctypes.c_int64)
    rho = np.zeros((C,) + tuple(int(g) for g in grid_a))
    _libg().oracle_spread(ctypes.c_long(N), ctypes.c_int(C), ctypes.c_int(w), P(grid_a, PI), P(i0, PI), P(Wd), P(q),
                          P(rho))                                           # (i)
    t2 = time.perf_counter()
    rho_hat = np.fft.fftn(rho, axes=(1, 2, 3))                             # (ii)
    phig = np.empty_like(rho)
    Dcache = multipliers if multipliers is not None else {}
    t_mult = 0.0
    for a, p in enumerate(exponents):
        if int(p) not in Dcache:
            tm0 = time.perf_counter()
            Dcache[int(p)] = multiplier(int(p), box, grid_a, w, c, r_c, c_w, zero_mode)
            t_mult += time.perf_counter() - tm0
        phig[a] = np.fft.ifftn(Dcache[int(p)] * rho_hat[a]).real * np.prod(grid_a)   # (iii) + inverse
    t3 = time.perf_counter()
    phi = np.empty((C, N))
    grad = np.empty((C, N, 3))
    _libg().oracle_gather(ctypes.c_long(N), ctypes.c_int(C), ctypes.c_int(w), P(grid_a, PI), P(i0, PI), P(Wd), P(dWd),
                          P(np.ascontiguousarray(phig)), P(phi), P(grad))
    grad = np.einsum("ed,and->ane", Hi, grad)
    F = -np.einsum("an,and->nd", q, grad)
    E_ch = 0.5 * np.einsum("an,an->a", q, phi)
    t4 = time.perf_counter()
    if timings is not None:
        timings.update(window=t1 - t0, spread=t2 - t1, fft_scale=t3 - t2 - t_mult, multipliers=t_mult,
                       gather=t4 - t3, total=t4 - t0)
    return float(E_ch.sum()), E_ch, phi, F
