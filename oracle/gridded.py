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


def stencil(pos, box, grid, w):
    """(i0 (N,3) int, z (N,3,w) float): first grid index and window arguments (reading R4).

    R4 fixes the arithmetic that decides the integer i0 (so that the oracle and the kernel take
    the same decision for atoms sitting exactly on a grid point): s = x * (1/L); s -= floor(s);
    u' = s * M - w/2;  i0 = ceil(u');  delta = i0 - u';  z_t = (t + delta) / (w/2) - 1, each
    operation rounded to float64 separately."""
    pos = np.asarray(pos, dtype=np.float64)
    box = np.asarray(box, dtype=np.float64)
    grid = np.asarray(grid)
    s = pos * (1.0 / box)
    s = s - np.floor(s)                           # wrap into [0, 1)
    s = np.where(s >= 1.0, 0.0, s)                # guard the rounding case s == 1
    u = s * grid.astype(np.float64) - w / 2.0
    cu = np.ceil(u)
    i0 = cu.astype(np.int64)
    delta = cu - u                                # in [0, 1)
    t = np.arange(w)
    z = (t[None, None, :] + delta[:, :, None]) / (w / 2.0) - 1.0
    return i0, z


def window_hat_1d(psi_w, w, h, L, M):
    """W^_pswf(k_d) = omega lambda_0 psi_0^{c_w}(omega k_d / c_w), omega = w h / 2, at the M
    signed DFT frequencies of one dimension.  Eq. (22)."""
    m = np.fft.fftfreq(M, d=1.0 / M)              # 0,1,..,-1 signed integers
    kd = 2 * np.pi * m / L
    omega = w * h / 2.0
    arg = omega * kd / psi_w.c
    val = omega * psi_w.lambda0 * psi_w(np.clip(arg, -1, 1))
    return m, kd, np.where(np.abs(arg) <= 1.0, val, np.nan)


def multiplier(p, box, grid, w, c, r_c, c_w, zero_mode=True):
    """D_p(m) on the full (Mx,My,Mz) DFT grid (readings R10, R11).  Eq. (25)."""
    box = np.asarray(box, dtype=np.float64)
    grid = np.asarray(grid)
    h = box / grid
    psi_w = PSWF0(c_w)
    moll = Mollifier(c, r_c)
    ms, ks, Wh = zip(*[window_hat_1d(psi_w, w, h[d], box[d], grid[d]) for d in range(3)])
    KX, KY, KZ = np.meshgrid(*ks, indexing="ij")
    kn = np.sqrt(KX ** 2 + KY ** 2 + KZ ** 2)
    What = Wh[0][:, None, None] * Wh[1][None, :, None] * Wh[2][None, None, :]
    nyq = np.zeros(tuple(grid), dtype=bool)
    for d in range(3):
        if grid[d] % 2 == 0:
            sl = [slice(None)] * 3
            sl[d] = grid[d] // 2
            nyq[tuple(sl)] = True
    inside = (kn * r_c < c) & ~nyq
    inside[0, 0, 0] = False
    Ph = np.zeros(tuple(grid))
    Ph[inside] = moll.Phi_hat(p, kn[inside])
    with np.errstate(invalid="ignore"):
        D = np.where(inside, Ph / What ** 2, 0.0)
    if np.isnan(D).any():
        raise ValueError("window transform used outside its band (grid too coarse for c_w)")
    if zero_mode:
        D[0, 0, 0] = moll.Phi0(p) / What[0, 0, 0] ** 2
    return D * np.prod(h) / np.prod(grid)


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
    box = np.asarray(box, dtype=np.float64)
    h = box / grid
    psi_w = PSWF0(c_w)
    i0, z = stencil(pos, box, grid, w)
    Wd = psi_w(z)
    # d/dr_i psi((x_g - r_i)/omega) = -psi'(z)/omega, omega = w h/2
    dWd = -psi_w.deriv(z, 1) / (w * h[None, :, None] / 2.0)
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
    h = np.asarray(box, dtype=np.float64) / np.asarray(grid)
    return float(c * h.max() / (eta * np.pi))


def default_c_w(w, eta=0.5):
    """Reading R3: window bandwidth c_w = w (3.55 - 1.55 eta)."""
    return float(w * (3.55 - 1.55 * eta))
