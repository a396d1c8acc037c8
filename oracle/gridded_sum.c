/* Oracle B's two atom loops in plain C (float64), for configurations too large for the numpy loops.
 *
 * TEST INFRASTRUCTURE ONLY (see oracle/__init__.py).  Shares nothing with the CUDA path.
 *
 * These are the loops of oracle/gridded.py spread() and gather(), Eq. (20)-(21),(24), PAPER.md:276-296,
 * written out: the first grid index i0 and the window values W_d(t) / derivative values dW_d(t) of every
 * atom are computed by gridded.py (stencil(), the Legendre series of psi_0^{c_w}) and passed in; the FFTs
 * and the multiplier stay in numpy.  No blocking, no reordering: atom by atom, point by point.
 *
 *   spread:  rho[a][ix][iy][iz] += q[a][j] Wx[j][tx] Wy[j][ty] Wz[j][tz],  i = (i0 + t) mod M
 *   gather:  phi[a][j]   = sum_t Wx Wy Wz   g[a][ix][iy][iz]
 *            grad[a][j][0..2] = the same with dWx, dWy, dWz in turn (derivatives along the grid axes)
 *
 * Threads: spread runs one channel per thread (no two threads touch the same grid), gather one atom.
 */
#include <stdint.h>
#include <stdlib.h>
#ifdef _OPENMP
#include <omp.h>
#endif

int oracle_gridded_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

static inline long wrap(long i, long M) {
    long r = i % M;
    return r < 0 ? r + M : r;
}

/* W: [N][3][w] window values; i0: [N][3]; q: [C][N]; rho: [C][Mx][My][Mz], zeroed by the caller */
int oracle_spread(long N, int C, int w, const int64_t *grid, const int64_t *i0, const double *W,
                  const double *q, double *rho) {
    const long Mx = grid[0], My = grid[1], Mz = grid[2];
#pragma omp parallel for schedule(static)
    for (int a = 0; a < C; ++a) {
        double *ra = rho + (long)a * Mx * My * Mz;
        for (long j = 0; j < N; ++j) {
            const double *Wx = W + (j * 3 + 0) * w, *Wy = W + (j * 3 + 1) * w, *Wz = W + (j * 3 + 2) * w;
            const double qa = q[(long)a * N + j];
            for (int tx = 0; tx < w; ++tx) {
                const long ix = wrap(i0[3 * j + 0] + tx, Mx);
                for (int ty = 0; ty < w; ++ty) {
                    const long iy = wrap(i0[3 * j + 1] + ty, My);
                    const double wxy = Wx[tx] * Wy[ty];
                    for (int tz = 0; tz < w; ++tz) {
                        const long iz = wrap(i0[3 * j + 2] + tz, Mz);
                        ra[(ix * My + iy) * Mz + iz] += qa * (wxy * Wz[tz]);
                    }
                }
            }
        }
    }
    return 0;
}

/* g: [C][Mx][My][Mz]; W, dW: [N][3][w]; phi: [C][N]; grad: [C][N][3] */
int oracle_gather(long N, int C, int w, const int64_t *grid, const int64_t *i0, const double *W,
                  const double *dW, const double *g, double *phi, double *grad) {
    const long Mx = grid[0], My = grid[1], Mz = grid[2];
#pragma omp parallel for schedule(static)
    for (long j = 0; j < N; ++j) {
        const double *Wx = W + (j * 3 + 0) * w, *Wy = W + (j * 3 + 1) * w, *Wz = W + (j * 3 + 2) * w;
        const double *Dx = dW + (j * 3 + 0) * w, *Dy = dW + (j * 3 + 1) * w, *Dz = dW + (j * 3 + 2) * w;
        for (int a = 0; a < C; ++a) {
            const double *ga = g + (long)a * Mx * My * Mz;
            double v = 0.0, gx = 0.0, gy = 0.0, gz = 0.0;
            for (int tx = 0; tx < w; ++tx) {
                const long ix = wrap(i0[3 * j + 0] + tx, Mx);
                for (int ty = 0; ty < w; ++ty) {
                    const long iy = wrap(i0[3 * j + 1] + ty, My);
                    for (int tz = 0; tz < w; ++tz) {
                        const long iz = wrap(i0[3 * j + 2] + tz, Mz);
                        const double val = ga[(ix * My + iy) * Mz + iz];
                        v += Wx[tx] * Wy[ty] * Wz[tz] * val;
                        gx += Dx[tx] * Wy[ty] * Wz[tz] * val;
                        gy += Wx[tx] * Dy[ty] * Wz[tz] * val;
                        gz += Wx[tx] * Wy[ty] * Dz[tz] * val;
                    }
                }
            }
            phi[(long)a * N + j] = v;
            grad[((long)a * N + j) * 3 + 0] = gx;
            grad[((long)a * N + j) * 3 + 1] = gy;
            grad[((long)a * N + j) * 3 + 2] = gz;
        }
    }
    return 0;
}
