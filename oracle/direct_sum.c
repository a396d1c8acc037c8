/* Oracle A in plain C: direct non-uniform Fourier sums of PAPER.md Eq. (5)-(6), float64.
 *
 * TEST INFRASTRUCTURE ONLY (see oracle/__init__.py).  Shares nothing with the CUDA path.
 *
 * For every channel a (exponent p_a) and every mode k_m = 2 pi m h^-T of the cell h (rows =
 * lattice vectors; orthorhombic: k = 2 pi (mx/Lx, my/Ly, mz/Lz)) of the
 * HALF mode set passed in (one of each +-k pair; rho(-k) = conj rho(k) and Phi^ is even, so
 * each listed mode counts twice in the full sum of Eq. (5)):
 *
 *   rho_a(k) = sum_j q_j^a e^{i k.r_j}                                        Eq. (6)
 *   E_a      = (1/2V) [ 2 sum_half Phi^_a(k) |rho_a(k)|^2 + Phi0_a Qnet_a^2 ]   Eq. (5)
 *   phi_i^a  = (1/V)  [ 2 sum_half Phi^_a(k) Re(e^{-ik.r_i} rho_a(k)) + Phi0_a Qnet_a ]
 *   F_i      = -dE/dr_i = -(1/V) sum_a q_i^a 2 sum_half Phi^_a(k) k Im(e^{-ik.r_i} rho_a(k))
 *
 * Phi^_a(k) (already r_c^(3-p) S^_p(k r_c), (S60)) and the zero-mode constants Phi0_a are
 * computed by oracle/kernels.py and passed in.  The only rearrangement of the definition is
 * e^{ik.r} = e^{2 pi i m.s} = e^{2 pi i mx sx} e^{2 pi i my sy} e^{2 pi i mz sz} in the fractional
 * coordinates s = r h^-1 the caller passes, with the three factors tabulated per atom by direct
 * cos/sin calls (no recurrences); the force needs the Cartesian k_m = sum_d m_d recip[d][.].
 */
#include <math.h>
#ifndef M_PI
#define M_PI 3.14159265358979323846
#endif
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

int oracle_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* fill tab[(m + mmax)] = e^{i 2 pi m r / L}, m = -mmax..mmax, as (re, im) pairs */
static void phase_table(double r, double L, int mmax, double *tab) {
    for (int m = -mmax; m <= mmax; ++m) {
        double ang = 2.0 * M_PI * (double)m * r / L;
        tab[2 * (m + mmax)] = cos(ang);
        tab[2 * (m + mmax) + 1] = sin(ang);
    }
}

int oracle_direct_sums(long N, const double *pos /*[N][3] fractional*/, int C, const double *q /*[C][N]*/,
                       const double *recip /*[3][3] = 2 pi h^-T*/, double V, long K, const int32_t *m /*[K][3]*/,
                       const double *Phi /*[C][K]*/, const double *Phi0 /*[C]*/, long n_sub,
                       const int64_t *sub /*[n_sub]*/, double *E_ch /*[C]*/,
                       double *phi /*[C][n_sub]*/, double *F /*[n_sub][3]*/) {
    const double box[3] = {1.0, 1.0, 1.0};   /* fractional coordinates: period 1 in every direction */
    int mmax[3] = {0, 0, 0};
    for (long k = 0; k < K; ++k)
        for (int d = 0; d < 3; ++d)
            if (abs(m[3 * k + d]) > mmax[d]) mmax[d] = abs(m[3 * k + d]);
    const long nrho = 2L * C * K;
    double *rho = (double *)calloc((size_t)(nrho > 0 ? nrho : 1), sizeof(double));
    if (!rho) return -1;
    int fail = 0;

    /* pass 1: structure factors */
#pragma omp parallel
    {
        double *loc = (double *)calloc((size_t)(nrho > 0 ? nrho : 1), sizeof(double));
        double *tx = (double *)malloc(sizeof(double) * 2 * (2 * mmax[0] + 1));
        double *ty = (double *)malloc(sizeof(double) * 2 * (2 * mmax[1] + 1));
        double *tz = (double *)malloc(sizeof(double) * 2 * (2 * mmax[2] + 1));
        if (!loc || !tx || !ty || !tz) {
#pragma omp atomic write
            fail = 1;
        } else {
#pragma omp for schedule(static)
            for (long j = 0; j < N; ++j) {
                phase_table(pos[3 * j + 0], box[0], mmax[0], tx);
                phase_table(pos[3 * j + 1], box[1], mmax[1], ty);
                phase_table(pos[3 * j + 2], box[2], mmax[2], tz);
                for (long k = 0; k < K; ++k) {
                    const double *ex = tx + 2 * (m[3 * k + 0] + mmax[0]);
                    const double *ey = ty + 2 * (m[3 * k + 1] + mmax[1]);
                    const double *ez = tz + 2 * (m[3 * k + 2] + mmax[2]);
                    double ar = ex[0] * ey[0] - ex[1] * ey[1], ai = ex[0] * ey[1] + ex[1] * ey[0];
                    double pr = ar * ez[0] - ai * ez[1], pi = ar * ez[1] + ai * ez[0];
                    for (int a = 0; a < C; ++a) {
                        double qa = q[(long)a * N + j];
                        loc[2 * ((long)a * K + k)] += qa * pr;
                        loc[2 * ((long)a * K + k) + 1] += qa * pi;
                    }
                }
            }
#pragma omp critical
            for (long t = 0; t < nrho; ++t) rho[t] += loc[t];
        }
        free(loc); free(tx); free(ty); free(tz);
    }
    if (fail) { free(rho); return -1; }

    /* energies */
    double *Qn = (double *)calloc((size_t)(C > 0 ? C : 1), sizeof(double));
    if (!Qn) { free(rho); return -1; }
    for (int a = 0; a < C; ++a) {
        double s = 0.0, Qnet = 0.0;
        for (long k = 0; k < K; ++k) {
            double re = rho[2 * ((long)a * K + k)], im = rho[2 * ((long)a * K + k) + 1];
            s += Phi[(long)a * K + k] * (re * re + im * im);
        }
        for (long j = 0; j < N; ++j) Qnet += q[(long)a * N + j];
        Qn[a] = Qnet;
        E_ch[a] = (2.0 * s + Phi0[a] * Qnet * Qnet) / (2.0 * V);
    }

    /* pass 2: potentials and forces on the requested atoms */
#pragma omp parallel
    {
        double *tx = (double *)malloc(sizeof(double) * 2 * (2 * mmax[0] + 1));
        double *ty = (double *)malloc(sizeof(double) * 2 * (2 * mmax[1] + 1));
        double *tz = (double *)malloc(sizeof(double) * 2 * (2 * mmax[2] + 1));
#pragma omp for schedule(static)
        for (long s = 0; s < n_sub; ++s) {
            long i = sub[s];
            phase_table(pos[3 * i + 0], box[0], mmax[0], tx);
            phase_table(pos[3 * i + 1], box[1], mmax[1], ty);
            phase_table(pos[3 * i + 2], box[2], mmax[2], tz);
            double Fi[3] = {0.0, 0.0, 0.0};
            for (int a = 0; a < C; ++a) {
                double ph = 0.0, g[3] = {0.0, 0.0, 0.0};
                for (long k = 0; k < K; ++k) {
                    const double *ex = tx + 2 * (m[3 * k + 0] + mmax[0]);
                    const double *ey = ty + 2 * (m[3 * k + 1] + mmax[1]);
                    const double *ez = tz + 2 * (m[3 * k + 2] + mmax[2]);
                    double ar = ex[0] * ey[0] - ex[1] * ey[1], ai = ex[0] * ey[1] + ex[1] * ey[0];
                    double pr = ar * ez[0] - ai * ez[1], pi = ar * ez[1] + ai * ez[0];
                    double re = rho[2 * ((long)a * K + k)], im = rho[2 * ((long)a * K + k) + 1];
                    /* t = e^{-ik.r_i} rho = (pr - i pi)(re + i im) */
                    double t_re = pr * re + pi * im, t_im = pr * im - pi * re;
                    double w = Phi[(long)a * K + k];
                    ph += w * t_re;
                    for (int d = 0; d < 3; ++d) {
                        const double kd = (double)m[3 * k + 0] * recip[0 * 3 + d] + (double)m[3 * k + 1] * recip[1 * 3 + d] +
                                          (double)m[3 * k + 2] * recip[2 * 3 + d];
                        g[d] += w * t_im * kd;
                    }
                }
                phi[(long)a * n_sub + s] = (2.0 * ph + Phi0[a] * Qn[a]) / V;
                for (int d = 0; d < 3; ++d) Fi[d] -= q[(long)a * N + i] * 2.0 * g[d] / V;
            }
            for (int d = 0; d < 3; ++d) F[3 * s + d] = Fi[d];
        }
        free(tx); free(ty); free(tz);
    }
    free(rho);
    free(Qn);
    return 0;
}
