/* ORACLE (C form) -- test infrastructure, not product code.
 *
 * The same definition as oracle/nbody_oracle.py, written as plain double
 * loops: direct summation of acceleration, jerk and potential (
 * Eq. 1; outputs L83), Plummer softening (L126, L132), self pair excluded
 * by index (L96), zero-distance pairs skipped when eps = 0 (L130-L132).
 * No blocking, no reordering: for each i, one pass over j in index order,
 * fp64 throughout.  OpenMP only spreads the independent i over host cores
 * ("The calculation of the force exerted on each particle is independent of
 * the calculations performed for other particles", L46).
 *
 * This is the implementation bench.py times as `cpu_baseline`
 * (`kind: "oracle"`) and the one the large-N parity tests use.  It shares no
 * code with paper_0707_0438_b200/csrc.  Pinned by tests/test_oracle_pins.py
 * (same pins as the numpy form).
 *
 * Build: gcc -O2 -fopenmp -shared -fPIC nbody_oracle.c -o liboracle.so -lm
 */
#include <math.h>
#include <stdint.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_JERK 1u

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* m[n_j], x[n_j][3], v[n_j][3] (v may be NULL when jerk is not wanted);
 * i_index[n_i] (>= 0: that j is the i-particle and is excluded; -1: external);
 * xi/vi [n_i][3] optional explicit i-state (NULL: taken from x, v at i_index).
 * acc[n_i][3], jerk[n_i][3] (may be NULL), pot[n_i].  Returns 0, or -1 on bad args. */
int oracle_force(int64_t n_j, const double *m, const double *x, const double *v,
                 double eps, int64_t n_i, const int64_t *i_index,
                 const double *xi, const double *vi, unsigned flags,
                 double *acc, double *jerk, double *pot)
{
    const int want_jerk = (flags & ORACLE_JERK) != 0;
    const double eps2 = eps * eps;
    if (n_j < 0 || n_i < 0 || !m || !x || !acc || !pot) return -1;
    if (want_jerk && (!v || !jerk)) return -1;
    for (int64_t k = 0; k < n_i; ++k) {
        int64_t idx = i_index ? i_index[k] : k;
        if (idx >= n_j) return -1;
        if (idx < 0 && !xi) return -1;
    }

#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t k = 0; k < n_i; ++k) {
        const int64_t self = i_index ? i_index[k] : k;
        double xk[3], vk[3] = {0.0, 0.0, 0.0};
        for (int d = 0; d < 3; ++d) {
            xk[d] = xi ? xi[3 * k + d] : x[3 * self + d];
            if (want_jerk) vk[d] = vi ? vi[3 * k + d] : v[3 * self + d];
        }
        double a[3] = {0.0, 0.0, 0.0}, jk[3] = {0.0, 0.0, 0.0}, p = 0.0;
        for (int64_t j = 0; j < n_j; ++j) {
            if (j == self) continue;
            const double rx = x[3 * j + 0] - xk[0];
            const double ry = x[3 * j + 1] - xk[1];
            const double rz = x[3 * j + 2] - xk[2];
            const double s = rx * rx + ry * ry + rz * rz + eps2;
            if (eps2 == 0.0 && s == 0.0) continue;
            const double s_m12 = 1.0 / sqrt(s);
            const double s_m32 = s_m12 / s;
            const double f = m[j] * s_m32;
            p -= m[j] * s_m12;
            a[0] += f * rx;
            a[1] += f * ry;
            a[2] += f * rz;
            if (want_jerk) {
                const double wx = v[3 * j + 0] - vk[0];
                const double wy = v[3 * j + 1] - vk[1];
                const double wz = v[3 * j + 2] - vk[2];
                const double rw = rx * wx + ry * wy + rz * wz;
                const double g = 3.0 * m[j] * rw * (s_m32 / s);
                jk[0] += f * wx - g * rx;
                jk[1] += f * wy - g * ry;
                jk[2] += f * wz - g * rz;
            }
        }
        for (int d = 0; d < 3; ++d) {
            acc[3 * k + d] = a[d];
            if (want_jerk) jerk[3 * k + d] = jk[d];
        }
        pot[k] = p;
    }
    return 0;
}

/* Nearest neighbour of each i-particle, own entry excluded by index, ties to
 * the lowest index (reading R20).  nn[k] = -1, r2[k] = INFINITY if there is no other particle. */
int oracle_nearest(int64_t n_j, const double *x, int64_t n_i, const int64_t *i_index,
                   const double *xi, int64_t *nn, double *r2out)
{
    if (n_j < 0 || n_i < 0 || !x || !nn || !r2out) return -1;
    for (int64_t k = 0; k < n_i; ++k) {
        int64_t idx = i_index ? i_index[k] : k;
        if (idx >= n_j) return -1;
        if (idx < 0 && !xi) return -1;
    }
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t k = 0; k < n_i; ++k) {
        const int64_t self = i_index ? i_index[k] : k;
        double xk[3];
        for (int d = 0; d < 3; ++d) xk[d] = xi ? xi[3 * k + d] : x[3 * self + d];
        int64_t best = -1;
        double bestr2 = INFINITY;
        for (int64_t j = 0; j < n_j; ++j) {
            if (j == self) continue;
            const double rx = x[3 * j + 0] - xk[0];
            const double ry = x[3 * j + 1] - xk[1];
            const double rz = x[3 * j + 2] - xk[2];
            const double r2 = rx * rx + ry * ry + rz * rz;
            if (r2 < bestr2) { bestr2 = r2; best = j; }
        }
        nn[k] = best;
        r2out[k] = bestr2;
    }
    return 0;
}

/* Hermite predictor (reading R8): Taylor series through the jerk. */
int oracle_predict(int64_t n, double t, const double *tj, const double *x, const double *v,
                   const double *a, const double *jerk, double *xp, double *vp)
{
    if (n < 0 || !tj || !x || !v || !a || !jerk || !xp || !vp) return -1;
    for (int64_t j = 0; j < n; ++j) {
        const double dt = t - tj[j];
        for (int d = 0; d < 3; ++d) {
            const int64_t q = 3 * j + d;
            xp[q] = x[q] + v[q] * dt + a[q] * (dt * dt / 2.0) + jerk[q] * (dt * dt * dt / 6.0);
            vp[q] = v[q] + a[q] * dt + jerk[q] * (dt * dt / 2.0);
        }
    }
    return 0;
}
