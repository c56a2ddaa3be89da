// nbk_hermite_common.h -- the pieces of reading R15 that both Hermite drivers share:
// the power-of-two level of a wanted step, the start-up step, the fp64 predictor of a due particle and
// the corrector.  One copy, used by the host driver
// (nbk_hermite.cpp), the device-resident driver's set-up (nbk_hermite_dev.cu) and its kernels
// (nbk_hermite_kernels.cu).  Plain C++ usable from host and device code; internal to the CUDA path.
//
// PAPER.md L68, L74 name the scheme (4th-order Hermite, block time steps) and print no formula; the
// start-up rule is reading R15: dt_0 = largest 2^-k <= min((eta / 4) |a| / |jerk|, dt_max).
#pragma once
#include <math.h>

#if defined(__CUDACC__)
#define NBK_HD __host__ __device__
#else
#define NBK_HD
#endif

namespace nbk {

constexpr int kTickLog2 = 52;   // time unit 2^-52: exact integer block times up to t = 2048
constexpr int kMaxLevel = 48;   // finest step 2^-48

// Level k of the largest step 2^-k <= want, clamped to [kmin, kMaxLevel] (kmin >= 0; dt_max itself may
// lie in [2^-48, 2) and is rounded down to a power of two first, see level_of_dt_max).
NBK_HD inline int level_for(double want, int kmin) {
    if (!(want > 0.0)) return kMaxLevel;
    int e;
    frexp(want, &e);            // want = f 2^e, f in [0.5, 1)  =>  2^(e-1) <= want < 2^e
    int k = -(e - 1);
    if (k < kmin) k = kmin;
    if (k > kMaxLevel) k = kMaxLevel;
    return k;
}

// Level of dt_max rounded down to a power of two, or -1 if that is outside [2^-kMaxLevel, 1]
// (dt_max >= 2 or < 2^-48: both drivers refuse it with NBK_EINVAL).
NBK_HD inline int level_of_dt_max(double dt_max) {
    if (!(dt_max > 0.0) || dt_max >= 2.0) return -1;
    int e;
    frexp(dt_max, &e);
    const int k = -(e - 1);
    return (k < 0 || k > kMaxLevel) ? -1 : k;
}

// Start-up level (reading R15): step (eta / 4) |a| / |jerk|, dt_max if either norm vanishes.
NBK_HD inline int startup_level(double norm_a, double norm_jerk, double eta, int kmin) {
    const double dtm = ldexp(1.0, -kmin);
    double want = dtm;
    if (norm_jerk > 0.0 && norm_a > 0.0) want = fmin(0.25 * eta * norm_a / norm_jerk, dtm);
    return level_for(want, kmin);
}

// New level after a corrected step (reading R15): Aarseth criterion
//   dt_A = sqrt(eta (|a1| |a2'| + |j1|^2) / (|j1| |a3| + |a2'|^2)),  a2' = a2 + a3 dt (end of the step),
// then the block rule: the step may halve as often as needed, may double once and only if dt_A >= 2 dt,
// 2 dt <= dt_max and the new block time T_new (in ticks of 2^-kTickLog2) is a multiple of 2 dt.
NBK_HD inline double norm3(const double* a) { return sqrt(a[0] * a[0] + a[1] * a[1] + a[2] * a[2]); }
NBK_HD inline int next_level_norms(double na, double nj, double n2, double n3, double eta, int k_old,
                                   int kmin, long long T_new) {
    const double dtm = ldexp(1.0, -kmin), dt_old = ldexp(1.0, -k_old);
    const double num = na * n2 + nj * nj, den = nj * n3 + n2 * n2;
    double want = dtm;
    if (den > 0.0) {
        const double dta = sqrt(eta * num / den);
        if (dta == dta && dta > 0.0) want = fmin(dta, dtm);
    }
    int k = k_old;
    if (want < dt_old) {
        const int kn = level_for(want, kmin);
        k = kn > k ? kn : k;
    } else if (want >= 2.0 * dt_old && k > kmin &&
               (T_new & ((1LL << (kTickLog2 - (k - 1))) - 1)) == 0) {
        k -= 1;
    }
    return k;
}
NBK_HD inline int next_level(const double* a1, const double* j1, const double* a2e, const double* a3,
                             double eta, int k_old, int kmin, long long T_new) {
    return next_level_norms(norm3(a1), norm3(j1), norm3(a2e), norm3(a3), eta, k_old, kmin, T_new);
}


// fp64 predictor of one component of a due particle over its own step dt (reading R8 / R15):
//   x_p = x + v dt + a0 dt^2/2 + j0 dt^3/6,  v_p = v + a0 dt + j0 dt^2/2.
NBK_HD inline void hermite_predict_component(double x, double v, double a0, double j0, double dt,
                                             double& xp, double& vp) {
    xp = x + v * dt + a0 * (dt * dt / 2.0) + j0 * (dt * dt * dt / 6.0);
    vp = v + a0 * dt + j0 * (dt * dt / 2.0);
}

// Corrector of one component (reading R15; fp64) -- the ONE copy of these coefficients in the product
// (host driver nbk_hermite.cpp, hd_correct_kernel and hd_steps_kernel through nbk_device.cuh):
//   a2 = [-6 (a0 - a1) - dt (4 j0 + 2 j1)] / dt^2,   a3 = [12 (a0 - a1) + 6 dt (j0 + j1)] / dt^3,
//   x1 = x_p + a2 dt^4/24 + a3 dt^5/120,  v1 = v_p + a2 dt^3/6 + a3 dt^4/24,  a2e = a2 + a3 dt.
// dt is a block step 2^-k, so 1/dt^2 and 1/dt^3 are exact powers of two and multiplying by them gives
// the bits of the division; the callers pass them (the device builds them from k's bit pattern).
NBK_HD inline void hermite_correct_component(double xp, double vp, double a0, double j0, double a1,
                                             double j1, double dt, double inv_dt2, double inv_dt3,
                                             double& x1, double& v1, double& a2e, double& a3) {
    const double da = a0 - a1;
    const double a2 = (-6.0 * da - dt * (4.0 * j0 + 2.0 * j1)) * inv_dt2;
    a3 = (12.0 * da + 6.0 * dt * (j0 + j1)) * inv_dt3;
    const double dt3 = dt * dt * dt, dt4 = dt3 * dt;
    x1 = xp + a2 * (dt4 / 24.0) + a3 * (dt4 * dt / 120.0);
    v1 = vp + a2 * (dt3 / 6.0) + a3 * (dt4 / 24.0);
    a2e = a2 + a3 * dt;
}

}  // namespace nbk
