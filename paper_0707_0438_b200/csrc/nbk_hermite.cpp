// nbk_hermite.cpp -- a8: host-side 4th-order Hermite predictor-corrector with power-of-two
// block time steps, driving the device force path through the public C ABI only.
//
// PAPER.md L68 ("4th order predictor-corrector Hermite ... a predictor step that predicts a
// particle's position and velocity, then the acceleration, its time derivative (jerk) and
// potential are computed by direct summation and a corrector step ..."), L72-L76 (corrector
// and step selection stay on the host in fp64), L74 (block time steps).  The paper prints
// none of the formulas; the ones below are DESIGN.md reading R15 (Makino & Aarseth 1992 form
// of the corrector, Aarseth step criterion, McMillan & Aarseth block rule).
//
// Per block step (call stack (5) of SURVEY.md):  pick the due block -> nbk_set_ti ->
// nbk_calc_firsthalf (device: predict all N, gather i, force, reduce) -> [host predicts the
// block's own particles in fp64 while the device works] -> nbk_calc_lasthalf -> corrector +
// new step on the host -> nbk_set_j_particles_f64 for the corrected particles only.
// The scheduler is O(n_active) per step: particles are kept in one list per power-of-two
// level; all particles of a level share their last-update time.
#include <chrono>
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <vector>

#include "../../include/nbk.h"
#include "nbk_hermite_common.h"

namespace {

using nbk::kMaxLevel;
using nbk::kTickLog2;
using nbk::level_for;

struct Clock {
    std::chrono::steady_clock::time_point t0 = std::chrono::steady_clock::now();
    double seconds() const {
        return std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count();
    }
};

using nbk::norm3;

struct Levels {
    std::vector<std::vector<int32_t>> list;
    std::vector<int32_t> pos;
    std::vector<int8_t> lev;
    explicit Levels(int64_t n) : list(kMaxLevel + 1), pos(n, -1), lev(n, -1) {}
    void insert(int32_t i, int k) {
        lev[i] = static_cast<int8_t>(k);
        pos[i] = static_cast<int32_t>(list[k].size());
        list[k].push_back(i);
    }
    void remove(int32_t i) {
        auto& l = list[lev[i]];
        const int32_t p = pos[i], last = l.back();
        l[p] = last;
        pos[last] = p;
        l.pop_back();
    }
    int finest() const {
        for (int k = kMaxLevel; k >= 0; --k)
            if (!list[k].empty()) return k;
        return -1;
    }
};

}  // namespace

extern "C" int nbk_hermite_evolve(nbk_ctx* ctx, int64_t n, const double* m, double* x, double* v,
                                  double eps, double t_end, double eta, double dt_max,
                                  nbk_hermite_stats* stats) {
    if (!ctx || n < 1 || !m || !x || !v || !(eps >= 0.0) || !(t_end >= 0.0) || !(eta > 0.0) ||
        !(dt_max > 0.0) || n > INT32_MAX)
        return NBK_EINVAL;
    const int kmin = nbk::level_of_dt_max(dt_max);  // dt_max rounded down to a power of two
    if (kmin < 0) return NBK_EINVAL;                // dt_max in [2^-48, 2): levels are indexed from 0
    const double dtm = std::ldexp(1.0, -kmin);
    if (t_end > 2047.0 || std::fmod(t_end, dtm) != 0.0) return NBK_EINVAL;
    const int64_t T_end = static_cast<int64_t>(std::ldexp(t_end, kTickLog2));
    const float eps2 = static_cast<float>(eps * eps);
    const uint32_t flags = NBK_JERK | NBK_POT;

    Clock wall;
    double gpu_s = 0.0;
    nbk_hermite_stats st;
    std::memset(&st, 0, sizeof(st));

    const size_t N = static_cast<size_t>(n);
    std::vector<double> a(3 * N), jk(3 * N), tl(N, 0.0);
    std::vector<float> fa(3 * N), fj(3 * N);
    std::vector<int32_t> act;
    act.reserve(N);
    std::vector<int> knew(N);
    const int64_t kParallelMin = 2048;   // blocks smaller than this are corrected by the calling thread
    // packed per-block buffers for set_j
    std::vector<double> bt(N), bm(N), bx(3 * N), bv(3 * N), ba(3 * N), bj(3 * N), xp(3 * N), vp(3 * N);
    Levels L(n);
    int rc;

    double prof[4] = {0, 0, 0, 0};  // set_ti+firsthalf, lasthalf, set_j, (unused)
    int slot = 0;
#define NBK_TIMED(call)                  \
    do {                                 \
        Clock c__;                       \
        rc = (call);                     \
        const double s__ = c__.seconds(); \
        gpu_s += s__;                    \
        prof[slot] += s__;               \
        if (rc != NBK_OK) return rc;     \
    } while (0)

    // t = 0: load everything, forces on all particles, first steps
    NBK_TIMED(nbk_set_j_particles_f64(ctx, n, nullptr, nullptr, m, x, v, nullptr, nullptr));
    NBK_TIMED(nbk_set_ti(ctx, 0.0));
    NBK_TIMED(nbk_calc_firsthalf(ctx, n, n, nullptr, nullptr, nullptr, eps2, flags));
    NBK_TIMED(nbk_calc_lasthalf(ctx, n, fa.data(), fj.data(), nullptr));
    st.interactions += n * n;
    for (size_t i = 0; i < N; ++i) {
        for (int c = 0; c < 3; ++c) { a[3 * i + c] = fa[3 * i + c]; jk[3 * i + c] = fj[3 * i + c]; }
        L.insert(static_cast<int32_t>(i),
                 nbk::startup_level(norm3(&a[3 * i]), norm3(&jk[3 * i]), eta, kmin));
    }
    NBK_TIMED(nbk_set_j_particles_f64(ctx, n, nullptr, tl.data(), m, x, v, a.data(), jk.data()));

    int64_t T = 0;
    while (T < T_end) {
        const int kf = L.finest();
        const int64_t step = int64_t(1) << (kTickLog2 - kf);
        const int64_t T_new = (T / step + 1) * step;
        if (T_new > T_end) break;
        const double t_new = std::ldexp(static_cast<double>(T_new), -kTickLog2);
        act.clear();
        for (int k = kf; k >= kmin; --k) {
            if (T_new % (int64_t(1) << (kTickLog2 - k)) != 0) break;
            act.insert(act.end(), L.list[k].begin(), L.list[k].end());
        }
        const int64_t ni = static_cast<int64_t>(act.size());

        slot = 0;
        NBK_TIMED(nbk_set_ti(ctx, t_new));
        NBK_TIMED(nbk_calc_firsthalf(ctx, n, ni, act.data(), nullptr, nullptr, eps2, flags));
        // host predictor (fp64) for the block's own particles, overlapped with the device
#pragma omp parallel for schedule(static) if (ni >= kParallelMin)
        for (int64_t q = 0; q < ni; ++q) {
            const size_t i = static_cast<size_t>(act[q]);
            const double dt = t_new - tl[i];
            for (int c = 0; c < 3; ++c) {
                const size_t k = 3 * i + c;
                nbk::hermite_predict_component(x[k], v[k], a[k], jk[k], dt, xp[3 * q + c], vp[3 * q + c]);
            }
        }
        slot = 1;
        NBK_TIMED(nbk_calc_lasthalf(ctx, ni, fa.data(), fj.data(), nullptr));

        // corrector, Aarseth step and block rule: independent per particle (large blocks run on all
        // host cores); the level lists are updated afterwards in block order, so the result does
        // not depend on the thread count
#pragma omp parallel for schedule(static) if (ni >= kParallelMin)
        for (int64_t q = 0; q < ni; ++q) {
            const int32_t ii = act[q];
            const size_t i = static_cast<size_t>(ii);
            const double dt = t_new - tl[i];  // the particle's own step: an exact power of two
            const double inv_dt2 = 1.0 / (dt * dt), inv_dt3 = 1.0 / (dt * dt * dt);
            double a1[3], j1[3], a2e[3], a3[3];
            for (int c = 0; c < 3; ++c) {
                const size_t k = 3 * i + c;
                a1[c] = fa[3 * q + c];
                j1[c] = fj[3 * q + c];
                nbk::hermite_correct_component(xp[3 * q + c], vp[3 * q + c], a[k], jk[k], a1[c], j1[c], dt,
                                               inv_dt2, inv_dt3, x[k], v[k], a2e[c], a3[c]);
                a[k] = a1[c];
                jk[k] = j1[c];
            }
            tl[i] = t_new;
            // Aarseth criterion and block rule
            const int k = nbk::next_level(a1, j1, a2e, a3, eta, L.lev[i], kmin, T_new);
            knew[q] = k;
            bt[q] = t_new;
            bm[q] = m[i];
            for (int c = 0; c < 3; ++c) {
                bx[3 * q + c] = x[3 * i + c];
                bv[3 * q + c] = v[3 * i + c];
                ba[3 * q + c] = a1[c];
                bj[3 * q + c] = j1[c];
            }
        }
        for (int64_t q = 0; q < ni; ++q) {
            const int32_t ii = act[q];
            if (knew[q] != L.lev[ii]) {
                L.remove(ii);
                L.insert(ii, knew[q]);
            }
        }
        slot = 2;
        NBK_TIMED(nbk_set_j_particles_f64(ctx, ni, act.data(), bt.data(), bm.data(), bx.data(),
                                          bv.data(), ba.data(), bj.data()));
        T = T_new;
        st.block_steps += 1;
        st.particle_steps += ni;
        st.interactions += ni * n;
        int b = 0;
        while ((int64_t(2) << b) <= ni && b < 31) ++b;
        st.ni_histogram[b] += 1;
    }
#undef NBK_TIMED
    st.t_reached = std::ldexp(static_cast<double>(T), -kTickLog2);
    st.wall_seconds = wall.seconds();
    st.gpu_call_seconds = gpu_s;
    if (stats) *stats = st;
    return NBK_OK;
}
