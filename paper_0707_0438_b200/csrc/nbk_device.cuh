// nbk_device.cuh -- device-side building blocks shared by the kernel sources: packed f32x2
// arithmetic, mbarrier / TMA bulk-copy helpers, the shared-memory tile ring's shape, and the
// i x j tile loops with the nearest-neighbour re-scan (L126-L128).
// Internal to the CUDA path.
#pragma once
#include "nbk_kernels.cuh"

#ifndef NBK_FOLD
#define NBK_FOLD 2     // j-tiles between folds of the fp32 accumulators into fp64 (power of two)
#endif

namespace nbk {

typedef unsigned long long u64;

// ---------------------------------------------------------------- packed fp32 pair helpers
__device__ __forceinline__ u64 fma2(u64 a, u64 b, u64 c) {
    u64 d;
    asm("fma.rn.ftz.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ u64 add2(u64 a, u64 b) {
    u64 d;
    asm("add.rn.ftz.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ u64 mul2(u64 a, u64 b) {
    u64 d;
    asm("mul.rn.ftz.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ u64 pack(float lo, float hi) {
    u64 d;
    asm("mov.b64 %0, {%1, %2};" : "=l"(d) : "f"(lo), "f"(hi));
    return d;
}
__device__ __forceinline__ void unpack(u64 d, float& lo, float& hi) {
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(d));
}
__device__ __forceinline__ float rsq(float x) {
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// ---------------------------------------------------------------- mbarrier / TMA bulk helpers
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    do {
        asm volatile(
            "{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            " selp.u32 %0, 1, 0, p;\n}"
            : "=r"(ok)
            : "r"(bar), "r"(parity)
            : "memory");
    } while (!ok);
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes,
                                         uint32_t bar) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
        ::"r"(dst), "l"(src), "r"(bytes), "r"(bar)
        : "memory");
}


__host__ __device__ __forceinline__ long long pair_start(long long k, long long P, int G) {
    return (k * P) / G;
}

// Shared memory of force_kernel:
//   [kStages full mbarriers | kStages empty mbarriers | pad to 128 B]
//   [kStages x narr x kTileJMax floats]  [nacc*I x threads doubles]
template <bool JERK>
struct Shape {
    static constexpr int narr = JERK ? 7 : 4;   // x y z m [vx vy vz]
    static constexpr int nacc = JERK ? 10 : 4;  // ax ay az pot [j1 xyz, j2 xyz]
    static constexpr int stage_floats = narr * kTileJMax;
};

template <int I, bool JERK>
constexpr size_t smem_bytes_of() {
    return 128 + sizeof(float) * kStages * Shape<JERK>::stage_floats +
           sizeof(double) * Shape<JERK>::nacc * I * warps_of(I) * 32 +
           8 * I * warps_of(I) * 32;   // nearest-neighbour (distance, tile) per thread and i
}

// One elected thread: bring j-tile `jt` (tj particles) into a ring slot.
template <bool JERK>
__device__ __forceinline__ void issue_tile(const JPred& j, int jt, int tj, float* stage,
                                           uint32_t bar) {
    const uint32_t bytes = tj * sizeof(float);
    constexpr uint32_t stride = kTileJMax * sizeof(float);
    const size_t off = static_cast<size_t>(jt) * tj;
    mbar_expect_tx(bar, bytes * Shape<JERK>::narr);
    const uint32_t dst = smem_u32(stage);
    bulk_g2s(dst + 0 * stride, j.x + off, bytes, bar);
    bulk_g2s(dst + 1 * stride, j.y + off, bytes, bar);
    bulk_g2s(dst + 2 * stride, j.z + off, bytes, bar);
    bulk_g2s(dst + 3 * stride, j.m + off, bytes, bar);
    if (JERK) {
        bulk_g2s(dst + 4 * stride, j.vx + off, bytes, bar);
        bulk_g2s(dst + 5 * stride, j.vy + off, bytes, bar);
        bulk_g2s(dst + 6 * stride, j.vz + off, bytes, bar);
    }
}

// ------------------------------------------------------------------- the i x j tile loops
// PAPER.md L91-L96 (kernel steps 1-4).  Per ordered pair (i, j), r = x_j - x_i, w = v_j - v_i,
// s = r.r + eps2:
//   pot  += m s^-1/2            (sign applied in reduce_kernel)
//   acc  += m s^-3/2 r
//   j1   += m s^-3/2 w ;  j2 += m s^-5/2 (r.w) r ;  jerk = j1 - 3 j2 (formed per partial row)
// The i-state is held negated (r = x_j + (-x_i) is one add).  sl[q] is the position of the
// i-particle's own j entry inside this tile (anything outside [0, tj) if it is elsewhere);
// MASK instantiations zero the mass of that entry.
// POT = false leaves the potential sum out (acc[q][3] stays 0).
// NN instantiations also keep, per i, the smallest s seen in this tile ("a
// comparison is added with each force calculation to maintain the particle with the minimum
// distance"); which j it was is found afterwards by re-scanning the one winning tile (nn_scan).
template <int I, bool JERK, bool EPS0, bool MASK, bool NN, bool POT = true>
__device__ __forceinline__ void tile_packed(const float* __restrict__ sx, int jbeg, int jend,
                                            const float (&ni)[I][6], const int (&sl)[I],
                                            u64 (&acc)[I][Shape<JERK>::nacc], float eps2,
                                            float (&tmin)[I]) {
    const u64 e2p = pack(eps2, eps2);
#pragma unroll 1
    for (int jj = jbeg; jj < jend; jj += 4) {
        const ulonglong2 X = *reinterpret_cast<const ulonglong2*>(sx + jj);
        const ulonglong2 Y = *reinterpret_cast<const ulonglong2*>(sx + kTileJMax + jj);
        const ulonglong2 Z = *reinterpret_cast<const ulonglong2*>(sx + 2 * kTileJMax + jj);
        const ulonglong2 M = *reinterpret_cast<const ulonglong2*>(sx + 3 * kTileJMax + jj);
        ulonglong2 VX, VY, VZ;
        if (JERK) {
            VX = *reinterpret_cast<const ulonglong2*>(sx + 4 * kTileJMax + jj);
            VY = *reinterpret_cast<const ulonglong2*>(sx + 5 * kTileJMax + jj);
            VZ = *reinterpret_cast<const ulonglong2*>(sx + 6 * kTileJMax + jj);
        }
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const u64 xj = h ? X.y : X.x, yj = h ? Y.y : Y.x, zj = h ? Z.y : Z.x;
            const u64 mj0 = h ? M.y : M.x;
#pragma unroll
            for (int q = 0; q < I; ++q) {
                u64 mj = mj0;
                if (MASK) {  // the i-particle's own entry contributes nothing
                    float mlo, mhi;
                    unpack(mj0, mlo, mhi);
                    mlo = (jj + 2 * h == sl[q]) ? 0.f : mlo;
                    mhi = (jj + 2 * h + 1 == sl[q]) ? 0.f : mhi;
                    mj = pack(mlo, mhi);
                }
                const u64 dx = add2(xj, pack(ni[q][0], ni[q][0]));
                const u64 dy = add2(yj, pack(ni[q][1], ni[q][1]));
                const u64 dz = add2(zj, pack(ni[q][2], ni[q][2]));
                u64 r2 = fma2(dx, dx, e2p);
                r2 = fma2(dy, dy, r2);
                r2 = fma2(dz, dz, r2);
                float r2a, r2b;
                unpack(r2, r2a, r2b);
                if (NN) {
                    float qa = r2a, qb = r2b;
                    if (MASK) {  // the own entry is nobody's neighbour
                        qa = (jj + 2 * h == sl[q]) ? __int_as_float(0x7f800000) : qa;
                        qb = (jj + 2 * h + 1 == sl[q]) ? __int_as_float(0x7f800000) : qb;
                    }
                    tmin[q] = fminf(tmin[q], fminf(qa, qb));
                }
                float ra = rsq(r2a), rb = rsq(r2b);
                u64 rinv, rinv2;
                if (EPS0) {  // zero-distance pairs contribute nothing
                    ra = r2a > 0.f ? ra : 0.f;
                    rb = r2b > 0.f ? rb : 0.f;
                    rinv = pack(ra, rb);
                    rinv2 = mul2(rinv, rinv);
                } else {
                    rinv = pack(ra, rb);
                    rinv2 = mul2(rinv, rinv);
                }
                const u64 mrinv = mul2(mj, rinv);
                if (POT) acc[q][3] = add2(acc[q][3], mrinv);   // (the integrator's kernels do not need the potential)
                const u64 mrinv3 = mul2(mrinv, rinv2);
                acc[q][0] = fma2(mrinv3, dx, acc[q][0]);
                acc[q][1] = fma2(mrinv3, dy, acc[q][1]);
                acc[q][2] = fma2(mrinv3, dz, acc[q][2]);
                if (JERK) {
                    const u64 vxj = h ? VX.y : VX.x, vyj = h ? VY.y : VY.x, vzj = h ? VZ.y : VZ.x;
                    const u64 dvx = add2(vxj, pack(ni[q][3], ni[q][3]));
                    const u64 dvy = add2(vyj, pack(ni[q][4], ni[q][4]));
                    const u64 dvz = add2(vzj, pack(ni[q][5], ni[q][5]));
                    u64 rv = mul2(dx, dvx);
                    rv = fma2(dy, dvy, rv);
                    rv = fma2(dz, dvz, rv);
                    acc[q][4] = fma2(mrinv3, dvx, acc[q][4]);
                    acc[q][5] = fma2(mrinv3, dvy, acc[q][5]);
                    acc[q][6] = fma2(mrinv3, dvz, acc[q][6]);
                    const u64 beta = mul2(mul2(rv, rinv2), mrinv3);
                    acc[q][7] = fma2(beta, dx, acc[q][7]);
                    acc[q][8] = fma2(beta, dy, acc[q][8]);
                    acc[q][9] = fma2(beta, dz, acc[q][9]);
                }
            }
        }
    }
}

// Nearest neighbour, second step: one warp re-scans the one j-tile whose minimum won, with the
// arithmetic of the tile loop (same s for the same pair), and returns the lowest j that attains the
// tile's minimum, the own entry left out by index (reading R20: ties go to the lowest index).
// r2out is the unsoftened squared distance of that pair in fp32.
__device__ __forceinline__ float sfma(float a, float b, float c) {
    float d;
    asm("fma.rn.ftz.f32 %0, %1, %2, %3;" : "=f"(d) : "f"(a), "f"(b), "f"(c));
    return d;
}
__device__ __forceinline__ float sadd(float a, float b) {
    float d;
    asm("add.rn.ftz.f32 %0, %1, %2;" : "=f"(d) : "f"(a), "f"(b));
    return d;
}
__device__ __forceinline__ void nn_scan(const JPred& j, int n_j, int tile, int tj, float nx,
                                        float ny, float nz, int self, float eps2, int lane,
                                        int* nn_out, float* r2_out) {
    float best = __int_as_float(0x7f800000);
    int bj = 0x7fffffff;
    if (tile >= 0) {
        const int j0 = tile * tj;
        for (int jj = j0 + lane; jj < j0 + tj && jj < n_j; jj += 32) {
            const float dx = sadd(j.x[jj], nx), dy = sadd(j.y[jj], ny), dz = sadd(j.z[jj], nz);
            const float s = sfma(dz, dz, sfma(dy, dy, sfma(dx, dx, eps2)));
            if (jj != self && s < best) { best = s; bj = jj; }   // ascending jj: first minimum kept
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const float ob = __shfl_xor_sync(0xffffffffu, best, o);
        const int oj = __shfl_xor_sync(0xffffffffu, bj, o);
        if (ob < best || (ob == best && oj < bj)) { best = ob; bj = oj; }
    }
    if (lane == 0) {
        if (bj == 0x7fffffff) {
            *nn_out = -1;
            *r2_out = __int_as_float(0x7f800000);
        } else {
            const float dx = sadd(j.x[bj], nx), dy = sadd(j.y[bj], ny), dz = sadd(j.z[bj], nz);
            *nn_out = bj;
            *r2_out = sfma(dz, dz, sfma(dy, dy, dx * dx));
        }
    }
}

// ------------------------------------------------------- Hermite predictor / corrector, one particle
// Predictor (reading R8), fp64, rounded once to fp32:
//   x_p = x + v dt + a dt^2/2 + jerk dt^3/6 ;  v_p = v + a dt + jerk dt^2/2 ;  dt = t - t_j
// o = x y z m vx vy vz.  One copy for predict_kernel, hd_predict_kernel and hd_steps_kernel, so that an
// i-particle predicted on its own has the bits of its j entry.
// CG: load through L2 (ld.global.cg) -- for the persistent stepping kernel, where other CTAs rewrite
// the state between two reads by this one and a line kept in L1 would be stale.
template <bool CG, typename T>
__device__ __forceinline__ T ld_state(const T* p) { return CG ? __ldcg(p) : *p; }

// one component: x_p (o_x) and v_p (o_v) from the raw state of a particle
__device__ __forceinline__ void predict_component(double x, double v, double ac, double jk, double dt,
                                                  double dt2, double dt3, float& o_x, float& o_v) {
    o_x = static_cast<float>(x + v * dt + ac * dt2 + jk * dt3);
    o_v = static_cast<float>(v + ac * dt + jk * dt2);
}

template <bool CG = false>
__device__ __forceinline__ void predict_one(const RawJ& raw, long long j, double t, float (&o)[7]) {
    const double dt = t - ld_state<CG>(raw.t + j);
    const double dt2 = dt * dt * 0.5, dt3 = dt * dt * dt * (1.0 / 6.0);
#pragma unroll
    for (int c = 0; c < 3; ++c)
        predict_component(ld_state<CG>(raw.x + c * raw.cap + j), ld_state<CG>(raw.v + c * raw.cap + j),
                          ld_state<CG>(raw.a + c * raw.cap + j), ld_state<CG>(raw.k + c * raw.cap + j), dt,
                          dt2, dt3, o[c], o[4 + c]);
    o[3] = ld_state<CG>(raw.m + j);
}

// Predictor + corrector of one component of a due particle (reading R15; fp64; formulas in
// nbk_hermite_common.h).  dt = 2^-k is a power of two, so the divisions by dt^2 and dt^3 are exact
// multiplications by 2^2k and 2^3k (same bits as the quotient).
__device__ __forceinline__ void correct_component(double x, double v, double a0, double j0, double a1,
                                                  double j1, int k, double& x1, double& v1,
                                                  double& a2e, double& a3) {
    // exact powers of two, written as bit patterns (k <= kMaxLevel = 48: exponents stay normal)
    const double dt = __longlong_as_double((1023LL - k) << 52);
    const double inv_dt2 = __longlong_as_double((1023LL + 2 * k) << 52);
    const double inv_dt3 = __longlong_as_double((1023LL + 3 * k) << 52);
    double xp, vp;
    hermite_predict_component(x, v, a0, j0, dt, xp, vp);
    hermite_correct_component(xp, vp, a0, j0, a1, j1, dt, inv_dt2, inv_dt3, x1, v1, a2e, a3);
}

// What a corrected particle writes: the fp64 state and the raw j-state the predictor reads.
__device__ __forceinline__ void store_corrected(const RawJ& raw, const HermiteState& hs, int i, int c,
                                                double x1, double v1, double a1, double j1) {
    const size_t e = 3 * static_cast<size_t>(i) + c;
    hs.x[e] = x1; hs.v[e] = v1; hs.a[e] = a1; hs.j[e] = j1;
    raw.x[c * raw.cap + i] = x1;
    raw.v[c * raw.cap + i] = static_cast<float>(v1);
    raw.a[c * raw.cap + i] = static_cast<float>(a1);
    raw.k[c * raw.cap + i] = static_cast<float>(j1);
}

// Level change of particle i: its level, the level counts and the per-index-block counts (integer
// atomics: order-independent).
__device__ __forceinline__ void store_level(const HermiteState& hs, DynHeader* h, int i, int k0, int k) {
    if (k == k0) return;
    hs.level[i] = static_cast<unsigned char>(k + 1);
    atomicAdd(reinterpret_cast<unsigned long long*>(&h->level_count[k0]), ~0ULL);   // -1
    atomicAdd(reinterpret_cast<unsigned long long*>(&h->level_count[k]), 1ULL);
    const int b = i >> 8;
    for (int l = k0 + 1; l <= k; ++l) atomicAdd(&hs.bc_ge[l * hs.nblk + b], 1);
    for (int l = k + 1; l <= k0; ++l) atomicAdd(&hs.bc_ge[l * hs.nblk + b], -1);
}

// Corrector, Aarseth step and block rule for one due particle i (reading R15; fp64): a1f, j1f are the
// new force and jerk (fp32 results of the force path).
__device__ __forceinline__ void correct_one(const RawJ& raw, const HermiteState& hs, DynHeader* h, int i,
                                            const float* a1f, const float* j1f, long long T_next,
                                            double t_next, double eta, int kmin) {
    const int k0 = hs.level[i] - 1;
    double a1[3], j1[3], a2e[3], a3[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const size_t e = 3 * static_cast<size_t>(i) + c;
        double x1, v1;
        a1[c] = a1f[c];
        j1[c] = j1f[c];
        correct_component(hs.x[e], hs.v[e], hs.a[e], hs.j[e], a1[c], j1[c], k0, x1, v1, a2e[c], a3[c]);
        store_corrected(raw, hs, i, c, x1, v1, a1[c], j1[c]);
    }
    raw.t[i] = t_next;
    store_level(hs, h, i, k0, next_level(a1, j1, a2e, a3, eta, k0, kmin, T_next));
}

// One ordered pair in scalar fp32 (the formulas of tile_packed with the jerk formed
// per pair: u = w - 3 (r.w) r / s, jerk += m s^-3/2 u).  nx.. = negated i-state; s7 += acc3, m/sqrt(s), jerk3.
template <bool JERK, bool EPS0>
__device__ __forceinline__ void pair_scalar(const float (&jv)[7], const float* ni, bool self, float eps2,
                                            float (&s7)[7]) {
    const float dx = jv[0] + ni[0], dy = jv[1] + ni[1], dz = jv[2] + ni[2];
    const float r2 = fmaf(dz, dz, fmaf(dy, dy, fmaf(dx, dx, eps2)));
    float rinv = rsq(r2);
    if (EPS0) rinv = r2 > 0.f ? rinv : 0.f;
    const float m = self ? 0.f : jv[3];       // L96: the own entry contributes nothing
    const float rinv2 = rinv * rinv, mrinv = m * rinv, mrinv3 = mrinv * rinv2;
    s7[0] = fmaf(mrinv3, dx, s7[0]);
    s7[1] = fmaf(mrinv3, dy, s7[1]);
    s7[2] = fmaf(mrinv3, dz, s7[2]);
    s7[3] += mrinv;
    if (JERK) {
        const float dvx = jv[4] + ni[3], dvy = jv[5] + ni[4], dvz = jv[6] + ni[5];
        const float rv = fmaf(dz, dvz, fmaf(dy, dvy, dx * dvx));
        const float g3 = -3.f * (rv * rinv2);
        s7[4] = fmaf(mrinv3, fmaf(g3, dx, dvx), s7[4]);
        s7[5] = fmaf(mrinv3, fmaf(g3, dy, dvy), s7[5]);
        s7[6] = fmaf(mrinv3, fmaf(g3, dz, dvz), s7[6]);
    }
}


// Bookkeeping of one finished block step (one thread).
__device__ __forceinline__ void step_bookkeeping(DynHeader* h, long long T_next, int n_act) {
    h->T_now = T_next;
    h->block_steps += 1;
    h->particle_steps += n_act;
    h->interactions += static_cast<long long>(n_act) * h->n;
    int b = 0;
    while ((2LL << b) <= n_act && b < 31) ++b;
    h->hist[b] += 1;
}

__device__ __forceinline__ float acc_take(u64& a) {
    float lo, hi;
    unpack(a, lo, hi);
    a = 0ull;
    return lo + hi;
}


}  // namespace nbk
