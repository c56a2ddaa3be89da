// nbk_kernels.cu -- sm_100a kernels of the direct-summation hot path.
//
//   a1  scatter_kernel   set_j staging -> raw j-state
//   a3  predict_kernel   Hermite predictor on the device (L68, L428; the paper runs it on
//                        the host, L78 -- moving it here is what north_star asks for)
//   a4+a5  force_kernel  i-gather + the i x j tile: acc, jerk, potential by direct summation
//                        (L68; Eq. 1; kernel steps 1-4 L91-L96; softening L126-L132)
//   a6  reduce_kernel    sum of the split-j partials (L112-L118, on the host in the paper)
//
// What is kept from the paper's 8800GTX design (L89-L102): i-particles live in registers, one
// thread owns whole i-particles, j-particles stream through shared memory in tiles, no use
// of Newton's third law (L98).  What is different on sm_100a:
//   * the inner loop is written in packed f32x2 arithmetic (FFMA2/FADD2/FMUL2): one
//     instruction handles two j-particles.  Measured on B200: a packed instruction occupies
//     the FP32 pipe for 2 cycles (same flop rate as scalar FFMA, half the issue slots), and 3
//     cycles when its three operands are three distinct register pairs not served by the
//     operand-reuse cache (register-file read bandwidth is two registers per cycle).
//   * one persistent CTA per SM (8, 12 or 16 warps for 4, 2 or 1 i-particles per thread).
//     The warp scheduler favours one CTA over its neighbours on the same SM, so several
//     independent CTAs per SM end one after the other and the last runs alone; one CTA whose
//     warps walk the same tile ring finishes together.
//   * j-tiles are brought in by TMA bulk copies (cp.async.bulk) into a 6-slot ring with one
//     "full" (transaction-count) and one "empty" (one arrival per warp) mbarrier per slot;
//     no __syncthreads in the steady state.  All lanes read the same shared-memory address
//     (LDS.128 broadcast, no bank conflicts).
//   * the (i-tile, j-tile) pair list is cut into G equal contiguous ranges ("stream-K"):
//     every SM gets the same work for any n_i, n_j; a CTA that crosses an i-tile boundary
//     writes one partial row per i-tile it touched and reduce_kernel adds the rows in fp64.
//     The paper's n_i < 4096 split-j special case (L112) becomes the general path.
//   * accumulation is hierarchical: fp32 inside one j-tile, fp64 (shared memory, one private
//     slot per thread) across tiles, fp64 across CTAs -- needed for the 1e-5 potential bound.
//   * the i-particle's own j entry is left out by INDEX (L96; oracle reading R6): only in the
//     j-tiles that hold the own entry of one of the warp's i-particles a second copy of the
//     loop runs that zeroes that entry's mass.  All other tiles run the unmasked loop.
#include "nbk_kernels.cuh"

#ifndef NBK_USE_RCP
#define NBK_USE_RCP 0
#endif
#ifndef NBK_UNROLL
#define NBK_UNROLL 1   // trips of the 4-j step of the packed tile loop unrolled together
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
__device__ __forceinline__ float rcp(float x) {
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
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

#ifdef NBK_TRACE
__device__ long long nbk_trace_buf[3 * 4096];
#endif

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
// NN instantiations also keep, per i, the smallest s seen in this tile ("a
// comparison is added with each force calculation to maintain the particle with the minimum
// distance"); which j it was is found afterwards by re-scanning the one winning tile (nn_scan).
template <int I, bool JERK, bool EPS0, bool MASK, bool NN>
__device__ __forceinline__ void tile_packed(const float* __restrict__ sx, int jbeg, int jend,
                                            const float (&ni)[I][6], const int (&sl)[I],
                                            u64 (&acc)[I][Shape<JERK>::nacc], float eps2,
                                            float (&tmin)[I]) {
    const u64 e2p = pack(eps2, eps2);
    constexpr int kUnroll = NBK_UNROLL;
#pragma unroll kUnroll
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
                } else if (NBK_USE_RCP) {
                    rinv = pack(ra, rb);
                    rinv2 = pack(rcp(r2a), rcp(r2b));
                } else {
                    rinv = pack(ra, rb);
                    rinv2 = mul2(rinv, rinv);
                }
                const u64 mrinv = mul2(mj, rinv);
                acc[q][3] = add2(acc[q][3], mrinv);
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

template <int I, bool JERK, bool EPS0, bool MASK>
__device__ __forceinline__ void tile_scalar(const float* __restrict__ sx, int jbeg, int jend,
                                            const float (&ni)[I][6], const int (&sl)[I],
                                            float (&acc)[I][Shape<JERK>::nacc], float eps2) {
#pragma unroll 2
    for (int jj = jbeg; jj < jend; ++jj) {
        const float xj = sx[jj], yj = sx[kTileJMax + jj], zj = sx[2 * kTileJMax + jj];
        const float mj0 = sx[3 * kTileJMax + jj];
        float vxj = 0.f, vyj = 0.f, vzj = 0.f;
        if (JERK) {
            vxj = sx[4 * kTileJMax + jj]; vyj = sx[5 * kTileJMax + jj]; vzj = sx[6 * kTileJMax + jj];
        }
#pragma unroll
        for (int q = 0; q < I; ++q) {
            const float mj = (MASK && jj == sl[q]) ? 0.f : mj0;
            const float dx = xj + ni[q][0], dy = yj + ni[q][1], dz = zj + ni[q][2];
            const float r2 = fmaf(dz, dz, fmaf(dy, dy, fmaf(dx, dx, eps2)));
            float rinv = rsq(r2);
            if (EPS0) rinv = r2 > 0.f ? rinv : 0.f;
            const float rinv2 = (!EPS0 && NBK_USE_RCP) ? rcp(r2) : rinv * rinv;
            const float mrinv = mj * rinv;
            acc[q][3] += mrinv;
            const float mrinv3 = mrinv * rinv2;
            acc[q][0] = fmaf(mrinv3, dx, acc[q][0]);
            acc[q][1] = fmaf(mrinv3, dy, acc[q][1]);
            acc[q][2] = fmaf(mrinv3, dz, acc[q][2]);
            if (JERK) {
                const float dvx = vxj + ni[q][3], dvy = vyj + ni[q][4], dvz = vzj + ni[q][5];
                const float rv = fmaf(dz, dvz, fmaf(dy, dvy, dx * dvx));
                acc[q][4] = fmaf(mrinv3, dvx, acc[q][4]);
                acc[q][5] = fmaf(mrinv3, dvy, acc[q][5]);
                acc[q][6] = fmaf(mrinv3, dvz, acc[q][6]);
                const float beta = (rv * rinv2) * mrinv3;
                acc[q][7] = fmaf(beta, dx, acc[q][7]);
                acc[q][8] = fmaf(beta, dy, acc[q][8]);
                acc[q][9] = fmaf(beta, dz, acc[q][9]);
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

template <bool PACKED> struct AccT { typedef float type; };
template <> struct AccT<true> { typedef u64 type; };

__device__ __forceinline__ float acc_take(u64& a) {
    float lo, hi;
    unpack(a, lo, hi);
    a = 0ull;
    return lo + hi;
}
__device__ __forceinline__ float acc_take(float& a) {
    const float s = a;
    a = 0.f;
    return s;
}

// ------------------------------------------------------------------------------ force kernel
template <int I, bool JERK, bool EPS0, bool PACKED, bool NN>
__global__ void __launch_bounds__(warps_of(I) * 32, 1) force_kernel(const ForceArgs a) {
    using S = Shape<JERK>;
    constexpr int NACC = S::nacc;
    constexpr int W = warps_of(I);
    constexpr int T = W * 32;
    typedef typename AccT<PACKED>::type acc_t;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const uint32_t full0 = smem_u32(smem_raw);
    const uint32_t empty0 = full0 + 8 * kStages;
    float* stages = reinterpret_cast<float*>(smem_raw + 128);
    double* sacc = reinterpret_cast<double*>(smem_raw + 128 +
                                             sizeof(float) * kStages * S::stage_floats);
    float* snn_best = reinterpret_cast<float*>(sacc + NACC * I * T);   // [I][T]
    int* snn_tile = reinterpret_cast<int*>(snn_best + I * T);          // [I][T]

    const int tid = threadIdx.x;
    const int lane = tid & 31;
    const int warp = tid >> 5;
#ifdef NBK_TRACE
    long long trace_t0 = 0;
    if (tid == 0) asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(trace_t0));
#endif
    // launch plan: from the host (kernel parameters) or, for the device-resident integrator, from
    // the step header (made by hd_begin_kernel with the same function the host planner runs)
    Decomp dplan = a.d;
    bool tail_on = a.tail.enabled != 0;
    if constexpr (I == 1) {
        if (a.dyn) {
            if (a.dyn->done || a.dyn->n_act <= 0) return;
            dplan = a.dyn->plan;
            if (static_cast<int>(blockIdx.x) >= dplan.G) return;
            tail_on = a.dyn->fused != 0;
        }
    }
    const Decomp& d = (I == 1) ? dplan : a.d;
    const int wjn = d.wj;
    const int wj = warp % wjn;           // which slice of each j-tile this warp takes
    const int wi = warp / wjn;           // which 32*I-wide group of the i-tile
    const int jlen = d.tj / wjn;
    const int jbeg = wj * jlen;

    const long long p0 = pair_start(blockIdx.x, d.P, d.G);
    const long long p1 = pair_start(blockIdx.x + 1LL, d.P, d.G);
    const int n_local = static_cast<int>(p1 - p0);
    const int it_first = static_cast<int>(p0 / d.njt);
    const int jt_first = static_cast<int>(p0 - static_cast<long long>(it_first) * d.njt);

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < kStages; ++s) {
            mbar_init(full0 + 8 * s, 1);
            mbar_init(empty0 + 8 * s, W);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < kPrefetch; ++s)
            if (s < n_local)
                issue_tile<JERK>(a.j, (jt_first + s) % d.njt, d.tj, stages + s * S::stage_floats,
                                 full0 + 8 * s);
    }

    float ni[I][6];     // negated i-state: -x -y -z -vx -vy -vz
    int self[I];        // the i-particle's own j index, or -1
    acc_t acc[I][NACC];
    float nn_best[I], tmin[I];   // NN: smallest s so far / in the current tile, and its j-tile
    int nn_tile[I];

    int it = it_first;
    int jt = jt_first;
    bool fresh = true;

    for (int n = 0; n < n_local; ++n) {
        // producer: keep the ring kPrefetch tiles ahead; a slot is refilled once every warp has
        // arrived on its "empty" barrier (tile m - kStages was the slot's previous tenant)
        if (tid == 0) {
            const int m = n + kPrefetch;
            if (m < n_local) {
                const int slot = m % kStages;
                if (m >= kStages) mbar_wait(empty0 + 8 * slot, ((m / kStages) - 1) & 1);
                issue_tile<JERK>(a.j, (jt_first + m) % d.njt, d.tj,
                                 stages + slot * S::stage_floats, full0 + 8 * slot);
            }
        }
        if (fresh) {
            // a4: i-gather (Fig. 1: "Data for particle i is taken directly from global memory")
#pragma unroll
            for (int q = 0; q < I; ++q) {
                const int il = wi * 32 * I + q * 32 + lane;
                const long long i = static_cast<long long>(it) * d.ti + il;
                float x = 0.f, y = 0.f, z = 0.f, vx = 0.f, vy = 0.f, vz = 0.f;
                int idx = -1;
                if (i < d.n_i) {
                    if (I == 1 && a.tail.inline_index) idx = a.tail.i_inline[i];
                    else idx = a.i_index ? a.i_index[i] : static_cast<int>(i);
                    if (idx >= 0) {
                        x = a.j.x[idx]; y = a.j.y[idx]; z = a.j.z[idx];
                        if (JERK) { vx = a.j.vx[idx]; vy = a.j.vy[idx]; vz = a.j.vz[idx]; }
                    }
                    if (a.xi) { x = a.xi[3 * i]; y = a.xi[3 * i + 1]; z = a.xi[3 * i + 2]; }
                    if (JERK && a.vi) { vx = a.vi[3 * i]; vy = a.vi[3 * i + 1]; vz = a.vi[3 * i + 2]; }
                }
                ni[q][0] = -x; ni[q][1] = -y; ni[q][2] = -z;
                ni[q][3] = -vx; ni[q][4] = -vy; ni[q][5] = -vz;
                self[q] = idx;
                nn_best[q] = tmin[q] = __int_as_float(0x7f800000);
                nn_tile[q] = -1;
#pragma unroll
                for (int v = 0; v < NACC; ++v) {
                    sacc[(q * NACC + v) * T + tid] = 0.0;
                    acc[q][v] = acc_t(0);
                }
            }
            fresh = false;
        }

        const int slot = n % kStages;
        mbar_wait(full0 + 8 * slot, (n / kStages) & 1);
        const float* sx = stages + slot * S::stage_floats;

        // does this tile hold the own entry of one of this warp's i-particles?
        int sl[I];
        bool mine = false;
        const int jbase = jt * d.tj;
#pragma unroll
        for (int q = 0; q < I; ++q) {
            sl[q] = self[q] - jbase;
            mine |= static_cast<unsigned>(sl[q]) < static_cast<unsigned>(d.tj);
        }
        if (__any_sync(0xffffffffu, mine)) {
            if constexpr (PACKED) tile_packed<I, JERK, EPS0, true, NN>(sx, jbeg, jbeg + jlen, ni, sl, acc, a.eps2, tmin);
            else tile_scalar<I, JERK, EPS0, true>(sx, jbeg, jbeg + jlen, ni, sl, acc, a.eps2);
        } else {
            if constexpr (PACKED) tile_packed<I, JERK, EPS0, false, NN>(sx, jbeg, jbeg + jlen, ni, sl, acc, a.eps2, tmin);
            else tile_scalar<I, JERK, EPS0, false>(sx, jbeg, jbeg + jlen, ni, sl, acc, a.eps2);
        }

        if (NN) {
#pragma unroll
            for (int q = 0; q < I; ++q) {
                if (tmin[q] < nn_best[q]) { nn_best[q] = tmin[q]; nn_tile[q] = jt; }
                tmin[q] = __int_as_float(0x7f800000);
            }
        }
        // this warp is done with the ring slot
        __syncwarp();
        if (lane == 0) mbar_arrive(empty0 + 8 * slot);

        // second level: fold this tile's fp32 sums into the thread's private fp64 slots
#pragma unroll
        for (int q = 0; q < I; ++q) {
#pragma unroll
            for (int v = 0; v < NACC; ++v)
                sacc[(q * NACC + v) * T + tid] += static_cast<double>(acc_take(acc[q][v]));
        }

        const bool last_of_tile = (jt == d.njt - 1) || (n == n_local - 1);
        if (last_of_tile) {
            // one partial row per (CTA, i-tile touched): 8 floats per i.  When wjn warps split
            // the j-tiles, the warp with slice 0 adds the wjn private sums of each i (fixed order).
            if (NN) {
#pragma unroll
                for (int q = 0; q < I; ++q) {
                    snn_best[q * T + tid] = nn_best[q];
                    snn_tile[q * T + tid] = nn_tile[q];
                }
            }
            if (wjn > 1) __syncthreads();   // uniform: every warp ends the segment at the same n
            const long long row = static_cast<long long>(blockIdx.x) * d.maxseg + (it - it_first);
            if (wj == 0) {
#pragma unroll
                for (int q = 0; q < I; ++q) {
                    const int il = wi * 32 * I + q * 32 + lane;
                    if (NN) {   // slices hold disjoint tiles' parts: smallest s, then lowest tile
                        float b = snn_best[q * T + tid];
                        int bt = snn_tile[q * T + tid];
                        for (int w = 1; w < wjn; ++w) {
                            const float ob = snn_best[q * T + tid + 32 * w];
                            const int ot = snn_tile[q * T + tid + 32 * w];
                            if (ob < b || (ob == b && ot < bt)) { b = ob; bt = ot; }
                        }
                        a.nn_partial[row * d.ti + il] = make_float2(b, __int_as_float(bt));
                    }
                    const double* sa = sacc + (q * NACC) * T + tid;
                    double t[NACC];
#pragma unroll
                    for (int v = 0; v < NACC; ++v) t[v] = sa[v * T];
                    for (int w = 1; w < wjn; ++w) {
#pragma unroll
                        for (int v = 0; v < NACC; ++v) t[v] += sa[v * T + 32 * w];
                    }
                    float4 o0, o1;
                    o0.x = static_cast<float>(t[0]);
                    o0.y = static_cast<float>(t[1]);
                    o0.z = static_cast<float>(t[2]);
                    o0.w = static_cast<float>(t[3]);
                    if (JERK) {
                        o1.x = static_cast<float>(t[4] - 3.0 * t[7 % NACC]);
                        o1.y = static_cast<float>(t[5 % NACC] - 3.0 * t[8 % NACC]);
                        o1.z = static_cast<float>(t[6 % NACC] - 3.0 * t[9 % NACC]);
                    } else {
                        o1.x = o1.y = o1.z = 0.f;
                    }
                    o1.w = 0.f;
                    float4* dst = reinterpret_cast<float4*>(a.partial + (row * d.ti + il) * 8);
                    dst[0] = o0;
                    dst[1] = o1;
                }
            }
            if (wjn > 1) __syncthreads();   // slots are zeroed again by the next segment's gather
            fresh = true;
        }
        if (++jt == d.njt) { jt = 0; ++it; }
    }
    // a6 in the same launch for small blocks (PAPER.md L118 sums the partial forces on the host;
    // here the last CTA to arrive does it, rows in CTA order => same bits whoever is last)
    if constexpr (I == 1) {
        if (tail_on) {
            __shared__ int is_last;
            __threadfence();
            __syncthreads();
            if (tid == 0) {
                const unsigned ticket = atomicAdd(a.tail.counter, 1u);
                is_last = (ticket == static_cast<unsigned>(d.G) - 1u);
                if (is_last) *a.tail.counter = 0u;
            }
            __syncthreads();
            if (is_last) {
                __threadfence();
                constexpr int NV = JERK ? 7 : 4;
                constexpr int RY = T / 32;          // row lanes per i
                const int tx = tid & 31, ty = tid >> 5;
                double s[NV];
#pragma unroll
                for (int v = 0; v < NV; ++v) s[v] = 0.0;
#pragma unroll 4
                for (int k = ty; k < d.G; k += RY) {
                    const float4* p = reinterpret_cast<const float4*>(
                        a.partial + (static_cast<long long>(k) * d.maxseg * d.ti + tx) * 8);
                    const float4 u = __ldcg(p);
                    s[0] += u.x; s[1] += u.y; s[2] += u.z; s[3] += u.w;
                    if (JERK) {
                        const float4 w = __ldcg(p + 1);
                        s[4 % NV] += w.x; s[5 % NV] += w.y; s[6 % NV] += w.z;
                    }
                }
#pragma unroll
                for (int v = 0; v < NV; ++v) sacc[v * T + tid] = s[v];
                __syncthreads();
                for (int st = RY >> 1; st > 0; st >>= 1) {
                    if (ty < st) {
#pragma unroll
                        for (int v = 0; v < NV; ++v) sacc[v * T + tid] += sacc[v * T + tid + st * 32];
                    }
                    __syncthreads();
                }
                if (NN) {
                    // smallest s over the CTAs' rows (ties: lowest tile), then re-scan that tile
                    float b = __int_as_float(0x7f800000);
                    int bt = -1;
                    for (int k = ty; k < d.G; k += RY) {
                        const float2 c = __ldcg(a.nn_partial + static_cast<long long>(k) * d.maxseg * d.ti + tx);
                        const int ct = __float_as_int(c.y);
                        if (c.x < b || (c.x == b && ct < bt)) { b = c.x; bt = ct; }
                    }
                    snn_best[tid] = b;
                    snn_tile[tid] = bt;
                    __syncthreads();
                    for (int st = RY >> 1; st > 0; st >>= 1) {
                        if (ty < st) {
                            const float ob = snn_best[tid + st * 32];
                            const int ot = snn_tile[tid + st * 32];
                            if (ob < snn_best[tid] || (ob == snn_best[tid] && ot < snn_tile[tid])) {
                                snn_best[tid] = ob;
                                snn_tile[tid] = ot;
                            }
                        }
                        __syncthreads();
                    }
                    for (int i = warp; i < d.n_i; i += W) {   // one warp per i-particle
                        int idx = a.tail.inline_index ? a.tail.i_inline[i]
                                                      : (a.i_index ? a.i_index[i] : i);
                        float x = 0.f, y = 0.f, z = 0.f;
                        if (idx >= 0) { x = a.j.x[idx]; y = a.j.y[idx]; z = a.j.z[idx]; }
                        if (a.xi) { x = a.xi[3 * i]; y = a.xi[3 * i + 1]; z = a.xi[3 * i + 2]; }
                        int nn;
                        float r2;
                        nn_scan(a.j, d.n_j, snn_tile[i], d.tj, -x, -y, -z, idx, a.eps2, lane, &nn, &r2);
                        if (lane == 0) {
                            a.nn_index[i] = nn;
                            a.nn_r2[i] = r2;
                            if (a.tail.host_out) {
                                a.tail.host_out[7 * d.n_i + i] = __int_as_float(nn);
                                a.tail.host_out[8 * d.n_i + i] = r2;
                            }
                        }
                    }
                }
                if (ty == 0 && tx < d.n_i) {
                    const int n = d.n_i;
                    float r[7];
                    r[0] = static_cast<float>(sacc[0 * T + tid]);
                    r[1] = static_cast<float>(sacc[1 * T + tid]);
                    r[2] = static_cast<float>(sacc[2 * T + tid]);
                    r[6] = static_cast<float>(-sacc[3 * T + tid]);
                    r[3] = JERK ? static_cast<float>(sacc[(4 % NV) * T + tid]) : 0.f;
                    r[4] = JERK ? static_cast<float>(sacc[(5 % NV) * T + tid]) : 0.f;
                    r[5] = JERK ? static_cast<float>(sacc[(6 % NV) * T + tid]) : 0.f;
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        a.tail.acc[3 * tx + c] = r[c];
                        a.tail.jerk[3 * tx + c] = r[3 + c];
                    }
                    a.tail.pot[tx] = r[6];
                    if (a.tail.host_out) {
#pragma unroll
                        for (int c = 0; c < 3; ++c) {
                            a.tail.host_out[3 * tx + c] = r[c];
                            a.tail.host_out[3 * n + 3 * tx + c] = r[3 + c];
                        }
                        a.tail.host_out[6 * n + tx] = r[6];
                    }
                }
            }
        }
    }
#ifdef NBK_TRACE
    if (tid == 0 && blockIdx.x < 4096) {
        long long t1;
        unsigned smid;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t1));
        asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
        nbk_trace_buf[3 * blockIdx.x] = trace_t0;
        nbk_trace_buf[3 * blockIdx.x + 1] = t1;
        nbk_trace_buf[3 * blockIdx.x + 2] = smid;
    }
#endif
}

// ----------------------------------------------------------------------------- reduce kernel
// PAPER.md L118 ("stored in global memory, after which they are ... summed", done on the host
// there).  256 threads = ix i-particles x (256 / ix) lanes over the partial rows; ix = 32 for
// n_i >= 32, else the next power of two >= n_i so that small blocks still use every thread.
// All i of a block lie in one i-tile (ix divides 32 divides ti); the CTAs that worked on that
// tile are found from the first/last i-tile tables the host filled (no division on the device).
template <bool JERK, bool NN>
__global__ void __launch_bounds__(256) reduce_kernel(const ReduceArgs a, int ix_log2) {
    __shared__ double sh[7][256];
    __shared__ float shb[NN ? 256 : 1];
    __shared__ int sht[NN ? 256 : 1];
    __shared__ int krange[2];
    __shared__ int s_first[kMaxCtas], s_last[kMaxCtas];
    Decomp dplan = a.d;
    if (a.dyn) {   // device-resident integrator: same plan as the force kernel made
        if (a.dyn->done || a.dyn->n_act <= 0 || a.dyn->fused) return;   // fused: already reduced
        dplan = a.dyn->plan;
        ix_log2 = 5;
    }
    const Decomp& d = dplan;
    const int ix = 1 << ix_log2, ry = 256 >> ix_log2;
    const int tid = threadIdx.x;
    const int tx = tid & (ix - 1), ty = tid >> ix_log2;
    // grid-stride over blocks of ix i-particles (the dyn launch has a fixed grid)
    for (long long i0 = static_cast<long long>(blockIdx.x) * ix; i0 < d.n_i;
         i0 += static_cast<long long>(gridDim.x) * ix) {
    const long long i = i0 + tx;
    const bool valid = i < d.n_i;
    const int it = static_cast<int>(i0 / d.ti);
    if (tid < d.G) {
        if (a.dyn) {
            const long long q0 = (static_cast<long long>(tid) * d.P) / d.G;
            const long long q1 = ((static_cast<long long>(tid) + 1) * d.P) / d.G;
            s_first[tid] = static_cast<int>(q0 / d.njt);
            s_last[tid] = static_cast<int>((q1 - 1) / d.njt);
        } else {
            s_first[tid] = a.it_first[tid];
            s_last[tid] = a.it_last[tid];
        }
    }
    __syncthreads();
    if (tid < d.G) {
        const bool in = s_first[tid] <= it && it <= s_last[tid];
        if (in && (tid == 0 || s_last[tid - 1] < it)) krange[0] = tid;
        if (in && (tid == d.G - 1 || s_first[tid + 1] > it)) krange[1] = tid;
    }
    __syncthreads();
    double s[7] = {0, 0, 0, 0, 0, 0, 0};
    float nb = __int_as_float(0x7f800000);
    int nt = -1;
    if (valid) {
        const int il = static_cast<int>(i - static_cast<long long>(it) * d.ti);
        const int k0 = krange[0], k1 = krange[1];
#pragma unroll 4
        for (int k = k0 + ty; k <= k1; k += ry) {
            const int seg = it - s_first[k];
            const long long row = static_cast<long long>(k) * d.maxseg + seg;
            if (NN) {
                const float2 c = a.nn_partial[row * d.ti + il];
                const int ct = __float_as_int(c.y);
                if (c.x < nb || (c.x == nb && ct < nt)) { nb = c.x; nt = ct; }
            }
            const float4* p = reinterpret_cast<const float4*>(a.partial + (row * d.ti + il) * 8);
            const float4 u = p[0];
            s[0] += u.x; s[1] += u.y; s[2] += u.z; s[3] += u.w;
            if (JERK) {
                const float4 v = p[1];
                s[4] += v.x; s[5] += v.y; s[6] += v.z;
            }
        }
    }
#pragma unroll
    for (int v = 0; v < 7; ++v) sh[v][tid] = s[v];
    if (NN) { shb[tid] = nb; sht[tid] = nt; }
    __syncthreads();
    for (int st = ry >> 1; st > 0; st >>= 1) {   // fixed-order tree: deterministic result
        if (ty < st) {
#pragma unroll
            for (int v = 0; v < 7; ++v) sh[v][tid] += sh[v][tid + st * ix];
            if (NN) {
                const float ob = shb[tid + st * ix];
                const int ot = sht[tid + st * ix];
                if (ob < shb[tid] || (ob == shb[tid] && ot < sht[tid])) { shb[tid] = ob; sht[tid] = ot; }
            }
        }
        __syncthreads();
    }
    if (NN && ty == 0 && valid) {
        a.nn_best[i] = shb[tid];
        a.nn_tile[i] = sht[tid];
    }
    if (ty == 0 && valid) {
        a.acc[3 * i + 0] = static_cast<float>(sh[0][tid]);
        a.acc[3 * i + 1] = static_cast<float>(sh[1][tid]);
        a.acc[3 * i + 2] = static_cast<float>(sh[2][tid]);
        a.pot[i] = static_cast<float>(-sh[3][tid]);
        a.jerk[3 * i + 0] = static_cast<float>(sh[4][tid]);
        a.jerk[3 * i + 1] = static_cast<float>(sh[5][tid]);
        a.jerk[3 * i + 2] = static_cast<float>(sh[6][tid]);
    }
    __syncthreads();   // shared arrays are reused by the next block of i-particles
    }
}

// One warp per i-particle: find the index inside the winning tile (two-kernel path).
__global__ void __launch_bounds__(256) nn_scan_kernel(const NnScanArgs a) {
    const int lane = threadIdx.x & 31;
    const int i = blockIdx.x * 8 + (threadIdx.x >> 5);
    if (i >= a.n_i) return;
    const int idx = a.i_index ? a.i_index[i] : i;
    float x = 0.f, y = 0.f, z = 0.f;
    if (idx >= 0) { x = a.j.x[idx]; y = a.j.y[idx]; z = a.j.z[idx]; }
    if (a.xi) { x = a.xi[3 * i]; y = a.xi[3 * i + 1]; z = a.xi[3 * i + 2]; }
    int nn;
    float r2;
    nn_scan(a.j, a.n_j, a.nn_tile[i], a.tj, -x, -y, -z, idx, a.eps2, lane, &nn, &r2);
    if (lane == 0) {
        a.nn_index[i] = nn;
        a.nn_r2[i] = r2;
    }
}

// --------------------------------------------------- batched acc + pot calls
// the GRAPE treecode sends, per group of <= ncrit particles, an
// interaction list and asks for the acceleration (no jerk, no neighbours) on the group's particles;
// one library call per group made the paper choose ncrit of 8192-32768.  Here all groups of a step
// go into one launch: the pair list is the concatenation over groups of their (i-tile, j-tile)
// pairs, cut into G equal ranges like the single-problem kernel; a CTA walks its range group by
// group.  Every (CTA, i-tile) segment writes one partial row (row = segment index + CTA index is
// unique and ordered); batch_reduce_kernel adds each i-tile's rows in CTA order (deterministic).
struct BatchCursor {
    int g, it, jt, nit, njt;
    long long joff, seg;
};
__device__ __forceinline__ void batch_load_group(const BatchArgs& a, BatchCursor& c) {
    c.njt = a.njt[c.g];
    c.nit = (a.i_end[c.g] - a.i_off[c.g] + a.ti - 1) / a.ti;
    c.joff = a.j_off[c.g];
    c.seg = a.seg_prefix[c.g];
}
__device__ __forceinline__ void batch_seek(const BatchArgs& a, long long p, BatchCursor& c) {
    int lo = 0, hi = a.n_groups - 1;     // largest g with pair_prefix[g] <= p
    while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if (a.pair_prefix[mid] <= p) lo = mid; else hi = mid - 1;
    }
    c.g = lo;
    batch_load_group(a, c);
    const long long r = p - a.pair_prefix[lo];
    c.it = static_cast<int>(r / c.njt);
    c.jt = static_cast<int>(r - static_cast<long long>(c.it) * c.njt);
}
__device__ __forceinline__ void batch_advance(const BatchArgs& a, BatchCursor& c) {
    if (++c.jt == c.njt) {
        c.jt = 0;
        if (++c.it == c.nit) {
            c.it = 0;
            if (++c.g < a.n_groups) batch_load_group(a, c);
        }
    }
}

template <bool EPS0>
__global__ void __launch_bounds__(512, 1) batch_kernel(const BatchArgs a) {
    constexpr int I = 1, W = 16, T = 512, NACC = 4;
    using S = Shape<false>;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const uint32_t full0 = smem_u32(smem_raw);
    const uint32_t empty0 = full0 + 8 * kStages;
    float* stages = reinterpret_cast<float*>(smem_raw + 128);
    double* sacc = reinterpret_cast<double*>(smem_raw + 128 + sizeof(float) * kStages * S::stage_floats);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wjn = a.wj;
    const int wj = warp % wjn, wi = warp / wjn;
    const int jlen = a.tj / wjn, jbeg = wj * jlen;
    const long long p0 = pair_start(blockIdx.x, a.P, a.G);
    const long long p1 = pair_start(blockIdx.x + 1LL, a.P, a.G);
    const int n_local = static_cast<int>(p1 - p0);
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < kStages; ++s) {
            mbar_init(full0 + 8 * s, 1);
            mbar_init(empty0 + 8 * s, W);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    auto issue = [&](const BatchCursor& c, int slot) {
        const uint32_t bytes = a.tj * sizeof(float);
        constexpr uint32_t stride = kTileJMax * sizeof(float);
        const size_t off = static_cast<size_t>(c.joff) + static_cast<size_t>(c.jt) * a.tj;
        const uint32_t bar = full0 + 8 * slot;
        mbar_expect_tx(bar, bytes * 4);
        const uint32_t dst = smem_u32(stages + slot * S::stage_floats);
        bulk_g2s(dst + 0 * stride, a.x + off, bytes, bar);
        bulk_g2s(dst + 1 * stride, a.y + off, bytes, bar);
        bulk_g2s(dst + 2 * stride, a.z + off, bytes, bar);
        bulk_g2s(dst + 3 * stride, a.m + off, bytes, bar);
    };
    BatchCursor pc;          // producer's cursor (thread 0 only), kPrefetch tiles ahead
    if (tid == 0) {
        batch_seek(a, p0, pc);
        for (int s = 0; s < kPrefetch && s < n_local; ++s) {
            issue(pc, s);
            batch_advance(a, pc);
        }
    }
    BatchCursor c;
    batch_seek(a, p0, c);
    float ni[I][6];
    int sl[I] = {-1};
    u64 acc[I][NACC];
    float tmin[I];
    bool fresh = true;
    for (int n = 0; n < n_local; ++n) {
        if (tid == 0) {
            const int mth = n + kPrefetch;
            if (mth < n_local) {
                const int slot = mth % kStages;
                if (mth >= kStages) mbar_wait(empty0 + 8 * slot, ((mth / kStages) - 1) & 1);
                issue(pc, slot);
                batch_advance(a, pc);
            }
        }
        if (fresh) {
            const int il = wi * 32 + lane;
            const int i_lo = a.i_off[c.g], n_i = a.i_end[c.g] - i_lo;
            const int i = c.it * a.ti + il;
            float x = 0.f, y = 0.f, z = 0.f;
            if (i < n_i) {
                const float* p = a.xi + 3 * static_cast<size_t>(i_lo + i);
                x = p[0]; y = p[1]; z = p[2];
            }
            ni[0][0] = -x; ni[0][1] = -y; ni[0][2] = -z;
            ni[0][3] = ni[0][4] = ni[0][5] = 0.f;
#pragma unroll
            for (int v = 0; v < NACC; ++v) {
                sacc[v * T + tid] = 0.0;
                acc[0][v] = 0ull;
            }
            fresh = false;
        }
        const int slot = n % kStages;
        mbar_wait(full0 + 8 * slot, (n / kStages) & 1);
        tile_packed<I, false, EPS0, false, false>(stages + slot * S::stage_floats, jbeg, jbeg + jlen,
                                                  ni, sl, acc, a.eps2, tmin);
        __syncwarp();
        if (lane == 0) mbar_arrive(empty0 + 8 * slot);
#pragma unroll
        for (int v = 0; v < NACC; ++v) sacc[v * T + tid] += static_cast<double>(acc_take(acc[0][v]));
        if (c.jt == c.njt - 1 || n == n_local - 1) {   // end of this CTA's part of the i-tile
            if (wjn > 1) __syncthreads();
            const long long row = c.seg + c.it + blockIdx.x;
            if (wj == 0) {
                const int il = wi * 32 + lane;
                double t[NACC];
#pragma unroll
                for (int v = 0; v < NACC; ++v) t[v] = sacc[v * T + tid];
                for (int w = 1; w < wjn; ++w) {
#pragma unroll
                    for (int v = 0; v < NACC; ++v) t[v] += sacc[v * T + tid + 32 * w];
                }
                float4 o;
                o.x = static_cast<float>(t[0]); o.y = static_cast<float>(t[1]);
                o.z = static_cast<float>(t[2]); o.w = static_cast<float>(t[3]);
                *reinterpret_cast<float4*>(a.partial + (row * a.ti + il) * 4) = o;
            }
            if (wjn > 1) __syncthreads();
            fresh = true;
        }
        batch_advance(a, c);
    }
}

// one block per i-tile (segment): add the rows of the CTAs that worked on it, in CTA order
__global__ void batch_reduce_kernel(const BatchArgs a) {
    const long long s = blockIdx.x;
    int lo = 0, hi = a.n_groups - 1;
    while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if (a.seg_prefix[mid] <= s) lo = mid; else hi = mid - 1;
    }
    const int g = lo;
    const int it = static_cast<int>(s - a.seg_prefix[g]);
    const int i_lo = a.i_off[g], n_i = a.i_end[g] - i_lo;
    const int il = threadIdx.x;
    const int i = it * a.ti + il;
    if (i >= n_i) return;
    const long long pl = a.pair_prefix[g] + static_cast<long long>(it) * a.njt[g];
    const long long ph = pl + a.njt[g] - 1;
    long long k0 = (pl * a.G) / a.P;
    while (k0 + 1 < a.G && pair_start(k0 + 1, a.P, a.G) <= pl) ++k0;
    while (k0 > 0 && pair_start(k0, a.P, a.G) > pl) --k0;
    long long k1 = (ph * a.G) / a.P;
    while (k1 + 1 < a.G && pair_start(k1 + 1, a.P, a.G) <= ph) ++k1;
    while (k1 > 0 && pair_start(k1, a.P, a.G) > ph) --k1;
    double t[4] = {0, 0, 0, 0};
    for (long long k = k0; k <= k1; ++k) {
        const float4 o = *reinterpret_cast<const float4*>(a.partial + ((s + k) * a.ti + il) * 4);
        t[0] += o.x; t[1] += o.y; t[2] += o.z; t[3] += o.w;
    }
    const size_t e = static_cast<size_t>(i_lo + i);
    a.acc[3 * e + 0] = static_cast<float>(t[0]);
    a.acc[3 * e + 1] = static_cast<float>(t[1]);
    a.acc[3 * e + 2] = static_cast<float>(t[2]);
    a.pot[e] = static_cast<float>(-t[3]);
}

// caller's lists (m [n], x [n][3]) -> packed SoA, each list padded to a multiple of tj
__global__ void batch_pack_kernel(const BatchPackArgs a) {
    const long long q = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (q >= a.n_padded) return;
    int lo = 0, hi = a.n_groups - 1;
    while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if (a.dst_off[mid] <= q) lo = mid; else hi = mid - 1;
    }
    const long long r = q - a.dst_off[lo];
    const long long len = a.src_len[lo];
    float x = 1e18f, y = 1e18f, z = 1e18f, m = 0.f;
    if (r < len) {
        const long long sidx = a.src_off[lo] + r;
        x = a.xj[3 * sidx]; y = a.xj[3 * sidx + 1]; z = a.xj[3 * sidx + 2];
        m = a.mj[sidx];
    }
    a.x[q] = x; a.y[q] = y; a.z[q] = z; a.m[q] = m;
}

// ------------------------------------------------- device-resident Hermite integrator (8(f)-1)
// the host round trip per block step is what is left once the force runs on
// the device; with fp64 on the device the corrector, the time-step choice and the block scheduler
// can stay there too.  Scheme and formulas: DESIGN.md reading R15 (the same ones the host driver
// nbk_hermite_evolve uses).
//
// Particles sit in one list per power-of-two level k (step 2^-k); all particles of a level share
// their last-update time, so the next block time follows from the finest occupied level and the
// particles due are those with level >= kstar: no pass over N to find them.
// Called by every thread of one CTA (>= 64 threads): hd_begin_kernel for the first step, the last
// block of hd_correct_kernel for all later ones.
__device__ void hd_begin_body(DynHeader* h) {
    __shared__ long long cnt[kMaxLevel + 1];
    __shared__ long long cost[kPlanCandidates];
    __shared__ Decomp cand[kPlanCandidates];
    __shared__ long long s_nact;
    const int tid = threadIdx.x;
    if (h->done) return;
    if (tid <= kMaxLevel) cnt[tid] = h->level_count[tid];
    __syncthreads();
    if (tid == 0) {
        s_nact = -1;
        int kf = -1;
        for (int k = kMaxLevel; k >= 0; --k)
            if (cnt[k] > 0) { kf = k; break; }
        long long T_next = 0;
        if (kf >= 0) {
            const long long step = 1LL << (kTickLog2 - kf);
            T_next = (h->T_now / step + 1) * step;
        }
        if (kf < 0 || T_next > h->T_end) {
            h->done = 1;
            h->n_act = 0;
        } else {
            int kstar = kf;
            long long n_act = 0;
            for (int k = kf; k >= h->kmin; --k) {
                if (T_next & ((1LL << (kTickLog2 - k)) - 1)) break;
                kstar = k;
                n_act += cnt[k];
            }
            h->T_next = T_next;
            h->t_next = ldexp(static_cast<double>(T_next), -kTickLog2);
            h->kstar = kstar;
            h->n_act = static_cast<int>(n_act);
            s_nact = n_act;
        }
    }
    __syncthreads();
    if (s_nact < 0) return;
    if (tid < kPlanCandidates)   // the launch plan of this step: candidates in parallel
        cost[tid] = plan_candidate(s_nact, h->n, h->num_sms, 1, h->max_partial_floats, tid, &cand[tid]);
    __syncthreads();
    if (tid == 0) {
        int bc = -1;
        for (int c = 0; c < kPlanCandidates; ++c)
            if (cost[c] >= 0 && (bc < 0 || cost[c] < cost[bc])) bc = c;
        h->plan = cand[bc];
        h->fused = cand[bc].nit == 1 && cand[bc].n_i <= kFusedMaxI;
    }
}

__global__ void hd_begin_kernel(DynHeader* h) {   // one CTA of 64 threads
    hd_begin_body(h);
}

// a3 for the device-resident integrator: predict every j to t_next and, in the same pass, list the
// particles that are due in ascending index order (block offsets from the per-block level counts,
// ballot prefix inside the block), so that every run takes the same launch shapes and slots.
__global__ void __launch_bounds__(256) hd_predict_kernel(const RawJ raw, DynHeader* h,
                                                         const HermiteState hs, long long n_pad,
                                                         float* px, float* py, float* pz, float* pm,
                                                         float* pvx, float* pvy, float* pvz) {
    __shared__ int red[8];
    __shared__ int wsum[8];
    if (h->done) return;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const long long j = static_cast<long long>(blockIdx.x) * 256 + tid;
    const long long n_j = h->n;
    const int kstar = h->kstar;
    // offset of this index block in act: due particles of all blocks before it
    int part = 0;
    for (int b = tid; b < static_cast<int>(blockIdx.x); b += 256) part += hs.bc_ge[kstar * hs.nblk + b];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
    if (lane == 0) red[warp] = part;
    const double t = h->t_next;
    float o[7] = {1e18f, 1e18f, 1e18f, 0.f, 0.f, 0.f, 0.f};
    bool due = false;
    if (j < n_j) {
        const double dt = t - raw.t[j];
        const double dt2 = dt * dt * 0.5, dt3 = dt * dt * dt * (1.0 / 6.0);
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const double x = raw.x[c * raw.cap + j];
            const double v = raw.v[c * raw.cap + j];
            const double ac = raw.a[c * raw.cap + j];
            const double jk = raw.k[c * raw.cap + j];
            o[c] = static_cast<float>(x + v * dt + ac * dt2 + jk * dt3);
            o[4 + c] = static_cast<float>(v + ac * dt + jk * dt2);
        }
        o[3] = raw.m[j];
        due = hs.level[j] >= kstar;
    }
    const unsigned bal = __ballot_sync(0xffffffffu, due);
    if (lane == 0) wsum[warp] = __popc(bal);
    __syncthreads();
    if (due) {
        int pos = __popc(bal & ((1u << lane) - 1u));
        for (int w = 0; w < 8; ++w) {
            pos += red[w];
            if (w < warp) pos += wsum[w];
        }
        hs.act[pos] = static_cast<int32_t>(j);
    }
    if (j < n_pad) {
        px[j] = o[0]; py[j] = o[1]; pz[j] = o[2]; pm[j] = o[3];
        pvx[j] = o[4]; pvy[j] = o[5]; pvz[j] = o[6];
    }
}

__device__ __forceinline__ double norm3d(const double* a) {
    return sqrt(a[0] * a[0] + a[1] * a[1] + a[2] * a[2]);
}
__device__ __forceinline__ int level_for_dev(double want, int kmin) {
    if (!(want > 0.0)) return kMaxLevel;
    int e;
    frexp(want, &e);
    int k = -(e - 1);
    if (k < kmin) k = kmin;
    if (k > kMaxLevel) k = kMaxLevel;
    return k;
}

// a8 on the device: Hermite corrector, Aarseth step, block rule (fp64), one thread per due particle;
// writes the fp64 state, the level lists' counts and the raw j-state the predictor reads.
__global__ void hd_correct_kernel(const RawJ raw, DynHeader* h, const HermiteState hs,
                                  const float* acc, const float* jerk) {
    if (h->done) return;
    const int n_act = h->n_act;
    for (int q = blockIdx.x * blockDim.x + threadIdx.x; q < n_act; q += gridDim.x * blockDim.x) {
    const int i = hs.act[q];
    const int k0 = hs.level[i];
    const double dt = ldexp(1.0, -k0);
    const double dtm = ldexp(1.0, -h->kmin);
    const long long T_next = h->T_next;
    double a1[3], j1[3], a2e[3], a3[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const size_t e = 3 * static_cast<size_t>(i) + c;
        const double x = hs.x[e], v = hs.v[e], a0 = hs.a[e], j0 = hs.j[e];
        const double xp = x + v * dt + a0 * (dt * dt / 2.0) + j0 * (dt * dt * dt / 6.0);
        const double vp = v + a0 * dt + j0 * (dt * dt / 2.0);
        a1[c] = acc[3 * q + c];
        j1[c] = jerk[3 * q + c];
        const double da = a0 - a1[c];
        const double a2 = (-6.0 * da - dt * (4.0 * j0 + 2.0 * j1[c])) / (dt * dt);
        a3[c] = (12.0 * da + 6.0 * dt * (j0 + j1[c])) / (dt * dt * dt);
        const double dt3 = dt * dt * dt, dt4 = dt3 * dt;
        const double x1 = xp + a2 * (dt4 / 24.0) + a3[c] * (dt4 * dt / 120.0);
        const double v1 = vp + a2 * (dt3 / 6.0) + a3[c] * (dt4 / 24.0);
        a2e[c] = a2 + a3[c] * dt;
        hs.x[e] = x1; hs.v[e] = v1; hs.a[e] = a1[c]; hs.j[e] = j1[c];
        raw.x[c * raw.cap + i] = x1;
        raw.v[c * raw.cap + i] = static_cast<float>(v1);
        raw.a[c * raw.cap + i] = static_cast<float>(a1[c]);
        raw.k[c * raw.cap + i] = static_cast<float>(j1[c]);
    }
    raw.t[i] = h->t_next;
    const double na = norm3d(a1), nj = norm3d(j1), n2 = norm3d(a2e), n3 = norm3d(a3);
    const double num = na * n2 + nj * nj, den = nj * n3 + n2 * n2;
    double want = dtm;
    if (den > 0.0) {
        const double dta = sqrt(h->eta * num / den);
        if (dta == dta && dta > 0.0) want = fmin(dta, dtm);
    }
    int k = k0;
    if (want < dt) {
        const int kn = level_for_dev(want, h->kmin);
        k = kn > k ? kn : k;
    } else if (want >= 2.0 * dt && k > h->kmin && (T_next & ((1LL << (kTickLog2 - (k - 1))) - 1)) == 0) {
        k -= 1;
    }
    if (k != k0) {
        hs.level[i] = k;
        atomicAdd(reinterpret_cast<unsigned long long*>(&h->level_count[k0]), ~0ULL);   // -1
        atomicAdd(reinterpret_cast<unsigned long long*>(&h->level_count[k]), 1ULL);
        const int b = i >> 8;
        for (int l = k0 + 1; l <= k; ++l) atomicAdd(&hs.bc_ge[l * hs.nblk + b], 1);
        for (int l = k + 1; l <= k0; ++l) atomicAdd(&hs.bc_ge[l * hs.nblk + b], -1);
    }
    if (q == 0) {   // bookkeeping of the step (T_now is read only by the next hd_begin_kernel)
        h->T_now = T_next;
        h->block_steps += 1;
        h->particle_steps += n_act;
        h->interactions += static_cast<long long>(n_act) * h->n;
        int b = 0;
        while ((2LL << b) <= n_act && b < 31) ++b;
        h->hist[b] += 1;
    }
    }
    // the last block to finish prepares the next step (T_next, who is due, launch plan): one launch
    // less per block step than a separate hd_begin_kernel
    __shared__ int is_last;
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) {
        const unsigned ticket = atomicAdd(&h->ticket, 1u);
        is_last = (ticket == gridDim.x - 1u);
        if (is_last) h->ticket = 0u;
    }
    __syncthreads();
    if (is_last) {
        __threadfence();
        hd_begin_body(h);
    }
}

// ------------------------------------------------------------------ scatter (a1) / predict (a3)
template <typename T>
__global__ void scatter_kernel(const ScatterArgs s, const RawJ raw) {
    const long long k = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (k >= s.n) return;
    const long long ad = s.addr ? static_cast<long long>(s.addr[k]) : k;
    if (ad < 0 || ad >= s.n_max) return;
    const T* m = static_cast<const T*>(s.m);
    const T* x = static_cast<const T*>(s.x);
    const T* v = static_cast<const T*>(s.v);
    const T* ac = static_cast<const T*>(s.a);
    const T* jk = static_cast<const T*>(s.k);
    raw.m[ad] = static_cast<float>(m[k]);
    raw.t[ad] = s.tj ? s.tj[k] : 0.0;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        raw.x[c * raw.cap + ad] = static_cast<double>(x[3 * k + c]);
        raw.v[c * raw.cap + ad] = v ? static_cast<float>(v[3 * k + c]) : 0.f;
        raw.a[c * raw.cap + ad] = ac ? static_cast<float>(ac[3 * k + c]) : 0.f;
        raw.k[c * raw.cap + ad] = jk ? static_cast<float>(jk[3 * k + c]) : 0.f;
    }
}

// Hermite predictor (reading R8), fp64, rounded once to fp32:
//   x_p = x + v dt + a dt^2/2 + jerk dt^3/6 ;  v_p = v + a dt + jerk dt^2/2 ;  dt = t - t_j
__global__ void predict_kernel(const RawJ raw, double t, long long n_j, long long n_pad, float* px,
                               float* py, float* pz, float* pm, float* pvx, float* pvy,
                               float* pvz) {
    const long long j = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (j >= n_pad) return;
    // padding (n_j <= j < n_pad): massless and far away, so that it is nobody's neighbour
    float o[7] = {1e18f, 1e18f, 1e18f, 0.f, 0.f, 0.f, 0.f};
    if (j < n_j) {
        const double dt = t - raw.t[j];
        const double dt2 = dt * dt * 0.5, dt3 = dt * dt * dt * (1.0 / 6.0);
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const double x = raw.x[c * raw.cap + j];
            const double v = raw.v[c * raw.cap + j];
            const double ac = raw.a[c * raw.cap + j];
            const double jk = raw.k[c * raw.cap + j];
            o[c] = static_cast<float>(x + v * dt + ac * dt2 + jk * dt3);
            o[4 + c] = static_cast<float>(v + ac * dt + jk * dt2);
        }
        o[3] = raw.m[j];
    }
    px[j] = o[0]; py[j] = o[1]; pz[j] = o[2]; pm[j] = o[3];
    pvx[j] = o[4]; pvy[j] = o[5]; pvz[j] = o[6];
}

// The same predictor with a pending set_j of a few particles folded in (a1 + a3 in one launch):
// the thread that owns an updated address stores the new raw state and predicts from it.
__global__ void predict_upd_kernel(const RawJ raw, double t, long long n_j, long long n_pad,
                                   float* px, float* py, float* pz, float* pm, float* pvx,
                                   float* pvy, float* pvz, const InlineJ upd) {
    const long long j = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (j >= n_pad) return;
    // padding (n_j <= j < n_pad): massless and far away, so that it is nobody's neighbour
    float o[7] = {1e18f, 1e18f, 1e18f, 0.f, 0.f, 0.f, 0.f};
    if (j < n_j) {
        int hit = -1;
        for (int k = 0; k < upd.n; ++k)
            if (upd.addr[k] == j) hit = k;   // the last entry for an address wins
        double tj, x[3];
        float v[3], ac[3], jk[3], m;
        if (hit >= 0) {
            tj = upd.t[hit]; m = upd.m[hit];
            raw.t[j] = tj; raw.m[j] = m;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                x[c] = upd.x[hit][c]; v[c] = upd.v[hit][c]; ac[c] = upd.a[hit][c]; jk[c] = upd.k[hit][c];
                raw.x[c * raw.cap + j] = x[c]; raw.v[c * raw.cap + j] = v[c];
                raw.a[c * raw.cap + j] = ac[c]; raw.k[c * raw.cap + j] = jk[c];
            }
        } else {
            tj = raw.t[j]; m = raw.m[j];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                x[c] = raw.x[c * raw.cap + j]; v[c] = raw.v[c * raw.cap + j];
                ac[c] = raw.a[c * raw.cap + j]; jk[c] = raw.k[c * raw.cap + j];
            }
        }
        const double dt = t - tj;
        const double dt2 = dt * dt * 0.5, dt3 = dt * dt * dt * (1.0 / 6.0);
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const double vd = v[c], ad = ac[c], kd = jk[c];
            o[c] = static_cast<float>(x[c] + vd * dt + ad * dt2 + kd * dt3);
            o[4 + c] = static_cast<float>(vd + ad * dt + kd * dt2);
        }
        o[3] = m;
    }
    px[j] = o[0]; py[j] = o[1]; pz[j] = o[2]; pm[j] = o[3];
    pvx[j] = o[4]; pvy[j] = o[5]; pvz[j] = o[6];
}

// --------------------------------------------------------------------------------- launchers
template <int I, bool JERK, bool EPS0, bool PACKED, bool NN>
static cudaError_t prepare_nn() {
    auto fn = force_kernel<I, JERK, EPS0, PACKED, NN>;
    const size_t smem = smem_bytes_of<I, JERK>();
    cudaError_t err = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                           static_cast<int>(smem));
    if (err != cudaSuccess) return err;
    int nb = 0;
    err = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, fn, warps_of(I) * 32, smem);
    if (err != cudaSuccess) return err;
    return nb >= 1 ? cudaSuccess : cudaErrorLaunchOutOfResources;
}

// the nearest-neighbour form exists for the packed acc + jerk + pot kernels only
template <int I, bool JERK, bool EPS0, bool PACKED>
static cudaError_t prepare_of() {
    cudaError_t err = prepare_nn<I, JERK, EPS0, PACKED, false>();
    if (err != cudaSuccess) return err;
    if constexpr (JERK && PACKED) err = prepare_nn<I, JERK, EPS0, PACKED, true>();
    return err;
}

template <int I, bool JERK, bool EPS0, bool PACKED>
static cudaError_t launch_of(const ForceArgs& a, bool nn, cudaStream_t s) {
    const size_t smem = smem_bytes_of<I, JERK>();
    if constexpr (JERK && PACKED) {
        if (nn) {
            force_kernel<I, JERK, EPS0, PACKED, true><<<a.d.G, warps_of(I) * 32, smem, s>>>(a);
            return cudaGetLastError();
        }
    }
    if (nn) return cudaErrorInvalidValue;
    force_kernel<I, JERK, EPS0, PACKED, false><<<a.d.G, warps_of(I) * 32, smem, s>>>(a);
    return cudaGetLastError();
}

#define NBK_DISPATCH(CALL, ...)                                                         \
    do {                                                                                \
        const int key = (v.I == 1 ? 0 : v.I == 2 ? 1 : 2) * 8 + (v.jerk ? 4 : 0) +      \
                        (v.eps0 ? 2 : 0) + (v.packed ? 1 : 0);                          \
        switch (key) {                                                                  \
            case 0: return CALL<1, false, false, false>(__VA_ARGS__);                   \
            case 1: return CALL<1, false, false, true>(__VA_ARGS__);                    \
            case 2: return CALL<1, false, true, false>(__VA_ARGS__);                    \
            case 3: return CALL<1, false, true, true>(__VA_ARGS__);                     \
            case 4: return CALL<1, true, false, false>(__VA_ARGS__);                    \
            case 5: return CALL<1, true, false, true>(__VA_ARGS__);                     \
            case 6: return CALL<1, true, true, false>(__VA_ARGS__);                     \
            case 7: return CALL<1, true, true, true>(__VA_ARGS__);                      \
            case 8: return CALL<2, false, false, false>(__VA_ARGS__);                   \
            case 9: return CALL<2, false, false, true>(__VA_ARGS__);                    \
            case 10: return CALL<2, false, true, false>(__VA_ARGS__);                   \
            case 11: return CALL<2, false, true, true>(__VA_ARGS__);                    \
            case 12: return CALL<2, true, false, false>(__VA_ARGS__);                   \
            case 13: return CALL<2, true, false, true>(__VA_ARGS__);                    \
            case 14: return CALL<2, true, true, false>(__VA_ARGS__);                    \
            case 15: return CALL<2, true, true, true>(__VA_ARGS__);                     \
            case 16: return CALL<4, false, false, false>(__VA_ARGS__);                  \
            case 17: return CALL<4, false, false, true>(__VA_ARGS__);                   \
            case 18: return CALL<4, false, true, false>(__VA_ARGS__);                   \
            case 19: return CALL<4, false, true, true>(__VA_ARGS__);                    \
            case 20: return CALL<4, true, false, false>(__VA_ARGS__);                   \
            case 21: return CALL<4, true, false, true>(__VA_ARGS__);                    \
            case 22: return CALL<4, true, true, false>(__VA_ARGS__);                    \
            default: return CALL<4, true, true, true>(__VA_ARGS__);                     \
        }                                                                               \
    } while (0)

size_t force_smem_bytes(const Variant& v) {
    const int nacc = v.jerk ? 10 : 4, narr = v.jerk ? 7 : 4;
    return 128 + sizeof(float) * kStages * narr * kTileJMax +
           sizeof(double) * nacc * v.I * warps_of(v.I) * 32 + 8 * v.I * warps_of(v.I) * 32;
}

cudaError_t force_prepare(const Variant& v) { NBK_DISPATCH(prepare_of); }

cudaError_t launch_force(const Variant& v, const ForceArgs& a, cudaStream_t s) {
    NBK_DISPATCH(launch_of, a, v.nn, s);
}

cudaError_t launch_reduce(const Variant& v, const ReduceArgs& a, cudaStream_t s) {
    int ix_log2 = 5;
    while (ix_log2 > 0 && (1 << (ix_log2 - 1)) >= a.d.n_i) --ix_log2;
    const int ix = 1 << ix_log2;
    const unsigned grid = static_cast<unsigned>((a.d.n_i + ix - 1) / ix);
    if (v.jerk && v.nn) reduce_kernel<true, true><<<grid, 256, 0, s>>>(a, ix_log2);
    else if (v.jerk) reduce_kernel<true, false><<<grid, 256, 0, s>>>(a, ix_log2);
    else reduce_kernel<false, false><<<grid, 256, 0, s>>>(a, ix_log2);
    return cudaGetLastError();
}

size_t batch_smem_bytes() {
    return 128 + sizeof(float) * kStages * Shape<false>::stage_floats + sizeof(double) * 4 * 512;
}

cudaError_t batch_prepare() {
    cudaError_t e = cudaFuncSetAttribute(batch_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         static_cast<int>(batch_smem_bytes()));
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(batch_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                static_cast<int>(batch_smem_bytes()));
}

cudaError_t launch_batch_pack(const BatchPackArgs& a, cudaStream_t s) {
    if (a.n_padded <= 0) return cudaSuccess;
    batch_pack_kernel<<<static_cast<unsigned>((a.n_padded + 255) / 256), 256, 0, s>>>(a);
    return cudaGetLastError();
}

cudaError_t launch_batch(const BatchArgs& a, bool eps0, cudaStream_t s) {
    if (eps0) batch_kernel<true><<<a.G, 512, batch_smem_bytes(), s>>>(a);
    else batch_kernel<false><<<a.G, 512, batch_smem_bytes(), s>>>(a);
    return cudaGetLastError();
}

cudaError_t launch_batch_reduce(const BatchArgs& a, cudaStream_t s) {
    batch_reduce_kernel<<<static_cast<unsigned>(a.n_seg), a.ti, 0, s>>>(a);
    return cudaGetLastError();
}

cudaError_t launch_hd_begin(DynHeader* h, cudaStream_t st) {
    hd_begin_kernel<<<1, 64, 0, st>>>(h);
    return cudaGetLastError();
}

cudaError_t launch_hd_predict(const RawJ& raw, DynHeader* h, const HermiteState& hs, long long n_pad,
                              float* px, float* py, float* pz, float* pm, float* pvx, float* pvy,
                              float* pvz, cudaStream_t st) {
    const unsigned grid = static_cast<unsigned>((n_pad + 255) / 256);
    hd_predict_kernel<<<grid, 256, 0, st>>>(raw, h, hs, n_pad, px, py, pz, pm, pvx, pvy, pvz);
    return cudaGetLastError();
}

cudaError_t launch_hd_correct(const RawJ& raw, DynHeader* h, const HermiteState& hs, const float* acc,
                              const float* jerk, int n, cudaStream_t st) {
    int grid = (n + 127) / 128;
    if (grid > 64) grid = 64;   // grid-stride over the due particles; most steps hold a handful
    hd_correct_kernel<<<grid, 128, 0, st>>>(raw, h, hs, acc, jerk);
    return cudaGetLastError();
}

cudaError_t launch_reduce_dyn(const Variant& v, const ReduceArgs& a, int ni_max, cudaStream_t s) {
    unsigned grid = static_cast<unsigned>((ni_max + 31) / 32);
    if (grid > 296) grid = 296;   // grid-stride: most steps return at once (reduced by the force kernel)
    if (v.jerk) reduce_kernel<true, false><<<grid, 256, 0, s>>>(a, 5);
    else reduce_kernel<false, false><<<grid, 256, 0, s>>>(a, 5);
    return cudaGetLastError();
}

cudaError_t launch_nn_scan(const NnScanArgs& a, cudaStream_t s) {
    if (a.n_i <= 0) return cudaSuccess;
    nn_scan_kernel<<<(a.n_i + 7) / 8, 256, 0, s>>>(a);
    return cudaGetLastError();
}

__global__ void scatter_inline_kernel(const InlineJ p, const RawJ raw) {
    const int k = threadIdx.x;
    if (k >= p.n) return;
    const long long ad = p.addr[k];
    raw.m[ad] = p.m[k];
    raw.t[ad] = p.t[k];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        raw.x[c * raw.cap + ad] = p.x[k][c];
        raw.v[c * raw.cap + ad] = p.v[k][c];
        raw.a[c * raw.cap + ad] = p.a[k][c];
        raw.k[c * raw.cap + ad] = p.k[k][c];
    }
}

cudaError_t launch_scatter_inline(const InlineJ& p, const RawJ& raw, cudaStream_t st) {
    if (p.n <= 0) return cudaSuccess;
    scatter_inline_kernel<<<1, kInlineMaxJ, 0, st>>>(p, raw);
    return cudaGetLastError();
}

cudaError_t launch_scatter(const ScatterArgs& s, const RawJ& raw, cudaStream_t st) {
    if (s.n <= 0) return cudaSuccess;
    const unsigned grid = static_cast<unsigned>((s.n + 255) / 256);
    if (s.f64) scatter_kernel<double><<<grid, 256, 0, st>>>(s, raw);
    else scatter_kernel<float><<<grid, 256, 0, st>>>(s, raw);
    return cudaGetLastError();
}

cudaError_t launch_predict(const RawJ& raw, double t, long long n_j, long long n_pad, float* px,
                           float* py, float* pz, float* pm, float* pvx, float* pvy, float* pvz,
                           const InlineJ* upd, cudaStream_t st) {
    if (n_pad <= 0) return cudaSuccess;
    const unsigned grid = static_cast<unsigned>((n_pad + 255) / 256);
    if (upd && upd->n > 0)
        predict_upd_kernel<<<grid, 256, 0, st>>>(raw, t, n_j, n_pad, px, py, pz, pm, pvx, pvy, pvz, *upd);
    else
        predict_kernel<<<grid, 256, 0, st>>>(raw, t, n_j, n_pad, px, py, pz, pm, pvx, pvy, pvz);
    return cudaGetLastError();
}

}  // namespace nbk

#ifdef NBK_TRACE
extern "C" int nbk_debug_trace(long long* out, int n) {
    return static_cast<int>(cudaMemcpyFromSymbol(out, nbk::nbk_trace_buf, sizeof(long long) * 3 * n));
}
#endif
