// nbk_force.cu -- the i x j force kernel (a4 + a5), the split-j reduction (a6) and the nearest-
// neighbour re-scan; sm_100a.  The other kernels: nbk_state_kernels.cu (a1, a3),
// nbk_batch_kernels.cu, nbk_hermite_kernels.cu; shared device code: nbk_device.cuh.
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
//     slot per thread) across the tiles of a CTA; a CTA's sums for an i-tile are then rounded
//     ONCE to an fp32 partial row, and the rows of an i-particle (at most one per CTA) are
//     added in fp64 in a fixed order and rounded to the fp32 result -- needed for the 1e-5
//     potential bound (measured pot max 1.3e-7 at C3).
//   * the i-particle's own j entry is left out by INDEX (L96; oracle reading R6): only in the
//     j-tiles that hold the own entry of one of the warp's i-particles a second copy of the
//     loop runs that zeroes that entry's mass.  All other tiles run the unmasked loop.
#include "nbk_device.cuh"

namespace nbk {


// ------------------------------------------------------------------------------ force kernel
template <int I, bool JERK, bool EPS0, bool NN, bool DYN>
__global__ void __launch_bounds__(warps_of(I) * 32, 1) force_kernel(const ForceArgs a) {
    using S = Shape<JERK>;
    constexpr int NACC = S::nacc;
    constexpr int W = warps_of(I);
    constexpr int T = W * 32;
    // eps = 0 keeps the ring slots of a fold group until the group's sums are known to be finite
    // (see below), so the producer runs fewer tiles ahead; a tile lasts tens of microseconds
    constexpr int PF = EPS0 ? kPrefetch - NBK_FOLD : kPrefetch;
    typedef u64 acc_t;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const uint32_t full0 = smem_u32(smem_raw);
    const uint32_t empty0 = full0 + 8 * kStages;
    float* stages = reinterpret_cast<float*>(smem_raw + 128);
    double* sacc = reinterpret_cast<double*>(smem_raw + 128 +
                                             sizeof(float) * kStages * S::stage_floats);
    float* snn_best = reinterpret_cast<float*>(sacc + NACC * I * T);   // [I][T]
    int* snn_tile = reinterpret_cast<int*>(snn_best + I * T);          // [I][T]

    // Block-step forms only (I == 1, and the device-planned DYN forms): the I = 2 and 4 forms of the
    // host entry points run for milliseconds, are launched without the attribute, and their code is
    // left as it was (two more instructions ahead of the tile loop cost 1 % at C3 -- code placement).
    if constexpr (I == 1 || DYN) {
        pdl_trigger();
        pdl_wait();   // before anything the predictor (or the step header) wrote is read
    }
    const int tid = threadIdx.x;
    const int lane = tid & 31;
    const int warp = tid >> 5;
    // launch plan: from the host (kernel parameters) or, for the device-resident integrator, from
    // the step header (made by hd_begin_kernel with the same function the host planner runs)
    Decomp dplan = a.d;
    bool tail_on = a.tail.enabled != 0;
    if constexpr (DYN) {
        if (a.dyn->done || a.dyn->skip || a.dyn->n_act <= 0 || a.dyn->plan_I != I) return;
        dplan = a.dyn->plan;
        if (static_cast<int>(blockIdx.x) >= dplan.G) return;
        tail_on = a.dyn->fused != 0;
    }
    const Decomp& d = DYN ? dplan : a.d;
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
        for (int s = 0; s < PF; ++s)
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
    int held_slot[NBK_FOLD], held_jt[NBK_FOLD], nheld = 0;   // EPS0: tiles of the open fold group

    for (int n = 0; n < n_local; ++n) {
        // producer: keep the ring kPrefetch tiles ahead; a slot is refilled once every warp has
        // arrived on its "empty" barrier (tile m - kStages was the slot's previous tenant)
        if (tid == 0) {
            const int m = n + PF;
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
        // eps = 0 (zero-distance pairs contribute nothing).  Zero distance can
        // only occur at the own entry (guarded copy of the loop, as for eps > 0 where its mass is
        // zeroed) or between coincident distinct particles.  Every other tile runs the plain loop:
        // there a zero distance makes rsqrt = inf and the potential sum non-finite, which the
        // fold below tests once per group of NBK_FOLD tiles; only then the group is redone with
        // the guarded loop.  Common case: no per-pair compare-and-select at all.
        if (__any_sync(0xffffffffu, mine)) {
            tile_packed<I, JERK, EPS0, true, NN, !DYN>(sx, jbeg, jbeg + jlen, ni, sl, acc, a.eps2, tmin);
        } else {
            tile_packed<I, JERK, false, false, NN, !DYN>(sx, jbeg, jbeg + jlen, ni, sl, acc, a.eps2, tmin);
        }

        if (NN) {
#pragma unroll
            for (int q = 0; q < I; ++q) {
                if (tmin[q] < nn_best[q]) { nn_best[q] = tmin[q]; nn_tile[q] = jt; }
                tmin[q] = __int_as_float(0x7f800000);
            }
        }
        if constexpr (EPS0) {   // released after the fold group's check
#pragma unroll
            for (int h = 0; h < NBK_FOLD; ++h)
                if (h == nheld) { held_slot[h] = slot; held_jt[h] = jt; }
            ++nheld;
        } else {   // this warp is done with the ring slot
            __syncwarp();
            if (lane == 0) mbar_arrive(empty0 + 8 * slot);
        }

        // second level: fold the fp32 sums into the thread's private fp64 slots, every NBK_FOLD tiles
        // (fp32 stays within <= NBK_FOLD * 128 terms per packed half) and at the end of a segment
        const bool last_of_tile = (jt == d.njt - 1) || (n == n_local - 1);
        if (last_of_tile || (jt & (NBK_FOLD - 1)) == NBK_FOLD - 1) {
            if constexpr (EPS0) {
                bool bad = false;
#pragma unroll
                for (int q = 0; q < I; ++q) {
                    float lo, hi;
                    unpack(acc[q][DYN ? 0 : 3], lo, hi);   // DYN forms keep no potential sum: inf x 0 in acc x
                    bad |= !(fabsf(lo + hi) < __int_as_float(0x7f800000));
                }
                if (__any_sync(0xffffffffu, bad)) {   // a coincident pair: redo the group, guarded
#pragma unroll
                    for (int q = 0; q < I; ++q) {
#pragma unroll
                        for (int v = 0; v < NACC; ++v) acc[q][v] = acc_t(0);
                    }
#pragma unroll
                    for (int h = 0; h < NBK_FOLD; ++h) {
                        if (h >= nheld) break;
                        const float* hx = stages + held_slot[h] * S::stage_floats;
                        int hl[I];   // the guarded loop with the own-entry mask serves every tile
#pragma unroll
                        for (int q = 0; q < I; ++q) hl[q] = self[q] - held_jt[h] * d.tj;
                        tile_packed<I, JERK, true, true, NN, !DYN>(hx, jbeg, jbeg + jlen, ni, hl, acc, a.eps2, tmin);
                        if (NN) {   // the same minima as the first pass found
#pragma unroll
                            for (int q = 0; q < I; ++q) tmin[q] = __int_as_float(0x7f800000);
                        }
                    }
                }
                __syncwarp();
                if (lane == 0) {
#pragma unroll
                    for (int h = 0; h < NBK_FOLD; ++h)
                        if (h < nheld) mbar_arrive(empty0 + 8 * held_slot[h]);
                }
                nheld = 0;
            }
#pragma unroll
            for (int q = 0; q < I; ++q) {
#pragma unroll
                for (int v = 0; v < NACC; ++v)
                    sacc[(q * NACC + v) * T + tid] += static_cast<double>(acc_take(acc[q][v]));
            }
        }
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
    pdl_trigger();
    pdl_wait();   // every thread, also those of a launch that returns at once (the successor waits on us)
    Decomp dplan = a.d;
    if (a.dyn) {   // device-resident integrator: same plan as the force kernel made
        if (a.dyn->done || a.dyn->skip || a.dyn->n_act <= 0 || a.dyn->fused) return;   // fused: already reduced
        dplan = a.dyn->plan;
        // large steps have two or three rows per i-particle: one thread per particle (as launch_reduce chooses)
        const long long rows_per_i = (static_cast<long long>(dplan.njt) * dplan.G + dplan.P - 1) / dplan.P + 1;
        ix_log2 = (rows_per_i <= 4 && dplan.ti % 256 == 0) ? 8 : 5;
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
        if (a.sum64) {   // j-shard: the caller adds the ranks' sums before the one rounding
#pragma unroll
            for (int v = 0; v < 7; ++v) a.sum64[8 * i + v] = sh[v][tid];
            a.sum64[8 * i + 7] = 0.0;
        }
    }
    __syncthreads();   // shared arrays are reused by the next block of i-particles
    }
}

// One warp per i-particle: find the index inside the winning tile (two-kernel path).
__global__ void __launch_bounds__(256) nn_scan_kernel(const NnScanArgs a) {
    pdl_trigger();
    pdl_wait();
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


// --------------------------------------------------------------------------------- launchers
template <int I, bool JERK, bool EPS0, bool NN, bool DYN>
static cudaError_t prepare_one() {
    auto fn = force_kernel<I, JERK, EPS0, NN, DYN>;
    const size_t smem = smem_bytes_of<I, JERK>();
    cudaError_t err = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                           static_cast<int>(smem));
    if (err != cudaSuccess) return err;
    int nb = 0;
    err = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, fn, warps_of(I) * 32, smem);
    if (err != cudaSuccess) return err;
    return nb >= 1 ? cudaSuccess : cudaErrorLaunchOutOfResources;
}

// the nearest-neighbour form exists for the acc + jerk + pot kernels only; the device-planned (DYN)
// form for acc + jerk + pot with I = 1 and I = 4 (the device-resident integrator)
template <int I, bool JERK, bool EPS0>
static cudaError_t prepare_of() {
    cudaError_t err = prepare_one<I, JERK, EPS0, false, false>();
    if (err != cudaSuccess) return err;
    if constexpr (JERK) err = prepare_one<I, JERK, EPS0, true, false>();
    if (err != cudaSuccess) return err;
    if constexpr (JERK && (I == 1 || I == 4)) err = prepare_one<I, JERK, EPS0, false, true>();
    return err;
}

template <int I, bool JERK, bool EPS0>
static cudaError_t launch_of(const ForceArgs& a, bool nn, cudaStream_t s) {
    const size_t smem = smem_bytes_of<I, JERK>();
    if constexpr (JERK) {
        if (nn) {
            if constexpr (I == 1)
                return launch_pdl(force_kernel<I, JERK, EPS0, true, false>, a.d.G, warps_of(I) * 32, smem, s, a);
            force_kernel<I, JERK, EPS0, true, false><<<a.d.G, warps_of(I) * 32, smem, s>>>(a);
            return cudaGetLastError();
        }
    }
    if (nn) return cudaErrorInvalidValue;
    if constexpr (I == 1)
        return launch_pdl(force_kernel<I, JERK, EPS0, false, false>, a.d.G, warps_of(I) * 32, smem, s, a);
    force_kernel<I, JERK, EPS0, false, false><<<a.d.G, warps_of(I) * 32, smem, s>>>(a);
    return cudaGetLastError();
}

template <int I, bool EPS0>
static cudaError_t launch_dyn_of(const ForceArgs& a, cudaStream_t s) {
    return launch_pdl(force_kernel<I, true, EPS0, false, true>, a.d.G, warps_of(I) * 32,
                      smem_bytes_of<I, true>(), s, a);
}

#define NBK_DISPATCH(CALL, ...)                                                         \
    do {                                                                                \
        const int key = (v.I == 1 ? 0 : v.I == 2 ? 1 : 2) * 4 + (v.jerk ? 2 : 0) +      \
                        (v.eps0 ? 1 : 0);                                               \
        switch (key) {                                                                  \
            case 0: return CALL<1, false, false>(__VA_ARGS__);                          \
            case 1: return CALL<1, false, true>(__VA_ARGS__);                           \
            case 2: return CALL<1, true, false>(__VA_ARGS__);                           \
            case 3: return CALL<1, true, true>(__VA_ARGS__);                            \
            case 4: return CALL<2, false, false>(__VA_ARGS__);                          \
            case 5: return CALL<2, false, true>(__VA_ARGS__);                           \
            case 6: return CALL<2, true, false>(__VA_ARGS__);                           \
            case 7: return CALL<2, true, true>(__VA_ARGS__);                            \
            case 8: return CALL<4, false, false>(__VA_ARGS__);                          \
            case 9: return CALL<4, false, true>(__VA_ARGS__);                           \
            case 10: return CALL<4, true, false>(__VA_ARGS__);                          \
            default: return CALL<4, true, true>(__VA_ARGS__);                           \
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

cudaError_t launch_force_dyn(const Variant& v, const ForceArgs& a, cudaStream_t s) {
    if (!v.jerk || v.nn || !a.dyn) return cudaErrorInvalidValue;
    if (v.I == 1) return v.eps0 ? launch_dyn_of<1, true>(a, s) : launch_dyn_of<1, false>(a, s);
    if (v.I == 4) return v.eps0 ? launch_dyn_of<4, true>(a, s) : launch_dyn_of<4, false>(a, s);
    return cudaErrorInvalidValue;
}

cudaError_t launch_reduce(const Variant& v, const ReduceArgs& a, cudaStream_t s) {
    // ix i-particles x 256 / ix row lanes per CTA.  Small blocks have many rows per i-particle (every CTA
    // of the force launch worked on the one i-tile) and few i-particles: fewer i per CTA then gives more
    // CTAs and more row lanes (n_i = 256 at N = 16384: 8 CTAs x 16 rows per lane -> 128 CTAs x 1 row).
    int ix_log2 = 5;
    while (ix_log2 > 0 && (1 << (ix_log2 - 1)) >= a.d.n_i) --ix_log2;
    const long long rows_per_i = (static_cast<long long>(a.d.njt) * a.d.G + a.d.P - 1) / a.d.P + 1;   // at most
    while (ix_log2 > 0 && (a.d.n_i >> ix_log2) < 128 && (256 >> ix_log2) < rows_per_i) --ix_log2;
    // large blocks have two or three rows per i-particle: one thread per i-particle, no row lanes
    if (rows_per_i <= 4 && a.d.ti % 256 == 0 && a.d.n_i >= 256 * 32) ix_log2 = 8;
    const int ix = 1 << ix_log2;
    const unsigned grid = static_cast<unsigned>((a.d.n_i + ix - 1) / ix);
    if (v.jerk && v.nn) return launch_pdl(reduce_kernel<true, true>, grid, 256, 0, s, a, ix_log2);
    if (v.jerk) return launch_pdl(reduce_kernel<true, false>, grid, 256, 0, s, a, ix_log2);
    return launch_pdl(reduce_kernel<false, false>, grid, 256, 0, s, a, ix_log2);
}


cudaError_t launch_reduce_dyn(const Variant& v, const ReduceArgs& a, int ni_max, cudaStream_t s) {
    unsigned grid = static_cast<unsigned>((ni_max + 31) / 32);
    if (grid > 296) grid = 296;   // grid-stride: most steps return at once (reduced by the force kernel)
    if (v.jerk) return launch_pdl(reduce_kernel<true, false>, grid, 256, 0, s, a, 5);
    return launch_pdl(reduce_kernel<false, false>, grid, 256, 0, s, a, 5);
}

cudaError_t launch_nn_scan(const NnScanArgs& a, cudaStream_t s) {
    if (a.n_i <= 0) return cudaSuccess;
    return launch_pdl(nn_scan_kernel, static_cast<unsigned>((a.n_i + 7) / 8), 256, 0, s, a);
}


}  // namespace nbk
