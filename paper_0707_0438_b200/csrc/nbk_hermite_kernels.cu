// nbk_hermite_kernels.cu -- kernels of the device-resident Hermite integrator:
// step header, predictor + selection, fp64 corrector.  Host side: nbk_hermite_dev.cu.
#include "nbk_device.cuh"

namespace nbk {

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
    pdl_trigger();
    pdl_wait();
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
    pdl_trigger();
    pdl_wait();
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


// a8 on the device: Hermite corrector, Aarseth step, block rule (fp64), one thread per due particle;
// writes the fp64 state, the level lists' counts and the raw j-state the predictor reads.
__global__ void hd_correct_kernel(const RawJ raw, DynHeader* h, const HermiteState hs,
                                  const float* acc, const float* jerk) {
    pdl_trigger();
    pdl_wait();
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
    const int k = next_level(a1, j1, a2e, a3, h->eta, k0, h->kmin, T_next);
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


cudaError_t launch_hd_begin(DynHeader* h, cudaStream_t st) {
    return launch_pdl(hd_begin_kernel, 1, 64, 0, st, h);
}

cudaError_t launch_hd_predict(const RawJ& raw, DynHeader* h, const HermiteState& hs, long long n_pad,
                              float* px, float* py, float* pz, float* pm, float* pvx, float* pvy,
                              float* pvz, cudaStream_t st) {
    const unsigned grid = static_cast<unsigned>((n_pad + 255) / 256);
    return launch_pdl(hd_predict_kernel, grid, 256, 0, st, raw, h, hs, n_pad, px, py, pz, pm, pvx, pvy, pvz);
}

cudaError_t launch_hd_correct(const RawJ& raw, DynHeader* h, const HermiteState& hs, const float* acc,
                              const float* jerk, int n, cudaStream_t st) {
    int grid = (n + 127) / 128;
    if (grid > 64) grid = 64;   // grid-stride over the due particles; most steps hold a handful
    return launch_pdl(hd_correct_kernel, static_cast<unsigned>(grid), 128, 0, st, raw, h, hs, acc, jerk);
}


}  // namespace nbk
