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
// One CTA of 64 threads.  Steps that hd_steps_kernel takes (n_act <= steps_max_act) are only
// marked (skip): the launched chain predict -> force -> reduce -> correct returns at once.
__global__ void hd_begin_kernel(DynHeader* h) {
    __shared__ long long cnt[kMaxLevel + 1];
    __shared__ long long cost[2 * kPlanCandidates];
    __shared__ Decomp cand[2 * kPlanCandidates];
    __shared__ long long s_nact;
    pdl_trigger();
    pdl_wait();
    const int tid = threadIdx.x;
    if (h->done) return;
    if (h->error) {   // the stepping kernel gave up a wait: the state is undefined, run nothing more on it
        if (tid == 0) h->done = 1;
        return;
    }
    if (tid <= kMaxLevel) cnt[tid] = h->level_count[tid];
    __syncthreads();
    if (tid == 0) {
        s_nact = -1;
        h->skip = 0;
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
            if (n_act <= h->steps_max_act) h->skip = 1;
            else s_nact = n_act;
        }
    }
    __syncthreads();
    if (s_nact < 0) return;
    // the launch plan of this step: the candidates of I = 1 and I = 4 in parallel, then the host
    // planner's rule (cost x warps / measured speed of the form, plan_shape)
    if (tid < 2 * kPlanCandidates) {
        const int I = tid < kPlanCandidates ? 1 : 4;
        cost[tid] = plan_candidate(s_nact, h->n, h->num_sms, I, h->max_partial_floats, tid % kPlanCandidates,
                                   &cand[tid]);
    }
    __syncthreads();
    if (tid == 0) {
        int bc = -1;
        double best = 0.0;
        for (int c = h->steps_max_act > 0 ? kPlanCandidates : 0; c < 2 * kPlanCandidates; ++c) {
            if (cost[c] < 0) continue;   // (with the stepping kernel on, only large steps come here: I = 4)
            const int I = c < kPlanCandidates ? 1 : 4;
            const double w = static_cast<double>(cost[c]) * warps_of(I) / (I == 4 ? 1.0 : 0.86);
            if (bc < 0 || w < best * (1.0 - 1e-9)) { bc = c; best = w; }
        }
        if (bc < 0) {   // no candidate fits the partial-row buffer: stop here rather than launch a garbage plan
            h->error = 2;
            h->done = 1;
            return;
        }
        h->plan = cand[bc];
        h->plan_I = bc < kPlanCandidates ? 1 : 4;
        h->fused = h->plan_I == 1 && cand[bc].nit == 1 && cand[bc].n_i <= kFusedMaxI;
    }
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
    if (h->done || h->skip) return;
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
        predict_one(raw, j, t, o);
        due = hs.level[j] > kstar;   // level bytes hold k + 1
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
    if (h->done || h->skip) return;
    const int n_act = h->n_act;
    const long long T_next = h->T_next;
    const double t_next = h->t_next, eta = h->eta;
    const int kmin = h->kmin;
    for (int q = blockIdx.x * blockDim.x + threadIdx.x; q < n_act; q += gridDim.x * blockDim.x) {
        correct_one(raw, hs, h, hs.act[q], acc + 3 * q, jerk + 3 * q, T_next, t_next, eta, kmin);
        if (q == 0) step_bookkeeping(h, T_next, n_act);   // T_now is read only by the next hd_begin_kernel
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
    if (grid > 592) grid = 592;   // grid-stride over the due particles
    return launch_pdl(hd_correct_kernel, static_cast<unsigned>(grid), 128, 0, st, raw, h, hs, acc, jerk);
}


}  // namespace nbk
