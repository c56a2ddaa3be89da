// nbk_small_kernels.cu -- small_block_kernel: a block step of up to 32 i-particles in ONE launch
// (a3 + a4 + a5 + a6 of SURVEY.md 8(a); for small blocks the cost is everything
// around the pair sums; L112-L118: split j over the multiprocessors and add the partial forces).
//
// One CTA per SM.  CTA k owns the j-particles [k * chunk, (k + 1) * chunk): it predicts them to the
// current time straight from the raw state into shared memory (and, beside that, into the predicted
// arrays in global memory, so that nbk_get_predicted and later calls at the same time find them), predicts
// the i-particles itself (same formula: the bits of their j entries), sums the pairs -- lanes over j for
// up to 4 i-particles, lanes over i (tile_packed) with the 16 warps splitting the chunk otherwise --
// and writes one partial row per i-particle.  The last CTA to arrive adds the rows in CTA order and
// writes the results to device memory and to the mapped host buffer.  A pending set_j of a few
// particles (the corrected ones of the previous step) rides in the kernel parameters: the CTA that owns
// an updated address stores the raw state and predicts from it.
// No TMA ring, no mbarriers, no predictor launch, no reduce launch: 2 CTA barriers and one ticket.
#include "nbk_device.cuh"

namespace nbk {

namespace {

constexpr int kST = 512, kSWs = kST / 32;

struct SmallSmem {
    float ni[kFusedMaxI][6];          // negated predicted i-state
    int self[kFusedMaxI];
    double scratch[kSWs][32][7];      // cross-warp sums, lanes over i
    float red[kSWs][4][8];            // cross-warp sums, lanes over j
    int is_last;
};

// raw state of particle j, from the pending update if it is in it (the last entry for an address wins)
__device__ __forceinline__ void raw_or_update(const RawJ& raw, const InlineJ& upd, long long j, bool store,
                                              double (&x)[3], float (&v)[3], float (&a)[3], float (&k)[3],
                                              float& m, double& tj) {
    int hit = -1;
    for (int q = 0; q < upd.n; ++q)
        if (upd.addr[q] == j) hit = q;
    if (hit >= 0) {
        tj = upd.t[hit]; m = upd.m[hit];
#pragma unroll
        for (int c = 0; c < 3; ++c) { x[c] = upd.x[hit][c]; v[c] = upd.v[hit][c]; a[c] = upd.a[hit][c]; k[c] = upd.k[hit][c]; }
        if (store) {   // the owner of the address keeps the raw state up to date
            raw.t[j] = tj; raw.m[j] = m;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                raw.x[c * raw.cap + j] = x[c]; raw.v[c * raw.cap + j] = v[c];
                raw.a[c * raw.cap + j] = a[c]; raw.k[c * raw.cap + j] = k[c];
            }
        }
    } else {
        tj = raw.t[j]; m = raw.m[j];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            x[c] = raw.x[c * raw.cap + j]; v[c] = raw.v[c * raw.cap + j];
            a[c] = raw.a[c * raw.cap + j]; k[c] = raw.k[c * raw.cap + j];
        }
    }
}

__device__ __forceinline__ void predict_values(const double (&x)[3], const float (&v)[3], const float (&a)[3],
                                               const float (&k)[3], float m, double tj, double t, float (&o)[7]) {
    const double dt = t - tj;
    const double dt2 = dt * dt * 0.5, dt3 = dt * dt * dt * (1.0 / 6.0);
#pragma unroll
    for (int c = 0; c < 3; ++c) predict_component(x[c], v[c], a[c], k[c], dt, dt2, dt3, o[c], o[4 + c]);
    o[3] = m;
}

}  // namespace

size_t small_smem_bytes(int chunk) {
    const size_t nb = (static_cast<size_t>(chunk) + kTileJMax - 1) / kTileJMax;
    return nb * 7 * kTileJMax * sizeof(float) + sizeof(SmallSmem) + 16;
}

template <bool JERK, bool EPS0>
__global__ void __launch_bounds__(kST, 1) small_block_kernel(const SmallArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int nb256 = (a.chunk + kTileJMax - 1) / kTileJMax;
    float* tiles = reinterpret_cast<float*>(smem_raw);
    SmallSmem& S = *reinterpret_cast<SmallSmem*>(
        smem_raw + ((static_cast<size_t>(nb256) * 7 * kTileJMax * sizeof(float) + 15) & ~static_cast<size_t>(15)));
    pdl_trigger();
    pdl_wait();
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int G = gridDim.x, cta = blockIdx.x;
    const int j0 = cta * a.chunk, n_i = a.n_i;
    // ---- a3 for the i-particles (every CTA) and for the CTA's own j-particles
    if (tid < n_i) {
        const int idx = a.inline_index ? a.i_inline[tid] : (a.i_index ? a.i_index[tid] : tid);
        float o[7] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
        if (idx >= 0) {
            double x[3], tj;
            float v[3], ac[3], k[3], m;
            raw_or_update(a.raw, a.upd, idx, false, x, v, ac, k, m, tj);
            predict_values(x, v, ac, k, m, tj, a.t, o);
        }
        S.ni[tid][0] = -o[0]; S.ni[tid][1] = -o[1]; S.ni[tid][2] = -o[2];
        S.ni[tid][3] = -o[4]; S.ni[tid][4] = -o[5]; S.ni[tid][5] = -o[6];
        S.self[tid] = idx;
    }
    for (int jl = tid; jl < nb256 * kTileJMax; jl += kST) {
        const long long j = static_cast<long long>(j0) + jl;
        float o[7] = {1e18f, 1e18f, 1e18f, 0.f, 0.f, 0.f, 0.f};   // padding: massless, far away
        const bool own = jl < a.chunk;
        if (own && j < a.n_j) {
            double x[3], tj;
            float v[3], ac[3], k[3], m;
            raw_or_update(a.raw, a.upd, j, true, x, v, ac, k, m, tj);
            predict_values(x, v, ac, k, m, tj, a.t, o);
        }
        float* dst = tiles + (jl >> 8) * 7 * kTileJMax + (jl & 255);
#pragma unroll
        for (int c = 0; c < 7; ++c) dst[c * kTileJMax] = o[c];
        if (own && j < a.n_pad) {   // the predicted arrays other calls read (nbk_get_predicted, larger blocks)
#pragma unroll
            for (int c = 0; c < 7; ++c) a.pred[c][j] = o[c];
        }
    }
    __syncthreads();
    // ---- a4 + a5: pair sums over the chunk, one partial row [7 values] per i-particle
    float* row0 = a.partial + static_cast<size_t>(cta) * kFusedMaxI * 8;
    if (n_i <= 4) {   // lanes over j, the sums down a warp tree, the warps' sums in warp order (fp64)
        float s7[4][7];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
#pragma unroll
            for (int v = 0; v < 7; ++v) s7[q][v] = 0.f;
        }
        for (int jl = tid; jl < nb256 * kTileJMax; jl += kST) {
            const float* src = tiles + (jl >> 8) * 7 * kTileJMax + (jl & 255);
            float jv[7];
#pragma unroll
            for (int c = 0; c < 7; ++c) jv[c] = src[c * kTileJMax];
#pragma unroll
            for (int q = 0; q < 4; ++q)
                if (q < n_i) pair_scalar<JERK, EPS0>(jv, S.ni[q], S.self[q] == j0 + jl, a.eps2, s7[q]);
        }
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            if (q < n_i) {
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
                    for (int v = 0; v < 7; ++v) s7[q][v] += __shfl_xor_sync(0xffffffffu, s7[q][v], o);
                }
                if (lane < 7) {
                    float val = s7[q][0];
#pragma unroll
                    for (int v = 1; v < 7; ++v) val = lane == v ? s7[q][v] : val;
                    S.red[warp][q][lane] = val;
                }
            }
        }
        __syncthreads();
        if (tid < 8 * n_i) {
            const int q = tid >> 3, v = tid & 7;
            double t = 0.0;
            if (v < 7) {
#pragma unroll
                for (int w = 0; w < kSWs; ++w) t += static_cast<double>(S.red[w][q][v]);
            }
            row0[q * 8 + v] = static_cast<float>(t);
        }
    } else {          // lanes over i: the 16 warps split the chunk, warp 0 adds their sums in order
        const int g4 = a.chunk >> 2;
        const int jb = ((warp * g4) / kSWs) << 2, je = (((warp + 1) * g4) / kSWs) << 2;
        const bool valid = lane < n_i;
        float ni[1][6] = {{0.f, 0.f, 0.f, 0.f, 0.f, 0.f}};
        int self = -1;
        if (valid) {
#pragma unroll
            for (int c = 0; c < 6; ++c) ni[0][c] = S.ni[lane][c];
            self = S.self[lane];
        }
        constexpr int NA = Shape<JERK>::nacc;
        double d[NA];
        u64 acc[1][NA];
        float tmin[1] = {0.f};
#pragma unroll
        for (int v = 0; v < NA; ++v) { d[v] = 0.0; acc[0][v] = 0ull; }
        for (int b = jb >> 8; (b << 8) < je; ++b) {
            const int lo = max(jb, b << 8) - (b << 8), hi = min(je, (b + 1) << 8) - (b << 8);
            const float* sx = tiles + b * 7 * kTileJMax;
            int sl[1] = {self - j0 - (b << 8)};
            const bool own = static_cast<unsigned>(sl[0]) < static_cast<unsigned>(kTileJMax);
            if (__any_sync(0xffffffffu, own)) tile_packed<1, JERK, EPS0, true, false>(sx, lo, hi, ni, sl, acc, a.eps2, tmin);
            else tile_packed<1, JERK, EPS0, false, false>(sx, lo, hi, ni, sl, acc, a.eps2, tmin);
#pragma unroll
            for (int v = 0; v < NA; ++v) d[v] += static_cast<double>(acc_take(acc[0][v]));
        }
        double t7[7] = {d[0], d[1], d[2], d[3], 0.0, 0.0, 0.0};
        if (JERK) {
            t7[4] = d[4 % NA] - 3.0 * d[7 % NA];
            t7[5] = d[5 % NA] - 3.0 * d[8 % NA];
            t7[6] = d[6 % NA] - 3.0 * d[9 % NA];
        }
#pragma unroll
        for (int v = 0; v < 7; ++v) S.scratch[warp][lane][v] = t7[v];
        __syncthreads();
        if (warp == 0 && valid) {
#pragma unroll
            for (int w = 1; w < kSWs; ++w) {
#pragma unroll
                for (int v = 0; v < 7; ++v) t7[v] += S.scratch[w][lane][v];
            }
            float4* dst = reinterpret_cast<float4*>(row0 + lane * 8);
            dst[0] = make_float4(static_cast<float>(t7[0]), static_cast<float>(t7[1]), static_cast<float>(t7[2]),
                                 static_cast<float>(t7[3]));
            dst[1] = make_float4(static_cast<float>(t7[4]), static_cast<float>(t7[5]), static_cast<float>(t7[6]), 0.f);
        }
    }
    // ---- a6: the last CTA to arrive adds the rows in CTA order (same bits whoever is last)
    __threadfence();
    __syncthreads();
    if (tid == 0) {
        const unsigned ticket = atomicAdd(a.counter, 1u);
        S.is_last = ticket == static_cast<unsigned>(G) - 1u;
        if (S.is_last) *a.counter = 0u;
    }
    __syncthreads();
    if (!S.is_last) return;
    __threadfence();
    const int tx = tid & 31, ty = tid >> 5;   // i-particle, row lane
    double s[7] = {0, 0, 0, 0, 0, 0, 0};
    if (tx < n_i) {
#pragma unroll 4
        for (int k = ty; k < G; k += kSWs) {
            const float4* p = reinterpret_cast<const float4*>(a.partial + (static_cast<size_t>(k) * kFusedMaxI + tx) * 8);
            const float4 u = __ldcg(p), w = __ldcg(p + 1);
            s[0] += u.x; s[1] += u.y; s[2] += u.z; s[3] += u.w;
            s[4] += w.x; s[5] += w.y; s[6] += w.z;
        }
    }
#pragma unroll
    for (int v = 0; v < 7; ++v) S.scratch[ty][tx][v] = s[v];
    __syncthreads();
    for (int st = kSWs >> 1; st > 0; st >>= 1) {
        if (ty < st) {
#pragma unroll
            for (int v = 0; v < 7; ++v) S.scratch[ty][tx][v] += S.scratch[ty + st][tx][v];
        }
        __syncthreads();
    }
    if (ty == 0 && tx < n_i) {
        const int n = n_i;
        float r[7];
        r[0] = static_cast<float>(S.scratch[0][tx][0]);
        r[1] = static_cast<float>(S.scratch[0][tx][1]);
        r[2] = static_cast<float>(S.scratch[0][tx][2]);
        r[6] = static_cast<float>(-S.scratch[0][tx][3]);
        r[3] = JERK ? static_cast<float>(S.scratch[0][tx][4]) : 0.f;
        r[4] = JERK ? static_cast<float>(S.scratch[0][tx][5]) : 0.f;
        r[5] = JERK ? static_cast<float>(S.scratch[0][tx][6]) : 0.f;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            a.acc[3 * tx + c] = r[c];
            a.jerk[3 * tx + c] = r[3 + c];
        }
        a.pot[tx] = r[6];
        if (a.host_out) {
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                a.host_out[3 * tx + c] = r[c];
                a.host_out[3 * n + 3 * tx + c] = r[3 + c];
            }
            a.host_out[6 * n + tx] = r[6];
            __threadfence_system();   // the results are in host memory before the sequence word below
        }
    }
    // The host may wait for the results by polling one mapped word instead of waiting for the kernel to retire
    // (nbk_calc_lasthalf): written last, by one thread, after every result-writing thread's system fence.
    if (a.host_seq) {
        __syncthreads();
        if (tid == 0) *reinterpret_cast<volatile unsigned*>(a.host_seq) = a.seq;
    }
}

cudaError_t small_prepare(int chunk_max) {
    const int smem = static_cast<int>(small_smem_bytes(chunk_max));
    cudaError_t e;
    if ((e = cudaFuncSetAttribute(small_block_kernel<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(small_block_kernel<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(small_block_kernel<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem)) != cudaSuccess) return e;
    return cudaFuncSetAttribute(small_block_kernel<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
}

cudaError_t launch_small_block(const SmallArgs& a, bool jerk, bool eps0, int grid, cudaStream_t s) {
    const size_t smem = small_smem_bytes(a.chunk);
    if (jerk) {
        if (eps0) return launch_pdl(small_block_kernel<true, true>, grid, kST, smem, s, a);
        return launch_pdl(small_block_kernel<true, false>, grid, kST, smem, s, a);
    }
    if (eps0) return launch_pdl(small_block_kernel<false, true>, grid, kST, smem, s, a);
    return launch_pdl(small_block_kernel<false, false>, grid, kST, smem, s, a);
}

}  // namespace nbk
