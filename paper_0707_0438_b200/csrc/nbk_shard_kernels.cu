// nbk_shard_kernels.cu -- the kernels of the j-sharded path over several GPUs (SURVEY.md 8(e),
// 8(f)-4).  PAPER.md L112-L118: for small blocks the j-particles are cut into parts, every part
// gives a partial force on all i-particles, and the partial forces are summed afterwards; here
// the parts live on different GPUs and the sum is one all-reduce of n_i x 8 doubles.
//
//   shard_gather_kernel   owner of an i-particle publishes its predicted state (zeros elsewhere,
//                         so a sum over ranks is an exact copy from the owner)
//   shard_split_kernel    [n_i][8] exchanged state -> the xi, vi arrays of the force call
//   shard_finish_kernel   summed fp64 partials -> acc, jerk, pot in fp32 (one rounding)
#include "nbk_kernels.cuh"

namespace nbk {

__global__ void __launch_bounds__(256) shard_gather_kernel(const ShardGatherArgs a) {
    pdl_trigger();
    pdl_wait();
    const long long k = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (k >= a.n_i) return;
    const long long l = static_cast<long long>(a.i_global[k]) - a.j0;
    const bool mine = l >= 0 && l < a.n_local;
    a.i_local[k] = mine ? static_cast<int32_t>(l) : -1;
    float4 p = make_float4(0.f, 0.f, 0.f, 0.f), q = p;
    if (mine) {
        p = make_float4(a.j.x[l], a.j.y[l], a.j.z[l], 0.f);
        q = make_float4(a.j.vx[l], a.j.vy[l], a.j.vz[l], 0.f);
    }
    float4* o = reinterpret_cast<float4*>(a.xv + 8 * k);
    o[0] = p;
    o[1] = q;
}

__global__ void __launch_bounds__(256) shard_split_kernel(const float* xv, long long n_i, float* xi,
                                                          float* vi) {
    pdl_trigger();
    pdl_wait();
    const long long k = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (k >= n_i) return;
    const float4* s = reinterpret_cast<const float4*>(xv + 8 * k);
    const float4 p = s[0], q = s[1];
    xi[3 * k] = p.x; xi[3 * k + 1] = p.y; xi[3 * k + 2] = p.z;
    vi[3 * k] = q.x; vi[3 * k + 1] = q.y; vi[3 * k + 2] = q.z;
}

// sum64 row: acc(3), -pot, jerk(3), 0 -- the layout reduce_kernel writes
__global__ void __launch_bounds__(256) shard_finish_kernel(const double* sum64, long long n_i,
                                                           float* acc, float* jerk, float* pot) {
    pdl_trigger();
    pdl_wait();
    const long long k = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (k >= n_i) return;
    const double* s = sum64 + 8 * k;
    if (acc) {
        acc[3 * k] = static_cast<float>(s[0]);
        acc[3 * k + 1] = static_cast<float>(s[1]);
        acc[3 * k + 2] = static_cast<float>(s[2]);
    }
    if (pot) pot[k] = static_cast<float>(-s[3]);
    if (jerk) {
        jerk[3 * k] = static_cast<float>(s[4]);
        jerk[3 * k + 1] = static_cast<float>(s[5]);
        jerk[3 * k + 2] = static_cast<float>(s[6]);
    }
}

// Exchange 1 over peer memory: the state of i-particle k is read from its OWNER's published buffer
// (one 32-byte P2P load pair per particle) -- an all-gather written as loads.  __ldcv: never served
// from a stale L1 line of an earlier call.
__global__ void __launch_bounds__(256) shard_fetch_kernel(const ShardPeers peers, const int32_t* i_global,
                                                          long long n_i, float* xv) {
    pdl_trigger();
    pdl_wait();
    const long long k = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (k >= n_i) return;
    const long long g = i_global[k];
    int r = 0;
    while (r + 1 < peers.world && g >= peers.begin[r + 1]) ++r;
    const float4* src = reinterpret_cast<const float4*>(peers.ptr[r]) + 2 * k;
    float4* dst = reinterpret_cast<float4*>(xv) + 2 * k;
    dst[0] = __ldcv(src);
    dst[1] = __ldcv(src + 1);
}

// Exchange 2 fused with the final rounding: every rank adds the G ranks' fp64 partial rows itself, in
// rank order (same bits on every rank, whatever the interconnect does), and rounds once to fp32.
// A one-shot all-reduce as P2P loads: G x 64 bytes per i-particle over NVLink.
__global__ void __launch_bounds__(256) shard_combine_kernel(const ShardPeers peers, long long n_i,
                                                            float* acc, float* jerk, float* pot) {
    pdl_trigger();
    pdl_wait();
    const long long k = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (k >= n_i) return;
    double s[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    for (int r = 0; r < peers.world; ++r) {
        const double2* row = reinterpret_cast<const double2*>(peers.ptr[r]) + 4 * k;
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const double2 u = __ldcv(row + q);
            s[2 * q] += u.x;
            s[2 * q + 1] += u.y;
        }
    }
    if (acc) {
        acc[3 * k] = static_cast<float>(s[0]);
        acc[3 * k + 1] = static_cast<float>(s[1]);
        acc[3 * k + 2] = static_cast<float>(s[2]);
    }
    if (pot) pot[k] = static_cast<float>(-s[3]);
    if (jerk) {
        jerk[3 * k] = static_cast<float>(s[4]);
        jerk[3 * k + 1] = static_cast<float>(s[5]);
        jerk[3 * k + 2] = static_cast<float>(s[6]);
    }
}

static unsigned grid_of(long long n) { return static_cast<unsigned>((n + 255) / 256); }

cudaError_t launch_shard_gather(const ShardGatherArgs& a, cudaStream_t s) {
    if (a.n_i <= 0) return cudaSuccess;
    return launch_pdl(shard_gather_kernel, grid_of(a.n_i), 256, 0, s, a);
}

cudaError_t launch_shard_split(const float* xv, long long n_i, float* xi, float* vi,
                               cudaStream_t s) {
    if (n_i <= 0) return cudaSuccess;
    return launch_pdl(shard_split_kernel, grid_of(n_i), 256, 0, s, xv, n_i, xi, vi);
}

cudaError_t launch_shard_finish(const double* sum64, long long n_i, float* acc, float* jerk,
                                float* pot, cudaStream_t s) {
    if (n_i <= 0) return cudaSuccess;
    return launch_pdl(shard_finish_kernel, grid_of(n_i), 256, 0, s, sum64, n_i, acc, jerk, pot);
}

cudaError_t launch_shard_fetch(const ShardPeers& peers, const int32_t* i_global, long long n_i,
                               float* xv, cudaStream_t s) {
    if (n_i <= 0) return cudaSuccess;
    return launch_pdl(shard_fetch_kernel, grid_of(n_i), 256, 0, s, peers, i_global, n_i, xv);
}

cudaError_t launch_shard_combine(const ShardPeers& peers, long long n_i, float* acc, float* jerk,
                                 float* pot, cudaStream_t s) {
    if (n_i <= 0) return cudaSuccess;
    return launch_pdl(shard_combine_kernel, grid_of(n_i), 256, 0, s, peers, n_i, acc, jerk, pot);
}

}  // namespace nbk
