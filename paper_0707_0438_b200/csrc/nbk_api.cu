// nbk_api.cu -- the C ABI of include/nbk.h: context, workspaces, staging and launch logic.
// Every step of the path runs in the kernels of nbk_kernels.cu; this file only moves
// arguments, picks the launch shape and enqueues.  There is no CPU fallback: without a CUDA
// device nbk_open fails with NBK_ECUDA.
#include <cuda_runtime.h>

#include <chrono>
#include <climits>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "../../include/nbk.h"
#include "nbk_kernels.cuh"

using namespace nbk;

namespace {

inline long long round_up(long long a, long long b) { return (a + b - 1) / b * b; }

struct DeviceGuard {  // make the context's device current for the call, restore on exit
    int prev = -1;
    bool ok = true;
    explicit DeviceGuard(int dev) {
        if (cudaGetDevice(&prev) != cudaSuccess) prev = -1;
        if (prev != dev) ok = cudaSetDevice(dev) == cudaSuccess;
    }
    ~DeviceGuard() {
        int cur = -1;
        if (prev >= 0 && cudaGetDevice(&cur) == cudaSuccess && cur != prev) cudaSetDevice(prev);
    }
};

}  // namespace

struct nbk_ctx {
    int device = 0;
    cudaStream_t stream = nullptr;
    bool own_stream = false;
    long long n_max = 0, ni_max = 0, n_cap = 0;
    int num_sms = 0;

    RawJ raw{};
    float* pred = nullptr;  // 7 arrays of n_cap floats: x y z m vx vy vz
    double t = 0.0;
    bool pred_valid = false;
    long long pred_nj = -1;

    int32_t* d_iidx = nullptr;
    float* d_xi = nullptr;
    float* d_vi = nullptr;
    float* d_partial = nullptr;
    size_t partial_bytes = 0;
    float* d_result = nullptr;  // acc[3 n_i] | jerk[3 n_i] | pot[n_i] of the last call
    float* h_result = nullptr;  // pinned, mapped into the device address space
    float* h_result_dev = nullptr;  // device view of h_result
    unsigned* d_counter = nullptr;  // arrival counter of the fused small-block tail
    float2* d_nn_partial = nullptr; // nearest neighbour: per partial row (smallest s, its j-tile)
    float* d_nn_best = nullptr;     // [ni_max]
    int32_t* d_nn_tile = nullptr;   // [ni_max]
    int32_t* d_nn_index = nullptr;  // [ni_max] result
    float* d_nn_r2 = nullptr;       // [ni_max] result
    bool last_nn = false;           // the last firsthalf asked for nearest neighbours
    unsigned char* d_batch = nullptr;  // batched calls: one growable device arena
    size_t batch_bytes = 0;
    bool batch_ready = false;
    HermiteState hs{};              // device-resident integrator state (allocated on first use)
    long long hs_cap = 0;
    DynHeader* d_hdr = nullptr;
    DynHeader* h_hdr = nullptr;     // pinned
    bool host_has_result = false;   // the last firsthalf wrote h_result itself (no D2H needed)
    InlineJ pending;                // a small set_j not yet on the device (pending.n == 0: none)

    unsigned char* h_stage = nullptr;  // pinned staging for set_j
    unsigned char* d_stage = nullptr;
    size_t stage_bytes = 0;
    cudaEvent_t stage_free = nullptr;  // recorded after the H2D that reads h_stage
    unsigned char* h_istage = nullptr;  // pinned staging for i_index / xi / vi
    cudaEvent_t istage_free = nullptr;

    long long last_ni = -1;
    bool in_flight = false;
    int variant_scalar = 0;
    int force_I = 0;
    bool fused_ok = true;  // nbk_set_variant bit 8 switches the one-launch small-block path off
    int last_cuda = 0;
    long long last_launch[8] = {0, 0, 0, 0, 0, 0, 0, 0};

    bool timing = false;
    cudaEvent_t ev[4][2];
    bool ev_used[4] = {false, false, false, false};
};

namespace {

int cuda_fail(nbk_ctx* c, cudaError_t e) {
    c->last_cuda = static_cast<int>(e);
    (void)cudaGetLastError();
    return NBK_ECUDA;
}

#define NBK_CUDA(c, call)                                   \
    do {                                                    \
        cudaError_t e__ = (call);                           \
        if (e__ != cudaSuccess) return cuda_fail((c), e__); \
    } while (0)

struct TimeScope {  // CUDA events around one kernel on the context's stream
    nbk_ctx* c;
    int slot;
    TimeScope(nbk_ctx* c_, int slot_) : c(c_), slot(slot_) {
        if (c->timing) { cudaEventRecord(c->ev[slot][0], c->stream); c->ev_used[slot] = true; }
    }
    ~TimeScope() {
        if (c->timing) cudaEventRecord(c->ev[slot][1], c->stream);
    }
};

float* pred_arr(const nbk_ctx* c, int k) { return c->pred + static_cast<size_t>(k) * c->n_cap; }

JPred jpred_of(const nbk_ctx* c) {
    JPred j;
    j.x = pred_arr(c, 0); j.y = pred_arr(c, 1); j.z = pred_arr(c, 2); j.m = pred_arr(c, 3);
    j.vx = pred_arr(c, 4); j.vy = pred_arr(c, 5); j.vz = pred_arr(c, 6);
    return j;
}

void free_all(nbk_ctx* c) {
    cudaFree(c->raw.x); cudaFree(c->raw.v); cudaFree(c->raw.a); cudaFree(c->raw.k);
    cudaFree(c->raw.m); cudaFree(c->raw.t); cudaFree(c->pred);
    cudaFree(c->d_iidx); cudaFree(c->d_xi); cudaFree(c->d_vi);
    cudaFree(c->d_partial); cudaFree(c->d_result); cudaFree(c->d_stage); cudaFree(c->d_counter);
    cudaFree(c->d_batch);
    cudaFree(c->hs.x); cudaFree(c->hs.v); cudaFree(c->hs.a); cudaFree(c->hs.j);
    cudaFree(c->hs.level); cudaFree(c->hs.act); cudaFree(c->hs.bc_ge); cudaFree(c->d_hdr);
    if (c->h_hdr) cudaFreeHost(c->h_hdr);
    cudaFree(c->d_nn_partial); cudaFree(c->d_nn_best); cudaFree(c->d_nn_tile);
    cudaFree(c->d_nn_index); cudaFree(c->d_nn_r2);
    if (c->h_result) cudaFreeHost(c->h_result);
    if (c->h_stage) cudaFreeHost(c->h_stage);
    if (c->h_istage) cudaFreeHost(c->h_istage);
    if (c->stage_free) cudaEventDestroy(c->stage_free);
    if (c->istage_free) cudaEventDestroy(c->istage_free);
    for (int s = 0; s < 4; ++s)
        for (int e = 0; e < 2; ++e)
            if (c->ev[s][e]) cudaEventDestroy(c->ev[s][e]);
    if (c->own_stream && c->stream) cudaStreamDestroy(c->stream);
    (void)cudaGetLastError();
}

// A pending small set_j goes to the device on its own (before anything else touches the raw state).
int flush_pending(nbk_ctx* c) {
    if (c->pending.n > 0) {
        TimeScope ts(c, 0);
        NBK_CUDA(c, launch_scatter_inline(c->pending, c->raw, c->stream));
        c->pending.n = 0;
    }
    return NBK_OK;
}

int do_predict(nbk_ctx* c, long long n_j) {
    const long long n_pad = round_up(n_j, kTileJMax);
    bool fold = c->pending.n > 0;
    for (int k = 0; k < c->pending.n; ++k) fold = fold && c->pending.addr[k] < n_j;
    if (!fold) {
        const int rc = flush_pending(c);
        if (rc != NBK_OK) return rc;
    }
    TimeScope ts(c, 1);
    NBK_CUDA(c, launch_predict(c->raw, c->t, n_j, n_pad, pred_arr(c, 0), pred_arr(c, 1),
                               pred_arr(c, 2), pred_arr(c, 3), pred_arr(c, 4), pred_arr(c, 5),
                               pred_arr(c, 6), fold ? &c->pending : nullptr, c->stream));
    c->pending.n = 0;
    c->pred_valid = true;
    c->pred_nj = n_j;
    return NBK_OK;
}

}  // namespace

// ---------------------------------------------------------------------------- host planner
// Launch shape for (n_i, n_j): i-particles per thread I (=> warps per CTA), how many warps split
// each j-tile (wj; the other W / wj warps split the i-tile), the j-tile size tj, and the
// stream-K cut of the (i-tile, j-tile) pair list over G <= SMs persistent CTAs.
// Cost model (relative time of the slowest CTA): pairs per CTA x warps x (j-steps per warp per
// pair x I + fixed per-pair work) / speed(I), speed measured on B200.
namespace nbk {

void plan_shape(long long n_i, long long n_j, int num_sms, int force_I, size_t max_partial_floats,
                Variant* v, Decomp* d) {
    static const int kI[3] = {4, 2, 1};
    static const double kSpeed[3] = {1.0, 0.96, 0.86};
    double best = -1.0;
    for (int a = 0; a < 3; ++a) {
        const int I = kI[a];
        if (force_I > 0 && I != force_I) continue;
        Decomp cand;
        const long long c = plan_fixed_i(n_i, n_j, num_sms, I, max_partial_floats, &cand);
        if (c < 0) continue;
        // a CTA's warps share the FP32 pipe: time per pair grows with the warp count
        const double cost = static_cast<double>(c) * warps_of(I) / kSpeed[a];
        if (best < 0.0 || cost < best * (1.0 - 1e-9)) {
            best = cost;
            v->I = I;
            *d = cand;
        }
    }
}

size_t plan_partial_floats(const Decomp& d) {
    return static_cast<size_t>(d.G) * d.maxseg * d.ti * 8;
}

// G * maxseg * ti <= n_i rounded up to i-tiles + 2 rows of kMaxRowI per CTA (a CTA touches at
// most (its share of i-tiles) + 2 i-tiles; ti <= kMaxRowI).
size_t plan_partial_floats_bound(long long ni_max, int num_sms) {
    return 8 * (static_cast<size_t>(ni_max) + static_cast<size_t>(kMaxRowI) * (3 * static_cast<size_t>(num_sms) + 1));
}

}  // namespace nbk

namespace {

// h_inline: host i-indices to pass in the kernel parameters (small blocks from the host entry
// point; d_iidx is then unused); to_host: also write the results into the mapped host buffer.
int enqueue_force(nbk_ctx* c, long long n_j, long long n_i, const int32_t* d_iidx,
                  const float* d_xi, const float* d_vi, float eps2, uint32_t flags,
                  const int32_t* h_inline = nullptr, bool to_host = false) {
    if (!c->pred_valid || c->pred_nj != n_j) {
        const int rc = do_predict(c, n_j);
        if (rc != NBK_OK) return rc;
    }
    float* acc = c->d_result;
    float* jerk = acc + 3 * n_i;
    float* pot = acc + 6 * n_i;
    c->last_ni = n_i;
    c->in_flight = true;
    c->host_has_result = false;
    if (n_i == 0) return NBK_OK;
    if (n_j == 0) {
        NBK_CUDA(c, cudaMemsetAsync(acc, 0, sizeof(float) * 7 * n_i, c->stream));
        c->last_launch[7] = 0;
        return NBK_OK;
    }
    Variant v;
    Decomp d;
    v.jerk = (flags & NBK_JERK) != 0;
    v.eps0 = (flags & NBK_EPS0) != 0 || eps2 == 0.f;
    v.nn = (flags & NBK_NN) != 0;
    v.packed = c->variant_scalar == 0 || v.nn;   // the neighbour search exists in the packed form
    c->last_nn = v.nn;
    d.G = 0;
    plan_shape(n_i, n_j, c->num_sms, c->force_I, c->partial_bytes / sizeof(float), &v, &d);
    if (d.G < 1 || plan_partial_floats(d) * sizeof(float) > c->partial_bytes) return NBK_ENOMEM;

    ForceArgs fa;
    fa.dyn = nullptr;
    fa.j = jpred_of(c);
    fa.i_index = d_iidx; fa.xi = d_xi; fa.vi = d_vi;
    fa.partial = c->d_partial;
    fa.nn_partial = c->d_nn_partial;
    fa.nn_index = c->d_nn_index;
    fa.nn_r2 = c->d_nn_r2;
    fa.eps2 = eps2;
    fa.d = d;
    std::memset(&fa.tail, 0, sizeof(fa.tail));
    const bool fused = v.I == 1 && d.nit == 1 && n_i <= kFusedMaxI && c->fused_ok;
    if (h_inline && !fused) {  // planner chose another shape: stage the indices after all
        NBK_CUDA(c, cudaEventSynchronize(c->istage_free));
        std::memcpy(c->h_istage, h_inline, sizeof(int32_t) * n_i);
        NBK_CUDA(c, cudaMemcpyAsync(c->d_iidx, c->h_istage, sizeof(int32_t) * n_i,
                                    cudaMemcpyHostToDevice, c->stream));
        NBK_CUDA(c, cudaEventRecord(c->istage_free, c->stream));
        fa.i_index = c->d_iidx;
    }
    if (fused) {
        fa.tail.enabled = 1;
        fa.tail.counter = c->d_counter;
        fa.tail.acc = acc; fa.tail.jerk = jerk; fa.tail.pot = pot;
        fa.tail.host_out = to_host ? c->h_result_dev : nullptr;
        if (h_inline) {
            fa.tail.inline_index = 1;
            std::memcpy(fa.tail.i_inline, h_inline, sizeof(int32_t) * n_i);
        }
    }
    {
        TimeScope ts(c, 2);
        NBK_CUDA(c, launch_force(v, fa, c->stream));
    }
    c->last_launch[0] = d.G;
    c->last_launch[1] = warps_of(v.I) * 32;
    c->last_launch[2] = v.I;
    c->last_launch[3] = d.wj;
    c->last_launch[4] = d.tj;
    c->last_launch[5] = c->num_sms;
    c->last_launch[6] = static_cast<long long>(force_smem_bytes(v));
    c->last_launch[7] = fused ? 1 : 2;
    if (fused) {
        c->host_has_result = to_host;
        return NBK_OK;
    }
    ReduceArgs ra;
    ra.dyn = nullptr;
    ra.n_j = static_cast<int>(n_j);
    for (int k = 0; k < d.G; ++k) {
        const long long q0 = (static_cast<long long>(k) * d.P) / d.G;
        const long long q1 = ((static_cast<long long>(k) + 1) * d.P) / d.G;
        ra.it_first[k] = static_cast<int>(q0 / d.njt);
        ra.it_last[k] = static_cast<int>((q1 - 1) / d.njt);
    }
    ra.partial = c->d_partial;
    ra.nn_partial = c->d_nn_partial;
    ra.nn_best = c->d_nn_best;
    ra.nn_tile = c->d_nn_tile;
    ra.acc = acc; ra.jerk = jerk; ra.pot = pot;
    ra.d = d;
    {
        TimeScope ts(c, 3);
        NBK_CUDA(c, launch_reduce(v, ra, c->stream));
        if (v.nn) {
            NnScanArgs na;
            na.j = fa.j;
            na.i_index = fa.i_index; na.xi = d_xi;
            na.nn_best = c->d_nn_best; na.nn_tile = c->d_nn_tile;
            na.nn_index = c->d_nn_index; na.nn_r2 = c->d_nn_r2;
            na.n_i = static_cast<int>(n_i); na.n_j = static_cast<int>(n_j); na.tj = d.tj;
            na.eps2 = eps2;
            NBK_CUDA(c, launch_nn_scan(na, c->stream));
            c->last_launch[7] = 3;
        }
    }
    return NBK_OK;
}

template <typename T>
int set_j_host(nbk_ctx* c, long long n, const int32_t* addr, const double* tj, const T* m,
               const T* x, const T* v, const T* a, const T* jerk) {
    if (!c || n < 0 || (n > 0 && (!m || !x))) return NBK_EINVAL;
    if (n > c->n_max) return NBK_ERANGE;
    if (addr)
        for (long long k = 0; k < n; ++k)
            if (addr[k] < 0 || addr[k] >= c->n_max) return NBK_ERANGE;
    if (n == 0) return NBK_OK;
    DeviceGuard g(c->device);
    if (!g.ok) return cuda_fail(c, cudaErrorInvalidDevice);
    {
        const int rc = flush_pending(c);
        if (rc != NBK_OK) return rc;
    }
    if (n <= kInlineMaxJ) {  // a handful of particles: the data rides in the next predictor launch
        InlineJ& p = c->pending;
        p.n = static_cast<int>(n);
        for (int k = 0; k < p.n; ++k) {
            p.addr[k] = addr ? addr[k] : k;
            p.t[k] = tj ? tj[k] : 0.0;
            p.m[k] = static_cast<float>(m[k]);
            for (int q = 0; q < 3; ++q) {
                p.x[k][q] = static_cast<double>(x[3 * k + q]);
                p.v[k][q] = v ? static_cast<float>(v[3 * k + q]) : 0.f;
                p.a[k][q] = a ? static_cast<float>(a[3 * k + q]) : 0.f;
                p.k[k][q] = jerk ? static_cast<float>(jerk[3 * k + q]) : 0.f;
            }
        }
        c->pred_valid = false;
        return NBK_OK;
    }
    NBK_CUDA(c, cudaEventSynchronize(c->stage_free));
    // pack [tj | m | x | v | a | jerk | addr] into the pinned buffer: one H2D copy
    size_t off = 0;
    auto put = [&](const void* src, size_t bytes) -> size_t {
        const size_t at = off;
        if (src) std::memcpy(c->h_stage + at, src, bytes);
        off += (bytes + 15) & ~static_cast<size_t>(15);
        return at;
    };
    const size_t o_t = put(tj, sizeof(double) * n);
    const size_t o_m = put(m, sizeof(T) * n);
    const size_t o_x = put(x, sizeof(T) * 3 * n);
    const size_t o_v = put(v, sizeof(T) * 3 * n);
    const size_t o_a = put(a, sizeof(T) * 3 * n);
    const size_t o_k = put(jerk, sizeof(T) * 3 * n);
    const size_t o_ad = put(addr, sizeof(int32_t) * n);
    if (off > c->stage_bytes) return NBK_ENOMEM;
    NBK_CUDA(c, cudaMemcpyAsync(c->d_stage, c->h_stage, off, cudaMemcpyHostToDevice, c->stream));
    NBK_CUDA(c, cudaEventRecord(c->stage_free, c->stream));
    ScatterArgs s;
    s.n = n;
    s.addr = addr ? reinterpret_cast<const int32_t*>(c->d_stage + o_ad) : nullptr;
    s.tj = tj ? reinterpret_cast<const double*>(c->d_stage + o_t) : nullptr;
    s.m = c->d_stage + o_m;
    s.x = c->d_stage + o_x;
    s.v = v ? c->d_stage + o_v : nullptr;
    s.a = a ? c->d_stage + o_a : nullptr;
    s.k = jerk ? c->d_stage + o_k : nullptr;
    s.f64 = sizeof(T) == sizeof(double);
    s.n_max = c->n_max;
    {
        TimeScope ts(c, 0);
        NBK_CUDA(c, launch_scatter(s, c->raw, c->stream));
    }
    c->pred_valid = false;
    return NBK_OK;
}

}  // namespace

extern "C" {

int nbk_open(nbk_ctx** out, int device, int64_t n_max, int64_t ni_max, void* cuda_stream) {
    if (!out || n_max < 1 || ni_max < 1 || n_max > (1LL << 30) || ni_max > (1LL << 30))
        return NBK_EINVAL;
    *out = nullptr;
    nbk_ctx* c = new (std::nothrow) nbk_ctx();
    if (!c) return NBK_ENOMEM;
    std::memset(c->ev, 0, sizeof(c->ev));
    c->pending.n = 0;
    c->device = device;
    int rc = NBK_OK;
    auto fail = [&](int code, cudaError_t e) {
        if (code == NBK_ECUDA) c->last_cuda = static_cast<int>(e);
        rc = code;
    };
    DeviceGuard g(device);
    cudaError_t e = g.ok ? cudaSuccess : cudaErrorInvalidDevice;
    do {
        if (e != cudaSuccess) break;
        cudaDeviceProp prop;
        if ((e = cudaGetDeviceProperties(&prop, device)) != cudaSuccess) break;
        if (prop.major < 10) { e = cudaErrorNoKernelImageForDevice; break; }
        c->num_sms = prop.multiProcessorCount;
        if (cuda_stream) {
            c->stream = static_cast<cudaStream_t>(cuda_stream);
        } else {
            if ((e = cudaStreamCreateWithFlags(&c->stream, cudaStreamNonBlocking)) != cudaSuccess) break;
            c->own_stream = true;
        }
        c->n_max = n_max;
        c->ni_max = ni_max;
        c->n_cap = round_up(n_max, kTileJMax);
        c->raw.cap = c->n_cap;
        for (int I : {1, 2, 4})
            for (int jk = 0; jk < 2 && e == cudaSuccess; ++jk)
                for (int e0 = 0; e0 < 2 && e == cudaSuccess; ++e0)
                    for (int pk = 0; pk < 2 && e == cudaSuccess; ++pk) {
                        Variant v{I, jk != 0, e0 != 0, pk != 0};
                        e = force_prepare(v);
                    }
        if (e != cudaSuccess) break;
        const size_t cap = static_cast<size_t>(c->n_cap);
        if ((e = cudaMalloc(&c->raw.x, sizeof(double) * 3 * cap)) != cudaSuccess) break;
        if ((e = cudaMalloc(&c->raw.v, sizeof(float) * 3 * cap)) != cudaSuccess) break;
        if ((e = cudaMalloc(&c->raw.a, sizeof(float) * 3 * cap)) != cudaSuccess) break;
        if ((e = cudaMalloc(&c->raw.k, sizeof(float) * 3 * cap)) != cudaSuccess) break;
        if ((e = cudaMalloc(&c->raw.m, sizeof(float) * cap)) != cudaSuccess) break;
        if ((e = cudaMalloc(&c->raw.t, sizeof(double) * cap)) != cudaSuccess) break;
        if ((e = cudaMalloc(&c->pred, sizeof(float) * 7 * cap)) != cudaSuccess) break;
        if ((e = cudaMemsetAsync(c->raw.x, 0, sizeof(double) * 3 * cap, c->stream)) != cudaSuccess) break;
        if ((e = cudaMemsetAsync(c->raw.v, 0, sizeof(float) * 3 * cap, c->stream)) != cudaSuccess) break;
        if ((e = cudaMemsetAsync(c->raw.a, 0, sizeof(float) * 3 * cap, c->stream)) != cudaSuccess) break;
        if ((e = cudaMemsetAsync(c->raw.k, 0, sizeof(float) * 3 * cap, c->stream)) != cudaSuccess) break;
        if ((e = cudaMemsetAsync(c->raw.m, 0, sizeof(float) * cap, c->stream)) != cudaSuccess) break;
        if ((e = cudaMemsetAsync(c->raw.t, 0, sizeof(double) * cap, c->stream)) != cudaSuccess) break;
        if ((e = cudaMemsetAsync(c->pred, 0, sizeof(float) * 7 * cap, c->stream)) != cudaSuccess) break;
        const size_t ni = static_cast<size_t>(ni_max);
        if ((e = cudaMalloc(&c->d_iidx, sizeof(int32_t) * ni)) != cudaSuccess) break;
        if ((e = cudaMalloc(&c->d_xi, sizeof(float) * 3 * ni)) != cudaSuccess) break;
        if ((e = cudaMalloc(&c->d_vi, sizeof(float) * 3 * ni)) != cudaSuccess) break;
        if ((e = cudaMalloc(&c->d_result, sizeof(float) * 7 * ni)) != cudaSuccess) break;
        if ((e = cudaHostAlloc(&c->h_result, sizeof(float) * 9 * ni, cudaHostAllocMapped)) != cudaSuccess) break;
        if ((e = cudaHostGetDevicePointer(&c->h_result_dev, c->h_result, 0)) != cudaSuccess) break;
        if ((e = cudaMalloc(&c->d_counter, sizeof(unsigned))) != cudaSuccess) break;
        if ((e = cudaMemsetAsync(c->d_counter, 0, sizeof(unsigned), c->stream)) != cudaSuccess) break;
        c->partial_bytes = sizeof(float) * plan_partial_floats_bound(ni_max, c->num_sms);
        if ((e = cudaMalloc(&c->d_partial, c->partial_bytes)) != cudaSuccess) break;
        if ((e = cudaMalloc(&c->d_nn_partial, c->partial_bytes / 4)) != cudaSuccess) break;
        if ((e = cudaMalloc(&c->d_nn_best, sizeof(float) * ni)) != cudaSuccess) break;
        if ((e = cudaMalloc(&c->d_nn_tile, sizeof(int32_t) * ni)) != cudaSuccess) break;
        if ((e = cudaMalloc(&c->d_nn_index, sizeof(int32_t) * ni)) != cudaSuccess) break;
        if ((e = cudaMalloc(&c->d_nn_r2, sizeof(float) * ni)) != cudaSuccess) break;
        c->stage_bytes = static_cast<size_t>(n_max) * (8 + 8 + 4 * 24 + 4) + 16 * 8;
        if ((e = cudaMallocHost(&c->h_stage, c->stage_bytes)) != cudaSuccess) break;
        if ((e = cudaMalloc(&c->d_stage, c->stage_bytes)) != cudaSuccess) break;
        if ((e = cudaMallocHost(&c->h_istage, ni * 28 + 64)) != cudaSuccess) break;
        if ((e = cudaEventCreateWithFlags(&c->stage_free, cudaEventDisableTiming)) != cudaSuccess) break;
        if ((e = cudaEventCreateWithFlags(&c->istage_free, cudaEventDisableTiming)) != cudaSuccess) break;
        if ((e = cudaEventRecord(c->stage_free, c->stream)) != cudaSuccess) break;
        if ((e = cudaEventRecord(c->istage_free, c->stream)) != cudaSuccess) break;
        for (int s = 0; s < 4 && e == cudaSuccess; ++s)
            for (int k = 0; k < 2 && e == cudaSuccess; ++k) e = cudaEventCreate(&c->ev[s][k]);
        if (e != cudaSuccess) break;
        e = cudaStreamSynchronize(c->stream);
    } while (false);
    if (e != cudaSuccess)
        fail(e == cudaErrorMemoryAllocation ? NBK_ENOMEM : NBK_ECUDA, e);
    if (rc != NBK_OK) {
        free_all(c);
        delete c;
        return rc;
    }
    *out = c;
    return NBK_OK;
}

int nbk_close(nbk_ctx* c) {
    if (!c) return NBK_OK;
    DeviceGuard g(c->device);
    if (c->stream) cudaStreamSynchronize(c->stream);
    free_all(c);
    delete c;
    return NBK_OK;
}

int nbk_npipes(const nbk_ctx* c) {
    if (!c) return NBK_EINVAL;
    return c->ni_max > INT_MAX ? INT_MAX : static_cast<int>(c->ni_max);
}

int nbk_set_j_particles(nbk_ctx* c, int64_t n, const int32_t* addr, const double* tj,
                        const float* m, const float* x, const float* v, const float* a,
                        const float* jerk) {
    return set_j_host<float>(c, n, addr, tj, m, x, v, a, jerk);
}

int nbk_set_j_particles_f64(nbk_ctx* c, int64_t n, const int32_t* addr, const double* tj,
                            const double* m, const double* x, const double* v, const double* a,
                            const double* jerk) {
    return set_j_host<double>(c, n, addr, tj, m, x, v, a, jerk);
}

int nbk_set_j_particles_dev(nbk_ctx* c, int64_t n, const int32_t* addr, const double* tj,
                            const float* m, const float* x, const float* v, const float* a,
                            const float* jerk) {
    if (!c || n < 0 || (n > 0 && (!m || !x))) return NBK_EINVAL;
    if (n > c->n_max) return NBK_ERANGE;
    if (n == 0) return NBK_OK;
    DeviceGuard g(c->device);
    if (!g.ok) return cuda_fail(c, cudaErrorInvalidDevice);
    {
        const int rc = flush_pending(c);
        if (rc != NBK_OK) return rc;
    }
    ScatterArgs s;
    s.n = n; s.addr = addr; s.tj = tj; s.m = m; s.x = x; s.v = v; s.a = a; s.k = jerk;
    s.f64 = 0;
    s.n_max = c->n_max;
    {
        TimeScope ts(c, 0);
        NBK_CUDA(c, launch_scatter(s, c->raw, c->stream));
    }
    c->pred_valid = false;
    return NBK_OK;
}

int nbk_set_ti(nbk_ctx* c, double t) {
    if (!c) return NBK_EINVAL;
    if (!(t == t)) return NBK_EINVAL;
    if (t != c->t) c->pred_valid = false;
    c->t = t;
    return NBK_OK;
}

int nbk_predict(nbk_ctx* c, int64_t n_j) {
    if (!c || n_j < 0) return NBK_EINVAL;
    if (n_j > c->n_max) return NBK_ERANGE;
    DeviceGuard g(c->device);
    if (!g.ok) return cuda_fail(c, cudaErrorInvalidDevice);
    return do_predict(c, n_j);
}

int nbk_get_predicted(nbk_ctx* c, int64_t n_j, float* m, float* x, float* v) {
    if (!c || n_j < 0) return NBK_EINVAL;
    if (n_j > c->n_max) return NBK_ERANGE;
    if (!c->pred_valid || c->pred_nj < n_j) return NBK_ESTATE;
    if (n_j == 0) return NBK_OK;
    DeviceGuard g(c->device);
    if (!g.ok) return cuda_fail(c, cudaErrorInvalidDevice);
    std::vector<float> tmp;
    try {
        tmp.resize(static_cast<size_t>(7) * n_j);
    } catch (...) {
        return NBK_ENOMEM;
    }
    for (int k = 0; k < 7; ++k)
        NBK_CUDA(c, cudaMemcpyAsync(tmp.data() + static_cast<size_t>(k) * n_j, pred_arr(c, k),
                                    sizeof(float) * n_j, cudaMemcpyDeviceToHost, c->stream));
    NBK_CUDA(c, cudaStreamSynchronize(c->stream));
    const size_t n = static_cast<size_t>(n_j);
    for (size_t j = 0; j < n; ++j) {
        if (x) { x[3 * j] = tmp[j]; x[3 * j + 1] = tmp[n + j]; x[3 * j + 2] = tmp[2 * n + j]; }
        if (m) m[j] = tmp[3 * n + j];
        if (v) { v[3 * j] = tmp[4 * n + j]; v[3 * j + 1] = tmp[5 * n + j]; v[3 * j + 2] = tmp[6 * n + j]; }
    }
    return NBK_OK;
}

int nbk_calc_firsthalf(nbk_ctx* c, int64_t n_j, int64_t n_i, const int32_t* i_index,
                       const float* xi, const float* vi, float eps2, uint32_t flags) {
    if (!c || n_j < 0 || n_i < 0 || !(eps2 >= 0.f)) return NBK_EINVAL;
    if ((flags & NBK_NN) && !(flags & NBK_JERK)) return NBK_EINVAL;
    if (n_j > c->n_max || n_i > c->ni_max) return NBK_ERANGE;
    if (i_index) {
        for (int64_t k = 0; k < n_i; ++k) {
            if (i_index[k] < -1 || i_index[k] >= n_j) return NBK_ERANGE;
            if (i_index[k] < 0 && !xi) return NBK_EINVAL;
        }
    } else if (n_i > n_j) {
        return NBK_ERANGE;
    }
    DeviceGuard g(c->device);
    if (!g.ok) return cuda_fail(c, cudaErrorInvalidDevice);
    const int32_t* d_ii = nullptr;
    const float* d_x = nullptr;
    const float* d_v = nullptr;
    if (n_i > 0 && n_i <= kFusedMaxI && !xi && !vi)   // small block: indices ride in the launch
        return enqueue_force(c, n_j, n_i, nullptr, nullptr, nullptr, eps2, flags, i_index, true);
    if (n_i > 0 && (i_index || xi || vi)) {
        NBK_CUDA(c, cudaEventSynchronize(c->istage_free));
        const size_t ni = static_cast<size_t>(n_i);
        unsigned char* h = c->h_istage;
        if (i_index) {
            std::memcpy(h, i_index, 4 * ni);
            NBK_CUDA(c, cudaMemcpyAsync(c->d_iidx, h, 4 * ni, cudaMemcpyHostToDevice, c->stream));
            d_ii = c->d_iidx;
        }
        h += (4 * ni + 15) & ~static_cast<size_t>(15);
        if (xi) {
            std::memcpy(h, xi, 12 * ni);
            NBK_CUDA(c, cudaMemcpyAsync(c->d_xi, h, 12 * ni, cudaMemcpyHostToDevice, c->stream));
            d_x = c->d_xi;
        }
        h += (12 * ni + 15) & ~static_cast<size_t>(15);
        if (vi) {
            std::memcpy(h, vi, 12 * ni);
            NBK_CUDA(c, cudaMemcpyAsync(c->d_vi, h, 12 * ni, cudaMemcpyHostToDevice, c->stream));
            d_v = c->d_vi;
        }
        NBK_CUDA(c, cudaEventRecord(c->istage_free, c->stream));
    }
    return enqueue_force(c, n_j, n_i, d_ii, d_x, d_v, eps2, flags);
}

int nbk_calc_firsthalf_dev(nbk_ctx* c, int64_t n_j, int64_t n_i, const int32_t* i_index,
                           const float* xi, const float* vi, float eps2, uint32_t flags) {
    if (!c || n_j < 0 || n_i < 0 || !(eps2 >= 0.f)) return NBK_EINVAL;
    if ((flags & NBK_NN) && !(flags & NBK_JERK)) return NBK_EINVAL;
    if (n_j > c->n_max || n_i > c->ni_max) return NBK_ERANGE;
    if (!i_index && n_i > n_j) return NBK_ERANGE;
    DeviceGuard g(c->device);
    if (!g.ok) return cuda_fail(c, cudaErrorInvalidDevice);
    return enqueue_force(c, n_j, n_i, i_index, xi, vi, eps2, flags);
}

int nbk_calc_lasthalf(nbk_ctx* c, int64_t n_i, float* acc, float* jerk, float* pot) {
    if (!c || n_i < 0) return NBK_EINVAL;
    if (!c->in_flight || n_i != c->last_ni) return NBK_ESTATE;
    if (n_i == 0) return NBK_OK;
    DeviceGuard g(c->device);
    if (!g.ok) return cuda_fail(c, cudaErrorInvalidDevice);
    const size_t ni = static_cast<size_t>(n_i);
    if (!c->host_has_result)
        NBK_CUDA(c, cudaMemcpyAsync(c->h_result, c->d_result, sizeof(float) * 7 * ni,
                                    cudaMemcpyDeviceToHost, c->stream));
    NBK_CUDA(c, cudaStreamSynchronize(c->stream));
    if (acc) std::memcpy(acc, c->h_result, sizeof(float) * 3 * ni);
    if (jerk) std::memcpy(jerk, c->h_result + 3 * ni, sizeof(float) * 3 * ni);
    if (pot) std::memcpy(pot, c->h_result + 6 * ni, sizeof(float) * ni);
    return NBK_OK;
}

int nbk_calc_lasthalf_dev(nbk_ctx* c, int64_t n_i, float* acc, float* jerk, float* pot) {
    if (!c || n_i < 0) return NBK_EINVAL;
    if (!c->in_flight || n_i != c->last_ni) return NBK_ESTATE;
    if (n_i == 0) return NBK_OK;
    DeviceGuard g(c->device);
    if (!g.ok) return cuda_fail(c, cudaErrorInvalidDevice);
    const size_t ni = static_cast<size_t>(n_i);
    if (acc) NBK_CUDA(c, cudaMemcpyAsync(acc, c->d_result, sizeof(float) * 3 * ni, cudaMemcpyDeviceToDevice, c->stream));
    if (jerk) NBK_CUDA(c, cudaMemcpyAsync(jerk, c->d_result + 3 * ni, sizeof(float) * 3 * ni, cudaMemcpyDeviceToDevice, c->stream));
    if (pot) NBK_CUDA(c, cudaMemcpyAsync(pot, c->d_result + 6 * ni, sizeof(float) * ni, cudaMemcpyDeviceToDevice, c->stream));
    return NBK_OK;
}

int nbk_get_neighbours(nbk_ctx* c, int64_t n_i, int32_t* nn_index, float* nn_r2) {
    if (!c || n_i < 0) return NBK_EINVAL;
    if (!c->in_flight || n_i != c->last_ni || !c->last_nn) return NBK_ESTATE;
    if (n_i == 0) return NBK_OK;
    DeviceGuard g(c->device);
    if (!g.ok) return cuda_fail(c, cudaErrorInvalidDevice);
    const size_t ni = static_cast<size_t>(n_i);
    float* h = c->h_result + 7 * ni;   // [nn_index as int bits | nn_r2]
    if (!c->host_has_result) {
        NBK_CUDA(c, cudaMemcpyAsync(h, c->d_nn_index, sizeof(int32_t) * ni, cudaMemcpyDeviceToHost, c->stream));
        NBK_CUDA(c, cudaMemcpyAsync(h + ni, c->d_nn_r2, sizeof(float) * ni, cudaMemcpyDeviceToHost, c->stream));
    }
    NBK_CUDA(c, cudaStreamSynchronize(c->stream));
    if (nn_index) std::memcpy(nn_index, h, sizeof(int32_t) * ni);
    if (nn_r2) std::memcpy(nn_r2, h + ni, sizeof(float) * ni);
    return NBK_OK;
}

int nbk_get_neighbours_dev(nbk_ctx* c, int64_t n_i, int32_t* nn_index, float* nn_r2) {
    if (!c || n_i < 0) return NBK_EINVAL;
    if (!c->in_flight || n_i != c->last_ni || !c->last_nn) return NBK_ESTATE;
    if (n_i == 0) return NBK_OK;
    DeviceGuard g(c->device);
    if (!g.ok) return cuda_fail(c, cudaErrorInvalidDevice);
    const size_t ni = static_cast<size_t>(n_i);
    if (nn_index) NBK_CUDA(c, cudaMemcpyAsync(nn_index, c->d_nn_index, sizeof(int32_t) * ni, cudaMemcpyDeviceToDevice, c->stream));
    if (nn_r2) NBK_CUDA(c, cudaMemcpyAsync(nn_r2, c->d_nn_r2, sizeof(float) * ni, cudaMemcpyDeviceToDevice, c->stream));
    return NBK_OK;
}

// ---- a8 on the device: the whole block-step loop without host round trips ----
int nbk_hermite_evolve_dev(nbk_ctx* c, int64_t n, const double* m, double* x, double* v, double eps,
                           double t_end, double eta, double dt_max, nbk_hermite_stats* stats) {
    if (!c || n < 1 || !m || !x || !v || !(eps >= 0.0) || !(t_end >= 0.0) || !(eta > 0.0) ||
        !(dt_max > 0.0) || n > INT32_MAX)
        return NBK_EINVAL;
    if (n > c->n_max || n > c->ni_max) return NBK_ERANGE;
    int e0;
    std::frexp(dt_max, &e0);
    int kmin = -(e0 - 1);            // dt_max rounded down to a power of two
    if (kmin < -10) kmin = -10;
    if (kmin < 0 || kmin > kMaxLevel) return NBK_EINVAL;   // dt_max in (2^-48, 1]... 2^0
    const double dtm = std::ldexp(1.0, -kmin);
    if (t_end > 2047.0 || std::fmod(t_end, dtm) != 0.0) return NBK_EINVAL;
    DeviceGuard g(c->device);
    if (!g.ok) return cuda_fail(c, cudaErrorInvalidDevice);
    const auto wall0 = std::chrono::steady_clock::now();
    const size_t N = static_cast<size_t>(n);
    const float eps2 = static_cast<float>(eps * eps);
    const uint32_t flags = NBK_JERK | NBK_POT;
    int rc;

    if (c->hs_cap < n) {
        cudaFree(c->hs.x); cudaFree(c->hs.v); cudaFree(c->hs.a); cudaFree(c->hs.j);
        cudaFree(c->hs.level); cudaFree(c->hs.act); cudaFree(c->hs.bc_ge);
        c->hs = HermiteState{};
        c->hs_cap = 0;
        NBK_CUDA(c, cudaMalloc(&c->hs.x, sizeof(double) * 3 * N));
        NBK_CUDA(c, cudaMalloc(&c->hs.v, sizeof(double) * 3 * N));
        NBK_CUDA(c, cudaMalloc(&c->hs.a, sizeof(double) * 3 * N));
        NBK_CUDA(c, cudaMalloc(&c->hs.j, sizeof(double) * 3 * N));
        NBK_CUDA(c, cudaMalloc(&c->hs.level, sizeof(int) * N));
        NBK_CUDA(c, cudaMalloc(&c->hs.act, sizeof(int32_t) * N));
        NBK_CUDA(c, cudaMalloc(&c->hs.bc_ge, sizeof(int) * (kMaxLevel + 1) * ((N + 255) / 256)));
        c->hs_cap = n;
    }
    if (!c->d_hdr) NBK_CUDA(c, cudaMalloc(&c->d_hdr, sizeof(DynHeader)));
    if (!c->h_hdr) NBK_CUDA(c, cudaMallocHost(&c->h_hdr, sizeof(DynHeader)));

    // t = 0 through the ordinary entry points: forces on everybody, first steps (reading R15)
    std::vector<float> fa(3 * N), fj(3 * N);
    std::vector<double> a(3 * N), jk(3 * N), tl(N, 0.0);
    std::vector<int> lev(N);
    if ((rc = nbk_set_j_particles_f64(c, n, nullptr, nullptr, m, x, v, nullptr, nullptr)) != NBK_OK) return rc;
    if ((rc = nbk_set_ti(c, 0.0)) != NBK_OK) return rc;
    if ((rc = nbk_calc_firsthalf(c, n, n, nullptr, nullptr, nullptr, eps2, flags)) != NBK_OK) return rc;
    if ((rc = nbk_calc_lasthalf(c, n, fa.data(), fj.data(), nullptr)) != NBK_OK) return rc;
    DynHeader& H = *c->h_hdr;
    std::memset(&H, 0, sizeof(H));
    for (size_t i = 0; i < N; ++i) {
        double na = 0.0, nj = 0.0;
        for (int q = 0; q < 3; ++q) {
            a[3 * i + q] = fa[3 * i + q];
            jk[3 * i + q] = fj[3 * i + q];
            na += a[3 * i + q] * a[3 * i + q];
            nj += jk[3 * i + q] * jk[3 * i + q];
        }
        na = std::sqrt(na); nj = std::sqrt(nj);
        double want = dtm;
        if (nj > 0.0 && na > 0.0) want = std::fmin(0.25 * eta * na / nj, dtm);
        int k = kMaxLevel;
        if (want > 0.0) {
            int e;
            std::frexp(want, &e);
            k = -(e - 1);
            if (k < kmin) k = kmin;
            if (k > kMaxLevel) k = kMaxLevel;
        }
        lev[i] = k;
        H.level_count[k] += 1;
    }
    const int nblk = static_cast<int>((N + 255) / 256);
    c->hs.nblk = nblk;
    std::vector<int> bc(static_cast<size_t>(kMaxLevel + 1) * nblk, 0);
    for (size_t i = 0; i < N; ++i)
        for (int l = 0; l <= lev[i]; ++l) bc[static_cast<size_t>(l) * nblk + (i >> 8)] += 1;
    if ((rc = nbk_set_j_particles_f64(c, n, nullptr, tl.data(), m, x, v, a.data(), jk.data())) != NBK_OK) return rc;
    if ((rc = flush_pending(c)) != NBK_OK) return rc;
    H.T_now = 0;
    H.T_end = static_cast<long long>(std::ldexp(t_end, kTickLog2));
    H.kmin = kmin;
    H.n = static_cast<int>(n);
    H.num_sms = c->num_sms < kMaxCtas ? c->num_sms : kMaxCtas;
    H.max_partial_floats = c->partial_bytes / sizeof(float);
    H.eta = eta;
    H.interactions = n * n;
    NBK_CUDA(c, cudaMemcpyAsync(c->hs.x, x, sizeof(double) * 3 * N, cudaMemcpyHostToDevice, c->stream));
    NBK_CUDA(c, cudaMemcpyAsync(c->hs.v, v, sizeof(double) * 3 * N, cudaMemcpyHostToDevice, c->stream));
    NBK_CUDA(c, cudaMemcpyAsync(c->hs.a, a.data(), sizeof(double) * 3 * N, cudaMemcpyHostToDevice, c->stream));
    NBK_CUDA(c, cudaMemcpyAsync(c->hs.j, jk.data(), sizeof(double) * 3 * N, cudaMemcpyHostToDevice, c->stream));
    NBK_CUDA(c, cudaMemcpyAsync(c->hs.level, lev.data(), sizeof(int) * N, cudaMemcpyHostToDevice, c->stream));
    NBK_CUDA(c, cudaMemcpyAsync(c->hs.bc_ge, bc.data(), sizeof(int) * bc.size(), cudaMemcpyHostToDevice, c->stream));
    NBK_CUDA(c, cudaMemcpyAsync(c->d_hdr, &H, sizeof(H), cudaMemcpyHostToDevice, c->stream));
    NBK_CUDA(c, cudaStreamSynchronize(c->stream));   // the host vectors above may go away

    // one block step = begin, predict + select, force (+ reduce), correct; enqueued in batches with
    // no host synchronisation inside a batch; steps past t_end return at once (done flag)
    Variant vv{1, true, eps2 == 0.f, true, false};
    const long long n_pad = round_up(n, kTileJMax);
    const size_t ni_max = static_cast<size_t>(c->ni_max);
    ForceArgs f;
    std::memset(&f, 0, sizeof(f));
    f.j = jpred_of(c);
    f.i_index = c->hs.act;
    f.partial = c->d_partial;
    f.eps2 = eps2;
    f.d.n_j = static_cast<int>(n);
    f.tail.counter = c->d_counter;
    f.tail.acc = c->d_result;
    f.tail.jerk = c->d_result + 3 * ni_max;
    f.tail.pot = c->d_result + 6 * ni_max;
    f.dyn = c->d_hdr;
    f.d.G = H.num_sms;   // grid: one CTA per SM; CTAs beyond the plan's G return
    ReduceArgs r;
    std::memset(&r, 0, sizeof(r));
    r.partial = c->d_partial;
    r.acc = f.tail.acc; r.jerk = f.tail.jerk; r.pot = f.tail.pot;
    r.dyn = c->d_hdr;
    r.n_j = static_cast<int>(n);
    // the five launches of a block step are captured once into a CUDA graph and replayed
    const int kBatch = 256;
    cudaGraph_t graph = nullptr;
    cudaGraphExec_t gexec = nullptr;
    auto enqueue_step = [&]() -> cudaError_t {
        cudaError_t e;
        if ((e = launch_hd_begin(c->d_hdr, c->stream)) != cudaSuccess) return e;
        if ((e = launch_hd_predict(c->raw, c->d_hdr, c->hs, n_pad, pred_arr(c, 0), pred_arr(c, 1),
                                   pred_arr(c, 2), pred_arr(c, 3), pred_arr(c, 4), pred_arr(c, 5),
                                   pred_arr(c, 6), c->stream)) != cudaSuccess) return e;
        if ((e = launch_force(vv, f, c->stream)) != cudaSuccess) return e;
        if ((e = launch_reduce_dyn(vv, r, static_cast<int>(n), c->stream)) != cudaSuccess) return e;
        return launch_hd_correct(c->raw, c->d_hdr, c->hs, f.tail.acc, f.tail.jerk,
                                 static_cast<int>(n), c->stream);
    };
    NBK_CUDA(c, cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeRelaxed));
    cudaError_t ce = enqueue_step();
    cudaError_t ce2 = cudaStreamEndCapture(c->stream, &graph);
    if (ce != cudaSuccess || ce2 != cudaSuccess) {
        if (graph) cudaGraphDestroy(graph);
        return cuda_fail(c, ce != cudaSuccess ? ce : ce2);
    }
    ce = cudaGraphInstantiate(&gexec, graph, 0);
    if (ce != cudaSuccess) { cudaGraphDestroy(graph); return cuda_fail(c, ce); }
    for (;;) {
        for (int s = 0; s < kBatch && ce == cudaSuccess; ++s) ce = cudaGraphLaunch(gexec, c->stream);
        if (ce == cudaSuccess)
            ce = cudaMemcpyAsync(c->h_hdr, c->d_hdr, sizeof(DynHeader), cudaMemcpyDeviceToHost, c->stream);
        if (ce == cudaSuccess) ce = cudaStreamSynchronize(c->stream);
        if (ce != cudaSuccess || c->h_hdr->done) break;
    }
    cudaGraphExecDestroy(gexec);
    cudaGraphDestroy(graph);
    if (ce != cudaSuccess) return cuda_fail(c, ce);
    NBK_CUDA(c, cudaMemcpyAsync(x, c->hs.x, sizeof(double) * 3 * N, cudaMemcpyDeviceToHost, c->stream));
    NBK_CUDA(c, cudaMemcpyAsync(v, c->hs.v, sizeof(double) * 3 * N, cudaMemcpyDeviceToHost, c->stream));
    NBK_CUDA(c, cudaStreamSynchronize(c->stream));
    c->pred_valid = false;
    c->in_flight = false;
    if (stats) {
        std::memset(stats, 0, sizeof(*stats));
        stats->block_steps = c->h_hdr->block_steps;
        stats->particle_steps = c->h_hdr->particle_steps;
        stats->interactions = c->h_hdr->interactions;
        stats->t_reached = std::ldexp(static_cast<double>(c->h_hdr->T_now), -kTickLog2);
        for (int b = 0; b < 32; ++b) stats->ni_histogram[b] = c->h_hdr->hist[b];
        stats->wall_seconds =
            std::chrono::duration<double>(std::chrono::steady_clock::now() - wall0).count();
        stats->gpu_call_seconds = stats->wall_seconds;
    }
    return NBK_OK;
}

// ---- batched acc + pot calls -------------------------------------------------
namespace {

int batch_impl(nbk_ctx* c, int64_t n_groups, const int64_t* i_offset, const float* xi,
               const int64_t* j_offset, const float* mj, const float* xj, float eps2, uint32_t flags,
               float* acc, float* pot, bool dev) {
    if (!c || n_groups < 0 || !(eps2 >= 0.f) || (flags & (NBK_JERK | NBK_NN))) return NBK_EINVAL;
    if (n_groups == 0) return NBK_OK;
    if (!i_offset || !j_offset || i_offset[0] != 0 || j_offset[0] != 0) return NBK_EINVAL;
    for (int64_t g = 0; g < n_groups; ++g)
        if (i_offset[g + 1] < i_offset[g] || j_offset[g + 1] < j_offset[g]) return NBK_EINVAL;
    const int64_t ni_tot = i_offset[n_groups], nj_tot = j_offset[n_groups];
    if (ni_tot > INT32_MAX || n_groups > INT32_MAX) return NBK_ERANGE;
    if (ni_tot == 0) return NBK_OK;
    if (!xi || !acc || !pot || (nj_tot > 0 && (!mj || !xj))) return NBK_EINVAL;
    DeviceGuard g(c->device);
    if (!g.ok) return cuda_fail(c, cudaErrorInvalidDevice);
    if (!c->batch_ready) {
        NBK_CUDA(c, batch_prepare());
        c->batch_ready = true;
    }
    // launch form from the mean group size: the i-tile is the power of two >= mean n_i in [32, 512];
    // the 16 warps that do not fit the i-tile split the j-tiles (wj)
    std::vector<int> keep;
    int64_t sum_ni = 0;
    for (int64_t q = 0; q < n_groups; ++q)
        if (i_offset[q + 1] > i_offset[q] && j_offset[q + 1] > j_offset[q]) {
            keep.push_back(static_cast<int>(q));
            sum_ni += i_offset[q + 1] - i_offset[q];
        }
    const size_t ni = static_cast<size_t>(ni_tot);
    float* d_acc = acc;
    float* d_pot = pot;
    const int ng = static_cast<int>(keep.size());
    int ti = 32;
    if (ng > 0) while (ti < 512 && ti < sum_ni / ng) ti *= 2;
    const int wj = 512 / ti, tj = 128;
    std::vector<long long> pair_prefix(ng + 1, 0), seg_prefix(ng + 1, 0), joff(ng + 1, 0), src_off(ng + 1, 0);
    std::vector<int> ioff(ng + 1, 0), njt(ng > 0 ? ng : 1, 0);
    for (int q = 0; q < ng; ++q) {
        const int64_t gg = keep[q];
        const long long n_i = i_offset[gg + 1] - i_offset[gg], n_j = j_offset[gg + 1] - j_offset[gg];
        const long long nit = (n_i + ti - 1) / ti, nt = (n_j + tj - 1) / tj;
        njt[q] = static_cast<int>(nt);
        pair_prefix[q + 1] = pair_prefix[q] + nit * nt;
        seg_prefix[q + 1] = seg_prefix[q] + nit;
        joff[q + 1] = joff[q] + nt * tj;
    }
    const long long P = pair_prefix[ng], n_seg = seg_prefix[ng], n_padded = joff[ng];
    const int gmax = c->num_sms < kMaxCtas ? c->num_sms : kMaxCtas;
    const int G = static_cast<int>(P < gmax ? P : gmax);
    // arena: [x y z m | descriptors | partial | (host entry: xi, mj, xj, acc, pot)]
    size_t off = 0;
    auto take = [&](size_t bytes) { const size_t at = off; off += (bytes + 255) & ~static_cast<size_t>(255); return at; };
    const size_t o_x = take(4 * sizeof(float) * n_padded);
    const size_t o_pp = take(sizeof(long long) * (ng + 1)), o_sp = take(sizeof(long long) * (ng + 1));
    const size_t o_jo = take(sizeof(long long) * (ng + 1)), o_so = take(sizeof(long long) * (ng + 1));
    const size_t o_do = take(sizeof(long long) * (ng + 1));
    const size_t o_io = take(sizeof(int) * (ng + 1)), o_nt = take(sizeof(int) * (ng + 1));
    const size_t o_ie = take(sizeof(int) * (ng + 1)), o_sl = take(sizeof(long long) * (ng + 1));
    const size_t o_part = take(sizeof(float) * 4 * ti * static_cast<size_t>(n_seg + G));
    size_t o_xi = 0, o_mj = 0, o_xj = 0, o_acc = 0, o_pot = 0;
    if (!dev) {
        o_xi = take(sizeof(float) * 3 * ni);
        o_mj = take(sizeof(float) * nj_tot);
        o_xj = take(sizeof(float) * 3 * nj_tot);
        o_acc = take(sizeof(float) * 3 * ni);
        o_pot = take(sizeof(float) * ni);
    }
    if (off > c->batch_bytes) {
        NBK_CUDA(c, cudaStreamSynchronize(c->stream));
        cudaFree(c->d_batch);
        c->d_batch = nullptr;
        c->batch_bytes = 0;
        NBK_CUDA(c, cudaMalloc(&c->d_batch, off + off / 4));
        c->batch_bytes = off + off / 4;
    }
    unsigned char* B = c->d_batch;
    // descriptors of the non-empty groups: i offsets are the caller's (outputs keep the caller's order)
    std::vector<long long> src_len(ng > 0 ? ng : 1, 0);
    for (int q = 0; q < ng; ++q) {
        ioff[q] = static_cast<int>(i_offset[keep[q]]);
        src_off[q] = j_offset[keep[q]];
        src_len[q] = j_offset[keep[q] + 1] - j_offset[keep[q]];
    }
    std::vector<int> iend(ng > 0 ? ng : 1);
    for (int q = 0; q < ng; ++q) iend[q] = static_cast<int>(i_offset[keep[q] + 1]);
    if (ng > 0) src_off[ng] = j_offset[keep[ng - 1] + 1];
    if (!dev) {
        NBK_CUDA(c, cudaMemcpyAsync(B + o_xi, xi, sizeof(float) * 3 * ni, cudaMemcpyHostToDevice, c->stream));
        if (nj_tot > 0) {
            NBK_CUDA(c, cudaMemcpyAsync(B + o_mj, mj, sizeof(float) * nj_tot, cudaMemcpyHostToDevice, c->stream));
            NBK_CUDA(c, cudaMemcpyAsync(B + o_xj, xj, sizeof(float) * 3 * nj_tot, cudaMemcpyHostToDevice, c->stream));
        }
        d_acc = reinterpret_cast<float*>(B + o_acc);
        d_pot = reinterpret_cast<float*>(B + o_pot);
    }
    NBK_CUDA(c, cudaMemsetAsync(d_acc, 0, sizeof(float) * 3 * ni, c->stream));
    NBK_CUDA(c, cudaMemsetAsync(d_pot, 0, sizeof(float) * ni, c->stream));
    if (ng > 0) {
        // pageable host vectors: these copies complete before the call returns to the vectors' scope end
        NBK_CUDA(c, cudaMemcpyAsync(B + o_pp, pair_prefix.data(), sizeof(long long) * (ng + 1), cudaMemcpyHostToDevice, c->stream));
        NBK_CUDA(c, cudaMemcpyAsync(B + o_sp, seg_prefix.data(), sizeof(long long) * (ng + 1), cudaMemcpyHostToDevice, c->stream));
        NBK_CUDA(c, cudaMemcpyAsync(B + o_jo, joff.data(), sizeof(long long) * (ng + 1), cudaMemcpyHostToDevice, c->stream));
        NBK_CUDA(c, cudaMemcpyAsync(B + o_so, src_off.data(), sizeof(long long) * (ng + 1), cudaMemcpyHostToDevice, c->stream));
        NBK_CUDA(c, cudaMemcpyAsync(B + o_io, ioff.data(), sizeof(int) * (ng + 1), cudaMemcpyHostToDevice, c->stream));
        NBK_CUDA(c, cudaMemcpyAsync(B + o_nt, njt.data(), sizeof(int) * ng, cudaMemcpyHostToDevice, c->stream));
        NBK_CUDA(c, cudaMemcpyAsync(B + o_ie, iend.data(), sizeof(int) * ng, cudaMemcpyHostToDevice, c->stream));
        NBK_CUDA(c, cudaMemcpyAsync(B + o_sl, src_len.data(), sizeof(long long) * ng, cudaMemcpyHostToDevice, c->stream));
        BatchPackArgs pk;
        pk.mj = dev ? mj : reinterpret_cast<const float*>(B + o_mj);
        pk.xj = dev ? xj : reinterpret_cast<const float*>(B + o_xj);
        pk.src_off = reinterpret_cast<const long long*>(B + o_so);
        pk.dst_off = reinterpret_cast<const long long*>(B + o_jo);
        pk.src_len = reinterpret_cast<const long long*>(B + o_sl);
        float* px = reinterpret_cast<float*>(B + o_x);
        pk.x = px; pk.y = px + n_padded; pk.z = px + 2 * n_padded; pk.m = px + 3 * n_padded;
        pk.n_groups = ng;
        pk.n_padded = n_padded;
        NBK_CUDA(c, launch_batch_pack(pk, c->stream));
        BatchArgs ba;
        ba.x = pk.x; ba.y = pk.y; ba.z = pk.z; ba.m = pk.m;
        ba.xi = dev ? xi : reinterpret_cast<const float*>(B + o_xi);
        ba.pair_prefix = reinterpret_cast<const long long*>(B + o_pp);
        ba.seg_prefix = reinterpret_cast<const long long*>(B + o_sp);
        ba.j_off = reinterpret_cast<const long long*>(B + o_jo);
        ba.i_off = reinterpret_cast<const int*>(B + o_io);
        ba.njt = reinterpret_cast<const int*>(B + o_nt);
        ba.i_end = reinterpret_cast<const int*>(B + o_ie);
        ba.partial = reinterpret_cast<float*>(B + o_part);
        ba.acc = d_acc; ba.pot = d_pot;
        ba.n_groups = ng; ba.ti = ti; ba.tj = tj; ba.wj = wj;
        ba.P = P; ba.n_seg = n_seg; ba.G = G; ba.eps2 = eps2;
        {
            TimeScope ts(c, 2);
            NBK_CUDA(c, launch_batch(ba, (flags & NBK_EPS0) != 0 || eps2 == 0.f, c->stream));
        }
        {
            TimeScope ts(c, 3);
            NBK_CUDA(c, launch_batch_reduce(ba, c->stream));
        }
        c->last_launch[0] = G; c->last_launch[1] = 512; c->last_launch[2] = 1; c->last_launch[3] = wj;
        c->last_launch[4] = tj; c->last_launch[5] = c->num_sms;
        c->last_launch[6] = static_cast<long long>(batch_smem_bytes()); c->last_launch[7] = 3;
    }
    if (!dev) {
        NBK_CUDA(c, cudaMemcpyAsync(acc, d_acc, sizeof(float) * 3 * ni, cudaMemcpyDeviceToHost, c->stream));
        NBK_CUDA(c, cudaMemcpyAsync(pot, d_pot, sizeof(float) * ni, cudaMemcpyDeviceToHost, c->stream));
    }
    // the descriptor vectors live on this stack frame: wait until their copies have been consumed
    NBK_CUDA(c, cudaStreamSynchronize(c->stream));
    return NBK_OK;
}

}  // namespace

int nbk_calc_batch(nbk_ctx* c, int64_t n_groups, const int64_t* i_offset, const float* xi,
                   const int64_t* j_offset, const float* mj, const float* xj, float eps2,
                   uint32_t flags, float* acc, float* pot) {
    return batch_impl(c, n_groups, i_offset, xi, j_offset, mj, xj, eps2, flags, acc, pot, false);
}

int nbk_calc_batch_dev(nbk_ctx* c, int64_t n_groups, const int64_t* i_offset, const float* xi,
                       const int64_t* j_offset, const float* mj, const float* xj, float eps2,
                       uint32_t flags, float* acc, float* pot) {
    return batch_impl(c, n_groups, i_offset, xi, j_offset, mj, xj, eps2, flags, acc, pot, true);
}

int nbk_sync(nbk_ctx* c) {
    if (!c) return NBK_EINVAL;
    DeviceGuard g(c->device);
    NBK_CUDA(c, cudaStreamSynchronize(c->stream));
    return NBK_OK;
}

int nbk_set_timing(nbk_ctx* c, int enable) {
    if (!c) return NBK_EINVAL;
    c->timing = enable != 0;
    for (int s = 0; s < 4; ++s) c->ev_used[s] = false;
    return NBK_OK;
}

int nbk_get_timing(nbk_ctx* c, float ms[4]) {
    if (!c || !ms) return NBK_EINVAL;
    DeviceGuard g(c->device);
    NBK_CUDA(c, cudaStreamSynchronize(c->stream));
    for (int s = 0; s < 4; ++s) {
        ms[s] = 0.f;
        if (c->ev_used[s]) NBK_CUDA(c, cudaEventElapsedTime(&ms[s], c->ev[s][0], c->ev[s][1]));
        c->ev_used[s] = false;
    }
    return NBK_OK;
}

int nbk_last_launch(const nbk_ctx* c, int64_t out[8]) {
    if (!c || !out) return NBK_EINVAL;
    for (int k = 0; k < 8; ++k) out[k] = c->last_launch[k];
    return NBK_OK;
}

int nbk_plan(int64_t n_i, int64_t n_j, int num_sms, int force_i, int64_t out[12]) {
    if (n_i < 1 || n_j < 1 || num_sms < 1 || !out || n_i > (1LL << 30) || n_j > (1LL << 30) ||
        !(force_i == 0 || force_i == 1 || force_i == 2 || force_i == 4))
        return NBK_EINVAL;
    Variant v{0, true, false, true};
    Decomp d;
    d.G = 0;
    plan_shape(n_i, n_j, num_sms, force_i, plan_partial_floats_bound(n_i, num_sms), &v, &d);
    if (d.G < 1) return NBK_ENOMEM;
    out[0] = v.I; out[1] = warps_of(v.I) * 32; out[2] = d.ti; out[3] = d.tj; out[4] = d.wj;
    out[5] = d.nit; out[6] = d.njt; out[7] = d.P; out[8] = d.G; out[9] = d.maxseg;
    out[10] = static_cast<int64_t>(plan_partial_floats(d));
    out[11] = static_cast<int64_t>(plan_partial_floats_bound(n_i, num_sms));
    return NBK_OK;
}

int nbk_set_variant(nbk_ctx* c, int variant) {
    if (!c || variant < 0) return NBK_EINVAL;
    const int I = (variant >> 4) & 15;
    if (!(I == 0 || I == 1 || I == 2 || I == 4)) return NBK_EINVAL;
    c->variant_scalar = variant & 1;
    c->force_I = I;
    c->fused_ok = (variant & 0x100) == 0;
    return NBK_OK;
}

int nbk_last_cuda_error(const nbk_ctx* c) { return c ? c->last_cuda : 0; }

const char* nbk_strerror(int status) {
    switch (status) {
        case NBK_OK: return "ok";
        case NBK_EINVAL: return "invalid argument";
        case NBK_ERANGE: return "address or count out of range for this context";
        case NBK_ENOMEM: return "out of memory";
        case NBK_ECUDA: return "CUDA error (see nbk_last_cuda_error)";
        case NBK_ESTATE: return "call order violated";
        default: return "unknown status";
    }
}

const char* nbk_version(void) { return "nbk 0.1 (sm_100a)"; }

}  // extern "C"
