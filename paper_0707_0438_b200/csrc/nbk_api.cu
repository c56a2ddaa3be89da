// nbk_api.cu -- the C ABI of include/nbk.h: context, workspaces, staging and launch logic.
// Every step of the path runs in the kernels of nbk_force.cu / nbk_state_kernels.cu; this file only moves
// arguments, picks the launch shape and enqueues.  There is no CPU fallback: without a CUDA
// device nbk_open fails with NBK_ECUDA.
#include <cuda_runtime.h>

#include <chrono>
#include <climits>
#include <cmath>
#include <cstdlib>
#include <atomic>
#include <cstring>
#include <functional>
#include <new>
#include <vector>

#include "nbk_ctx.cuh"

using namespace nbk;

namespace nbk {

bool pdl_enabled() {
    static const bool on = [] {
        const char* e = std::getenv("NBK_PDL");
        return !(e && e[0] == '0');
    }();
    return on;
}

// Page-locked host memory (cudaHostAlloc / cudaHostRegister, e.g. a pinned torch tensor): the DMA engine
// can read and write it directly, so large transfers skip the copy through the library's staging buffer.
bool is_pinned_host(const void* p) {
    if (!p) return true;   // absent arrays do not decide
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, p) != cudaSuccess) {
        (void)cudaGetLastError();
        return false;
    }
    return at.type == cudaMemoryTypeHost;
}
constexpr long long kDirectMin = 4096;   // particles from which a pinned caller array is copied directly

int cuda_fail(nbk_ctx* c, cudaError_t e) {
    c->last_cuda = static_cast<int>(e);
    (void)cudaGetLastError();
    return NBK_ECUDA;
}

JPred jpred_of(const nbk_ctx* c) {
    JPred j;
    j.x = pred_arr(c, 0); j.y = pred_arr(c, 1); j.z = pred_arr(c, 2); j.m = pred_arr(c, 3);
    j.vx = pred_arr(c, 4); j.vy = pred_arr(c, 5); j.vz = pred_arr(c, 6);
    return j;
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

}  // namespace nbk

namespace {

void free_all(nbk_ctx* c) {
    if (!c->caller_workspace) {   // otherwise these are pieces of the caller's buffer
        cudaFree(c->raw.x); cudaFree(c->raw.v); cudaFree(c->raw.a); cudaFree(c->raw.k);
        cudaFree(c->raw.m); cudaFree(c->raw.t); cudaFree(c->pred);
        cudaFree(c->d_iidx); cudaFree(c->d_xi); cudaFree(c->d_vi);
        cudaFree(c->d_partial); cudaFree(c->d_result); cudaFree(c->d_stage); cudaFree(c->d_counter);
        cudaFree(c->d_nn_partial); cudaFree(c->d_nn_best); cudaFree(c->d_nn_tile);
        cudaFree(c->d_nn_index); cudaFree(c->d_nn_r2);
    }
    cudaFree(c->d_batch);
    cudaFree(c->hs.x); cudaFree(c->hs.v); cudaFree(c->hs.a); cudaFree(c->hs.j);
    cudaFree(c->hs.level); cudaFree(c->hs.act); cudaFree(c->hs.bc_ge); cudaFree(c->hs.flag); cudaFree(c->hs.rows); cudaFree(c->d_hdr);
    if (c->h_hdr) cudaFreeHost(c->h_hdr);
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
                  const int32_t* h_inline = nullptr, bool to_host = false,
                  double* sum64 = nullptr) {
    eps2 = flushed_eps2(eps2);
    float* acc = c->d_result;
    float* jerk = acc + 3 * n_i;
    float* pot = acc + 6 * n_i;
    // A block of <= 32 particles of the j-set: ONE launch that predicts, sums and reduces (nbk_small_kernels.cu)
    {
        const int G = c->num_sms < kMaxCtas ? c->num_sms : kMaxCtas;
        const long long n_pad = round_up(n_j, kTileJMax);
        const long long chunk = round_up((n_pad + G - 1) / G, 4);
        bool small = n_i >= 1 && n_i <= kFusedMaxI && n_j >= 1 && !d_xi && !d_vi && !sum64 && c->fused_ok &&
                     !(flags & NBK_NN) && chunk <= kSmallMaxChunk &&
                     plan_partial_floats_bound(c->ni_max, c->num_sms) >= static_cast<size_t>(G) * kFusedMaxI * 8;
        if (small && h_inline)
            for (long long k = 0; k < n_i; ++k) small = small && h_inline[k] >= 0;
        if (small) {
            bool fold = true;
            for (int k = 0; k < c->pending.n; ++k) fold = fold && c->pending.addr[k] < n_j;
            if (!fold) {
                const int rc = flush_pending(c);
                if (rc != NBK_OK) return rc;
            }
            SmallArgs sa;
            sa.raw = c->raw;
            sa.t = c->t;
            sa.n_j = static_cast<int>(n_j);
            sa.n_pad = static_cast<int>(n_pad);
            sa.chunk = static_cast<int>(chunk);
            for (int k = 0; k < 7; ++k) sa.pred[k] = pred_arr(c, k);
            sa.n_i = static_cast<int>(n_i);
            sa.inline_index = h_inline ? 1 : 0;
            std::memset(sa.i_inline, 0, sizeof(sa.i_inline));
            if (h_inline) std::memcpy(sa.i_inline, h_inline, sizeof(int32_t) * n_i);
            sa.i_index = d_iidx;
            sa.eps2 = eps2;
            sa.partial = c->d_partial;
            sa.counter = c->d_counter;
            sa.acc = acc; sa.jerk = jerk; sa.pot = pot;
            sa.host_out = to_host ? c->h_result_dev : nullptr;
            sa.host_seq = to_host ? c->h_seq_dev : nullptr;
            sa.seq = ++c->small_seq;
            if (sa.seq == 0) sa.seq = ++c->small_seq;   // 0 is the word's initial value
            sa.upd = c->pending;
            if (!c->small_ready) {
                NBK_CUDA(c, small_prepare(kSmallMaxChunk));
                c->small_ready = true;
            }
            c->last_ni = n_i;
            c->in_flight = true;
            c->last_nn = false;
            {
                TimeScope ts(c, 2);
                NBK_CUDA(c, launch_small_block(sa, (flags & NBK_JERK) != 0, (flags & NBK_EPS0) != 0 || eps2 == 0.f, G,
                                               c->stream));
            }
            c->pending.n = 0;
            c->pred_valid = true;
            c->pred_nj = n_j;
            c->host_has_result = to_host;
            c->poll_result = to_host;
            c->last_launch[0] = G; c->last_launch[1] = 512; c->last_launch[2] = 1; c->last_launch[3] = 16;
            c->last_launch[4] = chunk; c->last_launch[5] = c->num_sms;
            c->last_launch[6] = static_cast<long long>(small_smem_bytes(sa.chunk)); c->last_launch[7] = 1;
            return NBK_OK;
        }
    }
    if (!c->pred_valid || c->pred_nj != n_j) {
        const int rc = do_predict(c, n_j);
        if (rc != NBK_OK) return rc;
    }
    c->last_ni = n_i;
    c->in_flight = true;
    c->host_has_result = false;
    c->poll_result = false;
    if (n_i == 0) return NBK_OK;
    if (n_j == 0) {
        NBK_CUDA(c, cudaMemsetAsync(acc, 0, sizeof(float) * 7 * n_i, c->stream));
        if (sum64) NBK_CUDA(c, cudaMemsetAsync(sum64, 0, sizeof(double) * 8 * n_i, c->stream));
        c->last_launch[7] = 0;
        return NBK_OK;
    }
    Variant v;
    Decomp d;
    v.jerk = (flags & NBK_JERK) != 0;
    v.eps0 = (flags & NBK_EPS0) != 0 || eps2 == 0.f;
    v.nn = (flags & NBK_NN) != 0;
    c->last_nn = v.nn;
    d.G = 0;
    plan_shape(n_i, n_j, c->num_sms, c->force_I, c->partial_bytes / sizeof(float), &v, &d);
    if (d.G < 1 || plan_partial_floats(d) * sizeof(float) > c->partial_bytes) return NBK_ENOMEM;
    if ((d.P + d.G - 1) / d.G > INT_MAX) return NBK_ERANGE;   // the kernel counts a CTA's pairs in an int

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
    const bool fused = v.I == 1 && d.nit == 1 && n_i <= kFusedMaxI && c->fused_ok && !sum64;
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
    ra.sum64 = sum64;
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
    {   // padded size of [tj | m | x | v | a | jerk | addr], checked before anything is copied
        const size_t un = static_cast<size_t>(n);
        auto pad = [](size_t b) { return (b + 15) & ~static_cast<size_t>(15); };
        const size_t need = pad(sizeof(double) * un) + pad(sizeof(T) * un) + 4 * pad(sizeof(T) * 3 * un) +
                            pad(sizeof(int32_t) * un);
        if (need > c->stage_bytes) return NBK_ENOMEM;
    }
    NBK_CUDA(c, cudaEventSynchronize(c->stage_free));
    // pack [tj | m | x | v | a | jerk | addr] into the pinned buffer: one H2D copy
    size_t off = 0;
    std::function<size_t(const void*, size_t)> put = [&](const void* src, size_t bytes) -> size_t {
        const size_t at = off;
        if (src) std::memcpy(c->h_stage + at, src, bytes);
        off += (bytes + 15) & ~static_cast<size_t>(15);
        return at;
    };
    // caller arrays in pinned memory: one asynchronous copy per array straight from them; the call
    // waits for the copies before it returns (the caller may reuse its arrays at once, nbk.h)
    const bool direct = n >= kDirectMin && is_pinned_host(tj) && is_pinned_host(m) && is_pinned_host(x) &&
                        is_pinned_host(v) && is_pinned_host(a) && is_pinned_host(jerk) && is_pinned_host(addr);
    cudaError_t derr = cudaSuccess;
    if (direct) {
        put = [&](const void* src, size_t bytes) -> size_t {
            const size_t at = off;
            if (src && derr == cudaSuccess)
                derr = cudaMemcpyAsync(c->d_stage + at, src, bytes, cudaMemcpyHostToDevice, c->stream);
            off += (bytes + 15) & ~static_cast<size_t>(15);
            return at;
        };
    }
    const size_t o_t = put(tj, sizeof(double) * n);
    const size_t o_m = put(m, sizeof(T) * n);
    const size_t o_x = put(x, sizeof(T) * 3 * n);
    const size_t o_v = put(v, sizeof(T) * 3 * n);
    const size_t o_a = put(a, sizeof(T) * 3 * n);
    const size_t o_k = put(jerk, sizeof(T) * 3 * n);
    const size_t o_ad = put(addr, sizeof(int32_t) * n);
    if (direct) {
        NBK_CUDA(c, derr);
        NBK_CUDA(c, cudaEventRecord(c->stage_free, c->stream));
        NBK_CUDA(c, cudaEventSynchronize(c->stage_free));
    } else {
        NBK_CUDA(c, cudaMemcpyAsync(c->d_stage, c->h_stage, off, cudaMemcpyHostToDevice, c->stream));
        NBK_CUDA(c, cudaEventRecord(c->stage_free, c->stream));
    }
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

namespace {

// Device memory of a context comes either from cudaMalloc (nbk_open) or, piece by piece and
// 256-byte aligned, from one caller-owned buffer (nbk_open_ws; nbk_workspace_bytes adds up the
// same pieces in the same order).
struct DeviceArena {
    unsigned char* base = nullptr;
    size_t cap = 0, off = 0;
    cudaError_t take(void** p, size_t bytes) {
        if (!base) return cudaMalloc(p, bytes);
        const size_t at = (off + 255) & ~static_cast<size_t>(255);
        off = at + bytes;
        if (off > cap) return cudaErrorMemoryAllocation;
        *p = base + at;
        return cudaSuccess;
    }
};

size_t workspace_total(long long n_max, long long ni_max, int num_sms) {
    const size_t cap = static_cast<size_t>(round_up(n_max, kTileJMax)), ni = static_cast<size_t>(ni_max);
    const size_t pb = sizeof(float) * plan_partial_floats_bound(ni_max, num_sms);
    const size_t sb = static_cast<size_t>(n_max) * (8 + 8 + 4 * 24 + 4) + 16 * 8;
    const size_t pieces[] = {24 * cap, 12 * cap, 12 * cap, 12 * cap, 4 * cap, 8 * cap, 28 * cap,   // raw, pred
                             4 * ni, 12 * ni, 12 * ni, 28 * ni, sizeof(unsigned),                   // i staging, result
                             pb, pb / 4, 4 * ni, 4 * ni, 4 * ni, 4 * ni, sb};                       // partial, nn, stage
    size_t off = 0;
    for (size_t b : pieces) off = ((off + 255) & ~static_cast<size_t>(255)) + b;
    return off;
}

int open_impl(nbk_ctx** out, int device, int64_t n_max, int64_t ni_max, void* cuda_stream,
              void* workspace, size_t workspace_bytes) {
    if (!out || n_max < 1 || ni_max < 1 || n_max > (1LL << 30) || ni_max > (1LL << 30))
        return NBK_EINVAL;
    *out = nullptr;
    nbk_ctx* c = new (std::nothrow) nbk_ctx();
    if (!c) return NBK_ENOMEM;
    DeviceArena arena;
    arena.base = static_cast<unsigned char*>(workspace);
    arena.cap = workspace_bytes;
    c->caller_workspace = workspace != nullptr;
    auto dalloc = [&](void** p, size_t bytes) { return arena.take(p, bytes); };
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
                for (int e0 = 0; e0 < 2 && e == cudaSuccess; ++e0) {
                    Variant v{I, jk != 0, e0 != 0, false};
                    e = force_prepare(v);
                }
        if (e != cudaSuccess) break;
        const size_t cap = static_cast<size_t>(c->n_cap);
        if ((e = dalloc(reinterpret_cast<void**>(&c->raw.x), sizeof(double) * 3 * cap)) != cudaSuccess) break;
        if ((e = dalloc(reinterpret_cast<void**>(&c->raw.v), sizeof(float) * 3 * cap)) != cudaSuccess) break;
        if ((e = dalloc(reinterpret_cast<void**>(&c->raw.a), sizeof(float) * 3 * cap)) != cudaSuccess) break;
        if ((e = dalloc(reinterpret_cast<void**>(&c->raw.k), sizeof(float) * 3 * cap)) != cudaSuccess) break;
        if ((e = dalloc(reinterpret_cast<void**>(&c->raw.m), sizeof(float) * cap)) != cudaSuccess) break;
        if ((e = dalloc(reinterpret_cast<void**>(&c->raw.t), sizeof(double) * cap)) != cudaSuccess) break;
        if ((e = dalloc(reinterpret_cast<void**>(&c->pred), sizeof(float) * 7 * cap)) != cudaSuccess) break;
        if ((e = cudaMemsetAsync(c->raw.x, 0, sizeof(double) * 3 * cap, c->stream)) != cudaSuccess) break;
        if ((e = cudaMemsetAsync(c->raw.v, 0, sizeof(float) * 3 * cap, c->stream)) != cudaSuccess) break;
        if ((e = cudaMemsetAsync(c->raw.a, 0, sizeof(float) * 3 * cap, c->stream)) != cudaSuccess) break;
        if ((e = cudaMemsetAsync(c->raw.k, 0, sizeof(float) * 3 * cap, c->stream)) != cudaSuccess) break;
        if ((e = cudaMemsetAsync(c->raw.m, 0, sizeof(float) * cap, c->stream)) != cudaSuccess) break;
        if ((e = cudaMemsetAsync(c->raw.t, 0, sizeof(double) * cap, c->stream)) != cudaSuccess) break;
        if ((e = cudaMemsetAsync(c->pred, 0, sizeof(float) * 7 * cap, c->stream)) != cudaSuccess) break;
        const size_t ni = static_cast<size_t>(ni_max);
        if ((e = dalloc(reinterpret_cast<void**>(&c->d_iidx), sizeof(int32_t) * ni)) != cudaSuccess) break;
        if ((e = dalloc(reinterpret_cast<void**>(&c->d_xi), sizeof(float) * 3 * ni)) != cudaSuccess) break;
        if ((e = dalloc(reinterpret_cast<void**>(&c->d_vi), sizeof(float) * 3 * ni)) != cudaSuccess) break;
        if ((e = dalloc(reinterpret_cast<void**>(&c->d_result), sizeof(float) * 7 * ni)) != cudaSuccess) break;
        const size_t seq_at = (9 * ni + 15) / 16 * 16;   // the sequence word on a 64-byte line of its own behind the results
        if ((e = cudaHostAlloc(&c->h_result, sizeof(float) * (seq_at + 16), cudaHostAllocMapped)) != cudaSuccess) break;
        if ((e = cudaHostGetDevicePointer(&c->h_result_dev, c->h_result, 0)) != cudaSuccess) break;
        std::memset(c->h_result + seq_at, 0, sizeof(float) * 16);
        c->h_seq = reinterpret_cast<volatile unsigned*>(c->h_result + seq_at);
        c->h_seq_dev = reinterpret_cast<unsigned*>(c->h_result_dev + seq_at);
        if ((e = dalloc(reinterpret_cast<void**>(&c->d_counter), sizeof(unsigned))) != cudaSuccess) break;
        if ((e = cudaMemsetAsync(c->d_counter, 0, sizeof(unsigned), c->stream)) != cudaSuccess) break;
        c->partial_bytes = sizeof(float) * plan_partial_floats_bound(ni_max, c->num_sms);
        if ((e = dalloc(reinterpret_cast<void**>(&c->d_partial), c->partial_bytes)) != cudaSuccess) break;
        if ((e = dalloc(reinterpret_cast<void**>(&c->d_nn_partial), c->partial_bytes / 4)) != cudaSuccess) break;
        if ((e = dalloc(reinterpret_cast<void**>(&c->d_nn_best), sizeof(float) * ni)) != cudaSuccess) break;
        if ((e = dalloc(reinterpret_cast<void**>(&c->d_nn_tile), sizeof(int32_t) * ni)) != cudaSuccess) break;
        if ((e = dalloc(reinterpret_cast<void**>(&c->d_nn_index), sizeof(int32_t) * ni)) != cudaSuccess) break;
        if ((e = dalloc(reinterpret_cast<void**>(&c->d_nn_r2), sizeof(float) * ni)) != cudaSuccess) break;
        c->stage_bytes = static_cast<size_t>(n_max) * (8 + 8 + 4 * 24 + 4) + 16 * 8;
        if ((e = cudaMallocHost(&c->h_stage, c->stage_bytes)) != cudaSuccess) break;
        if ((e = dalloc(reinterpret_cast<void**>(&c->d_stage), c->stage_bytes)) != cudaSuccess) break;
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

}  // namespace

int nbk_open(nbk_ctx** out, int device, int64_t n_max, int64_t ni_max, void* cuda_stream) {
    return open_impl(out, device, n_max, ni_max, cuda_stream, nullptr, 0);
}

int nbk_open_ws(nbk_ctx** out, int device, int64_t n_max, int64_t ni_max, void* cuda_stream,
                void* workspace, int64_t workspace_bytes) {
    if (!workspace || workspace_bytes <= 0 || (reinterpret_cast<uintptr_t>(workspace) & 255u)) return NBK_EINVAL;
    return open_impl(out, device, n_max, ni_max, cuda_stream, workspace, static_cast<size_t>(workspace_bytes));
}

int64_t nbk_workspace_bytes(int device, int64_t n_max, int64_t ni_max) {
    if (n_max < 1 || ni_max < 1 || n_max > (1LL << 30) || ni_max > (1LL << 30)) return NBK_EINVAL;
    int sms = 0;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device) != cudaSuccess) {
        (void)cudaGetLastError();
        return NBK_ECUDA;
    }
    return static_cast<int64_t>(workspace_total(n_max, ni_max, sms));
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
    if (!c->host_has_result && n_i >= kDirectMin && (acc || jerk || pot) && is_pinned_host(acc) &&
        is_pinned_host(jerk) && is_pinned_host(pot)) {   // pinned caller arrays: device -> caller directly
        if (acc) NBK_CUDA(c, cudaMemcpyAsync(acc, c->d_result, sizeof(float) * 3 * ni, cudaMemcpyDeviceToHost, c->stream));
        if (jerk) NBK_CUDA(c, cudaMemcpyAsync(jerk, c->d_result + 3 * ni, sizeof(float) * 3 * ni, cudaMemcpyDeviceToHost, c->stream));
        if (pot) NBK_CUDA(c, cudaMemcpyAsync(pot, c->d_result + 6 * ni, sizeof(float) * ni, cudaMemcpyDeviceToHost, c->stream));
        NBK_CUDA(c, cudaStreamSynchronize(c->stream));
        return NBK_OK;
    }
    if (!c->host_has_result)
        NBK_CUDA(c, cudaMemcpyAsync(c->h_result, c->d_result, sizeof(float) * 7 * ni,
                                    cudaMemcpyDeviceToHost, c->stream));
    if (c->host_has_result && c->poll_result && !c->timing) {
        // One-launch small block: its last CTA wrote the results into h_result (mapped) and then the sequence
        // word.  Seeing the word is enough -- no need to wait for the kernel to retire and the driver to notice
        // (the per-call overhead is what a block step of a few particles costs).  The stream
        // is asked now and then so that a failed launch ends the wait.
        const unsigned want = c->small_seq;
        for (unsigned spins = 1; *c->h_seq != want; ++spins) {
            if ((spins & 2047u) == 0) {
                const cudaError_t q = cudaStreamQuery(c->stream);
                if (q == cudaSuccess) {
                    if (*c->h_seq == want) break;
                    return cuda_fail(c, cudaErrorUnknown);   // the kernel retired without writing the word
                }
                if (q != cudaErrorNotReady) return cuda_fail(c, q);
            }
        }
        std::atomic_thread_fence(std::memory_order_acquire);
    } else {
        NBK_CUDA(c, cudaStreamSynchronize(c->stream));
    }
    if (acc) std::memcpy(acc, c->h_result, sizeof(float) * 3 * ni);
    if (jerk) std::memcpy(jerk, c->h_result + 3 * ni, sizeof(float) * 3 * ni);
    if (pot) std::memcpy(pot, c->h_result + 6 * ni, sizeof(float) * ni);
    return NBK_OK;
}

int nbk_calc_lasthalf_f64(nbk_ctx* c, int64_t n_i, double* acc, double* jerk, double* pot) {
    if (!c || n_i < 0) return NBK_EINVAL;
    if (!c->in_flight || n_i != c->last_ni) return NBK_ESTATE;
    const int rc = nbk_calc_lasthalf(c, n_i, nullptr, nullptr, nullptr);   // waits, fills h_result
    if (rc != NBK_OK) return rc;
    const size_t ni = static_cast<size_t>(n_i);
    const float* h = c->h_result;
    for (size_t k = 0; k < 3 * ni; ++k) {
        if (acc) acc[k] = h[k];
        if (jerk) jerk[k] = h[3 * ni + k];
    }
    if (pot)
        for (size_t k = 0; k < ni; ++k) pot[k] = h[6 * ni + k];
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

// ---- j-sharding over several GPUs -----------------
int nbk_shard_gather_i_dev(nbk_ctx* c, int64_t n_local, int64_t j0, int64_t n_i,
                           const int32_t* i_global, int32_t* i_local, float* xv) {
    if (!c || n_local < 0 || n_i < 0 || j0 < 0) return NBK_EINVAL;
    if (n_i > 0 && (!i_global || !i_local || !xv)) return NBK_EINVAL;
    if (n_local > c->n_max || n_i > c->ni_max) return NBK_ERANGE;
    if (n_i == 0) return NBK_OK;
    DeviceGuard g(c->device);
    if (!g.ok) return cuda_fail(c, cudaErrorInvalidDevice);
    if (n_local > 0 && (!c->pred_valid || c->pred_nj != n_local)) {
        const int rc = do_predict(c, n_local);
        if (rc != NBK_OK) return rc;
    }
    ShardGatherArgs a;
    a.j = jpred_of(c);
    a.i_global = i_global; a.i_local = i_local; a.xv = xv;
    a.n_i = n_i; a.j0 = j0; a.n_local = n_local;
    NBK_CUDA(c, launch_shard_gather(a, c->stream));
    return NBK_OK;
}

int nbk_shard_calc_partial_dev(nbk_ctx* c, int64_t n_local, int64_t n_i, const int32_t* i_local,
                               const float* xv, float eps2, uint32_t flags, double* sum64) {
    if (!c || n_local < 0 || n_i < 0 || !(eps2 >= 0.f)) return NBK_EINVAL;
    if (flags & NBK_NN) return NBK_EINVAL;   // the neighbour search is per shard: not combined here
    if (n_i > 0 && (!i_local || !xv || !sum64)) return NBK_EINVAL;
    if (n_local > c->n_max || n_i > c->ni_max) return NBK_ERANGE;
    DeviceGuard g(c->device);
    if (!g.ok) return cuda_fail(c, cudaErrorInvalidDevice);
    NBK_CUDA(c, launch_shard_split(xv, n_i, c->d_xi, c->d_vi, c->stream));
    return enqueue_force(c, n_local, n_i, i_local, c->d_xi, c->d_vi, eps2, flags, nullptr, false,
                         sum64);
}

int nbk_shard_finish_dev(nbk_ctx* c, int64_t n_i, const double* sum64, float* acc, float* jerk,
                         float* pot) {
    if (!c || n_i < 0) return NBK_EINVAL;
    if (n_i > 0 && !sum64) return NBK_EINVAL;
    DeviceGuard g(c->device);
    if (!g.ok) return cuda_fail(c, cudaErrorInvalidDevice);
    NBK_CUDA(c, launch_shard_finish(sum64, n_i, acc, jerk, pot, c->stream));
    return NBK_OK;
}

int nbk_shard_fetch_i_dev(nbk_ctx* c, int64_t n_i, int32_t world, const int32_t* i_global,
                          const int64_t* shard_begin, const void* const* peer_xv, float* xv) {
    if (!c || n_i < 0 || world < 1 || world > kMaxPeers || !shard_begin || !peer_xv) return NBK_EINVAL;
    if (n_i > 0 && (!i_global || !xv)) return NBK_EINVAL;
    if (n_i > c->ni_max) return NBK_ERANGE;
    ShardPeers p;
    std::memset(&p, 0, sizeof(p));
    p.world = world;
    for (int r = 0; r < world; ++r) {
        if (!peer_xv[r] || shard_begin[r] > shard_begin[r + 1]) return NBK_EINVAL;
        p.ptr[r] = peer_xv[r];
        p.begin[r] = shard_begin[r];
    }
    p.begin[world] = shard_begin[world];
    DeviceGuard g(c->device);
    if (!g.ok) return cuda_fail(c, cudaErrorInvalidDevice);
    NBK_CUDA(c, launch_shard_fetch(p, i_global, n_i, xv, c->stream));
    return NBK_OK;
}

int nbk_shard_combine_dev(nbk_ctx* c, int64_t n_i, int32_t world, const void* const* peer_sum64,
                          float* acc, float* jerk, float* pot) {
    if (!c || n_i < 0 || world < 1 || world > kMaxPeers || !peer_sum64) return NBK_EINVAL;
    ShardPeers p;
    std::memset(&p, 0, sizeof(p));
    p.world = world;
    for (int r = 0; r < world; ++r) {
        if (!peer_sum64[r]) return NBK_EINVAL;
        p.ptr[r] = peer_sum64[r];
    }
    DeviceGuard g(c->device);
    if (!g.ok) return cuda_fail(c, cudaErrorInvalidDevice);
    NBK_CUDA(c, launch_shard_combine(p, n_i, acc, jerk, pot, c->stream));
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
    Variant v{0, true, false, false};
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
    if (!c || variant < 0 || (variant & ~0x1f0)) return NBK_EINVAL;
    const int I = (variant >> 4) & 15;
    if (!(I == 0 || I == 1 || I == 2 || I == 4)) return NBK_EINVAL;
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
