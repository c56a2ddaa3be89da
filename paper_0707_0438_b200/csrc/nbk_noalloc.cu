// nbk_noalloc.cu -- nbk_calc_noalloc_dev: the split-j force evaluation for callers that must not
// allocate device memory.
//
// Who this is for.  Every other way into the library goes through nbk_open, which calls cudaMalloc /
// cudaHostAlloc for the j-state, the partial rows and the staging buffers.  Some callers cannot do that:
//   - a plug-in inside a process whose own memory pool (a framework's caching allocator, a simulation
//     code that sized its arrays to the last byte of HBM at start-up) already owns the device memory
//     budget, so a cudaMalloc from a library either fails or takes memory the host promised elsewhere;
//   - a step loop with a latency bound, because cudaMalloc / cudaFree take the driver's allocation lock
//     and cudaFree waits for the whole device: one call stalls every stream of the process;
//   - codes run under a "no allocation after initialisation" rule, where each allocation site has to
//     be justified and the simplest answer is to have none.
// They get this one call.  It has no context: the j-particles and the results are the caller's own
// device arrays, and the only memory the method needs beyond them -- the partial force rows of the
// split-j scheme (3.2) and one arrival counter per i-tile -- lives in the
// file-scope __device__ array below, which is part of the library's image: every GPU that loads
// libnbk.so holds those NBK_NOALLOC_SCRATCH_BYTES (4 MiB + 256 B) from the moment the module is loaded
// until the process exits, whether this call is used or not.
//
// What follows from the scratch being one array per GPU:
//   - the sizes are bounded: n_i <= NBK_NOALLOC_MAX_NI, n_j <= NBK_NOALLOC_MAX_NJ; beyond that the call
//     returns NBK_ERANGE and does nothing (use a context);
//   - every call on a device uses the same array.  Calls on ONE stream are ordered by the stream and
//     are safe.  Calls of one process whose kernels can overlap on the GPU (different streams, from one
//     host thread or from several) write the same rows and counters: a data race, wrong results.
//     Order them with events or use one stream.  (Another process has its own copy of the array.);
//   - the array keeps what the last call left.  The rows need no clearing (every row a call reads it
//     has written itself); the arrival counters must start at zero, so each call enqueues a
//     cudaMemsetAsync of the counter block in front of its kernel (and the kernel's last CTA of a tile
//     puts its counter back to zero as well).
//
// The name of a __device__ array is, in host code, a host-side handle and not a device address:
// handing it to a kernel or to cudaMemsetAsync makes the GPU touch an unrelated (or unmapped) address.
// The address comes from cudaGetSymbolAddress, asked once per device with that device current
// (scratch_of below), and that pointer is what the launches get.  The FIRST call on a device does this
// set-up (it may make the runtime load the module); make that first call outside any stream capture.
//
// The arithmetic is include/nbk.h's: r = x_j - x_i, w = v_j - v_i, s = r.r + eps2, fp32 per pair with
// rsqrt, fp32 sums over one tile of 256 j-particles folded into fp64, partial rows stored in fp32, the
// rows of an i-particle added in fp64 in split order (so results repeat bit for bit), one rounding.
// It is a plain kernel (one i-particle per thread, j-tiles staged through shared memory as in PAPER.md
// L91-L96) -- the tuned TMA / packed-arithmetic path stays behind nbk_calc_firsthalf.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdint>
#include <mutex>

#include "../../include/nbk.h"

namespace {

constexpr int kTileI = 128;     // i-particles per CTA, one per thread
constexpr int kTileJ = 256;     // j-particles staged in shared memory at a time
constexpr int kMaxSplit = 32;   // most CTAs that share one i-tile's j-range
constexpr int kRowFloats = 8;   // ax ay az sum(m/sqrt s) jx jy jz 0
constexpr int kMaxTilesI = NBK_NOALLOC_MAX_NI / kTileI;
constexpr size_t kRowsBytes = sizeof(float) * kRowFloats * NBK_NOALLOC_MAX_NI * kMaxSplit;
constexpr size_t kCounterBytes = 256;  // kMaxTilesI unsigned counters, padded to the alignment
static_assert(NBK_NOALLOC_MAX_NI % kTileI == 0, "whole i-tiles");
static_assert(kMaxTilesI * sizeof(unsigned) <= kCounterBytes, "counters fit their block");
static_assert(kRowsBytes + kCounterBytes == NBK_NOALLOC_SCRATCH_BYTES, "nbk.h states the size");
constexpr int kMaxDevices = 64;

// The scratch: [kMaxSplit][n_i padded to whole tiles][8] floats of partial rows, then the counters.
static __device__ __align__(256) unsigned char g_noalloc_scratch[NBK_NOALLOC_SCRATCH_BYTES];

template <bool JERK>
__global__ void __launch_bounds__(kTileI)
noalloc_force_kernel(const float* __restrict__ m, const float* __restrict__ x,
                     const float* __restrict__ v, int n_j, const int32_t* __restrict__ i_index, int n_i,
                     float eps2, int eps0, int n_split, int j_per_split, float* rows, unsigned* arrived,
                     float* __restrict__ acc, float* __restrict__ jerk, float* __restrict__ pot) {
    __shared__ float4 s_pm[kTileJ];
    __shared__ float4 s_vel[JERK ? kTileJ : 1];
    __shared__ int s_last;

    const int tile = blockIdx.x, split = blockIdx.y;
    const int k = tile * kTileI + threadIdx.x;
    const int ni_pad = gridDim.x * kTileI;
    int self = -1;
    float xi = 0.f, yi = 0.f, zi = 0.f, vxi = 0.f, vyi = 0.f, vzi = 0.f;
    bool live = k < n_i;
    if (live) {
        self = i_index ? i_index[k] : k;
        if (self < 0 || self >= n_j) {
            live = false;  // documented: such an entry gets zeros
            self = -1;
        } else {
            xi = x[3 * (size_t)self], yi = x[3 * (size_t)self + 1], zi = x[3 * (size_t)self + 2];
            if (JERK) vxi = v[3 * (size_t)self], vyi = v[3 * (size_t)self + 1], vzi = v[3 * (size_t)self + 2];
        }
    }

    const int j0 = split * j_per_split;
    const int j1 = min(n_j, j0 + j_per_split);
    double A0 = 0, A1 = 0, A2 = 0, P = 0, J0 = 0, J1 = 0, J2 = 0;
    for (int jt = j0; jt < j1; jt += kTileJ) {
        const int cnt = min(kTileJ, j1 - jt);
        __syncthreads();
        for (int t = threadIdx.x; t < cnt; t += kTileI) {
            const size_t j = (size_t)(jt + t);
            s_pm[t] = make_float4(x[3 * j], x[3 * j + 1], x[3 * j + 2], m[j]);
            if (JERK) s_vel[t] = make_float4(v[3 * j], v[3 * j + 1], v[3 * j + 2], 0.f);
        }
        __syncthreads();
        float ax = 0.f, ay = 0.f, az = 0.f, ps = 0.f, jx = 0.f, jy = 0.f, jz = 0.f;
#pragma unroll 4
        for (int t = 0; t < cnt; ++t) {
            const float4 pm = s_pm[t];
            const float dx = pm.x - xi, dy = pm.y - yi, dz = pm.z - zi;
            const float s = fmaf(dx, dx, fmaf(dy, dy, fmaf(dz, dz, eps2)));
            // own entry left out by index; with NBK_EPS0 so is any pair at distance 0 (L130-L132)
            const bool skip = (jt + t == self) || (eps0 && s == 0.f);
            const float rinv = skip ? 0.f : rsqrtf(s);
            const float rinv2 = rinv * rinv;
            const float mr = pm.w * rinv;     // m s^(-1/2)
            const float mr3 = mr * rinv2;     // m s^(-3/2)
            ps += mr;
            ax = fmaf(mr3, dx, ax), ay = fmaf(mr3, dy, ay), az = fmaf(mr3, dz, az);
            if (JERK) {
                const float4 vv = s_vel[t];
                const float wx = vv.x - vxi, wy = vv.y - vyi, wz = vv.z - vzi;
                const float rw = fmaf(dx, wx, fmaf(dy, wy, dz * wz));
                const float c = -3.f * rw * rinv2;  // -3 (r.w)/s
                jx = fmaf(mr3, fmaf(c, dx, wx), jx);
                jy = fmaf(mr3, fmaf(c, dy, wy), jy);
                jz = fmaf(mr3, fmaf(c, dz, wz), jz);
            }
        }
        A0 += ax, A1 += ay, A2 += az, P += ps, J0 += jx, J1 += jy, J2 += jz;
    }

    // partial row of (split, k) -- every thread of the CTA writes its own, dead lanes write zeros
    float4* row = reinterpret_cast<float4*>(rows + ((size_t)split * ni_pad + k) * kRowFloats);
    const bool on = live;
    __stcg(row, make_float4(on ? (float)A0 : 0.f, on ? (float)A1 : 0.f, on ? (float)A2 : 0.f, on ? (float)P : 0.f));
    __stcg(row + 1, make_float4(on ? (float)J0 : 0.f, on ? (float)J1 : 0.f, on ? (float)J2 : 0.f, 0.f));

    // the CTA that arrives last at this i-tile's counter adds the tile's rows (split-j sum)
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) s_last = (atomicAdd(&arrived[tile], 1u) == (unsigned)(n_split - 1));
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    if (k < n_i) {
        double a0 = 0, a1 = 0, a2 = 0, p = 0, q0 = 0, q1 = 0, q2 = 0;
        for (int sp = 0; sp < n_split; ++sp) {  // fixed order: the result does not depend on arrival order
            const float4* r = reinterpret_cast<const float4*>(rows + ((size_t)sp * ni_pad + k) * kRowFloats);
            const float4 u = __ldcg(r), w = __ldcg(r + 1);
            a0 += u.x, a1 += u.y, a2 += u.z, p += u.w, q0 += w.x, q1 += w.y, q2 += w.z;
        }
        if (acc) acc[3 * (size_t)k] = (float)a0, acc[3 * (size_t)k + 1] = (float)a1, acc[3 * (size_t)k + 2] = (float)a2;
        if (pot) pot[k] = (float)(-p);
        if (jerk) jerk[3 * (size_t)k] = (float)q0, jerk[3 * (size_t)k + 1] = (float)q1, jerk[3 * (size_t)k + 2] = (float)q2;
    }
    if (threadIdx.x == 0) arrived[tile] = 0u;  // leave the counter as the next call needs it
}

struct DeviceScratch {
    unsigned char* ptr = nullptr;  // device address of g_noalloc_scratch on this device
    int num_sms = 0;
};
DeviceScratch g_dev[kMaxDevices];
std::mutex g_dev_mutex;

// Device address of the scratch array on `device`, which must be the current device.  The symbol is
// looked up once per device: each device that loads the module has its own copy at its own address.
cudaError_t scratch_of(int device, DeviceScratch* out) {
    std::lock_guard<std::mutex> lock(g_dev_mutex);
    DeviceScratch& d = g_dev[device];
    if (!d.ptr) {
        void* p = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
        if (e != cudaSuccess) return e;
        int sms = 0;
        e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device);
        if (e != cudaSuccess) return e;
        d.num_sms = sms > 0 ? sms : 1;
        d.ptr = static_cast<unsigned char*>(p);
    }
    *out = d;
    return cudaSuccess;
}

struct CurrentDevice {  // make `dev` current for the call, put the caller's device back afterwards
    int prev = -1;
    cudaError_t err = cudaSuccess;
    explicit CurrentDevice(int dev) {
        err = cudaGetDevice(&prev);
        if (err != cudaSuccess) { prev = -1; return; }
        if (prev != dev) err = cudaSetDevice(dev);
    }
    ~CurrentDevice() {
        int cur = -1;
        if (prev >= 0 && cudaGetDevice(&cur) == cudaSuccess && cur != prev) cudaSetDevice(prev);
    }
};

int fail(int* cuda_error, cudaError_t e) {
    if (cuda_error) *cuda_error = static_cast<int>(e);
    cudaGetLastError();  // leave no sticky launch error behind for the caller's next CUDA call
    return NBK_ECUDA;
}

}  // namespace

extern "C" int nbk_calc_noalloc_dev(int device, void* cuda_stream, int64_t n_j, const float* m,
                                    const float* x, const float* v, int64_t n_i,
                                    const int32_t* i_index, float eps2, uint32_t flags, float* acc,
                                    float* jerk, float* pot, int* cuda_error) {
    if (cuda_error) *cuda_error = 0;
    if (device < 0 || device >= kMaxDevices || n_j < 0 || n_i < 0) return NBK_EINVAL;
    if (!(eps2 >= 0.f) || std::isinf(eps2)) return NBK_EINVAL;
    if (flags & ~(NBK_JERK | NBK_POT | NBK_EPS0)) return NBK_EINVAL;  // NBK_NN: use a context
    if (n_i > NBK_NOALLOC_MAX_NI || n_j > NBK_NOALLOC_MAX_NJ) return NBK_ERANGE;
    const bool want_jerk = (flags & NBK_JERK) != 0;
    if (n_j > 0 && (!m || !x || (want_jerk && !v))) return NBK_EINVAL;
    if (n_i == 0) return NBK_OK;
    // the kernels flush subnormals: a subnormal eps2 is eps2 = 0 and needs the zero-distance mask too
    if (eps2 < 1.17549435e-38f) eps2 = 0.f;
    const int eps0 = ((flags & NBK_EPS0) || eps2 == 0.f) ? 1 : 0;

    CurrentDevice cur(device);
    if (cur.err != cudaSuccess) return fail(cuda_error, cur.err);
    DeviceScratch sc;
    cudaError_t e = scratch_of(device, &sc);
    if (e != cudaSuccess) return fail(cuda_error, e);
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    float* rows = reinterpret_cast<float*>(sc.ptr);
    unsigned* arrived = reinterpret_cast<unsigned*>(sc.ptr + kRowsBytes);

    // launch shape: enough (i-tile, j-split) CTAs for four per SM, j-splits of whole tiles
    const int tiles_i = static_cast<int>((n_i + kTileI - 1) / kTileI);
    const long long tiles_j = (n_j + kTileJ - 1) / kTileJ;
    long long n_split = (4LL * sc.num_sms + tiles_i - 1) / tiles_i;
    if (n_split > kMaxSplit) n_split = kMaxSplit;
    if (n_split > tiles_j) n_split = tiles_j;
    if (n_split < 1) n_split = 1;
    const long long j_per_split = tiles_j > 0 ? (tiles_j + n_split - 1) / n_split * kTileJ : kTileJ;
    n_split = n_j > 0 ? (n_j + j_per_split - 1) / j_per_split : 1;

    e = cudaMemsetAsync(arrived, 0, kCounterBytes, stream);  // counters start every call at zero
    if (e != cudaSuccess) return fail(cuda_error, e);
    if (!want_jerk && jerk) {  // same convention as lasthalf: no NBK_JERK, jerk reads zero
        e = cudaMemsetAsync(jerk, 0, sizeof(float) * 3 * static_cast<size_t>(n_i), stream);
        if (e != cudaSuccess) return fail(cuda_error, e);
    }
    const dim3 grid(static_cast<unsigned>(tiles_i), static_cast<unsigned>(n_split));
    if (want_jerk)
        noalloc_force_kernel<true><<<grid, kTileI, 0, stream>>>(
            m, x, v, static_cast<int>(n_j), i_index, static_cast<int>(n_i), eps2, eps0,
            static_cast<int>(n_split), static_cast<int>(j_per_split), rows, arrived, acc, jerk, pot);
    else
        noalloc_force_kernel<false><<<grid, kTileI, 0, stream>>>(
            m, x, nullptr, static_cast<int>(n_j), i_index, static_cast<int>(n_i), eps2, eps0,
            static_cast<int>(n_split), static_cast<int>(j_per_split), rows, arrived, acc, nullptr, pot);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(cuda_error, e);
    return NBK_OK;
}
