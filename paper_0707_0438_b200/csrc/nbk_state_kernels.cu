// nbk_state_kernels.cu -- a1 (set_j scatter) and a3 (Hermite predictor) kernels and their launchers.
#include "nbk_device.cuh"

namespace nbk {

// ------------------------------------------------------------------ scatter (a1) / predict (a3)
template <typename T>
__global__ void scatter_kernel(const ScatterArgs s, const RawJ raw) {
    pdl_trigger();
    pdl_wait();
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

// Hermite predictor (reading R8): predict_one, nbk_device.cuh
__global__ void predict_kernel(const RawJ raw, double t, long long n_j, long long n_pad, float* px,
                               float* py, float* pz, float* pm, float* pvx, float* pvy,
                               float* pvz) {
    pdl_trigger();
    pdl_wait();
    const long long j = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (j >= n_pad) return;
    // padding (n_j <= j < n_pad): massless and far away, so that it is nobody's neighbour
    float o[7] = {1e18f, 1e18f, 1e18f, 0.f, 0.f, 0.f, 0.f};
    if (j < n_j) predict_one(raw, j, t, o);
    px[j] = o[0]; py[j] = o[1]; pz[j] = o[2]; pm[j] = o[3];
    pvx[j] = o[4]; pvy[j] = o[5]; pvz[j] = o[6];
}

// The same predictor with a pending set_j of a few particles folded in (a1 + a3 in one launch):
// the thread that owns an updated address stores the new raw state and predicts from it.
__global__ void predict_upd_kernel(const RawJ raw, double t, long long n_j, long long n_pad,
                                   float* px, float* py, float* pz, float* pm, float* pvx,
                                   float* pvy, float* pvz, const InlineJ upd) {
    pdl_trigger();
    pdl_wait();
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


__global__ void scatter_inline_kernel(const InlineJ p, const RawJ raw) {
    pdl_trigger();
    pdl_wait();
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
    return launch_pdl(scatter_inline_kernel, 1, kInlineMaxJ, 0, st, p, raw);
}

cudaError_t launch_scatter(const ScatterArgs& s, const RawJ& raw, cudaStream_t st) {
    if (s.n <= 0) return cudaSuccess;
    const unsigned grid = static_cast<unsigned>((s.n + 255) / 256);
    if (s.f64) return launch_pdl(scatter_kernel<double>, grid, 256, 0, st, s, raw);
    return launch_pdl(scatter_kernel<float>, grid, 256, 0, st, s, raw);
}

cudaError_t launch_predict(const RawJ& raw, double t, long long n_j, long long n_pad, float* px,
                           float* py, float* pz, float* pm, float* pvx, float* pvy, float* pvz,
                           const InlineJ* upd, cudaStream_t st) {
    if (n_pad <= 0) return cudaSuccess;
    const unsigned grid = static_cast<unsigned>((n_pad + 255) / 256);
    if (upd && upd->n > 0)
        return launch_pdl(predict_upd_kernel, grid, 256, 0, st, raw, t, n_j, n_pad, px, py, pz, pm, pvx, pvy,
                          pvz, *upd);
    return launch_pdl(predict_kernel, grid, 256, 0, st, raw, t, n_j, n_pad, px, py, pz, pm, pvx, pvy, pvz);
}


}  // namespace nbk
