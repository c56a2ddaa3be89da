// nbk_ctx.cuh -- the context behind the C ABI and the helpers shared by the host-side sources
// (nbk_api.cu, nbk_hermite_dev.cu, nbk_batch.cu).  Internal; not part of include/nbk.h.
#pragma once
#include <cuda_runtime.h>

#include <cstdint>

#include "../../include/nbk.h"
#include "nbk_kernels.cuh"

namespace nbk {


inline long long round_up(long long a, long long b) { return (a + b - 1) / b * b; }

// The kernels' arithmetic flushes subnormals to zero (.ftz): a subnormal eps2 IS eps2 = 0 to them, so
// it must select the zero-distance mask like an exact 0 does.
inline float flushed_eps2(float eps2) { return eps2 < 1.17549435e-38f ? 0.f : eps2; }

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


}  // namespace nbk

struct nbk_ctx {
    int device = 0;
    cudaStream_t stream = nullptr;
    bool own_stream = false;
    bool caller_workspace = false;  // device buffers of nbk_open live in the caller's workspace
    long long n_max = 0, ni_max = 0, n_cap = 0;
    int num_sms = 0;

    nbk::RawJ raw{};
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
    bool small_ready = false;            // small_block_kernel's shared-memory limit has been raised
    nbk::HermiteState hs{};              // device-resident integrator state (allocated on first use)
    long long hs_cap = 0;
    unsigned hs_seq = 0;                 // steps the stepping kernel has taken in this context (tags of its rows and flags)
    size_t hs_rows_bytes = 0;
    nbk::DynHeader* d_hdr = nullptr;
    nbk::DynHeader* h_hdr = nullptr;     // pinned
    bool host_has_result = false;   // the last firsthalf wrote h_result itself (no D2H needed)
    volatile unsigned* h_seq = nullptr;  // mapped word behind h_result: small_block_kernel's "results are in host memory" mark
    unsigned* h_seq_dev = nullptr;
    unsigned small_seq = 0;              // value the last small-block launch writes there
    bool poll_result = false;            // lasthalf may poll h_seq instead of synchronising the stream
    nbk::InlineJ pending;                // a small set_j not yet on the device (pending.n == 0: none)

    unsigned char* h_stage = nullptr;  // pinned staging for set_j
    unsigned char* d_stage = nullptr;
    size_t stage_bytes = 0;
    cudaEvent_t stage_free = nullptr;  // recorded after the H2D that reads h_stage
    unsigned char* h_istage = nullptr;  // pinned staging for i_index / xi / vi
    cudaEvent_t istage_free = nullptr;

    long long last_ni = -1;
    bool in_flight = false;
    int force_I = 0;
    bool fused_ok = true;  // nbk_set_variant bit 8 switches the one-launch small-block path off
    int last_cuda = 0;
    long long last_launch[8] = {0, 0, 0, 0, 0, 0, 0, 0};

    bool timing = false;
    cudaEvent_t ev[4][2];
    bool ev_used[4] = {false, false, false, false};
};


namespace nbk {

int cuda_fail(nbk_ctx* c, cudaError_t e);

#define NBK_CUDA(c, call)                                        \
    do {                                                         \
        cudaError_t e__ = (call);                                \
        if (e__ != cudaSuccess) return nbk::cuda_fail((c), e__); \
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

inline float* pred_arr(const nbk_ctx* c, int k) { return c->pred + static_cast<size_t>(k) * c->n_cap; }
JPred jpred_of(const nbk_ctx* c);
// A pending small set_j goes to the device on its own (before anything else touches the raw state).
int flush_pending(nbk_ctx* c);

}  // namespace nbk
