// nbk_hermite_dev.cu -- nbk_hermite_evolve_dev: the Hermite block-step loop resident on the device
// (SURVEY.md 8(f)-1).  Host side only: state upload, CUDA-graph replay of the rounds (persistent stepping
// kernel + the chain of launches for the large steps), termination check; the kernels are in
// nbk_hermite_steps.cu and nbk_hermite_kernels.cu.
#include <chrono>
#include <climits>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <vector>

#include "nbk_ctx.cuh"

using namespace nbk;

namespace {
inline long long round_up_ll(long long a, long long b) { return (a + b - 1) / b * b; }
}  // namespace

extern "C" {
// ---- a8 on the device: the whole block-step loop without host round trips ----
int nbk_hermite_evolve_dev(nbk_ctx* c, int64_t n, const double* m, double* x, double* v, double eps,
                           double t_end, double eta, double dt_max, nbk_hermite_stats* stats) {
    if (!c || n < 1 || !m || !x || !v || !(eps >= 0.0) || !(t_end >= 0.0) || !(eta > 0.0) ||
        !(dt_max > 0.0) || n > INT32_MAX)
        return NBK_EINVAL;
    if (n > c->n_max || n > c->ni_max) return NBK_ERANGE;
    const int kmin = level_of_dt_max(dt_max);   // dt_max rounded down to a power of two
    if (kmin < 0) return NBK_EINVAL;            // dt_max in [2^-48, 2)
    const double dtm = std::ldexp(1.0, -kmin);
    if (t_end > 2047.0 || std::fmod(t_end, dtm) != 0.0) return NBK_EINVAL;
    DeviceGuard g(c->device);
    if (!g.ok) return cuda_fail(c, cudaErrorInvalidDevice);
    const auto wall0 = std::chrono::steady_clock::now();
    const size_t N = static_cast<size_t>(n);
    const float eps2 = flushed_eps2(static_cast<float>(eps * eps));
    const uint32_t flags = NBK_JERK | NBK_POT;
    int rc;

    if (c->hs_cap < n) {
        cudaFree(c->hs.x); cudaFree(c->hs.v); cudaFree(c->hs.a); cudaFree(c->hs.j);
        cudaFree(c->hs.level); cudaFree(c->hs.act); cudaFree(c->hs.bc_ge); cudaFree(c->hs.flag); cudaFree(c->hs.rows);
        c->hs = HermiteState{};
        c->hs_rows_bytes = 0;
        c->hs_cap = 0;
        NBK_CUDA(c, cudaMalloc(&c->hs.x, sizeof(double) * 3 * N));
        NBK_CUDA(c, cudaMalloc(&c->hs.v, sizeof(double) * 3 * N));
        NBK_CUDA(c, cudaMalloc(&c->hs.a, sizeof(double) * 3 * N));
        NBK_CUDA(c, cudaMalloc(&c->hs.j, sizeof(double) * 3 * N));
        NBK_CUDA(c, cudaMalloc(&c->hs.level, (N + 15) / 16 * 16));
        NBK_CUDA(c, cudaMalloc(&c->hs.act, sizeof(int32_t) * N));
        NBK_CUDA(c, cudaMalloc(&c->hs.bc_ge, sizeof(int) * (kMaxLevel + 1) * ((N + 255) / 256)));
        NBK_CUDA(c, cudaMalloc(&c->hs.flag, sizeof(unsigned long long) * kStepsMaxAct));
        NBK_CUDA(c, cudaMemset(c->hs.flag, 0, sizeof(unsigned long long) * kStepsMaxAct));
        c->hs_cap = n;
    }
    if (!c->d_hdr) NBK_CUDA(c, cudaMalloc(&c->d_hdr, sizeof(DynHeader)));
    if (!c->h_hdr) NBK_CUDA(c, cudaMallocHost(&c->h_hdr, sizeof(DynHeader)));

    int env_max_act = -1;   // test knob NBK_STEPS_MAX_ACT (include/nbk.h): a whole number 0..kStepsMaxAct, else NBK_EINVAL
    if (const char* e = std::getenv("NBK_STEPS_MAX_ACT")) {
        char* end = nullptr;
        const long val = std::strtol(e, &end, 10);
        if (end == e || *end != '\0' || val < 0 || val > kStepsMaxAct) return NBK_EINVAL;
        env_max_act = static_cast<int>(val);
    }

    // t = 0 through the ordinary entry points: forces on everybody, first steps (reading R15)
    std::vector<float> fa(3 * N), fj(3 * N);
    std::vector<double> a(3 * N), jk(3 * N), tl(N, 0.0);
    std::vector<unsigned char> lev((N + 15) / 16 * 16, 0);   // k + 1
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
        const int k = startup_level(std::sqrt(na), std::sqrt(nj), eta, kmin);
        lev[i] = static_cast<unsigned char>(k + 1);
        H.level_count[k] += 1;
    }
    const int nblk = static_cast<int>((N + 255) / 256);
    c->hs.nblk = nblk;
    std::vector<int> bc(static_cast<size_t>(kMaxLevel + 1) * nblk, 0);
    for (size_t i = 0; i < N; ++i)
        for (int l = 0; l < lev[i]; ++l) bc[static_cast<size_t>(l) * nblk + (i >> 8)] += 1;
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
    NBK_CUDA(c, cudaMemcpyAsync(c->hs.level, lev.data(), lev.size(), cudaMemcpyHostToDevice, c->stream));
    NBK_CUDA(c, cudaMemcpyAsync(c->hs.bc_ge, bc.data(), sizeof(int) * bc.size(), cudaMemcpyHostToDevice, c->stream));

    // Block steps of up to max_act due particles run inside the persistent stepping kernel
    // (nbk_hermite_steps.cu); it returns at the first larger step, which the chain of launches
    // hd_begin -> hd_predict -> force (I = 1 or 4, the device planner's choice) -> reduce -> hd_correct
    // takes; then the stepping kernel again.  One graph holds kIterPerGraph such rounds; they are enqueued
    // in batches with no host synchronisation inside a batch, and rounds past t_end return at once.
    const int G = H.num_sms;
    int max_act = kStepsMaxAct;
    if (env_max_act >= 0) max_act = env_max_act;
    if (max_act > kStepsMaxAct) max_act = kStepsMaxAct;
    if (max_act > G * (kStepsThreads / 32)) max_act = G * (kStepsThreads / 32);   // one due particle per warp
    const int chunk = static_cast<int>(round_up_ll((n + G - 1) / G, 4));
    const int n_lev = static_cast<int>(round_up_ll(n, 16 * kStepsThreads));
    if (steps_smem_bytes(chunk, n_lev) > 220 * 1024 || n_lev / (16 * kStepsThreads) > kStepsMaxVec) max_act = 0;   // does not fit one SM: chain of launches only
    if (max_act > 0) {
        int per_sm = 0;
        NBK_CUDA(c, steps_prepare(chunk, n_lev, &per_sm));
        if (per_sm < 1) max_act = 0;
    }
    if (max_act > 0) {   // the stepping kernel's rows: its own buffer, zeroed once (tags only grow, hs_seq)
        const size_t need = static_cast<size_t>(G) * max_act * 8 * sizeof(unsigned long long);
        if (c->hs_rows_bytes < need) {
            cudaFree(c->hs.rows);
            c->hs.rows = nullptr;
            c->hs_rows_bytes = 0;
            NBK_CUDA(c, cudaMalloc(&c->hs.rows, need));
            NBK_CUDA(c, cudaMemsetAsync(c->hs.rows, 0, need, c->stream));
            c->hs_rows_bytes = need;
        }
    }
    if (c->hs_seq >= (1u << 31)) {   // 32-bit tags: start over long before they wrap (a zeroed word = no step yet;
                                     // one call would need more than 2^31 steps to wrap by itself)
        if (c->hs.rows) NBK_CUDA(c, cudaMemsetAsync(c->hs.rows, 0, c->hs_rows_bytes, c->stream));
        NBK_CUDA(c, cudaMemsetAsync(c->hs.flag, 0, sizeof(unsigned long long) * kStepsMaxAct, c->stream));
        c->hs_seq = 0;
    }
    H.steps_max_act = max_act;
    H.seq = c->hs_seq;
    NBK_CUDA(c, cudaMemcpyAsync(c->d_hdr, &H, sizeof(H), cudaMemcpyHostToDevice, c->stream));
    NBK_CUDA(c, cudaStreamSynchronize(c->stream));   // the host vectors above may go away

    Variant v1{1, true, eps2 == 0.f, false}, v4{4, true, eps2 == 0.f, false};
    const long long n_pad = round_up_ll(n, kTileJMax);
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
    r.sum64 = nullptr;
    r.n_j = static_cast<int>(n);
    StepsArgs sa;
    sa.raw = c->raw;
    sa.h = c->d_hdr;
    sa.hs = c->hs;
    sa.eps2 = eps2;
    sa.chunk = chunk;
    sa.n_lev = n_lev;
    sa.max_act = max_act;
    sa.max_steps = 1 << 20;
    auto enqueue_round = [&](bool cooperative) -> cudaError_t {
        cudaError_t e;
        if (max_act > 0 && (e = launch_hd_steps(sa, eps2 == 0.f, G, cooperative, c->stream)) != cudaSuccess) return e;
        if ((e = launch_hd_begin(c->d_hdr, c->stream)) != cudaSuccess) return e;
        if ((e = launch_hd_predict(c->raw, c->d_hdr, c->hs, n_pad, pred_arr(c, 0), pred_arr(c, 1),
                                   pred_arr(c, 2), pred_arr(c, 3), pred_arr(c, 4), pred_arr(c, 5),
                                   pred_arr(c, 6), c->stream)) != cudaSuccess) return e;
        // without the stepping kernel the planner may pick I = 1: both forms are launched, one returns at once
        if (max_act == 0 && (e = launch_force_dyn(v1, f, c->stream)) != cudaSuccess) return e;
        if ((e = launch_force_dyn(v4, f, c->stream)) != cudaSuccess) return e;
        if ((e = launch_reduce_dyn(v1, r, static_cast<int>(n), c->stream)) != cudaSuccess) return e;
        return launch_hd_correct(c->raw, c->d_hdr, c->hs, f.tail.acc, f.tail.jerk,
                                 static_cast<int>(n), c->stream);
    };
    // inside a graph consecutive kernels are joined by programmatic dependent-launch edges
    // (nbk_kernels.cuh), between graph launches the stream serialises fully
    const int kIterPerGraph = 8, kGraphsPerBatch = 32;
    cudaGraph_t graph = nullptr;
    cudaGraphExec_t gexec = nullptr;
    cudaError_t ce = cudaSuccess;
    for (int attempt = 0; attempt < 2; ++attempt) {   // cooperative launch of the stepping kernel, else plain
        const bool cooperative = attempt == 0;
        NBK_CUDA(c, cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeRelaxed));
        ce = cudaSuccess;
        for (int s = 0; s < kIterPerGraph && ce == cudaSuccess; ++s) ce = enqueue_round(cooperative);
        cudaError_t ce2 = cudaStreamEndCapture(c->stream, &graph);
        if (ce == cudaSuccess) ce = ce2;
        if (ce == cudaSuccess) ce = cudaGraphInstantiate(&gexec, graph, 0);
        if (ce == cudaSuccess) {
            // nbk_last_launch after this call: out[0] CTAs of the stepping kernel (0: off), out[1] its threads,
            // out[7] 2 = captured as a cooperative launch (co-residency checked by the driver), 1 = plain launch
            // (co-residency by construction: one CTA per SM, occupancy checked in steps_prepare), 0 = no stepping kernel
            c->last_launch[0] = max_act > 0 ? G : 0;
            c->last_launch[1] = max_act > 0 ? kStepsThreads : 0;
            c->last_launch[2] = 0; c->last_launch[3] = 0; c->last_launch[4] = max_act;
            c->last_launch[5] = G; c->last_launch[6] = 0;
            c->last_launch[7] = max_act > 0 ? (cooperative ? 2 : 1) : 0;
            break;
        }
        if (graph) cudaGraphDestroy(graph);
        graph = nullptr;
        gexec = nullptr;
        (void)cudaGetLastError();
        if (max_act == 0) break;
    }
    if (ce != cudaSuccess) return cuda_fail(c, ce);
    for (;;) {
        for (int s = 0; s < kGraphsPerBatch && ce == cudaSuccess; ++s) ce = cudaGraphLaunch(gexec, c->stream);
        if (ce == cudaSuccess)
            ce = cudaMemcpyAsync(c->h_hdr, c->d_hdr, sizeof(DynHeader), cudaMemcpyDeviceToHost, c->stream);
        if (ce == cudaSuccess) ce = cudaStreamSynchronize(c->stream);
        if (ce != cudaSuccess || c->h_hdr->done || c->h_hdr->error) break;
    }
    c->hs_seq = c->h_hdr->seq;   // tags of the stepping kernel's rows and flags never repeat in this context
    cudaGraphExecDestroy(gexec);
    cudaGraphDestroy(graph);
    if (ce != cudaSuccess) return cuda_fail(c, ce);
    if (c->h_hdr->error) {   // a wait inside the stepping kernel gave up: its tags are not to be trusted again
        c->hs_seq = c->h_hdr->seq + (1u << 24);
        if (c->h_hdr->error == 2) return NBK_ERANGE;   // no launch plan fits this context's partial rows
        return cuda_fail(c, cudaErrorLaunchTimeout);
    }
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

}  // extern "C"
