// nbk_kernels.cuh -- launch-side declarations shared by the kernel sources (nbk_force.cu, nbk_*_kernels.cu)
// and the host sources (nbk_api.cu, nbk_hermite_dev.cu, nbk_batch.cu).
// Internal to the CUDA path; nothing here is part of the C ABI (include/nbk.h).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "nbk_hermite_common.h"

namespace nbk {

constexpr int kTileJMax = 256;  // largest j-tile (particles); ring slots are sized for it
constexpr int kStages = 6;      // tile ring depth
constexpr int kPrefetch = 4;    // tiles the producer runs ahead (kStages - kPrefetch = drift slack)
constexpr int kMaxI = 4;        // max i-particles per thread
constexpr int kMaxRowI = 1024;  // max (warps * 32 * I): i-rows one CTA writes per (segment)
constexpr int kMaxCtas = 256;   // max CTAs of a force launch (one per SM; B200 has 148)

// ---- programmatic dependent launch (sm_90+).  A block step is a chain of short kernels (predict ->
// force -> reduce -> correct): each kernel of the chain is launched with programmatic stream
// serialisation, lets its successor be scheduled as soon as all of its own CTAs are resident
// (pdl_trigger at entry) and waits for its predecessor's completion and memory flush before it
// touches global memory (pdl_wait).  That hides the launch and CTA-scheduling latency between
// dependent kernels (2-3 us per edge), which is what a small block step is made of.
// Without the launch attribute both instructions do nothing.  NBK_PDL=0 in the environment turns
// the attribute off.
bool pdl_enabled();
#ifdef __CUDACC__
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kernel)(KArgs...), unsigned grid, unsigned block, size_t smem,
                              cudaStream_t s, Args&&... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid, 1, 1);
    cfg.blockDim = dim3(block, 1, 1);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = pdl_enabled() ? 1 : 0;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}
#endif

// warps per CTA for each i-per-thread count: one CTA per SM, registers decide the warp count
__host__ __device__ constexpr int warps_of(int I) { return I == 4 ? 8 : (I == 2 ? 12 : 16); }

// Predicted j-state, structure of arrays, each padded to a multiple of kTileJMax with m = 0.
struct JPred {
    const float* x;
    const float* y;
    const float* z;
    const float* m;
    const float* vx;
    const float* vy;
    const float* vz;
};

// Work decomposition ("stream-K" over the (i-tile, j-tile) pair list, i-major):
// pair p = it * njt + jt;  CTA k owns pairs [k*P/G, (k+1)*P/G).
struct Decomp {
    int n_i;          // active i-particles
    int n_j;          // j-particles (unpadded)
    int ti;           // i-particles per CTA tile = (W / wj) * 32 * I
    int tj;           // j-particles per tile (64, 128 or 256)
    int wj;           // warps that split each j-tile; W / wj warps split the i-tile
    int nit;          // i-tiles
    int njt;          // j-tiles
    long long P;      // nit * njt
    int G;            // CTAs
    int maxseg;       // max i-tiles one CTA touches
};

struct Variant {
    int I;        // 1, 2 or 4
    bool jerk;
    bool eps0;
    bool nn;      // nearest neighbour too (instantiated for the jerk forms only)
};

// Planner for one i-per-thread count I: choose wj and tj and cut the pair list.  Runs on the host
// (plan_shape tries I = 4, 2, 1) and on the device (the device-resident integrator plans its own
// block steps with I = 1).  Cost of a candidate = pairs per CTA x (j-steps per warp per pair x I +
// per-tile work); returns it, or -1 if no candidate fits max_partial_floats.
constexpr int kPlanCandidates = 15;   // wj in {1,2,4,8,16} x tj in {256,128,64}
__host__ __device__ inline long long plan_candidate(long long n_i, long long n_j, int num_sms, int I,
                                                    unsigned long long max_partial_floats, int c,
                                                    Decomp* d) {
    const int W = warps_of(I);
    const int wj = 1 << (c / 3), tj = 256 >> (c % 3);
    if (wj > W || W % wj || tj / wj < 4) return -1;
    const long long ti = static_cast<long long>(W / wj) * 32 * I;
    const long long nit = (n_i + ti - 1) / ti;
    const long long njt = (n_j + tj - 1) / tj;
    const long long P = nit * njt;
    const long long gmax = num_sms < kMaxCtas ? num_sms : kMaxCtas;
    const long long G = P < gmax ? P : gmax;
    const long long per = (P + G - 1) / G;
    const long long maxseg = (per - 1 + njt - 1) / njt + 1;
    if (static_cast<unsigned long long>(G) * maxseg * ti * 8 > max_partial_floats) return -1;
    d->n_i = static_cast<int>(n_i);
    d->n_j = static_cast<int>(n_j);
    d->ti = static_cast<int>(ti);
    d->tj = tj;
    d->wj = wj;
    d->nit = static_cast<int>(nit);
    d->njt = static_cast<int>(njt);
    d->P = P;
    d->G = static_cast<int>(G);
    d->maxseg = static_cast<int>(maxseg);
    return per * (static_cast<long long>(tj / wj) * I + 6 * I + 24);
}

__host__ __device__ inline long long plan_fixed_i(long long n_i, long long n_j, int num_sms, int I,
                                                  unsigned long long max_partial_floats, Decomp* d) {
    long long best = -1;
    for (int c = 0; c < kPlanCandidates; ++c) {   // first of the cheapest wins
        Decomp cand;
        const long long cost = plan_candidate(n_i, n_j, num_sms, I, max_partial_floats, c, &cand);
        if (cost >= 0 && (best < 0 || cost < best)) {
            best = cost;
            *d = cand;
        }
    }
    return best;
}

// Host planner (nbk_api.cu): the best of I = 4, 2, 1 (cost x warps / measured speed of that form).
// force_I > 0 pins I.  Fills *v (I only; flags are the caller's) and *d; d->G stays untouched if no
// candidate fits max_partial_floats.
void plan_shape(long long n_i, long long n_j, int num_sms, int force_I, size_t max_partial_floats,
                Variant* v, Decomp* d);
// Floats of partial storage a plan needs, and the bound nbk_open allocates for (ni_max, num_sms).
size_t plan_partial_floats(const Decomp& d);
size_t plan_partial_floats_bound(long long ni_max, int num_sms);

// ---- device-resident Hermite integrator: all block-step state lives here ------
// kTickLog2 (time unit 2^-52) and kMaxLevel (finest step 2^-48): nbk_hermite_common.h
struct DynHeader {
    long long T_now, T_end, T_next;     // block times in ticks
    double t_next;                      // T_next in time units
    int kstar;                          // particles with level >= kstar are due at T_next
    int n_act;                          // how many (from the level counts)
    int done;                           // T_next would pass T_end: every kernel returns at once
    int kmin;                           // coarsest level (dt_max = 2^-kmin)
    int n;                              // particles
    int num_sms;
    unsigned long long max_partial_floats;
    double eta;
    long long block_steps, particle_steps, interactions;
    long long level_count[kMaxLevel + 1];
    long long hist[32];
    Decomp plan;                        // launch plan of the current step (made once, hd_begin_kernel)
    int plan_I;                         // i-particles per thread of that plan: which force kernel runs
    int fused;                          // the force kernel's last CTA reduces (small block)
    int skip;                           // this step is left to hd_steps_kernel: the launched chain returns
    int steps_max_act;                  // hd_steps_kernel takes steps of up to this many due particles (0: off)
    int error;                          // 1: a wait of hd_steps_kernel on another CTA's tagged rows / flags gave up; 2: hd_begin_kernel found no launch plan that fits
    unsigned seq;                       // hd_steps_kernel: steps it has taken so far
};
struct HermiteState {        // fp64 integrator state, [n][3] row-major; level[n]
    double* x;
    double* v;
    double* a;
    double* j;
    unsigned char* level;    // [n rounded up to 16] step level k (dt = 2^-k) of every particle as k + 1, 0 beyond n
    int32_t* act;            // [n] indices of the particles due at T_next, ascending
    int* bc_ge;              // [kMaxLevel + 1][nblk]: particles of index block b (256 indices) with
                             // level >= k; gives each block its offset into act without a scan
    int nblk;
    unsigned long long* flag;  // [kStepsMaxAct] stepping kernel: (step number << 32 | new level) of each particle of the last step
    unsigned long long* rows;  // [ctas][max_act][8] stepping kernel: partial rows, (step number << 32 | value bits)
};

constexpr int kFusedMaxI = 32;  // largest i-block served by the one-launch small-block path

// Small-block tail (n_i <= kFusedMaxI, one i-tile, I = 1): the last CTA to finish sums the partial
// rows itself (fixed order) and writes the results, so a block step is one launch; the i-indices
// travel in the kernel parameters and the results can go straight to mapped host memory.
struct FusedTail {
    int enabled;                   // 0: partial rows only, reduce_kernel follows
    int inline_index;              // 1: i-indices are i_inline[], not ForceArgs::i_index
    int32_t i_inline[kFusedMaxI];
    unsigned* counter;             // device, zero between launches (the last CTA resets it)
    float* acc;                    // device result [n_i][3]
    float* jerk;                   // device result [n_i][3]
    float* pot;                    // device result [n_i]
    float* host_out;               // mapped pinned copy acc|jerk|pot (7 n_i floats) or nullptr
};

struct ForceArgs {
    JPred j;
    const int32_t* i_index;  // [n_i] or nullptr (identity)
    const float* xi;         // [n_i][3] or nullptr
    const float* vi;         // [n_i][3] or nullptr
    float* partial;          // [k*maxseg+seg][ti][8]
    float2* nn_partial;      // [k*maxseg+seg][ti] (smallest s, its j-tile as int bits); NN only
    int32_t* nn_index;       // [n_i] results of the nearest-neighbour search (NN only)
    float* nn_r2;            // [n_i]
    float eps2;
    Decomp d;
    FusedTail tail;
    const DynHeader* dyn;    // DYN instantiations: n_i and the launch plan come from the device
};

struct ReduceArgs {
    int it_first[kMaxCtas];  // first / last i-tile CTA k works on (host-filled from the pair split)
    int it_last[kMaxCtas];
    const float* partial;
    const float2* nn_partial;  // NN only
    float* nn_best;            // [n_i] smallest s over all rows (NN only)
    int32_t* nn_tile;          // [n_i] its j-tile
    float* acc;   // [n_i][3]
    float* jerk;  // [n_i][3]
    float* pot;   // [n_i]
    double* sum64;  // nullable [n_i][8]: the fp64 sums before rounding (acc3, -pot, jerk3, 0): j-shards
    Decomp d;
    const DynHeader* dyn;    // non-null: plan on the device (and return if the force kernel reduced)
    int n_j;                 // dyn only
};

struct RawJ {        // raw j-state kept for the predictor, structure of arrays of capacity cap
    double* x;       // [3][cap]
    float* v;        // [3][cap]
    float* a;        // [3][cap]
    float* k;        // [3][cap]  (jerk)
    float* m;        // [cap]
    double* t;       // [cap]
    long long cap;
};

size_t force_smem_bytes(const Variant& v);
// Raises the dynamic shared-memory limit of the instantiation and checks that one CTA fits an SM.
cudaError_t force_prepare(const Variant& v);
cudaError_t launch_force(const Variant& v, const ForceArgs& a, cudaStream_t s);
// DYN instantiation (I = 1 or 4, acc + jerk + pot): the plan and n_i come from a.dyn on the device
cudaError_t launch_force_dyn(const Variant& v, const ForceArgs& a, cudaStream_t s);
cudaError_t launch_reduce(const Variant& v, const ReduceArgs& a, cudaStream_t s);
// Nearest neighbour, second step for the two-kernel path: one warp per i re-scans the winning tile.
struct NnScanArgs {
    JPred j;
    const int32_t* i_index;
    const float* xi;
    const float* nn_best;
    const int32_t* nn_tile;
    int32_t* nn_index;
    float* nn_r2;
    int n_i, n_j, tj;
    float eps2;
};
cudaError_t launch_nn_scan(const NnScanArgs& a, cudaStream_t s);

// j-sharding over several GPUs: nbk_shard_kernels.cu
struct ShardGatherArgs {
    JPred j;                  // this rank's predicted j-state (addresses are local)
    const int32_t* i_global;  // [n_i] global j address of each i-particle
    int32_t* i_local;         // [n_i] out: address in this shard, or -1 if another rank owns it
    float* xv;                // [n_i][8] out: x y z 0 vx vy vz 0 of owned i-particles, 0 elsewhere
    long long n_i;
    long long j0;             // global address of local address 0
    long long n_local;
};
cudaError_t launch_shard_gather(const ShardGatherArgs& a, cudaStream_t s);
cudaError_t launch_shard_split(const float* xv, long long n_i, float* xi, float* vi, cudaStream_t s);
cudaError_t launch_shard_finish(const double* sum64, long long n_i, float* acc, float* jerk,
                                float* pot, cudaStream_t s);
// The same two exchanges over peer memory (NVLink P2P loads from the other ranks' symmetric buffers)
// instead of NCCL collectives: ptr[r] is rank r's buffer as mapped into this process.
constexpr int kMaxPeers = 16;
struct ShardPeers {
    const void* ptr[kMaxPeers];
    long long begin[kMaxPeers + 1];   // shard r owns global addresses [begin[r], begin[r+1]) (fetch only)
    int world;
};
cudaError_t launch_shard_fetch(const ShardPeers& peers, const int32_t* i_global, long long n_i,
                               float* xv, cudaStream_t s);
cudaError_t launch_shard_combine(const ShardPeers& peers, long long n_i, float* acc, float* jerk,
                                 float* pot, cudaStream_t s);

// set_j scatter: staged particles -> raw SoA at addr (nullptr: identity).  x, v as fp32 or fp64.
struct ScatterArgs {
    long long n;
    const int32_t* addr;
    const double* tj;
    const void* m;      // float or double
    const void* x;      // [n][3] float or double
    const void* v;      // may be nullptr
    const void* a;      // may be nullptr
    const void* k;      // may be nullptr
    int f64;            // 1: m, x, v, a, k are double
    long long n_max;    // addresses outside [0, n_max) are skipped
};
cudaError_t launch_scatter(const ScatterArgs& s, const RawJ& raw, cudaStream_t st);

// set_j of a few particles with the data in the kernel parameters (no staging copy): what a
// block step of a handful of corrected particles needs.
constexpr int kInlineMaxJ = 16;
struct InlineJ {
    int n;
    int32_t addr[kInlineMaxJ];
    double t[kInlineMaxJ];
    double x[kInlineMaxJ][3];     // kept in fp64 (see RawJ)
    float m[kInlineMaxJ];
    float v[kInlineMaxJ][3];
    float a[kInlineMaxJ][3];
    float k[kInlineMaxJ][3];
};
cudaError_t launch_scatter_inline(const InlineJ& p, const RawJ& raw, cudaStream_t st);

// a3: predict raw -> predicted arrays for j < n_j, m = 0 padding for n_j <= j < n_pad.  upd (may be
// nullptr): a pending small set_j whose addresses are all < n_j, stored and used in the same launch.
cudaError_t launch_predict(const RawJ& raw, double t, long long n_j, long long n_pad, float* px,
                           float* py, float* pz, float* pm, float* pvx, float* pvy, float* pvz,
                           const InlineJ* upd, cudaStream_t st);

// ---- a block step of <= kFusedMaxI i-particles in one launch (nbk_small_kernels.cu): predictor for the
// CTA's own j-particles and for the i-particles, pair sums, reduction by the last CTA.
constexpr int kSmallMaxChunk = 2048;   // j-particles per CTA at most (shared memory): n_j <= SMs x 2048
struct SmallArgs {
    RawJ raw;
    double t;                 // prediction time
    int n_j, n_pad;           // j-particles, and the padded count the predicted arrays are filled to
    int chunk;                // j-particles per CTA, multiple of 4; grid x chunk >= n_pad
    float* pred[7];           // predicted arrays x y z m vx vy vz (also written: other calls read them)
    int n_i;
    int inline_index;         // 1: i-indices are i_inline[], else i_index (nullptr: identity)
    int32_t i_inline[kFusedMaxI];
    const int32_t* i_index;
    float eps2;
    float* partial;           // [cta][kFusedMaxI][8]
    unsigned* counter;        // zero between launches (the last CTA resets it)
    float* acc;               // results [n_i][3], [n_i][3], [n_i]
    float* jerk;
    float* pot;
    float* host_out;          // mapped pinned copy acc|jerk|pot (7 n_i floats) or nullptr
    unsigned* host_seq;       // mapped pinned word: set to `seq` after host_out is complete (nullptr: not wanted)
    unsigned seq;
    InlineJ upd;              // a pending set_j of a few particles (upd.n may be 0), all addresses < n_j
};
size_t small_smem_bytes(int chunk);
cudaError_t small_prepare(int chunk_max);
cudaError_t launch_small_block(const SmallArgs& a, bool jerk, bool eps0, int grid, cudaStream_t s);

// ---- batched acc + pot calls: many (i-group, j-list) problems in one launch ----
struct BatchArgs {
    const float* x;            // packed j-lists, SoA, each list padded to a multiple of 128 (m = 0 far away)
    const float* y;
    const float* z;
    const float* m;
    const float* xi;           // [n_i_total][3] i-positions, groups back to back (caller's order)
    const long long* pair_prefix;  // [n_groups + 1] pairs (chunks x j-tiles) before group g
    const long long* seg_prefix;   // [n_groups + 1] chunks before group g
    const long long* j_off;        // [n_groups] start of the group's padded list in x, y, z, m
    const int* i_off;              // [n_groups] start / end of the group's i-particles in xi and the
    const int* i_end;              //            outputs (the caller's offsets)
    const int* njt;                // [n_groups] j-tiles of the group's list
    float* partial;                // [chunk + worker][ci][4]
    float* acc;                    // [n_i_total][3]  (reduce)
    float* pot;                    // [n_i_total]     (reduce)
    int n_groups;                  // non-empty groups only
    int ci;                        // i-particles per chunk = 32 * ipl / slices
    int ipl;                       // i-particles per lane (1 or 2)
    int slices;                    // lanes of a warp split this many ways over a tile's j-particles (1, 2, 4)
    long long P;                   // pairs in all
    long long n_seg;               // chunks in all
    long long G;                   // workers (warps) that take a range of the pair list
    float eps2;
};
struct BatchPackArgs {
    const float* mj;               // caller's lists: [n_j_total], [n_j_total][3]
    const float* xj;
    const long long* src_off;      // [n_groups] start and length of the caller's list of each group
    const long long* src_len;
    const long long* dst_off;      // [n_groups + 1] padded offsets
    float* x; float* y; float* z; float* m;
    int n_groups;
    long long n_padded;
};
cudaError_t launch_batch_pack(const BatchPackArgs& a, cudaStream_t s);
cudaError_t batch_prepare();
size_t batch_smem_bytes();
cudaError_t launch_batch(const BatchArgs& a, bool eps0, cudaStream_t s);
cudaError_t launch_batch_reduce(const BatchArgs& a, cudaStream_t s);

// device-resident integrator kernels (one block step = begin, predict+select, force, reduce, correct)
// hd_steps_kernel (nbk_hermite_steps.cu): whole block steps of up to max_act due particles inside one
// persistent kernel, one CTA per SM; the phases of a step are ordered by per-word step tags on the partial
// rows and per-particle flags (no grid barrier, no counter).
constexpr int kStepsThreads = 512;     // 16 warps per CTA
constexpr int kStepsMaxAct = 1024;     // largest step the stepping kernel can hold (due list in shared memory)
constexpr int kStepsMaxVec = 16;       // 16-byte loads of level bytes per thread at most: n <= 131072
struct StepsArgs {
    RawJ raw;
    DynHeader* h;
    HermiteState hs;
    float eps2;
    int chunk;             // j-particles per CTA (multiple of 4); G * chunk >= n
    int n_lev;             // n rounded up to a multiple of 16 * kStepsThreads (level bytes every CTA keeps)
    int max_act;           // steps with more due particles end the launch (the chain of launches takes them)
    int max_steps;         // block steps per launch at most
};
size_t steps_smem_bytes(int chunk, int n_lev);
cudaError_t steps_prepare(int chunk, int n_lev, int* ctas_per_sm);
cudaError_t launch_hd_steps(const StepsArgs& a, bool eps0, int grid, bool cooperative, cudaStream_t st);
cudaError_t launch_hd_begin(DynHeader* h, cudaStream_t st);
cudaError_t launch_hd_predict(const RawJ& raw, DynHeader* h, const HermiteState& hs, long long n_pad,
                              float* px, float* py, float* pz, float* pm, float* pvx, float* pvy,
                              float* pvz, cudaStream_t st);
cudaError_t launch_hd_correct(const RawJ& raw, DynHeader* h, const HermiteState& hs, const float* acc,
                              const float* jerk, int n, cudaStream_t st);
cudaError_t launch_reduce_dyn(const Variant& v, const ReduceArgs& a, int ni_max, cudaStream_t s);

}  // namespace nbk
