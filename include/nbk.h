/* nbk.h -- C ABI of the B200-native direct N-body force library ("N-Body Kernels").
 *
 * The boundary is shaped on the GRAPE-6-style call list of the paper's `kirin` library
 * (App. A: GPU_open, GPU_close, GPU_npipes, GPU_set_j_particle,
 * GPU_set_ti, GPUcalc_firsthalf, GPUcalc_lasthalf) and on its statement of the data that
 * crosses it (L80-L83: in  m, x, v;  out  a, jerk, potential).  Names and signatures are
 * this build's own.  Differences from the paper's library, all asked for by
 * BASELINE.json's north_star: j-particle prediction runs on the device (the paper predicts
 * on the host and uploads all N every block step, L78, L428); split-j partial sums are
 * reduced on the device (the paper sums them on the host, L118).
 *
 * What is computed (Eq. 1; "acceleration, its time derivative (jerk) and
 * potential ... by direct summation" L68; softening L126, L132; self term L96; DESIGN.md
 * readings R1-R8), G = 1, r = x_j - x_i, w = v_j - v_i, s = r.r + eps2:
 *
 *     acc_i  =  sum_j m_j r s^(-3/2)
 *     jerk_i =  sum_j m_j [ w s^(-3/2) - 3 (r.w) r s^(-5/2) ]
 *     pot_i  = -sum_j m_j s^(-1/2)
 *
 * over all j in [0, n_j) except the i-particle's own j entry; with NBK_EPS0 pairs with
 * s == 0 contribute nothing.  Pairwise arithmetic is fp32 (FMA + rsqrt.approx); the sums over
 * one j-tile are fp32, a CTA adds its tiles in fp64 and rounds its share once to an fp32 partial
 * row, the partial rows of an i-particle (at most one per CTA) are added in fp64 in a fixed order;
 * results are returned in fp32.
 *
 * Conventions
 *   - Every function returns NBK_OK (0) or a negative nbk_status; nothing throws or aborts.
 *     NaN/Inf in results is not an error.  After NBK_ECUDA, nbk_last_cuda_error() gives the
 *     cudaError_t value.
 *   - "host" pointers are ordinary host memory (pageable is fine; the library stages through
 *     its own pinned buffers).  If every array of a call of >= 4096 particles lies in page-locked
 *     memory (cudaHostAlloc / cudaHostRegister, a pinned torch tensor), set_j and lasthalf copy
 *     straight from / into the caller's arrays instead; semantics are unchanged (the call returns
 *     once the caller's arrays may be reused / hold the results).  "device" pointers (functions ending in _dev) are device
 *     memory on the context's device; the library only enqueues work on the context's
 *     stream and does not synchronise.
 *   - The caller owns every array it passes.  Host arrays may be reused as soon as the call
 *     returns; device arrays once the work enqueued on the stream has run.
 *   - Vectors are row-major [n][3], C order.
 *   - One context = one device = one stream = one caller thread at a time.
 */
#ifndef NBK_H_
#define NBK_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct nbk_ctx nbk_ctx;

typedef enum nbk_status {
    NBK_OK = 0,
    NBK_EINVAL = -1,  /* NULL / negative / inconsistent argument */
    NBK_ERANGE = -2,  /* address, n_j or n_i beyond what the context was opened for */
    NBK_ENOMEM = -3,  /* host or device allocation failed */
    NBK_ECUDA = -4,   /* a CUDA call failed: see nbk_last_cuda_error() */
    NBK_ESTATE = -5   /* call order violated (e.g. lasthalf with no firsthalf in flight) */
} nbk_status;

/* flags of nbk_calc_firsthalf */
#define NBK_JERK 1u /* also compute the jerk (needs v of the j-particles)                */
#define NBK_POT 2u  /* kept for GRAPE-style callers: the potential is always computed    */
#define NBK_EPS0 4u /* mask pairs with s == 0; forced on if eps2==0 */
#define NBK_NN 8u   /* also find each i-particle's nearest neighbour (L126-L128); needs NBK_JERK */

/* ---- life cycle (GPU_open / GPU_close / GPU_npipes) ----------------- */

/* Create a context on CUDA device `device` able to hold n_max j-particles and to serve up to
 * ni_max i-particles per call.  `cuda_stream` is a cudaStream_t (e.g. a torch stream's
 * .cuda_stream) on which all work is enqueued; NULL = the library creates its own non-blocking
 * stream.  Note that the handle of CUDA's legacy default stream IS NULL (torch's default stream has
 * .cuda_stream == 0): a caller that mixes its own work on the default stream with _dev calls must
 * pass a real stream here or order the two with events.
 * All device and pinned memory is allocated here, none later. */
int nbk_open(nbk_ctx** out, int device, int64_t n_max, int64_t ni_max, void* cuda_stream);

/* The same with the context's device buffers carved out of ONE caller-owned device buffer (e.g. a
 * torch tensor), so that the caller's allocator owns the memory: `workspace` is a device pointer
 * aligned to 256 bytes holding at least nbk_workspace_bytes(device, n_max, ni_max) bytes; it must
 * outlive the context and is not freed by nbk_close.  Pinned host staging, and the buffers that
 * nbk_hermite_evolve_dev and nbk_calc_batch allocate on first use, stay the library's. */
int nbk_open_ws(nbk_ctx** out, int device, int64_t n_max, int64_t ni_max, void* cuda_stream,
                void* workspace, int64_t workspace_bytes);
/* Bytes of workspace nbk_open_ws needs on `device` (depends on its SM count), or a negative status. */
int64_t nbk_workspace_bytes(int device, int64_t n_max, int64_t ni_max);

/* Free everything the context owns (waits for its stream first).  NULL is accepted. */
int nbk_close(nbk_ctx* ctx);

/* GRAPE callers ask how many i-particles one call takes (48 on GRAPE-6Af, L102; "can be
 * configured", L426).  Here any n_i <= ni_max is accepted; this returns ni_max clipped to
 * INT_MAX.  Negative nbk_status on a NULL context. */
int nbk_npipes(const nbk_ctx* ctx);

/* ---- a1: load j-particles (GPU_set_j_particle, L427; batched) ---------------------------- */

/* Store n particles into the device j-state at addresses addr[k] (NULL: k itself), each
 * 0 <= addr < n_max.  tj[n] last-update times (NULL: 0), m[n], x[n][3], v[n][3] (NULL: 0),
 * a[n][3], jerk[n][3] (NULL: 0, i.e. the particle is not moved by the predictor).
 * Positions are kept in fp64 on the device so the predictor rounds once; the _f64 form takes
 * double x, v straight from an fp64 integrator.  Host pointers.  The copy is asynchronous on
 * the context's stream from a pinned staging buffer the library owns. */
int nbk_set_j_particles(nbk_ctx* ctx, int64_t n, const int32_t* addr, const double* tj,
                        const float* m, const float* x, const float* v, const float* a,
                        const float* jerk);
int nbk_set_j_particles_f64(nbk_ctx* ctx, int64_t n, const int32_t* addr, const double* tj,
                            const double* m, const double* x, const double* v, const double* a,
                            const double* jerk);
/* Same as nbk_set_j_particles with DEVICE pointers; nothing is staged, nothing synchronises. */
int nbk_set_j_particles_dev(nbk_ctx* ctx, int64_t n, const int32_t* addr, const double* tj,
                            const float* m, const float* x, const float* v, const float* a,
                            const float* jerk);

/* ---- a2/a3: set time and predict (GPU_set_ti, L428; predictor L68, reading R8) ---------- */

/* Record the time t to which j-particles are predicted.  Cheap: marks the predicted state
 * stale; the predictor kernel runs on the device at the next nbk_predict / firsthalf. */
int nbk_set_ti(nbk_ctx* ctx, double t);

/* Run the predictor now for j in [0, n_j):  dt = t - tj (fp64),
 *   x_p = x + v dt + a dt^2/2 + jerk dt^3/6,  v_p = v + a dt + jerk dt^2/2,
 * evaluated in fp64 and rounded once to the fp32 arrays the force kernel reads.
 * firsthalf calls this itself when the predicted state is stale. */
int nbk_predict(nbk_ctx* ctx, int64_t n_j);

/* Read back the predicted fp32 state (host pointers, any may be NULL); synchronises.
 * For tests of a3 and for callers that want the positions the forces were evaluated at. */
int nbk_get_predicted(nbk_ctx* ctx, int64_t n_j, float* m, float* x, float* v);

/* ---- a4-a6: force on a block of i-particles (GPUcalc_firsthalf, L429) -------------------- */

/* Enqueue prediction (if stale), the i x j force kernel and the split-j reduction for n_i
 * i-particles against j-particles [0, n_j).  Asynchronous: returns once the work is queued.
 *   i_index[n_i]  i_index[k] >= 0: i-particle k is j-particle i_index[k]; its predicted
 *                 state is gathered on the device and its own j entry is left out of the
 *                 sums.  -1: external test particle (needs xi; no j is left out).
 *                 NULL: i_index[k] = k.
 *   xi, vi        optional [n_i][3] explicit i-state overriding the gathered one (vi NULL:
 *                 gathered velocity, or 0 for external particles).
 *   eps2          softening length squared (>= 0).
 *   flags         NBK_JERK | NBK_POT | NBK_EPS0.
 * Host pointers (copied before return). */
int nbk_calc_firsthalf(nbk_ctx* ctx, int64_t n_j, int64_t n_i, const int32_t* i_index,
                       const float* xi, const float* vi, float eps2, uint32_t flags);
/* Same with DEVICE pointers, which must stay valid until the enqueued work has run. */
int nbk_calc_firsthalf_dev(nbk_ctx* ctx, int64_t n_j, int64_t n_i, const int32_t* i_index,
                           const float* xi, const float* vi, float eps2, uint32_t flags);

/* ---- a7: read back (GPUcalc_lasthalf, L430) ----------------------------------------------- */

/* Wait for the last firsthalf and copy acc[n_i][3], jerk[n_i][3], pot[n_i] to HOST arrays
 * (any may be NULL; jerk is zero if NBK_JERK was not set).  n_i must equal firsthalf's.
 * After a one-launch small block (n_i <= 32 particles of the j-set) the wait is a poll of a word in
 * mapped host memory that the kernel writes after the results, not a stream synchronisation: the call
 * returns as soon as the results are in host memory; the stream itself may take a microsecond longer to
 * drain (nbk_sync waits for that). */
int nbk_calc_lasthalf(nbk_ctx* ctx, int64_t n_i, float* acc, float* jerk, float* pot);
/* Same into double arrays (GRAPE-style callers keep doubles); the values are the fp32 results. */
int nbk_calc_lasthalf_f64(nbk_ctx* ctx, int64_t n_i, double* acc, double* jerk, double* pot);
/* Same to DEVICE arrays, asynchronous on the stream, no synchronisation. */
int nbk_calc_lasthalf_dev(nbk_ctx* ctx, int64_t n_i, float* acc, float* jerk, float* pot);

/* ---- the same force evaluation for callers that must not allocate --------------------------------
 * nbk_open allocates device and pinned memory, so everything above needs a caller that may call
 * cudaMalloc.  Not every caller can: a plug-in in a process whose memory pool has already taken the
 * device's memory (a library-side cudaMalloc then fails or eats what the host application counted
 * on), a step loop that cannot afford cudaMalloc / cudaFree stalling the device, a code that forbids
 * allocation after start-up.  nbk_calc_noalloc_dev is the one entry point for them.  It takes no
 * context and calls no cudaMalloc, cudaFree, cudaHostAlloc or any routine that allocates: inputs
 * and outputs are the caller's device arrays, and the split-j partial rows and
 * their arrival counters sit in a fixed array of NBK_NOALLOC_SCRATCH_BYTES that is part of the
 * library's device image -- each GPU that loads libnbk.so carries it until the process exits.
 *
 *   device, cuda_stream   the device the arrays live on and a cudaStream_t of that device to enqueue
 *                         on (NULL: the legacy default stream).  Asynchronous: nothing waits.
 *   m[n_j], x[n_j][3], v[n_j][3]   the j-particles' state at the time of the evaluation, fp32, already
 *                         predicted by the caller (no predictor runs here); v may be NULL without NBK_JERK.
 *   i_index[n_i]          i-particle k is j-particle i_index[k]; its own j entry is left out of its
 *                         sums.  NULL: i_index[k] = k.  An entry outside [0, n_j) gets zeros.
 *   eps2, flags           as nbk_calc_firsthalf; NBK_NN is refused (NBK_EINVAL).
 *   acc[n_i][3], jerk[n_i][3], pot[n_i]   results (any may be NULL; jerk is zero without NBK_JERK).
 *   cuda_error            optional HOST int: the cudaError_t behind an NBK_ECUDA return, else 0.
 * All array pointers are DEVICE pointers.  Sums as defined at the top of this file: fp32 per pair,
 * fp64 across tiles and splits in a fixed order (repeatable bit for bit), results rounded once.
 *
 * Limits, and what sharing one array means:
 *   - n_i <= NBK_NOALLOC_MAX_NI and n_j <= NBK_NOALLOC_MAX_NJ, else NBK_ERANGE and nothing is enqueued.
 *   - The first call on a device looks up the array's device address (cudaGetSymbolAddress, with that
 *     device current; this can make the runtime load the library's device code).  Make that first
 *     call before starting any stream capture.
 *   - All calls on a device use the same array.  Calls on one stream are ordered and safe; calls of a
 *     process that can overlap on the GPU (two streams without an event between them) race on the
 *     rows and counters and give wrong results.  The counters are zeroed on the stream at the start
 *     of every call; the rows are written before they are read, so old contents never matter. */
#define NBK_NOALLOC_MAX_NI 4096
#define NBK_NOALLOC_MAX_NJ 16777216
#define NBK_NOALLOC_SCRATCH_BYTES (4194304 + 256)
int nbk_calc_noalloc_dev(int device, void* cuda_stream, int64_t n_j, const float* m, const float* x,
                         const float* v, int64_t n_i, const int32_t* i_index, float eps2,
                         uint32_t flags, float* acc, float* jerk, float* pot, int* cuda_error);

/* ---- nearest neighbour ("the GRAPE hardware also calculates the nearest
 * neighbour of every particle that is being updated ... done as part of the force calculation";
 * SURVEY.md 8(f)-2) ------------------------------------------------------------------------------ */

/* After a firsthalf with NBK_NN: nn_index[n_i] = the j in [0, n_j) with the smallest softened
 * squared distance s = r.r + eps2 to i-particle k as the kernel computes it in fp32, the own entry
 * left out by index, ties to the lowest j (-1 if there is no other j); nn_r2[n_i] = its unsoftened
 * squared distance in fp32 (inf if none).  The search rides in the force kernel (one min per pair);
 * the index is recovered by re-scanning the one j-tile that held the minimum.  Host arrays (either
 * may be NULL); waits for the stream.  NBK_ESTATE if the last firsthalf had no NBK_NN. */
int nbk_get_neighbours(nbk_ctx* ctx, int64_t n_i, int32_t* nn_index, float* nn_r2);
/* Same to DEVICE arrays, asynchronous on the stream. */
int nbk_get_neighbours_dev(nbk_ctx* ctx, int64_t n_i, int32_t* nn_index, float* nn_r2);

/* ---- batched acceleration + potential calls --------------------------------
 * the GRAPE treecode asks, for each group of particles, for the
 * acceleration (no jerk, no neighbours) due to that group's interaction list; with one library
 * call per group the paper needed groups of 8192-32768 particles.  Here all groups of a step are
 * one call and one force launch (the tree walk itself is the caller's).
 *   i_offset[n_groups + 1], j_offset[n_groups + 1]   HOST arrays, ascending from 0: group g owns
 *       i-particles [i_offset[g], i_offset[g+1]) of xi / acc / pot and list entries
 *       [j_offset[g], j_offset[g+1]) of mj / xj.
 *   xi[n_i][3], mj[n_j], xj[n_j][3]    inputs;  acc[n_i][3], pot[n_i]  outputs
 *       (host pointers for nbk_calc_batch, device pointers for nbk_calc_batch_dev).
 * For every i of group g:  acc_i = sum_j m_j r s^(-3/2),  pot_i = -sum_j m_j s^(-1/2) over the
 * group's list, r = x_j - x_i, s = r.r + eps2.  Nothing is left out by index: a list entry at the
 * i-particle's own position adds 0 to acc and -m_j/eps to pot for eps2 > 0 (GRAPE callers subtract
 * it), and is skipped with NBK_EPS0 or eps2 == 0.  flags: NBK_POT | NBK_EPS0 (NBK_JERK, NBK_NN:
 * NBK_EINVAL).  i-particles of a group with an empty list get zeros.  Independent of the context's
 * j-state; the library keeps its own growable device arena for the packed lists.  Both forms
 * return after the work has run (the host form has then filled acc and pot). */
int nbk_calc_batch(nbk_ctx* ctx, int64_t n_groups, const int64_t* i_offset, const float* xi,
                   const int64_t* j_offset, const float* mj, const float* xj, float eps2,
                   uint32_t flags, float* acc, float* pot);
int nbk_calc_batch_dev(nbk_ctx* ctx, int64_t n_groups, const int64_t* i_offset, const float* xi,
                       const int64_t* j_offset, const float* mj, const float* xj, float eps2,
                       uint32_t flags, float* acc, float* pot);

/* ---- a8: host Hermite driver (reading R15) ------------------- */

typedef struct nbk_hermite_stats {
    int64_t block_steps;      /* force calls made                                    */
    int64_t particle_steps;   /* sum of n_i over block steps                         */
    int64_t interactions;     /* sum of n_i * n over block steps                     */
    double wall_seconds;      /* whole run, host clock                               */
    double gpu_call_seconds;  /* host time spent inside nbk_* calls (incl. waiting)  */
    double t_reached;
    int64_t ni_histogram[32]; /* bucket b counts block steps with 2^b <= n_i < 2^(b+1) */
} nbk_hermite_stats;

/* Integrate n particles from t = 0 to t_end with the 4th-order Hermite predictor-corrector,
 * power-of-two block time steps and the Aarseth criterion (eta, dt_max), host arithmetic in
 * fp64, forces from this context (which must have n_max >= n, ni_max >= n).
 * m[n], x[n][3], v[n][3] are HOST fp64 arrays, updated in place to the state at t_end
 * (t_end must be a multiple of dt_max so that all particles are synchronised there).
 * dt_max is rounded down to a power of two and must lie in [2^-48, 2): step levels are 2^-k with
 * k in [0, 48]; anything else (dt_max >= 2 included), t_end > 2047 or eta <= 0 is NBK_EINVAL.
 * stats may be NULL. */
int nbk_hermite_evolve(nbk_ctx* ctx, int64_t n, const double* m, double* x, double* v,
                       double eps, double t_end, double eta, double dt_max,
                       nbk_hermite_stats* stats);

/* The same integration with the whole block-step loop on the device (PAPER.md
 * L346, L368 name it as what fp64 GPUs make possible).  After the forces at t = 0, block steps of up to
 * 1024 due particles run inside one persistent kernel (one CTA per SM, every CTA keeps its share of the
 * j-particles' state and every particle's step level in shared memory: scheduler, predictor, pair sums,
 * reduction and fp64 corrector of a step without leaving the kernel); larger steps are five stream-ordered
 * launches -- step header + launch plan made on the device, predictor + selection of the particles due,
 * i x j force kernel (1 or 4 i-particles per thread, the device planner's choice), reduction, fp64
 * corrector + Aarseth step + block rule.  Everything is replayed from a CUDA graph in batches with no
 * host synchronisation in between.  For n > 131072 (or when the state does not fit shared memory) every
 * step takes the launches.  Same scheme, formulas, arguments and argument limits as nbk_hermite_evolve;
 * results are bitwise repeatable; stats->gpu_call_seconds equals wall_seconds.  NBK_ECUDA with
 * nbk_last_cuda_error() == cudaErrorLaunchTimeout means a wait inside the persistent kernel gave up
 * (another process holding SMs for seconds; the first CTA to give up raises an abort word and the others
 * leave within milliseconds): the state is then undefined.  NBK_ERANGE after the forces at t = 0 means no
 * launch plan of a large step fits the context's partial-row buffer (open it with a larger ni_max).  Test
 * knob: the environment variable NBK_STEPS_MAX_ACT (a whole number 0..1024, read at each call; anything else
 * is NBK_EINVAL) caps the step size the persistent kernel takes; 0 sends every step through the launches.
 * After the call nbk_last_launch reports the persistent kernel: out[0] its CTAs (0: not used), out[1] its
 * threads, out[4] the step-size cap, out[7] 2 if it was captured as a cooperative launch (the driver checks
 * that all CTAs are co-resident), 1 if as a plain launch (co-residency by construction: one CTA per SM). */
int nbk_hermite_evolve_dev(nbk_ctx* ctx, int64_t n, const double* m, double* x, double* v,
                           double eps, double t_end, double eta, double dt_max,
                           nbk_hermite_stats* stats);

/* ---- utilities --------------------------------------------------------------------------- */

/* ---- j-sharding over several GPUs --------------------------------------
 * "the j-particles are divided in blocks ... the partial forces are stored ...
 * after which they are summed".  Stretched over devices: rank r of G holds the j-particles with
 * global addresses [j0_r, j0_r + n_local_r) in its own context (local address = global - j0_r),
 * every rank computes the partial sums of ALL active i-particles against its own j-particles, and
 * one all-reduce(sum) of n_i x 8 doubles gives every rank the total.  The library does the three
 * device steps; the two all-reduces between them are the caller's (torch.distributed / NCCL; the
 * Python class ShardedForce in paper_0707_0438_b200/sharded.py strings them together).  All
 * pointers are DEVICE pointers; everything is enqueued on the context's stream, nothing waits.
 *
 * 1. nbk_shard_gather_i_dev: predict (if stale), then for each i-particle k with global address
 *    i_global[k]: i_local[k] = its local address if this rank owns it, else -1;
 *    xv[k][0..7] = (x, y, z, 0, vx, vy, vz, 0) of its predicted fp32 state if owned, else zeros.
 *    Exactly one rank owns each i-particle, so all-reduce(sum) of xv over the ranks is an exact
 *    copy of the owner's state to everybody.
 * 2. nbk_shard_calc_partial_dev: the force kernel and split-j reduction of i-particles with the
 *    state xv (after the exchange) against local j-particles [0, n_local), the own entry of an
 *    owned i-particle (i_local[k] >= 0) left out; writes sum64[k][0..7] = (acc(3), -pot, jerk(3),
 *    0): the fp64 sum of this rank's fp32 partial rows (each CTA's share is rounded to fp32 once, as
 *    on one GPU), NOT yet rounded to the fp32 result (the fp32 results of this rank alone remain
 *    readable with nbk_calc_lasthalf*).  flags as nbk_calc_firsthalf; NBK_NN is refused
 *    (NBK_EINVAL).  n_local == 0 is allowed (sums are zero).
 * 3. nbk_shard_finish_dev: after all-reduce(sum) of sum64: acc, jerk, pot in fp32 (one rounding;
 *    pot = -sum64[k][3]); any output may be NULL.  Every rank gets bit-identical results because
 *    an all-reduce returns the same bits on every rank. */
int nbk_shard_gather_i_dev(nbk_ctx* ctx, int64_t n_local, int64_t j0, int64_t n_i,
                           const int32_t* i_global, int32_t* i_local, float* xv);
int nbk_shard_calc_partial_dev(nbk_ctx* ctx, int64_t n_local, int64_t n_i, const int32_t* i_local,
                               const float* xv, float eps2, uint32_t flags, double* sum64);
int nbk_shard_finish_dev(nbk_ctx* ctx, int64_t n_i, const double* sum64, float* acc, float* jerk,
                         float* pot);

/* The same two exchanges as loads from PEER memory (NVLink / NVSwitch P2P) instead of collectives,
 * for callers whose xv and sum64 buffers live in symmetric memory mapped into every rank (e.g.
 * torch.distributed._symmetric_memory).  `world` <= 16 ranks.  The caller separates the steps with a
 * cross-rank barrier on the stream (after gather_i; after calc_partial): two barriers per call, no
 * payload collective.
 *   nbk_shard_fetch_i_dev   replaces all-reduce 1: xv[k] (this rank's private [n_i][8] buffer) = row k
 *                           of the OWNER's published buffer, the owner found from shard_begin (HOST
 *                           array of world + 1 global addresses); peer_xv is a HOST array of `world`
 *                           device pointers, peer_xv[r] = rank r's buffer written by its gather_i.
 *   nbk_shard_combine_dev   replaces all-reduce 2 and finish: acc, jerk, pot = the sum over ranks r, in
 *                           rank order, of row k of peer_sum64[r] (HOST array of `world` device
 *                           pointers to the [n_i][8] fp64 buffers calc_partial wrote), rounded once.
 *                           Same bits on every rank. */
int nbk_shard_fetch_i_dev(nbk_ctx* ctx, int64_t n_i, int32_t world, const int32_t* i_global,
                          const int64_t* shard_begin, const void* const* peer_xv, float* xv);
int nbk_shard_combine_dev(nbk_ctx* ctx, int64_t n_i, int32_t world, const void* const* peer_sum64,
                          float* acc, float* jerk, float* pot);

/* Block until everything enqueued on the context's stream has run. */
int nbk_sync(nbk_ctx* ctx);

/* Kernel timing: when enabled, firsthalf/predict record CUDA events around each kernel on
 * the context's stream.  nbk_get_timing waits for them and returns the durations, in
 * milliseconds, of the LAST call's kernels: ms[0] scatter (set_j), ms[1] predict,
 * ms[2] i x j force tile, ms[3] reduce.  A kernel that did not run reports 0. */
int nbk_set_timing(nbk_ctx* ctx, int enable);
int nbk_get_timing(nbk_ctx* ctx, float ms[4]);

/* Launch shape of the last firsthalf: out[0] grid (CTAs, one per SM at most), out[1] threads
 * per CTA, out[2] i-particles per thread, out[3] warps splitting each j-tile, out[4] j-tile
 * size, out[5] SM count, out[6] dynamic shared memory bytes, out[7] number of kernels launched
 * by the last firsthalf (2: force + reduce; 1: small block -- predicted, summed and reduced by one
 * launch of 512-thread CTAs, out[3] = 16, out[4] = j-particles per CTA -- or, with external positions or
 * NBK_NN, reduced by the tiled force kernel's last
 * CTA; 3: force + reduce + neighbour re-scan).  After nbk_calc_batch: out[0] CTAs of 16 warps, out[2]
 * i-particles per lane (1, 2), out[3] ways the lanes of a warp split a j-tile (1, 2, 4), out[4] 128. */
int nbk_last_launch(const nbk_ctx* ctx, int64_t out[8]);

/* Host-only (no GPU needed): the launch plan firsthalf would use for (n_i, n_j) on a device with
 * num_sms SMs -- the split-j / stream-K decomposition of PAPER.md L112-L118 generalised.
 * force_i: 0 or a pinned i-per-thread count (1, 2, 4).  out[0] i per thread, out[1] threads per
 * CTA, out[2] i-tile, out[3] j-tile, out[4] warps splitting a j-tile, out[5] i-tiles,
 * out[6] j-tiles, out[7] pairs P, out[8] CTAs G, out[9] max i-tiles one CTA touches,
 * out[10] floats of partial rows needed, out[11] floats a context with ni_max = n_i holds.
 * CTA k works on pairs [k*P/G, (k+1)*P/G) of the i-major (i-tile, j-tile) list. */
int nbk_plan(int64_t n_i, int64_t n_j, int num_sms, int force_i, int64_t out[12]);

/* Test and measurement knob, not needed by callers: pins a launch shape the planner would not
 * pick so that the test matrix reaches every kernel form.  bits 4-7: pin the i-particles per
 * thread (1, 2, 4; 0 = planner's choice).  bit 8: switch off the one-launch path for blocks of
 * <= 32 i-particles (reduction by the last CTA, indices in the launch parameters, results
 * written to mapped host memory).  Any other bit: NBK_EINVAL.  All forms compute the same sums. */
int nbk_set_variant(nbk_ctx* ctx, int variant);

int nbk_last_cuda_error(const nbk_ctx* ctx);
const char* nbk_strerror(int status);
const char* nbk_version(void);

#ifdef __cplusplus
}
#endif
#endif /* NBK_H_ */
