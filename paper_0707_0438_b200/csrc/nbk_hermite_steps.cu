// nbk_hermite_steps.cu -- hd_steps_kernel: whole Hermite block steps inside ONE persistent kernel
// (what a small block step costs is the traffic and latency
// around the force, not the force; L346, L368: with fp64 on the device the rest of the integrator can
// sit beside it).
//
// One CTA per SM, 16 warps, all co-resident.  CTA k owns the j-particles [k * chunk, (k + 1) * chunk)
// and keeps their raw state (x fp64, v, a, jerk, m, t_j) in shared memory for the whole launch; every
// CTA also keeps the level of ALL particles (one byte each) and the level counts, so the scheduler
// runs in every CTA from shared memory alone.  One block step:
//   A  wait for the flags of the previous step's particles (one word each: step number and new level,
//      written by whoever corrected the particle) -> own level bytes and counts; owned particles among
//      them re-read their corrected raw state.  Header (next block time, threshold level, number due)
//      from the counts; due list in ascending index order by a scan of the level bytes.
//   B  predictor: own chunk from shared memory into the tile layout of the force loop (the predicted
//      j-state never goes to global memory), due particles from global raw state (every CTA predicts
//      them itself: same formula, same bits as their j entries); then the pair sums over the resident
//      chunk -- lanes over j for steps of a few particles, lanes over i (tile_packed) otherwise -- fp32
//      inside a warp's share, fp64 above; one partial row per (CTA, due particle).
//      Every value of a row travels in one 8-byte word together with the step number, so a row is
//      complete as soon as its words carry the current number: no fence, no counter, no barrier.
//   C  due particle q belongs to CTA (q mod G): all its threads fetch the G rows at once and spin until
//      they are all of this step; the rows are added in CTA order (fp64, lane tree then warps in order),
//      rounded once to fp32, and warp 0 runs the fp64 corrector (one lane per component), the Aarseth
//      step and the block rule, then sets the particle's flag.
// The launch ends when the run is finished, after max_steps steps, or at a step with more than
// max_act due particles, which the chain of launches (hd_begin -> hd_predict -> force -> reduce ->
// hd_correct) takes with the planner's launch shape.  Every sum is taken in a fixed order and the due
// list is ordered: bitwise repeatable.
#include "nbk_device.cuh"

namespace nbk {

namespace {

constexpr int kSW = kStepsThreads / 32;   // warps per CTA
constexpr int kLaneJMax = 4;              // steps of up to this many particles: lanes run over j
constexpr long long kSpinLimit = 1LL << 26;

// One failed poll of a wait on another CTA's tagged word.  Every 4096 polls the waiter looks at the launch's
// abort word (DynHeader::error); the waiter that runs out of polls raises it, so that all other CTAs leave
// within a few thousand polls of the first one giving up instead of each running out its own limit.
__device__ __forceinline__ bool spin_abort(long long& spins, DynHeader* h) {
    if ((++spins & 4095) != 0) return false;
    if (spins <= kSpinLimit && *reinterpret_cast<volatile int*>(&h->error) == 0) return false;
    atomicExch(&h->error, 1);
    return true;
}


// one value of a partial row and the number of the step it belongs to, in one 8-byte word
__device__ __forceinline__ unsigned long long row_word(float v, unsigned seq) {
    return (static_cast<unsigned long long>(seq) << 32) | static_cast<unsigned long long>(__float_as_uint(v));
}
__device__ __forceinline__ void st_row(unsigned long long* p, unsigned long long w) {
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(w) : "memory");
}
__device__ __forceinline__ ulonglong2 ld_row2(const unsigned long long* p) {   // two words, each valid on its own
    ulonglong2 v;
    asm volatile("ld.relaxed.gpu.global.v2.u64 {%0, %1}, [%2];" : "=l"(v.x), "=l"(v.y) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ unsigned long long ld_acquire64(const unsigned long long* p) {
    unsigned long long v;
    asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}

struct StepsSmem {
    int act[kStepsMaxAct];             // due particles of the current step, ascending
    float ni[kStepsMaxAct][6];         // their negated predicted state
    double scratch[kSW][32][7];        // cross-warp sums (lanes over i)
    float red[kSW][kLaneJMax][8];      // cross-warp sums (lanes over j)
    int cnt[kMaxLevel + 1];            // particles per level
    long long hist[32];                // CTA 0: steps by log2(size), written back at the end
    int wsum[kSW];
    int err;
};

// shared memory: tiles | raw chunk (x, t fp64; v, a, k, m fp32) | level bytes | StepsSmem
struct Layout {
    float* tiles;      // [nb256][7][256]
    double* rx;        // [3][chunk]
    double* rt;        // [chunk]
    float* rv;         // [3][chunk]
    float* ra;
    float* rk;
    float* rm;         // [chunk]
    unsigned char* lev;  // [n_lev]: level + 1, 0 beyond n
    StepsSmem* S;
};
__host__ __device__ inline size_t layout_bytes(int chunk, int n_lev) {
    const size_t nb = (static_cast<size_t>(chunk) + kTileJMax - 1) / kTileJMax;
    size_t b = nb * 7 * kTileJMax * sizeof(float);
    b += sizeof(double) * 4 * chunk + sizeof(float) * 10 * chunk;
    b = (b + 15) & ~static_cast<size_t>(15);
    b += static_cast<size_t>(n_lev);
    b = (b + 15) & ~static_cast<size_t>(15);
    return b + sizeof(StepsSmem);
}
__device__ inline Layout layout_of(unsigned char* p, int chunk, int n_lev) {
    Layout L;
    const size_t nb = (static_cast<size_t>(chunk) + kTileJMax - 1) / kTileJMax;
    L.tiles = reinterpret_cast<float*>(p);
    p += nb * 7 * kTileJMax * sizeof(float);
    L.rx = reinterpret_cast<double*>(p); p += sizeof(double) * 3 * chunk;
    L.rt = reinterpret_cast<double*>(p); p += sizeof(double) * chunk;
    L.rv = reinterpret_cast<float*>(p); p += sizeof(float) * 3 * chunk;
    L.ra = reinterpret_cast<float*>(p); p += sizeof(float) * 3 * chunk;
    L.rk = reinterpret_cast<float*>(p); p += sizeof(float) * 3 * chunk;
    L.rm = reinterpret_cast<float*>(p); p += sizeof(float) * chunk;
    p = reinterpret_cast<unsigned char*>((reinterpret_cast<uintptr_t>(p) + 15) & ~static_cast<uintptr_t>(15));
    L.lev = p; p += n_lev;
    p = reinterpret_cast<unsigned char*>((reinterpret_cast<uintptr_t>(p) + 15) & ~static_cast<uintptr_t>(15));
    L.S = reinterpret_cast<StepsSmem*>(p);
    return L;
}

// raw state of particle j (global, through L2) into slot jl of the CTA's resident chunk
__device__ __forceinline__ void fetch_raw(const RawJ& raw, const Layout& L, int chunk, int j, int jl) {
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        L.rx[c * chunk + jl] = __ldcg(raw.x + c * raw.cap + j);
        L.rv[c * chunk + jl] = __ldcg(raw.v + c * raw.cap + j);
        L.ra[c * chunk + jl] = __ldcg(raw.a + c * raw.cap + j);
        L.rk[c * chunk + jl] = __ldcg(raw.k + c * raw.cap + j);
    }
    L.rm[jl] = __ldcg(raw.m + j);
    L.rt[jl] = __ldcg(raw.t + j);
}

}  // namespace

size_t steps_smem_bytes(int chunk, int n_lev) { return layout_bytes(chunk, n_lev) + 16; }

template <bool EPS0>
__global__ void __launch_bounds__(kStepsThreads, 1) hd_steps_kernel(const StepsArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const Layout L = layout_of(smem_raw, a.chunk, a.n_lev);
    StepsSmem& S = *L.S;
    const int nb256 = (a.chunk + kTileJMax - 1) / kTileJMax;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int G = gridDim.x, cta = blockIdx.x;
    DynHeader* h = a.h;
    const RawJ& raw = a.raw;
    const HermiteState& hs = a.hs;
    const int n = h->n, kmin = h->kmin, chunk = a.chunk;
    const double eta = h->eta;
    const long long T_end = h->T_end;
    long long T_now = h->T_now;
    const unsigned seq0 = h->seq;          // steps taken by earlier launches: flags carry seq0 + step + 1
    const int j0 = cta * chunk;
    unsigned long long* rows = hs.rows;   // [cta][max_act][8] words
    if (h->done || h->error) return;
    // ---- set-up: resident copies of the chunk's raw state, of every particle's level, of the counts
    for (int jl = tid; jl < chunk; jl += kStepsThreads)
        if (j0 + jl < n) fetch_raw(raw, L, chunk, j0 + jl, jl);
    for (int i = 16 * tid; i < a.n_lev; i += 16 * kStepsThreads)   // level bytes (k + 1; 0 beyond n), 16 per load
        *reinterpret_cast<uint4*>(L.lev + i) = i < n ? *reinterpret_cast<const uint4*>(hs.level + i) : make_uint4(0u, 0u, 0u, 0u);
    if (tid <= kMaxLevel) S.cnt[tid] = static_cast<int>(h->level_count[tid]);
    if (tid < 32) S.hist[tid] = 0;
    if (tid == 0) S.err = 0;
    int n_prev = 0, stop = 0;
    long long steps_done = 0, psteps = 0;
    __syncthreads();

    for (int step = 0;; ++step) {
        // --------------------------------------------- A: last step's changes, header, due list
        for (int q = tid; q < n_prev; q += kStepsThreads) {
            const int i = S.act[q];
            const unsigned want = seq0 + static_cast<unsigned>(step);   // the previous step's number
            unsigned long long f;
            long long spins = 0;
            while (static_cast<unsigned>((f = ld_acquire64(hs.flag + q)) >> 32) != want) {
                if (spin_abort(spins, h)) { S.err = 1; break; }   // never hang the device
            }
            const int nl = static_cast<int>(f & 0xffu), ol = L.lev[i] - 1;
            if (nl != ol) {
                L.lev[i] = static_cast<unsigned char>(nl + 1);
                atomicSub(&S.cnt[ol], 1);
                atomicAdd(&S.cnt[nl], 1);
            }
            if (i >= j0 && i < j0 + chunk) fetch_raw(raw, L, chunk, i, i - j0);
        }
        __syncthreads();
        // header, by every warp for itself (no broadcast, no barrier): finest occupied level -> next block
        // time -> threshold level -> number due
        int kstar, n_act = 0;
        long long T_next = 0;
        {
            const int c0 = S.cnt[lane], c1 = lane + 32 <= kMaxLevel ? S.cnt[lane + 32] : 0;
            const unsigned m0 = __ballot_sync(0xffffffffu, c0 > 0), m1 = __ballot_sync(0xffffffffu, c1 > 0);
            const int kf = m1 ? 63 - __clz(m1) : (m0 ? 31 - __clz(m0) : -1);
            kstar = kf;
            if (kf >= 0) {
                const int sh = kTickLog2 - kf;
                T_next = ((T_now >> sh) + 1) << sh;
            }
            if (S.err) {
                stop = 3;
            } else if (kf < 0 || T_next > T_end) {
                stop = 2;   // the run is finished
            } else {
                // T_next is a multiple of 2^-k (in ticks of 2^-52) for every k >= 52 - ctz(T_next): those
                // levels are due, down to the coarsest one in use
                kstar = max(kmin, kTickLog2 - (__ffsll(T_next) - 1));
                n_act = (lane >= kstar ? c0 : 0) + (lane + 32 >= kstar ? c1 : 0);
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) n_act += __shfl_xor_sync(0xffffffffu, n_act, o);
                if (n_act > a.max_act || step >= a.max_steps) stop = 1;
            }
        }
        if (stop) break;
        const double t_next = static_cast<double>(T_next) * 0x1p-52;   // = ldexp(T_next, -kTickLog2), exact scaling
        const unsigned seq = seq0 + static_cast<unsigned>(step) + 1u;   // this step's number (never 0)
        {   // due = level >= kstar.  Level bytes hold level + 1 (0: no particle), all below 128, so
            // (byte + 0x80 - (kstar + 1)) has its top bit set exactly for the due ones.  A warp scans a
            // contiguous region, 16 bytes per lane and load with the lanes side by side (no bank
            // conflicts); ascending order = (load, lane, byte).
            const int nvec = a.n_lev / (16 * kStepsThreads);   // loads per thread, at most kStepsMaxVec
            const unsigned char* wbase = L.lev + warp * nvec * 512;
            const unsigned add = 0x01010101u * static_cast<unsigned>(0x80 - (kstar + 1));
            int c = 0;
#pragma unroll 4
            for (int o = 0; o < nvec; ++o) {
                const uint4 w = *reinterpret_cast<const uint4*>(wbase + (o * 32 + lane) * 16);
                c += __popc((w.x + add) & 0x80808080u) + __popc((w.y + add) & 0x80808080u) +
                     __popc((w.z + add) & 0x80808080u) + __popc((w.w + add) & 0x80808080u);
            }
            int tot = c;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) tot += __shfl_xor_sync(0xffffffffu, tot, o);
            if (lane == 0) S.wsum[warp] = tot;
            __syncthreads();
            if (tot > 0) {   // few warps: positions of this warp's due particles, load by load
                int pos = 0;
#pragma unroll
                for (int w = 0; w < kSW; ++w) pos += w < warp ? S.wsum[w] : 0;
                for (int o = 0; o < nvec; ++o) {
                    const unsigned char* p = wbase + (o * 32 + lane) * 16;
                    const uint4 w = *reinterpret_cast<const uint4*>(p);
                    const unsigned m[4] = {(w.x + add) & 0x80808080u, (w.y + add) & 0x80808080u,
                                           (w.z + add) & 0x80808080u, (w.w + add) & 0x80808080u};
                    const int cl = __popc(m[0]) + __popc(m[1]) + __popc(m[2]) + __popc(m[3]);
                    if (__ballot_sync(0xffffffffu, cl > 0) == 0u) continue;
                    int incl = cl;
#pragma unroll
                    for (int d = 1; d < 32; d <<= 1) {
                        const int up = __shfl_up_sync(0xffffffffu, incl, d);
                        if (lane >= d) incl += up;
                    }
                    int at = pos + incl - cl;
                    const int first = static_cast<int>(p - L.lev);
#pragma unroll
                    for (int k = 0; k < 4; ++k) {
                        unsigned mm = m[k];
                        while (mm) {
                            const int bit = __ffs(mm) - 1;   // 7, 15, 23 or 31
                            mm &= mm - 1;
                            S.act[at++] = first + 4 * k + (bit >> 3);
                        }
                    }
                    pos += __shfl_sync(0xffffffffu, incl, 31);
                }
            }
        }
        __syncthreads();
        // ------------------------------------------- B: predict the due particles and the own chunk
        for (int q = tid; q < n_act; q += kStepsThreads) {
            float o[7];
            predict_one<true>(raw, S.act[q], t_next, o);
            S.ni[q][0] = -o[0]; S.ni[q][1] = -o[1]; S.ni[q][2] = -o[2];
            S.ni[q][3] = -o[4]; S.ni[q][4] = -o[5]; S.ni[q][5] = -o[6];
        }
        // chunk slots start at warp 1, so that warp 0 (busy with the due particles) gets the padding
        for (int jl = (tid + kStepsThreads - 32) % kStepsThreads; jl < nb256 * kTileJMax; jl += kStepsThreads) {
            float o[7] = {1e18f, 1e18f, 1e18f, 0.f, 0.f, 0.f, 0.f};   // padding: massless, far away
            if (jl < chunk && j0 + jl < n) {
                const double dt = t_next - L.rt[jl];
                const double dt2 = dt * dt * 0.5, dt3 = dt * dt * dt * (1.0 / 6.0);
#pragma unroll
                for (int c = 0; c < 3; ++c)
                    predict_component(L.rx[c * chunk + jl], L.rv[c * chunk + jl], L.ra[c * chunk + jl],
                                      L.rk[c * chunk + jl], dt, dt2, dt3, o[c], o[4 + c]);
                o[3] = L.rm[jl];
            }
            float* dst = L.tiles + (jl >> 8) * 7 * kTileJMax + (jl & 255);
#pragma unroll
            for (int c = 0; c < 7; ++c) dst[c * kTileJMax] = o[c];
        }
        __syncthreads();
        // ---------------------------------------------------------------------- B: the pair sums
        if (n_act <= kLaneJMax) {
            // a few due particles: every thread takes j-particles of the chunk (one each for chunks of up
            // to 512), runs over the due particles, and the sums go down a warp tree
            float s7[kLaneJMax][7];
#pragma unroll
            for (int q = 0; q < kLaneJMax; ++q) {
#pragma unroll
                for (int v = 0; v < 7; ++v) s7[q][v] = 0.f;
            }
            for (int jl = tid; jl < nb256 * kTileJMax; jl += kStepsThreads) {
                const float* src = L.tiles + (jl >> 8) * 7 * kTileJMax + (jl & 255);
                float jv[7];
#pragma unroll
                for (int c = 0; c < 7; ++c) jv[c] = src[c * kTileJMax];
#pragma unroll
                for (int q = 0; q < kLaneJMax; ++q)
                    if (q < n_act) pair_scalar<true, EPS0>(jv, S.ni[q], S.act[q] == j0 + jl, a.eps2, s7[q]);
            }
#pragma unroll
            for (int q = 0; q < kLaneJMax; ++q) {
                if (q < n_act) {
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
            if (tid < 8 * n_act) {   // the warps' sums in warp order (fp64), one value per thread
                const int q = tid >> 3, v = tid & 7;
                double t = 0.0;
                if (v < 7) {
#pragma unroll
                    for (int w = 0; w < kSW; ++w) t += static_cast<double>(S.red[w][q][v]);
                }
                st_row(rows + (static_cast<size_t>(cta) * a.max_act + q) * 8 + v, row_word(static_cast<float>(t), seq));
            }
        } else {
            // nit i-tiles of 32 due particles (lane = particle); wj warps split the chunk for one i-tile,
            // kSW / wj i-tiles run side by side, in rounds
            const int nit = (n_act + 31) >> 5;
            // wj warps per i-tile, kSW / wj i-tiles per round: the split with the least (rounds x (chunk / wj + a
            // round's fixed part, about a tenth of a chunk)); e.g. 24 tiles: 3 rounds of half chunks, not 2 of whole
            int wj = kSW, best = 1 << 30;
            for (int w = kSW; w >= 1; w >>= 1) {
                const int rounds = (nit * w + kSW - 1) / kSW;
                const int cost = rounds * (160 / w + 16);
                if (cost < best) { best = cost; wj = w; }
            }
            const int ng = kSW / wj;
            const int ws = warp % wj, wg = warp / wj;
            const int g4 = chunk >> 2;                        // groups of 4 j-particles in the chunk
            const int jb = ((ws * g4) / wj) << 2, je = (((ws + 1) * g4) / wj) << 2;
            for (int r = 0; r * ng < nit; ++r) {
                const int it = r * ng + wg;
                const int q = it * 32 + lane;
                const bool valid = it < nit && q < n_act;
                float ni[1][6] = {{0.f, 0.f, 0.f, 0.f, 0.f, 0.f}};
                int self = -1;
                if (valid) {
#pragma unroll
                    for (int c = 0; c < 6; ++c) ni[0][c] = S.ni[q][c];
                    self = S.act[q];
                }
                double d[10];
#pragma unroll
                for (int v = 0; v < 10; ++v) d[v] = 0.0;
                if (it < nit) {
                    u64 acc[1][10];
                    float tmin[1] = {0.f};
#pragma unroll
                    for (int v = 0; v < 10; ++v) acc[0][v] = 0ull;
                    for (int b = jb >> 8; (b << 8) < je; ++b) {   // 256-particle blocks of the slice
                        const int lo = max(jb, b << 8) - (b << 8), hi = min(je, (b + 1) << 8) - (b << 8);
                        const float* sx = L.tiles + b * 7 * kTileJMax;
                        int sl[1] = {self - j0 - (b << 8)};
                        const bool own = static_cast<unsigned>(sl[0]) < static_cast<unsigned>(kTileJMax);
                        if (__any_sync(0xffffffffu, own)) tile_packed<1, true, EPS0, true, false, false>(sx, lo, hi, ni, sl, acc, a.eps2, tmin);
                        else tile_packed<1, true, EPS0, false, false, false>(sx, lo, hi, ni, sl, acc, a.eps2, tmin);
#pragma unroll
                        for (int v = 0; v < 10; ++v) d[v] += static_cast<double>(acc_take(acc[0][v]));
                    }
                }
                double t7[7] = {d[0], d[1], d[2], d[3], d[4] - 3.0 * d[7], d[5] - 3.0 * d[8], d[6] - 3.0 * d[9]};
                if (wj > 1) {   // the wj slices of one i-tile: added by the warp with slice 0, in order
#pragma unroll
                    for (int v = 0; v < 7; ++v) S.scratch[warp][lane][v] = t7[v];
                    __syncthreads();
                    if (ws == 0) {
#pragma unroll
                        for (int w = 1; w < kSW; ++w) {
                            if (w < wj) {
#pragma unroll
                                for (int v = 0; v < 7; ++v) t7[v] += S.scratch[warp + w][lane][v];
                            }
                        }
                    }
                }
                if (ws == 0 && valid) {
                    unsigned long long* dst = rows + (static_cast<size_t>(cta) * a.max_act + q) * 8;
#pragma unroll
                    for (int v = 0; v < 7; ++v) st_row(dst + v, row_word(static_cast<float>(t7[v]), seq));
                }
                if (wj > 1) __syncthreads();   // scratch is reused by the next round
            }
        }
        // ------------------------------------------------------ C: reduce + correct, by the owning CTA
        // Due particle q belongs to CTA q mod G.  All its threads fetch the G rows at once (thread =
        // (row, half): one round trip), wait until every word carries this step's number, and add the
        // rows in CTA order: lanes of a warp by a fixed tree, then the warps in order.
        for (int myq = cta; myq < n_act; myq += G) {
            const int my_i = S.act[myq];
            const int k0 = L.lev[my_i] - 1;
            double old_state = 0.0;   // warp 0: the particle's fp64 state, one lane per value (x v a j) x (3)
            if (warp == 0 && lane < 12) {
                const double* arr = lane < 3 ? hs.x : lane < 6 ? hs.v : lane < 9 ? hs.a : hs.j;
                old_state = __ldcg(arr + 3 * static_cast<size_t>(my_i) + lane % 3);
            }
            const int k = tid >> 1, hf = tid & 1;
            double v4[4] = {0.0, 0.0, 0.0, 0.0};
            if (k < G) {
                const unsigned long long* p = rows + (static_cast<size_t>(k) * a.max_act + myq) * 8 + 4 * hf;
                ulonglong2 w0, w1;
                long long spins = 0;
                for (;;) {
                    w0 = ld_row2(p);
                    w1 = ld_row2(p + 2);
                    const bool ok = static_cast<unsigned>(w0.x >> 32) == seq && static_cast<unsigned>(w0.y >> 32) == seq &&
                                    static_cast<unsigned>(w1.x >> 32) == seq &&
                                    (hf || static_cast<unsigned>(w1.y >> 32) == seq);   // word 7 is not used
                    if (ok) break;
                    if (spin_abort(spins, h)) { S.err = 1; break; }   // never hang the device
                }
                v4[0] = __uint_as_float(static_cast<unsigned>(w0.x)); v4[1] = __uint_as_float(static_cast<unsigned>(w0.y));
                v4[2] = __uint_as_float(static_cast<unsigned>(w1.x)); v4[3] = hf ? 0.0 : __uint_as_float(static_cast<unsigned>(w1.y));
            }
#pragma unroll
            for (int o = 2; o < 32; o <<= 1) {
#pragma unroll
                for (int e = 0; e < 4; ++e) v4[e] += __shfl_xor_sync(0xffffffffu, v4[e], o);
            }
            if (lane < 2) {
#pragma unroll
                for (int e = 0; e < 4; ++e) S.scratch[warp][lane][e] = v4[e];
            }
            __syncthreads();
            if (warp == 0 && !S.err) {   // (a wait gave up: the rows are not this step's -- correct nothing, publish no flag)
                double sv = 0.0;   // lane v < 7: sum v (acc3, m/sqrt(s), jerk3)
                if (lane < 8) {
#pragma unroll
                    for (int w = 0; w < kSW; ++w) sv += S.scratch[w][lane >> 2][lane & 3];
                }
                // lane c < 3 corrects component c
                const int c = lane % 3;
                const double x = __shfl_sync(0xffffffffu, old_state, c), v = __shfl_sync(0xffffffffu, old_state, 3 + c);
                const double a0 = __shfl_sync(0xffffffffu, old_state, 6 + c), jk0 = __shfl_sync(0xffffffffu, old_state, 9 + c);
                const double a1 = static_cast<float>(__shfl_sync(0xffffffffu, sv, c));       // one rounding to fp32
                const double j1 = static_cast<float>(__shfl_sync(0xffffffffu, sv, 4 + c));
                double x1, v1, a2e, a3;
                correct_component(x, v, a0, jk0, a1, j1, k0, x1, v1, a2e, a3);
                if (lane < 3) store_corrected(raw, hs, my_i, c, x1, v1, a1, j1);
                // squared norms over the three component lanes, (c0 + c1) + c2, in every lane; lane e < 4 takes
                // the root of norm e (|a1|, |j1|, |a2'|, |a3|): four square roots side by side
                const double sq[4] = {a1 * a1, j1 * j1, a2e * a2e, a3 * a3};
                double mine = 0.0;
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const double tot = (__shfl_sync(0xffffffffu, sq[e], 0) + __shfl_sync(0xffffffffu, sq[e], 1)) +
                                       __shfl_sync(0xffffffffu, sq[e], 2);
                    mine = lane == e ? tot : mine;
                }
                mine = sqrt(mine);
                const double na = __shfl_sync(0xffffffffu, mine, 0), nj = __shfl_sync(0xffffffffu, mine, 1);
                const double n2 = __shfl_sync(0xffffffffu, mine, 2), n3 = __shfl_sync(0xffffffffu, mine, 3);
                __syncwarp();   // the component lanes' stores happen before lane 0's fence (cumulative) and flag
                if (lane == 0) {
                    raw.t[my_i] = t_next;
                    const int kn = next_level_norms(na, nj, n2, n3, eta, k0, kmin, T_next);
                    store_level(hs, h, my_i, k0, kn);
                    __threadfence();   // state, level tables, then the flag: step number and new level
                    const unsigned long long f = (static_cast<unsigned long long>(seq) << 32) |
                                                 static_cast<unsigned long long>(kn);
                    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(hs.flag + myq), "l"(f) : "memory");
                }
            }
            __syncthreads();   // scratch is reused by the CTA's next particle
        }
        if (cta == 0 && tid == 0) {
            int b = 0;
            while ((2LL << b) <= n_act && b < 31) ++b;
            S.hist[b] += 1;
        }
        steps_done += 1;
        psteps += n_act;
        n_prev = n_act;
        T_now = T_next;
    }
    if (cta == 0) {   // bookkeeping of the whole launch
        if (tid == 0) {
            h->T_now = T_now;
            h->seq = seq0 + static_cast<unsigned>(steps_done);
            h->block_steps += steps_done;
            h->particle_steps += psteps;
            h->interactions += psteps * n;
            if (stop == 2) { h->done = 1; h->n_act = 0; }
            if (stop == 3) h->error = 1;
        }
        if (tid < 32) h->hist[tid] += S.hist[tid];
    }
}

cudaError_t steps_prepare(int chunk, int n_lev, int* ctas_per_sm) {
    const size_t smem = steps_smem_bytes(chunk, n_lev);
    int nb = 0, nb1 = 0;
    cudaError_t e;
    if ((e = cudaFuncSetAttribute(hd_steps_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem))) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(hd_steps_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(smem))) != cudaSuccess) return e;
    if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, hd_steps_kernel<false>, kStepsThreads, smem)) != cudaSuccess) return e;
    if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb1, hd_steps_kernel<true>, kStepsThreads, smem)) != cudaSuccess) return e;
    *ctas_per_sm = nb < nb1 ? nb : nb1;
    return cudaSuccess;
}

cudaError_t launch_hd_steps(const StepsArgs& a, bool eps0, int grid, bool cooperative, cudaStream_t st) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(static_cast<unsigned>(grid), 1, 1);
    cfg.blockDim = dim3(kStepsThreads, 1, 1);
    cfg.dynamicSmemBytes = steps_smem_bytes(a.chunk, a.n_lev);
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeCooperative;
    at[0].val.cooperative = cooperative ? 1 : 0;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    if (eps0) return cudaLaunchKernelEx(&cfg, hd_steps_kernel<true>, a);
    return cudaLaunchKernelEx(&cfg, hd_steps_kernel<false>, a);
}

}  // namespace nbk

