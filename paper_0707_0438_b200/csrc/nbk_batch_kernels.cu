// nbk_batch_kernels.cu -- kernels of the batched acc + pot calls: list packing,
// the segmented stream-K force kernel, the ordered reduction.  Host side: nbk_batch.cu.
#include "nbk_device.cuh"

namespace nbk {

// --------------------------------------------------- batched acc + pot calls
// the GRAPE treecode sends, per group of <= ncrit particles, an
// interaction list and asks for the acceleration (no jerk, no neighbours) on the group's particles;
// one library call per group made the paper choose ncrit of 8192-32768.  Here all groups of a step
// go into one launch, and the unit that is scheduled is small enough for groups of a few particles:
//   * a chunk is ci = 32 I / S i-particles of one group: I per lane (1 or 2), or, for small groups, the
//     warp's lanes split S = 2 or 4 ways over the j-particles of a tile (lane = slice x particle);
//   * the pair list is the concatenation over groups of their (chunk, j-tile) pairs, cut into equal
//     contiguous ranges over ALL WARPS of the grid (stream-K at warp granularity); a warp walks its
//     range on its own: its own ring of j-tiles filled by TMA bulk copies that one of its lanes
//     issues, its own mbarriers, no CTA-wide synchronisation anywhere;
//   * every (warp, chunk) segment writes one partial row (row = chunk index + warp index is unique
//     and ordered); batch_reduce_kernel adds each chunk's rows in warp order (deterministic).
constexpr int kBW = 16;          // warps per CTA
constexpr int kBTj = 128;        // j-particles per tile
constexpr int kBStages = 4;      // tiles in a warp's ring

struct BatchCursor {
    int g, it, jt, nit, njt;
    long long joff, seg;
};
__device__ __forceinline__ void batch_load_group(const BatchArgs& a, BatchCursor& c) {
    c.njt = a.njt[c.g];
    c.nit = (a.i_end[c.g] - a.i_off[c.g] + a.ci - 1) / a.ci;
    c.joff = a.j_off[c.g];
    c.seg = a.seg_prefix[c.g];
}
__device__ __forceinline__ void batch_seek(const BatchArgs& a, long long p, BatchCursor& c) {
    int lo = 0, hi = a.n_groups - 1;     // largest g with pair_prefix[g] <= p
    while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if (a.pair_prefix[mid] <= p) lo = mid; else hi = mid - 1;
    }
    c.g = lo;
    batch_load_group(a, c);
    const long long r = p - a.pair_prefix[lo];
    c.it = static_cast<int>(r / c.njt);
    c.jt = static_cast<int>(r - static_cast<long long>(c.it) * c.njt);
}
__device__ __forceinline__ void batch_advance(const BatchArgs& a, BatchCursor& c) {
    if (++c.jt == c.njt) {
        c.jt = 0;
        if (++c.it == c.nit) {
            c.it = 0;
            if (++c.g < a.n_groups) batch_load_group(a, c);
        }
    }
}

// acc + pot pair sums of I i-particles per lane over the j-particles jbeg, jbeg + jstep, ... < jend
// (4 at a time) of one tile: the arithmetic of tile_packed without the jerk terms.
// sx: x y z m, kBTj floats each.
template <int I, bool EPS0>
__device__ __forceinline__ void tile_acc(const float* __restrict__ sx, int jbeg, int jend, int jstep,
                                         const float (&ni)[I][3], u64 (&acc)[I][4], float eps2) {
    const u64 e2p = pack(eps2, eps2);
#pragma unroll 1
    for (int jj = jbeg; jj < jend; jj += jstep) {
        const ulonglong2 X = *reinterpret_cast<const ulonglong2*>(sx + jj);
        const ulonglong2 Y = *reinterpret_cast<const ulonglong2*>(sx + kBTj + jj);
        const ulonglong2 Z = *reinterpret_cast<const ulonglong2*>(sx + 2 * kBTj + jj);
        const ulonglong2 M = *reinterpret_cast<const ulonglong2*>(sx + 3 * kBTj + jj);
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const u64 xj = h ? X.y : X.x, yj = h ? Y.y : Y.x, zj = h ? Z.y : Z.x, mj = h ? M.y : M.x;
#pragma unroll
            for (int q = 0; q < I; ++q) {
                const u64 dx = add2(xj, pack(ni[q][0], ni[q][0]));
                const u64 dy = add2(yj, pack(ni[q][1], ni[q][1]));
                const u64 dz = add2(zj, pack(ni[q][2], ni[q][2]));
                u64 r2 = fma2(dx, dx, e2p);
                r2 = fma2(dy, dy, r2);
                r2 = fma2(dz, dz, r2);
                float r2a, r2b;
                unpack(r2, r2a, r2b);
                float ra = rsq(r2a), rb = rsq(r2b);
                if (EPS0) {   // zero-distance pairs contribute nothing
                    ra = r2a > 0.f ? ra : 0.f;
                    rb = r2b > 0.f ? rb : 0.f;
                }
                const u64 rinv = pack(ra, rb);
                const u64 rinv2 = mul2(rinv, rinv);
                const u64 mrinv = mul2(mj, rinv);
                acc[q][3] = add2(acc[q][3], mrinv);
                const u64 mrinv3 = mul2(mrinv, rinv2);
                acc[q][0] = fma2(mrinv3, dx, acc[q][0]);
                acc[q][1] = fma2(mrinv3, dy, acc[q][1]);
                acc[q][2] = fma2(mrinv3, dz, acc[q][2]);
            }
        }
    }
}

// One warp = one worker.  a.slices = S (1, 2, 4): the lanes split S ways over the j-particles of a tile,
// 32 / S lanes over i-particles (I = 1 only).
template <int I, bool EPS0>
__global__ void __launch_bounds__(kBW * 32, 1) batch_kernel(const BatchArgs a) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const long long wg = static_cast<long long>(blockIdx.x) * kBW + warp;   // worker index in the grid
    if (wg >= a.G) return;
    // this warp's shared memory: kBStages full barriers, then kBStages tiles of 4 x kBTj floats
    unsigned char* mine = smem_raw + static_cast<size_t>(warp) * (128 + sizeof(float) * kBStages * 4 * kBTj);
    const uint32_t full0 = smem_u32(mine);
    float* stages = reinterpret_cast<float*>(mine + 128);
    const long long p0 = pair_start(wg, a.P, static_cast<int>(a.G)), p1 = pair_start(wg + 1, a.P, static_cast<int>(a.G));
    const int n_local = static_cast<int>(p1 - p0);
    if (lane == 0) {
#pragma unroll
        for (int s = 0; s < kBStages; ++s) mbar_init(full0 + 8 * s, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncwarp();
    auto issue = [&](const BatchCursor& c, int slot) {
        constexpr uint32_t bytes = kBTj * sizeof(float);
        const size_t off = static_cast<size_t>(c.joff) + static_cast<size_t>(c.jt) * kBTj;
        const uint32_t bar = full0 + 8 * slot;
        mbar_expect_tx(bar, bytes * 4);
        const uint32_t dst = smem_u32(stages + slot * 4 * kBTj);
        bulk_g2s(dst + 0 * bytes, a.x + off, bytes, bar);
        bulk_g2s(dst + 1 * bytes, a.y + off, bytes, bar);
        bulk_g2s(dst + 2 * bytes, a.z + off, bytes, bar);
        bulk_g2s(dst + 3 * bytes, a.m + off, bytes, bar);
    };
    BatchCursor c;
    batch_seek(a, p0, c);
    BatchCursor pc = c;      // the producer lane's cursor, kBStages tiles ahead
    if (lane == 0) {
        for (int s = 0; s < kBStages && s < n_local; ++s) {
            issue(pc, s);
            batch_advance(a, pc);
        }
    }
    const int S = a.slices, isub = 32 / S;
    const int il0 = lane % isub, sl = lane / isub;   // particle and slice of this lane
    float ni[I][3];
    u64 acc[I][4];
    double d[I][4];
    bool fresh = true;
    for (int n = 0; n < n_local; ++n) {
        if (fresh) {
            const int i_lo = a.i_off[c.g], n_i = a.i_end[c.g] - i_lo;
#pragma unroll
            for (int q = 0; q < I; ++q) {
                const int i = c.it * a.ci + q * 32 + il0;
                float x = 0.f, y = 0.f, z = 0.f;
                if (i < n_i) {
                    const float* p = a.xi + 3 * static_cast<size_t>(i_lo + i);
                    x = p[0]; y = p[1]; z = p[2];
                }
                ni[q][0] = -x; ni[q][1] = -y; ni[q][2] = -z;
#pragma unroll
                for (int v = 0; v < 4; ++v) { acc[q][v] = 0ull; d[q][v] = 0.0; }
            }
            fresh = false;
        }
        const int slot = n % kBStages;
        mbar_wait(full0 + 8 * slot, (n / kBStages) & 1);
        tile_acc<I, EPS0>(stages + slot * 4 * kBTj, 4 * sl, kBTj, 4 * S, ni, acc, a.eps2);
        __syncwarp();   // every lane is done with the slot: refill it
        if (lane == 0 && n + kBStages < n_local) {
            issue(pc, slot);
            batch_advance(a, pc);
        }
        // fp32 inside one tile (<= 64 terms per packed half), fp64 above
#pragma unroll
        for (int q = 0; q < I; ++q) {
#pragma unroll
            for (int v = 0; v < 4; ++v) d[q][v] += static_cast<double>(acc_take(acc[q][v]));
        }
        if (c.jt == c.njt - 1 || n == n_local - 1) {   // end of this warp's part of the chunk
            const long long row = c.seg + c.it + wg;
#pragma unroll
            for (int q = 0; q < I; ++q) {
                for (int o = isub; o < 32; o <<= 1) {   // the slices of one particle, fixed order
#pragma unroll
                    for (int v = 0; v < 4; ++v) d[q][v] += __shfl_xor_sync(0xffffffffu, d[q][v], o);
                }
                if (sl == 0) {
                    float4 o4;
                    o4.x = static_cast<float>(d[q][0]); o4.y = static_cast<float>(d[q][1]);
                    o4.z = static_cast<float>(d[q][2]); o4.w = static_cast<float>(d[q][3]);
                    *reinterpret_cast<float4*>(a.partial + (row * a.ci + q * 32 + il0) * 4) = o4;
                }
            }
            fresh = true;
        }
        batch_advance(a, c);
    }
}

// thread = (chunk, particle of the chunk): add the rows of the warps that worked on the chunk, in warp order
__global__ void __launch_bounds__(256) batch_reduce_kernel(const BatchArgs a) {
    const int per = 256 / a.ci;                       // chunks per block
    const long long s = static_cast<long long>(blockIdx.x) * per + threadIdx.x / a.ci;
    const int il = threadIdx.x % a.ci;
    if (s >= a.n_seg) return;
    int lo = 0, hi = a.n_groups - 1;
    while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if (a.seg_prefix[mid] <= s) lo = mid; else hi = mid - 1;
    }
    const int g = lo;
    const int it = static_cast<int>(s - a.seg_prefix[g]);
    const int i_lo = a.i_off[g], n_i = a.i_end[g] - i_lo;
    const int i = it * a.ci + il;
    if (i >= n_i) return;
    // workers k0..k1 hold pairs of this chunk: owner(p) = ceil((p + 1) G / P) - 1
    const long long pl = a.pair_prefix[g] + static_cast<long long>(it) * a.njt[g];
    const long long ph = pl + a.njt[g] - 1;
    const long long k0 = ((pl + 1) * a.G + a.P - 1) / a.P - 1, k1 = ((ph + 1) * a.G + a.P - 1) / a.P - 1;
    double t[4] = {0, 0, 0, 0};
    for (long long k = k0; k <= k1; ++k) {
        const float4 o = *reinterpret_cast<const float4*>(a.partial + ((s + k) * a.ci + il) * 4);
        t[0] += o.x; t[1] += o.y; t[2] += o.z; t[3] += o.w;
    }
    const size_t e = static_cast<size_t>(i_lo + i);
    a.acc[3 * e + 0] = static_cast<float>(t[0]);
    a.acc[3 * e + 1] = static_cast<float>(t[1]);
    a.acc[3 * e + 2] = static_cast<float>(t[2]);
    a.pot[e] = static_cast<float>(-t[3]);
}

// caller's lists (m [n], x [n][3]) -> packed SoA, each list padded to a multiple of tj
__global__ void batch_pack_kernel(const BatchPackArgs a) {
    const long long q = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (q >= a.n_padded) return;
    int lo = 0, hi = a.n_groups - 1;
    while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if (a.dst_off[mid] <= q) lo = mid; else hi = mid - 1;
    }
    const long long r = q - a.dst_off[lo];
    const long long len = a.src_len[lo];
    float x = 1e18f, y = 1e18f, z = 1e18f, m = 0.f;
    if (r < len) {
        const long long sidx = a.src_off[lo] + r;
        x = a.xj[3 * sidx]; y = a.xj[3 * sidx + 1]; z = a.xj[3 * sidx + 2];
        m = a.mj[sidx];
    }
    a.x[q] = x; a.y[q] = y; a.z[q] = z; a.m[q] = m;
}


size_t batch_smem_bytes() {
    return static_cast<size_t>(kBW) * (128 + sizeof(float) * kBStages * 4 * kBTj);
}

cudaError_t batch_prepare() {
    const int smem = static_cast<int>(batch_smem_bytes());
    cudaError_t e;
    if ((e = cudaFuncSetAttribute(batch_kernel<1, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(batch_kernel<1, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(batch_kernel<2, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem)) != cudaSuccess) return e;
    return cudaFuncSetAttribute(batch_kernel<2, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
}

cudaError_t launch_batch_pack(const BatchPackArgs& a, cudaStream_t s) {
    if (a.n_padded <= 0) return cudaSuccess;
    batch_pack_kernel<<<static_cast<unsigned>((a.n_padded + 255) / 256), 256, 0, s>>>(a);
    return cudaGetLastError();
}

cudaError_t launch_batch(const BatchArgs& a, bool eps0, cudaStream_t s) {
    const unsigned grid = static_cast<unsigned>((a.G + kBW - 1) / kBW);
    const size_t smem = batch_smem_bytes();
    if (a.ipl == 2) {
        if (eps0) batch_kernel<2, true><<<grid, kBW * 32, smem, s>>>(a);
        else batch_kernel<2, false><<<grid, kBW * 32, smem, s>>>(a);
    } else {
        if (eps0) batch_kernel<1, true><<<grid, kBW * 32, smem, s>>>(a);
        else batch_kernel<1, false><<<grid, kBW * 32, smem, s>>>(a);
    }
    return cudaGetLastError();
}

cudaError_t launch_batch_reduce(const BatchArgs& a, cudaStream_t s) {
    const long long per = 256 / a.ci;
    batch_reduce_kernel<<<static_cast<unsigned>((a.n_seg + per - 1) / per), 256, 0, s>>>(a);
    return cudaGetLastError();
}


}  // namespace nbk
