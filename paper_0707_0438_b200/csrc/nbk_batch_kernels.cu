// nbk_batch_kernels.cu -- kernels of the batched acc + pot calls: list packing,
// the segmented stream-K force kernel, the ordered reduction.  Host side: nbk_batch.cu.
#include "nbk_device.cuh"

namespace nbk {

// --------------------------------------------------- batched acc + pot calls
// the GRAPE treecode sends, per group of <= ncrit particles, an
// interaction list and asks for the acceleration (no jerk, no neighbours) on the group's particles;
// one library call per group made the paper choose ncrit of 8192-32768.  Here all groups of a step
// go into one launch: the pair list is the concatenation over groups of their (i-tile, j-tile)
// pairs, cut into G equal ranges like the single-problem kernel; a CTA walks its range group by
// group.  Every (CTA, i-tile) segment writes one partial row (row = segment index + CTA index is
// unique and ordered); batch_reduce_kernel adds each i-tile's rows in CTA order (deterministic).
struct BatchCursor {
    int g, it, jt, nit, njt;
    long long joff, seg;
};
__device__ __forceinline__ void batch_load_group(const BatchArgs& a, BatchCursor& c) {
    c.njt = a.njt[c.g];
    c.nit = (a.i_end[c.g] - a.i_off[c.g] + a.ti - 1) / a.ti;
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

template <bool EPS0>
__global__ void __launch_bounds__(512, 1) batch_kernel(const BatchArgs a) {
    constexpr int I = 1, W = 16, T = 512, NACC = 4;
    using S = Shape<false>;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const uint32_t full0 = smem_u32(smem_raw);
    const uint32_t empty0 = full0 + 8 * kStages;
    float* stages = reinterpret_cast<float*>(smem_raw + 128);
    double* sacc = reinterpret_cast<double*>(smem_raw + 128 + sizeof(float) * kStages * S::stage_floats);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int wjn = a.wj;
    const int wj = warp % wjn, wi = warp / wjn;
    const int jlen = a.tj / wjn, jbeg = wj * jlen;
    const long long p0 = pair_start(blockIdx.x, a.P, a.G);
    const long long p1 = pair_start(blockIdx.x + 1LL, a.P, a.G);
    const int n_local = static_cast<int>(p1 - p0);
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < kStages; ++s) {
            mbar_init(full0 + 8 * s, 1);
            mbar_init(empty0 + 8 * s, W);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    auto issue = [&](const BatchCursor& c, int slot) {
        const uint32_t bytes = a.tj * sizeof(float);
        constexpr uint32_t stride = kTileJMax * sizeof(float);
        const size_t off = static_cast<size_t>(c.joff) + static_cast<size_t>(c.jt) * a.tj;
        const uint32_t bar = full0 + 8 * slot;
        mbar_expect_tx(bar, bytes * 4);
        const uint32_t dst = smem_u32(stages + slot * S::stage_floats);
        bulk_g2s(dst + 0 * stride, a.x + off, bytes, bar);
        bulk_g2s(dst + 1 * stride, a.y + off, bytes, bar);
        bulk_g2s(dst + 2 * stride, a.z + off, bytes, bar);
        bulk_g2s(dst + 3 * stride, a.m + off, bytes, bar);
    };
    BatchCursor pc;          // producer's cursor (thread 0 only), kPrefetch tiles ahead
    if (tid == 0) {
        batch_seek(a, p0, pc);
        for (int s = 0; s < kPrefetch && s < n_local; ++s) {
            issue(pc, s);
            batch_advance(a, pc);
        }
    }
    BatchCursor c;
    batch_seek(a, p0, c);
    float ni[I][6];
    int sl[I] = {-1};
    u64 acc[I][NACC];
    float tmin[I];
    bool fresh = true;
    for (int n = 0; n < n_local; ++n) {
        if (tid == 0) {
            const int mth = n + kPrefetch;
            if (mth < n_local) {
                const int slot = mth % kStages;
                if (mth >= kStages) mbar_wait(empty0 + 8 * slot, ((mth / kStages) - 1) & 1);
                issue(pc, slot);
                batch_advance(a, pc);
            }
        }
        if (fresh) {
            const int il = wi * 32 + lane;
            const int i_lo = a.i_off[c.g], n_i = a.i_end[c.g] - i_lo;
            const int i = c.it * a.ti + il;
            float x = 0.f, y = 0.f, z = 0.f;
            if (i < n_i) {
                const float* p = a.xi + 3 * static_cast<size_t>(i_lo + i);
                x = p[0]; y = p[1]; z = p[2];
            }
            ni[0][0] = -x; ni[0][1] = -y; ni[0][2] = -z;
            ni[0][3] = ni[0][4] = ni[0][5] = 0.f;
#pragma unroll
            for (int v = 0; v < NACC; ++v) {
                sacc[v * T + tid] = 0.0;
                acc[0][v] = 0ull;
            }
            fresh = false;
        }
        const int slot = n % kStages;
        mbar_wait(full0 + 8 * slot, (n / kStages) & 1);
        tile_packed<I, false, EPS0, false, false>(stages + slot * S::stage_floats, jbeg, jbeg + jlen,
                                                  ni, sl, acc, a.eps2, tmin);
        __syncwarp();
        if (lane == 0) mbar_arrive(empty0 + 8 * slot);
#pragma unroll
        for (int v = 0; v < NACC; ++v) sacc[v * T + tid] += static_cast<double>(acc_take(acc[0][v]));
        if (c.jt == c.njt - 1 || n == n_local - 1) {   // end of this CTA's part of the i-tile
            if (wjn > 1) __syncthreads();
            const long long row = c.seg + c.it + blockIdx.x;
            if (wj == 0) {
                const int il = wi * 32 + lane;
                double t[NACC];
#pragma unroll
                for (int v = 0; v < NACC; ++v) t[v] = sacc[v * T + tid];
                for (int w = 1; w < wjn; ++w) {
#pragma unroll
                    for (int v = 0; v < NACC; ++v) t[v] += sacc[v * T + tid + 32 * w];
                }
                float4 o;
                o.x = static_cast<float>(t[0]); o.y = static_cast<float>(t[1]);
                o.z = static_cast<float>(t[2]); o.w = static_cast<float>(t[3]);
                *reinterpret_cast<float4*>(a.partial + (row * a.ti + il) * 4) = o;
            }
            if (wjn > 1) __syncthreads();
            fresh = true;
        }
        batch_advance(a, c);
    }
}

// one block per i-tile (segment): add the rows of the CTAs that worked on it, in CTA order
__global__ void batch_reduce_kernel(const BatchArgs a) {
    const long long s = blockIdx.x;
    int lo = 0, hi = a.n_groups - 1;
    while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if (a.seg_prefix[mid] <= s) lo = mid; else hi = mid - 1;
    }
    const int g = lo;
    const int it = static_cast<int>(s - a.seg_prefix[g]);
    const int i_lo = a.i_off[g], n_i = a.i_end[g] - i_lo;
    const int il = threadIdx.x;
    const int i = it * a.ti + il;
    if (i >= n_i) return;
    const long long pl = a.pair_prefix[g] + static_cast<long long>(it) * a.njt[g];
    const long long ph = pl + a.njt[g] - 1;
    long long k0 = (pl * a.G) / a.P;
    while (k0 + 1 < a.G && pair_start(k0 + 1, a.P, a.G) <= pl) ++k0;
    while (k0 > 0 && pair_start(k0, a.P, a.G) > pl) --k0;
    long long k1 = (ph * a.G) / a.P;
    while (k1 + 1 < a.G && pair_start(k1 + 1, a.P, a.G) <= ph) ++k1;
    while (k1 > 0 && pair_start(k1, a.P, a.G) > ph) --k1;
    double t[4] = {0, 0, 0, 0};
    for (long long k = k0; k <= k1; ++k) {
        const float4 o = *reinterpret_cast<const float4*>(a.partial + ((s + k) * a.ti + il) * 4);
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
    return 128 + sizeof(float) * kStages * Shape<false>::stage_floats + sizeof(double) * 4 * 512;
}

cudaError_t batch_prepare() {
    cudaError_t e = cudaFuncSetAttribute(batch_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         static_cast<int>(batch_smem_bytes()));
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(batch_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                static_cast<int>(batch_smem_bytes()));
}

cudaError_t launch_batch_pack(const BatchPackArgs& a, cudaStream_t s) {
    if (a.n_padded <= 0) return cudaSuccess;
    batch_pack_kernel<<<static_cast<unsigned>((a.n_padded + 255) / 256), 256, 0, s>>>(a);
    return cudaGetLastError();
}

cudaError_t launch_batch(const BatchArgs& a, bool eps0, cudaStream_t s) {
    if (eps0) batch_kernel<true><<<a.G, 512, batch_smem_bytes(), s>>>(a);
    else batch_kernel<false><<<a.G, 512, batch_smem_bytes(), s>>>(a);
    return cudaGetLastError();
}

cudaError_t launch_batch_reduce(const BatchArgs& a, cudaStream_t s) {
    batch_reduce_kernel<<<static_cast<unsigned>(a.n_seg), a.ti, 0, s>>>(a);
    return cudaGetLastError();
}


}  // namespace nbk
