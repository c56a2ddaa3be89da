// nbk_batch.cu -- nbk_calc_batch[_dev]: many (i-group, interaction-list) acc + pot problems in one
// launch.  Host side only: descriptors, arena, launches; kernels in nbk_batch_kernels.cu.
#include <chrono>
#include <climits>
#include <cmath>
#include <cstring>
#include <vector>

#include "nbk_ctx.cuh"

using namespace nbk;

// ---- batched acc + pot calls -------------------------------------------------
namespace {

int batch_impl(nbk_ctx* c, int64_t n_groups, const int64_t* i_offset, const float* xi,
               const int64_t* j_offset, const float* mj, const float* xj, float eps2, uint32_t flags,
               float* acc, float* pot, bool dev) {
    if (!c || n_groups < 0 || !(eps2 >= 0.f) || (flags & (NBK_JERK | NBK_NN))) return NBK_EINVAL;
    eps2 = flushed_eps2(eps2);
    if (n_groups == 0) return NBK_OK;
    if (!i_offset || !j_offset || i_offset[0] != 0 || j_offset[0] != 0) return NBK_EINVAL;
    for (int64_t g = 0; g < n_groups; ++g)
        if (i_offset[g + 1] < i_offset[g] || j_offset[g + 1] < j_offset[g]) return NBK_EINVAL;
    const int64_t ni_tot = i_offset[n_groups], nj_tot = j_offset[n_groups];
    if (ni_tot > INT32_MAX || n_groups > INT32_MAX) return NBK_ERANGE;
    if (ni_tot == 0) return NBK_OK;
    if (!xi || !acc || !pot || (nj_tot > 0 && (!mj || !xj))) return NBK_EINVAL;
    DeviceGuard g(c->device);
    if (!g.ok) return cuda_fail(c, cudaErrorInvalidDevice);
    if (!c->batch_ready) {
        NBK_CUDA(c, batch_prepare());
        c->batch_ready = true;
    }
    // launch form from the mean group size: a chunk (what one warp works on) is 64 i-particles (two per
    // lane), 32, or -- small groups -- 16 or 8 with the lanes splitting each j-tile 2 or 4 ways
    std::vector<int> keep;
    int64_t sum_ni = 0;
    for (int64_t q = 0; q < n_groups; ++q)
        if (i_offset[q + 1] > i_offset[q] && j_offset[q + 1] > j_offset[q]) {
            keep.push_back(static_cast<int>(q));
            sum_ni += i_offset[q + 1] - i_offset[q];
        }
    const size_t ni = static_cast<size_t>(ni_tot);
    float* d_acc = acc;
    float* d_pot = pot;
    const int ng = static_cast<int>(keep.size());
    const long long mean = ng > 0 ? sum_ni / ng : 0;
    const int ipl = mean >= 96 ? 2 : 1;
    const int slices = mean >= 24 ? 1 : (mean >= 12 ? 2 : 4);
    const int ti = 32 * ipl / slices, tj = 128;   // ti: i-particles per chunk
    std::vector<long long> pair_prefix(ng + 1, 0), seg_prefix(ng + 1, 0), joff(ng + 1, 0), src_off(ng + 1, 0);
    std::vector<int> ioff(ng + 1, 0), njt(ng > 0 ? ng : 1, 0);
    for (int q = 0; q < ng; ++q) {
        const int64_t gg = keep[q];
        const long long n_i = i_offset[gg + 1] - i_offset[gg], n_j = j_offset[gg + 1] - j_offset[gg];
        const long long nit = (n_i + ti - 1) / ti, nt = (n_j + tj - 1) / tj;
        njt[q] = static_cast<int>(nt);
        pair_prefix[q + 1] = pair_prefix[q] + nit * nt;
        seg_prefix[q + 1] = seg_prefix[q] + nit;
        joff[q + 1] = joff[q] + nt * tj;
    }
    const long long P = pair_prefix[ng], n_seg = seg_prefix[ng], n_padded = joff[ng];
    const long long gmax = 16LL * (c->num_sms < kMaxCtas ? c->num_sms : kMaxCtas);   // workers: all warps of the grid
    const long long G = P < gmax ? P : gmax;
    if ((P + G - 1) / (G > 0 ? G : 1) > INT_MAX) return NBK_ERANGE;
    // arena: [x y z m | descriptors | partial | (host entry: xi, mj, xj, acc, pot)]
    size_t off = 0;
    auto take = [&](size_t bytes) { const size_t at = off; off += (bytes + 255) & ~static_cast<size_t>(255); return at; };
    const size_t o_x = take(4 * sizeof(float) * n_padded);
    const size_t o_pp = take(sizeof(long long) * (ng + 1)), o_sp = take(sizeof(long long) * (ng + 1));
    const size_t o_jo = take(sizeof(long long) * (ng + 1)), o_so = take(sizeof(long long) * (ng + 1));
    const size_t o_do = take(sizeof(long long) * (ng + 1));
    const size_t o_io = take(sizeof(int) * (ng + 1)), o_nt = take(sizeof(int) * (ng + 1));
    const size_t o_ie = take(sizeof(int) * (ng + 1)), o_sl = take(sizeof(long long) * (ng + 1));
    const size_t o_part = take(sizeof(float) * 4 * ti * static_cast<size_t>(n_seg + G));
    size_t o_xi = 0, o_mj = 0, o_xj = 0, o_acc = 0, o_pot = 0;
    if (!dev) {
        o_xi = take(sizeof(float) * 3 * ni);
        o_mj = take(sizeof(float) * nj_tot);
        o_xj = take(sizeof(float) * 3 * nj_tot);
        o_acc = take(sizeof(float) * 3 * ni);
        o_pot = take(sizeof(float) * ni);
    }
    if (off > c->batch_bytes) {
        NBK_CUDA(c, cudaStreamSynchronize(c->stream));
        cudaFree(c->d_batch);
        c->d_batch = nullptr;
        c->batch_bytes = 0;
        NBK_CUDA(c, cudaMalloc(&c->d_batch, off + off / 4));
        c->batch_bytes = off + off / 4;
    }
    unsigned char* B = c->d_batch;
    // descriptors of the non-empty groups: i offsets are the caller's (outputs keep the caller's order)
    std::vector<long long> src_len(ng > 0 ? ng : 1, 0);
    for (int q = 0; q < ng; ++q) {
        ioff[q] = static_cast<int>(i_offset[keep[q]]);
        src_off[q] = j_offset[keep[q]];
        src_len[q] = j_offset[keep[q] + 1] - j_offset[keep[q]];
    }
    std::vector<int> iend(ng > 0 ? ng : 1);
    for (int q = 0; q < ng; ++q) iend[q] = static_cast<int>(i_offset[keep[q] + 1]);
    if (ng > 0) src_off[ng] = j_offset[keep[ng - 1] + 1];
    if (!dev) {
        NBK_CUDA(c, cudaMemcpyAsync(B + o_xi, xi, sizeof(float) * 3 * ni, cudaMemcpyHostToDevice, c->stream));
        if (nj_tot > 0) {
            NBK_CUDA(c, cudaMemcpyAsync(B + o_mj, mj, sizeof(float) * nj_tot, cudaMemcpyHostToDevice, c->stream));
            NBK_CUDA(c, cudaMemcpyAsync(B + o_xj, xj, sizeof(float) * 3 * nj_tot, cudaMemcpyHostToDevice, c->stream));
        }
        d_acc = reinterpret_cast<float*>(B + o_acc);
        d_pot = reinterpret_cast<float*>(B + o_pot);
    }
    NBK_CUDA(c, cudaMemsetAsync(d_acc, 0, sizeof(float) * 3 * ni, c->stream));
    NBK_CUDA(c, cudaMemsetAsync(d_pot, 0, sizeof(float) * ni, c->stream));
    if (ng > 0) {
        // pageable host vectors: these copies complete before the call returns to the vectors' scope end
        NBK_CUDA(c, cudaMemcpyAsync(B + o_pp, pair_prefix.data(), sizeof(long long) * (ng + 1), cudaMemcpyHostToDevice, c->stream));
        NBK_CUDA(c, cudaMemcpyAsync(B + o_sp, seg_prefix.data(), sizeof(long long) * (ng + 1), cudaMemcpyHostToDevice, c->stream));
        NBK_CUDA(c, cudaMemcpyAsync(B + o_jo, joff.data(), sizeof(long long) * (ng + 1), cudaMemcpyHostToDevice, c->stream));
        NBK_CUDA(c, cudaMemcpyAsync(B + o_so, src_off.data(), sizeof(long long) * (ng + 1), cudaMemcpyHostToDevice, c->stream));
        NBK_CUDA(c, cudaMemcpyAsync(B + o_io, ioff.data(), sizeof(int) * (ng + 1), cudaMemcpyHostToDevice, c->stream));
        NBK_CUDA(c, cudaMemcpyAsync(B + o_nt, njt.data(), sizeof(int) * ng, cudaMemcpyHostToDevice, c->stream));
        NBK_CUDA(c, cudaMemcpyAsync(B + o_ie, iend.data(), sizeof(int) * ng, cudaMemcpyHostToDevice, c->stream));
        NBK_CUDA(c, cudaMemcpyAsync(B + o_sl, src_len.data(), sizeof(long long) * ng, cudaMemcpyHostToDevice, c->stream));
        BatchPackArgs pk;
        pk.mj = dev ? mj : reinterpret_cast<const float*>(B + o_mj);
        pk.xj = dev ? xj : reinterpret_cast<const float*>(B + o_xj);
        pk.src_off = reinterpret_cast<const long long*>(B + o_so);
        pk.dst_off = reinterpret_cast<const long long*>(B + o_jo);
        pk.src_len = reinterpret_cast<const long long*>(B + o_sl);
        float* px = reinterpret_cast<float*>(B + o_x);
        pk.x = px; pk.y = px + n_padded; pk.z = px + 2 * n_padded; pk.m = px + 3 * n_padded;
        pk.n_groups = ng;
        pk.n_padded = n_padded;
        NBK_CUDA(c, launch_batch_pack(pk, c->stream));
        BatchArgs ba;
        ba.x = pk.x; ba.y = pk.y; ba.z = pk.z; ba.m = pk.m;
        ba.xi = dev ? xi : reinterpret_cast<const float*>(B + o_xi);
        ba.pair_prefix = reinterpret_cast<const long long*>(B + o_pp);
        ba.seg_prefix = reinterpret_cast<const long long*>(B + o_sp);
        ba.j_off = reinterpret_cast<const long long*>(B + o_jo);
        ba.i_off = reinterpret_cast<const int*>(B + o_io);
        ba.njt = reinterpret_cast<const int*>(B + o_nt);
        ba.i_end = reinterpret_cast<const int*>(B + o_ie);
        ba.partial = reinterpret_cast<float*>(B + o_part);
        ba.acc = d_acc; ba.pot = d_pot;
        ba.n_groups = ng; ba.ci = ti; ba.ipl = ipl; ba.slices = slices;
        ba.P = P; ba.n_seg = n_seg; ba.G = G; ba.eps2 = eps2;
        {
            TimeScope ts(c, 2);
            NBK_CUDA(c, launch_batch(ba, (flags & NBK_EPS0) != 0 || eps2 == 0.f, c->stream));
        }
        {
            TimeScope ts(c, 3);
            NBK_CUDA(c, launch_batch_reduce(ba, c->stream));
        }
        c->last_launch[0] = (G + 15) / 16; c->last_launch[1] = 512; c->last_launch[2] = ipl; c->last_launch[3] = slices;
        c->last_launch[4] = tj; c->last_launch[5] = c->num_sms;
        c->last_launch[6] = static_cast<long long>(batch_smem_bytes()); c->last_launch[7] = 3;
    }
    if (!dev) {
        NBK_CUDA(c, cudaMemcpyAsync(acc, d_acc, sizeof(float) * 3 * ni, cudaMemcpyDeviceToHost, c->stream));
        NBK_CUDA(c, cudaMemcpyAsync(pot, d_pot, sizeof(float) * ni, cudaMemcpyDeviceToHost, c->stream));
    }
    // the descriptor vectors live on this stack frame: wait until their copies have been consumed
    NBK_CUDA(c, cudaStreamSynchronize(c->stream));
    return NBK_OK;
}

}  // namespace

extern "C" {


int nbk_calc_batch(nbk_ctx* c, int64_t n_groups, const int64_t* i_offset, const float* xi,
                   const int64_t* j_offset, const float* mj, const float* xj, float eps2,
                   uint32_t flags, float* acc, float* pot) {
    return batch_impl(c, n_groups, i_offset, xi, j_offset, mj, xj, eps2, flags, acc, pot, false);
}

int nbk_calc_batch_dev(nbk_ctx* c, int64_t n_groups, const int64_t* i_offset, const float* xi,
                       const int64_t* j_offset, const float* mj, const float* xj, float eps2,
                       uint32_t flags, float* acc, float* pot) {
    return batch_impl(c, n_groups, i_offset, xi, j_offset, mj, xj, eps2, flags, acc, pot, true);
}
}  // extern "C"
