// dvh.cuh -- dose-volume-histogram points on the device (plan evaluation).
//
// D_p of a structure = the ceil(p n_s / 100)-th largest dose among its n_s voxels (reading R10).  Exact
// selection by three rounds of radix histograms over an order-preserving integer image of the fp32 dose (11 + 11 + 10
// bits); the host only walks the (small) histograms between rounds.  Mean dose by fixed-order fp64 sums (bit-
// reproducible).  Not on the hot path.
#pragma once
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>
#include <cuda_runtime.h>

namespace imrt {

constexpr int DVH_BINS = 2048;
constexpr int DVH_MAX_PCTS = 16;
constexpr int DVH_SUM_BLOCKS = 592;      // grid of the count / sum kernel (fixed: the summation order depends on it)

struct DvhQuery {
    unsigned int prefix;   // bits of the selection key fixed so far
    unsigned int mask;     // which bits those are
};

struct DvhWork {
    unsigned int* hist;    // [n_structures * DVH_MAX_PCTS][DVH_BINS]
    unsigned int* cnt;     // [n_structures]
    double* sum;           // [n_structures]
    double* part;          // [DVH_SUM_BLOCKS][n_structures] per-block dose sums
    DvhQuery* query;       // [n_structures * n_pcts]
};

// ascending key <=> descending dose (total order on finite floats, -0 < +0)
__host__ __device__ __forceinline__ unsigned int dvh_key(float d) {
#ifdef __CUDA_ARCH__
    unsigned int u = __float_as_uint(d);
#else
    unsigned int u;
    memcpy(&u, &d, 4);
#endif
    u = (u & 0x80000000u) ? ~u : (u | 0x80000000u);   // ascending in d
    return ~u;                                        // descending in d
}
inline float dvh_unkey(unsigned int k) {
    unsigned int u = ~k;
    u = (u & 0x80000000u) ? (u & 0x7FFFFFFFu) : ~u;
    float d;
    memcpy(&d, &u, 4);
    return d;
}

// Voxel count and dose sum per structure.  Deterministic: a warp sums the doses of one structure at a time with a fixed
// butterfly, warps keep private per-structure sums, a block adds its warps' sums in warp order and writes one partial
// per structure; k_dvh_sum_final adds the blocks' partials in block order.  (Counts are integers: atomics commute.)
constexpr int DVH_SUM_WARPS = 8;
__global__ void __launch_bounds__(DVH_SUM_WARPS * 32) k_dvh_count_sum(const float* __restrict__ d, const uint8_t* __restrict__ sid, int n_v,
                                                                      int n_s, unsigned int* cnt, double* part) {
    extern __shared__ double dvh_wsum[];          // [DVH_SUM_WARPS][n_s]
    __shared__ unsigned int s_cnt[256];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int i = threadIdx.x; i < DVH_SUM_WARPS * n_s; i += blockDim.x) dvh_wsum[i] = 0.0;
    for (int i = threadIdx.x; i < 256; i += blockDim.x) s_cnt[i] = 0u;
    __syncthreads();
    const int n_round = (n_v + 31) & ~31;         // whole warps stay in the loop together
    for (int j = blockIdx.x * blockDim.x + threadIdx.x; j < n_round; j += gridDim.x * blockDim.x) {
        const bool in = j < n_v;
        const int sj = in ? (int)sid[j] : -1;
        const double dj = in ? (double)d[j] : 0.0;
        if (in) atomicAdd(&s_cnt[sj], 1u);
        unsigned int todo = __ballot_sync(0xffffffffu, in);
        while (todo) {                             // one structure of the warp's 32 voxels at a time
            const int s0 = __shfl_sync(0xffffffffu, sj, __ffs(todo) - 1);
            const bool mine = sj == s0;
            double v = mine ? dj : 0.0;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
            if (lane == 0) dvh_wsum[warp * n_s + s0] += v;
            todo &= ~__ballot_sync(0xffffffffu, mine);
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < n_s; i += blockDim.x) {
        double t = 0.0;
        for (int w = 0; w < DVH_SUM_WARPS; ++w) t += dvh_wsum[w * n_s + i];
        part[(size_t)blockIdx.x * n_s + i] = t;
        if (s_cnt[i]) atomicAdd(&cnt[i], s_cnt[i]);
    }
}
__global__ void k_dvh_sum_final(const double* __restrict__ part, int n_blocks, int n_s, double* sum) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_s) return;
    double t = 0.0;
    for (int b = 0; b < n_blocks; ++b) t += part[(size_t)b * n_s + i];
    sum[i] = t;
}

// One refinement round: every voxel votes in the histogram of each query of its structure whose prefix it matches.
__global__ void k_dvh_hist(const float* __restrict__ d, const uint8_t* __restrict__ sid, int n_v, const DvhQuery* __restrict__ query,
                           int n_pcts, int shift, unsigned int bin_mask, unsigned int* hist) {
    for (int j = blockIdx.x * blockDim.x + threadIdx.x; j < n_v; j += gridDim.x * blockDim.x) {
        const unsigned int k = dvh_key(d[j]);
        const int q0 = (int)sid[j] * n_pcts;
        for (int q = q0; q < q0 + n_pcts; ++q) {
            const DvhQuery Q = query[q];
            if ((k & Q.mask) == Q.prefix) atomicAdd(&hist[(size_t)q * DVH_BINS + ((k >> shift) & bin_mask)], 1u);
        }
    }
}

// host_dp [n_s][n_pcts], host_mean [n_s].  Synchronises the stream.
inline cudaError_t dvh_points(const DvhWork& W, const float* d, const uint8_t* sid, int n_v, int n_s, const double* pcts, int n_pcts,
                              double* host_dp, double* host_mean, cudaStream_t st, const char** what) {
    cudaError_t e;
#define DVH_TRY(x) do { e = (x); if (e != cudaSuccess) { *what = #x; return e; } } while (0)
    const int nq = n_s * n_pcts;
    std::vector<unsigned int> cnt(n_s);
    std::vector<double> sum(n_s);
    DVH_TRY(cudaMemsetAsync(W.cnt, 0, sizeof(unsigned int) * 256, st));
    DVH_TRY(cudaMemsetAsync(W.sum, 0, sizeof(double) * 256, st));
    const int grid = std::max(1, std::min((n_v + 255) / 256, 148 * 8));
    const int sum_blocks = std::max(1, std::min((n_v + 255) / 256, DVH_SUM_BLOCKS));
    k_dvh_count_sum<<<sum_blocks, DVH_SUM_WARPS * 32, sizeof(double) * DVH_SUM_WARPS * n_s, st>>>(d, sid, n_v, n_s, W.cnt, W.part);
    k_dvh_sum_final<<<(n_s + 63) / 64, 64, 0, st>>>(W.part, sum_blocks, n_s, W.sum);
    DVH_TRY(cudaGetLastError());
    DVH_TRY(cudaMemcpyAsync(cnt.data(), W.cnt, sizeof(unsigned int) * n_s, cudaMemcpyDeviceToHost, st));
    DVH_TRY(cudaMemcpyAsync(sum.data(), W.sum, sizeof(double) * n_s, cudaMemcpyDeviceToHost, st));
    DVH_TRY(cudaStreamSynchronize(st));

    std::vector<DvhQuery> query(nq, DvhQuery{0u, 0u});
    std::vector<long long> rank(nq, 0);   // 1-based rank among the voxels still matching the prefix
    for (int s = 0; s < n_s; ++s) {
        host_mean[s] = cnt[s] ? sum[s] / (double)cnt[s] : NAN;
        for (int i = 0; i < n_pcts; ++i) {
            long long r = (long long)std::ceil(pcts[i] * (double)cnt[s] / 100.0);
            r = std::max<long long>(1, std::min<long long>(r, cnt[s]));
            rank[s * n_pcts + i] = r;
        }
    }
    const int shifts[3] = {21, 10, 0}, bits[3] = {11, 11, 10};
    std::vector<unsigned int> hist((size_t)nq * DVH_BINS);
    for (int level = 0; level < 3; ++level) {
        const unsigned int bin_mask = (1u << bits[level]) - 1u;
        DVH_TRY(cudaMemcpyAsync(W.query, query.data(), sizeof(DvhQuery) * nq, cudaMemcpyHostToDevice, st));
        DVH_TRY(cudaMemsetAsync(W.hist, 0, sizeof(unsigned int) * (size_t)nq * DVH_BINS, st));
        k_dvh_hist<<<grid, 256, 0, st>>>(d, sid, n_v, W.query, n_pcts, shifts[level], bin_mask, W.hist);
        DVH_TRY(cudaGetLastError());
        DVH_TRY(cudaMemcpyAsync(hist.data(), W.hist, sizeof(unsigned int) * (size_t)nq * DVH_BINS, cudaMemcpyDeviceToHost, st));
        DVH_TRY(cudaStreamSynchronize(st));
        for (int q = 0; q < nq; ++q) {
            if (!cnt[q / n_pcts]) continue;
            const unsigned int* hq = &hist[(size_t)q * DVH_BINS];
            long long seen = 0;
            unsigned int b = 0;
            for (; b <= bin_mask; ++b) {
                if (seen + hq[b] >= rank[q]) break;
                seen += hq[b];
            }
            rank[q] -= seen;
            query[q].prefix |= b << shifts[level];
            query[q].mask |= bin_mask << shifts[level];
        }
    }
    for (int q = 0; q < nq; ++q) host_dp[q] = cnt[q / n_pcts] ? (double)dvh_unkey(query[q].prefix) : NAN;
#undef DVH_TRY
    return cudaSuccess;
}

}  // namespace imrt
