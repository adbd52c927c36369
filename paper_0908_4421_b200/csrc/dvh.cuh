// dvh.cuh -- dose-volume-histogram points on the device (plan evaluation).
//
// D_p of a structure = the ceil(p n_s / 100)-th largest dose among its n_s voxels (reading R10).  Exact
// selection by three rounds of radix histograms over an order-preserving integer image of the fp32 dose (11 + 11 + 10
// bits); the host only walks the (small) histograms between rounds.  Mean dose by fp64 atomics.  Not on the hot path.
#pragma once
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>
#include <cuda_runtime.h>

namespace imrt {

constexpr int DVH_BINS = 2048;
constexpr int DVH_MAX_PCTS = 16;

struct DvhQuery {
    unsigned int prefix;   // bits of the selection key fixed so far
    unsigned int mask;     // which bits those are
};

struct DvhWork {
    unsigned int* hist;    // [n_structures * DVH_MAX_PCTS][DVH_BINS]
    unsigned int* cnt;     // [n_structures]
    double* sum;           // [n_structures]
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

__global__ void k_dvh_count_sum(const float* __restrict__ d, const uint8_t* __restrict__ sid, int n_v, unsigned int* cnt, double* sum) {
    __shared__ double s_sum[256];
    __shared__ unsigned int s_cnt[256];
    for (int i = threadIdx.x; i < 256; i += blockDim.x) { s_sum[i] = 0.0; s_cnt[i] = 0u; }
    __syncthreads();
    for (int j = blockIdx.x * blockDim.x + threadIdx.x; j < n_v; j += gridDim.x * blockDim.x) {
        atomicAdd(&s_sum[sid[j]], (double)d[j]);
        atomicAdd(&s_cnt[sid[j]], 1u);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < 256; i += blockDim.x)
        if (s_cnt[i]) { atomicAdd(&sum[i], s_sum[i]); atomicAdd(&cnt[i], s_cnt[i]); }
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
    k_dvh_count_sum<<<grid, 256, 0, st>>>(d, sid, n_v, W.cnt, W.sum);
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
