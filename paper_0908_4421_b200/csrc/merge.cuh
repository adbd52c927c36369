// merge.cuh -- mixed-resolution row merging on the device (section 3.1: "for unspecified tissue we increased
// the voxel size in each dimension by a factor of 2"; reading R17).
//
// The rows of D (voxels) that carry the same group id are replaced by ONE row, their mean: the dose of a coarse voxel
// is the mean dose of the fine voxels it contains.  A column belongs to the merged row if any row of the group stores
// it; its value is (sum over the group's rows in ascending row order, in fp64) / (number of rows of the group), rounded
// to fp32 -- a fixed order, so the result is reproducible and equals the oracle's plain loop bit for bit.
//
// Plan-creation-side work, not on the hot path: a stable radix sort of (group, row) pairs lists every group's rows, one
// warp per group then marks the group's columns in a shared-memory bitmap (count pass: popcount; fill pass: prefix
// popcounts give every column its position, and the lanes walk the set bits, look each column up in the group's rows by
// binary search and add in row order).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace imrt {

constexpr int MERGE_WARPS = 8;

__global__ void k_merge_keys(const int* __restrict__ group, int n_v, int n_groups, unsigned int* keys, unsigned int* rows, int* flags) {
    int bad = 0;
    for (int j = blockIdx.x * blockDim.x + threadIdx.x; j < n_v; j += gridDim.x * blockDim.x) {
        const int g = group[j];
        bad |= (g < 0) | (g >= n_groups);
        keys[j] = (unsigned int)g;
        rows[j] = (unsigned int)j;
    }
    if (bad) flags[0] = 1;
}

// The raw CSR is checked here, BEFORE imrt_plan_create ever sees it (merging runs first): flags[1] = row_ptr does not start at
// 0 or decreases somewhere; flags[2] = a column outside [0, n_b) (it would index past the shared-memory bitmap below).
__global__ void k_merge_check_row_ptr(const int* __restrict__ row_ptr, int n_v, int* flags) {
    int bad = 0;
    for (int j = blockIdx.x * blockDim.x + threadIdx.x; j < n_v; j += gridDim.x * blockDim.x)
        bad |= (row_ptr[j] > row_ptr[j + 1]) | (j == 0 && row_ptr[0] != 0);
    if (bad) flags[1] = 1;
}
__global__ void k_merge_check_cols(const int* __restrict__ row_ptr, const int* __restrict__ col, int n_v, int n_b, int* flags) {
    if (flags[1]) return;                            // row_ptr cannot be trusted: do not follow it
    const int lane = threadIdx.x & 31, warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, n_warps = (gridDim.x * blockDim.x) >> 5;
    int bad = 0;
    for (int j = warp; j < n_v; j += n_warps)
        for (int p = row_ptr[j] + lane; p < row_ptr[j + 1]; p += 32) bad |= (col[p] < 0) | (col[p] >= n_b);
    if (bad) flags[2] = 1;
}

// group_ptr[g] = first position of the sorted keys that is >= g
__global__ void k_merge_group_ptr(const unsigned int* __restrict__ keys, int n_v, int n_groups, int* group_ptr) {
    const int g = blockIdx.x * blockDim.x + threadIdx.x;
    if (g > n_groups) return;
    int lo = 0, hi = n_v;
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if (keys[mid] < (unsigned int)g) lo = mid + 1; else hi = mid;
    }
    group_ptr[g] = lo;
}

// the warp's bitmap of the columns the rows of group g store; returns (to every lane) nothing -- callers popcount
__device__ __forceinline__ void merge_mark(const int* __restrict__ row_ptr, const int* __restrict__ col, const unsigned int* __restrict__ rows,
                                           int r0, int r1, uint32_t* bm, int words, int lane) {
    for (int w = lane; w < words; w += 32) bm[w] = 0u;
    __syncwarp();
    for (int t = r0; t < r1; ++t) {
        const int j = (int)rows[t];
        for (int p = row_ptr[j] + lane; p < row_ptr[j + 1]; p += 32) { const int c = col[p]; atomicOr(&bm[c >> 5], 1u << (c & 31)); }
    }
    __syncwarp();
}

__global__ void __launch_bounds__(MERGE_WARPS * 32) k_merge_count(const int* __restrict__ row_ptr, const int* __restrict__ col,
                                                                  const unsigned int* __restrict__ rows, const int* __restrict__ group_ptr,
                                                                  int n_groups, int words, int warps, int* cnt) {
    extern __shared__ uint32_t merge_smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (warp >= warps) return;
    uint32_t* bm = merge_smem + (size_t)warp * words;
    for (int g = blockIdx.x * warps + warp; g < n_groups; g += gridDim.x * warps) {
        merge_mark(row_ptr, col, rows, group_ptr[g], group_ptr[g + 1], bm, words, lane);
        int c = 0;
        for (int w = lane; w < words; w += 32) c += __popc(bm[w]);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
        if (lane == 0) cnt[g] = c;
        __syncwarp();
    }
}

__global__ void __launch_bounds__(MERGE_WARPS * 32) k_merge_fill(const int* __restrict__ row_ptr, const int* __restrict__ col,
                                                                 const float* __restrict__ val, const unsigned int* __restrict__ rows,
                                                                 const int* __restrict__ group_ptr, int n_groups, int words, int warps,
                                                                 const int* __restrict__ out_row_ptr, int* out_col, float* out_val) {
    extern __shared__ uint32_t merge_smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (warp >= warps) return;
    uint32_t* bm = merge_smem + (size_t)warp * 2 * words;
    uint32_t* pre = bm + words;
    for (int g = blockIdx.x * warps + warp; g < n_groups; g += gridDim.x * warps) {
        const int r0 = group_ptr[g], r1 = group_ptr[g + 1];
        merge_mark(row_ptr, col, rows, r0, r1, bm, words, lane);
        int running = 0;                             // exclusive prefix of the words' popcounts
        for (int base = 0; base < words; base += 32) {
            const int w = base + lane;
            const int c = w < words ? __popc(bm[w]) : 0;
            int inc = c;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += t; }
            if (w < words) pre[w] = (uint32_t)(running + inc - c);
            running += __shfl_sync(0xffffffffu, inc, 31);
        }
        __syncwarp();
        const int o0 = out_row_ptr[g];
        const double inv_n = (double)(r1 - r0);
        for (int w = lane; w < words; w += 32) {
            uint32_t bits = bm[w];
            int pos = o0 + (int)pre[w];
            while (bits) {
                const int b = __ffs(bits) - 1;
                bits &= bits - 1;
                const int c = 32 * w + b;
                double sum = 0.0;
                for (int t = r0; t < r1; ++t) {      // ascending row order: the order of the additions
                    const int j = (int)rows[t];
                    int lo = row_ptr[j], hi = row_ptr[j + 1];
                    while (lo < hi) {
                        const int mid = (lo + hi) >> 1;
                        if (col[mid] < c) lo = mid + 1; else hi = mid;
                    }
                    if (lo < row_ptr[j + 1] && col[lo] == c) sum += (double)val[lo];
                }
                out_col[pos] = c;
                out_val[pos] = (float)(sum / inv_n);
                ++pos;
            }
        }
        __syncwarp();
    }
}

}  // namespace imrt
