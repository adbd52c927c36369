// imrtgp.cu -- host side of libimrtgp: the C-ABI of include/imrtgp.h, plan construction (validation, explicit
// transpose, row blocks, nnz ranges), the three loop drivers and the read-backs.  Kernels live in kernels.cuh.
//
// Build: nvcc -gencode arch=compute_100a,code=sm_100a -lineinfo -O3 -shared -Xcompiler -fPIC (see ../build.py).
#include "../../include/imrtgp.h"

#include <algorithm>
#include <chrono>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>

#include <cub/block/block_scan.cuh>
#include <cub/device/device_radix_sort.cuh>
#include <cub/device/device_scan.cuh>

#include "dvh.cuh"
#include "kernels.cuh"
#include "layout.cuh"
#include "merge.cuh"

using namespace imrt;

// ------------------------------------------------------------------------------------------------ errors
static thread_local std::string g_create_error;

struct imrt_plan {
    DevPlan P;
    imrt_params prm;
    imrt_options opt;
    cudaStream_t stream;
    int n_sm;                         // CTAs of this plan's persistent passes (the SM count, or imrt_options.n_ctas)
    int n_sm_device;                  // SMs of the device
    size_t smem_bytes;
    int grid_p;                       // persistent kernel grid
    bool has_x;
    int64_t n_blk, n_nonempty, n_skipped, pack_bytes, n_quad_rows;
    std::vector<double> blk_cost;     // modelled, then measured, cost of every dose-pass block (host)
    int* cta_blk_w;
    int4* blk_w;
    std::vector<int> rp_tr;           // row pointers of the stream the transpose pass reads (host copy)
    std::vector<double> tr_share;     // share of that stream per CTA
    int tr_align;
    int n_rows_tr;                    // rows of that stream: n_b, or the number of row pairs
    int64_t tr_stream_bytes;          // bytes of that stream (values + voxel ids / offsets + bases)
    int64_t max_ranges, max_slots;
    TrRange* tr_range_w;
    int* rowslot_w;
    int* cta_rng_w;
    double tune_spread[2];            // slowest / mean CTA time of the dose pass before and after tuning
    std::vector<int> cta_blk_h;       // the dose-pass partition in use (host copy, for imrt_plan_get_tuning)
    std::vector<double> create_ms;    // phase times of plan creation (imrt_options.profile_create)
    // borrowed inputs
    const int32_t* row_ptr;
    const uint8_t* sid;
    // workspace pieces the host needs by name
    float* r_scratch;
    float* g_scratch;
    float* d_scratch;
    int* rowT_ptr_w;
    int* colT_w;
    float* valT_w;
    DvhWork dvh;
    DevPlan* rank_plans_w;            // device copies of the plans of co-resident ranks (imrt_plan_run_ranks)
    // conditional graph (driver 0)
    cudaGraph_t graph;
    cudaGraphExec_t graph_exec;
    std::string err;
};

static imrt_status fail(imrt_plan* p, imrt_status s, const char* fmt, ...) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    if (p) p->err = buf; else g_create_error = buf;
    return s;
}

#define CUDA_TRY(plan, expr)                                                                                       \
    do {                                                                                                           \
        cudaError_t e_ = (expr);                                                                                   \
        if (e_ != cudaSuccess)                                                                                     \
            return fail(plan, IMRT_STATUS_CUDA_ERROR, "%s: %s (%s:%d)", #expr, cudaGetErrorString(e_), __FILE__,  \
                        __LINE__);                                                                                 \
    } while (0)

// ------------------------------------------------------------------------------------------------ workspace
namespace {

struct Bump {                           // the same walk sizes the workspace and places the arrays
    unsigned char* base;
    size_t off;
    template <typename T>
    T* take(size_t n) {
        off = (off + 255) & ~(size_t)255;
        T* p = base ? reinterpret_cast<T*>(base + off) : nullptr;
        off += n * sizeof(T);
        return p;
    }
};

struct Bounds {
    int64_t max_blk, max_meta, max_ranges, max_slots, nnz_pad, nnz_pack;
    size_t sort_temp, max_pack;
};

Bounds bounds_for(int64_t n_v, int64_t n_b, int64_t nnz) {
    Bounds b;
    const int64_t slots = nnz + 3 * n_v;    // every row padded to a multiple of 4 slots
    b.max_blk = 4 * (slots / ROW_REC_SLOTS + 1) + 4 * (n_v / SEG_ROWS + 1) + n_v / 16 + 8 + 8 * TARGET_RECORDS;
    b.max_meta = n_v + b.max_blk * (META_HDR + 2 + 3) + 8;
    b.max_pack = (size_t)b.max_meta * 4 + (size_t)slots * 8 + (size_t)b.max_blk * (128 + 48) + 256;
    b.max_ranges = 2 * 1024 + n_b / RL_MAX + 2 * (n_b / RL_MAX + 1) + 4;
    b.max_slots = n_b + b.max_ranges + 4;
    b.nnz_pad = ((nnz + 3) & ~(int64_t)3) + 8;
    b.nnz_pack = nnz + 128 * n_b + 128;         // packed D^T: every row padded to a multiple of 128 entries
    b.sort_temp = (size_t)(16 << 20) + (size_t)nnz;
    return b;
}

struct Layout {
    State* st;
    float4* table;
    int4* blk;
    int4* pk;
    uint32_t* rowmeta;
    unsigned char* pack;
    int* cta_blk;
    int* rowT_ptr;
    int* colT;
    float* valT;
    float* valP;
    int* voxU;
    int* pairU;
    unsigned short* idP;
    unsigned int* baseP;
    int* rowP_ptr;
    TrRange* tr_range;
    int* rowslot_ptr;
    int* cta_rng;
    float* xbuf[2];
    float* g;
    float* rbuf[R_MAX + 1];
    double* Gpart[2];
    double* gslot[2];
    double* tr_obj;
    double* tr_lambda;
    double* tr_step_sq;
    int* tr_trials;
    float* r_scratch;
    float* g_scratch;
    float* d_scratch;
    int* flags;
    unsigned long long* cta_ns;
    DvhWork dvh;
    // build scratch
    int* quadU;
    unsigned char* covered;
    LayoutTotals* totals;
    DevPlan* rank_plans;
    int *seg_rec, *seg_meta, *seg_b128;
    long long *cost_fx, *cost_pre;
    unsigned int* keysA;
    unsigned int* keysB;
    unsigned int* valsA;
    unsigned int* valsB;
    void* sort_temp;
    size_t total;
};

Layout make_layout(void* base, int64_t n_v, int64_t n_b, int64_t nnz, int n_s, int max_iters) {
    const Bounds B = bounds_for(n_v, n_b, nnz);
    Bump w{static_cast<unsigned char*>(base), 0};
    Layout L;
    L.st = w.take<State>(1);
    L.table = w.take<float4>(MAX_STRUCTURES);
    L.blk = w.take<int4>(B.max_blk);
    L.pk = w.take<int4>(B.max_blk);
    L.rowmeta = w.take<uint32_t>(B.max_meta);
    L.pack = w.take<unsigned char>(B.max_pack);
    L.cta_blk = w.take<int>(1024 + 1);
    L.rowT_ptr = w.take<int>(n_b + 1);
    L.colT = w.take<int>(B.nnz_pad);
    L.valT = w.take<float>(B.nnz_pad);
    L.valP = w.take<float>(2 * B.nnz_pack);      // fp32 per entry, or float2 per entry of the row-pair stream
    L.voxU = w.take<int>(B.nnz_pack);
    L.pairU = w.take<int>(n_b / 2 + 4);
    L.idP = w.take<unsigned short>(B.nnz_pack);
    L.baseP = w.take<unsigned int>(B.nnz_pack / 32 + 4);
    L.rowP_ptr = w.take<int>(n_b + 1);
    L.tr_range = w.take<TrRange>(B.max_ranges);
    L.rowslot_ptr = w.take<int>(n_b + 1);
    L.cta_rng = w.take<int>(1024 + 1);
    for (int i = 0; i < 2; ++i) L.xbuf[i] = w.take<float>(n_b + 4);
    L.g = w.take<float>(n_b + 4);
    for (int i = 0; i <= R_MAX; ++i) L.rbuf[i] = w.take<float>(n_v + 4);
    for (int i = 0; i < 2; ++i) L.Gpart[i] = w.take<double>(1024 * R_MAX);
    for (int i = 0; i < 2; ++i) L.gslot[i] = w.take<double>(2 * B.max_slots);    // two sums per slot in the row-pair stream
    L.tr_obj = w.take<double>((size_t)max_iters + 1);
    L.tr_lambda = w.take<double>((size_t)max_iters + 1);
    L.tr_step_sq = w.take<double>((size_t)max_iters + 1);
    L.tr_trials = w.take<int>((size_t)max_iters + 1);
    L.r_scratch = w.take<float>(n_v + 4);
    L.g_scratch = w.take<float>(n_b + 4);
    L.d_scratch = w.take<float>(n_v + 4);
    L.flags = w.take<int>(16);
    L.cta_ns = w.take<unsigned long long>(4096);
    L.dvh.hist = w.take<unsigned int>((size_t)n_s * DVH_MAX_PCTS * DVH_BINS);
    L.dvh.cnt = w.take<unsigned int>((size_t)MAX_STRUCTURES);
    L.dvh.sum = w.take<double>((size_t)MAX_STRUCTURES);
    L.dvh.part = w.take<double>((size_t)DVH_SUM_BLOCKS * n_s);
    L.dvh.query = w.take<DvhQuery>((size_t)MAX_STRUCTURES * DVH_MAX_PCTS);
    L.quadU = w.take<int>(n_v / 4 + 2);
    L.covered = w.take<unsigned char>(n_v + 4);
    L.totals = w.take<LayoutTotals>(1);
    L.rank_plans = w.take<DevPlan>(MAX_WORLD);
    L.seg_rec = w.take<int>(n_v / SEG_ROWS + 4);
    L.seg_meta = w.take<int>(n_v / SEG_ROWS + 4);
    L.seg_b128 = w.take<int>(n_v / SEG_ROWS + 4);
    L.cost_fx = w.take<long long>(B.max_blk + 2);
    L.cost_pre = w.take<long long>(B.max_blk + 2);
    L.keysA = w.take<unsigned int>(nnz + 4);
    L.keysB = w.take<unsigned int>(nnz + 4);
    L.valsA = w.take<unsigned int>(nnz + 4);
    L.valsB = w.take<unsigned int>(nnz + 4);
    L.sort_temp = w.take<unsigned char>(B.sort_temp);
    L.total = (w.off + 255) & ~(size_t)255;
    return L;
}

// ------------------------------------------------------------------------------------------------ build kernels
__global__ void k_validate(const int* __restrict__ col, const float* __restrict__ val, long long nnz, int n_b, int* flags) {
    int bad_col = 0, bad_val = 0;
    for (long long p = blockIdx.x * (long long)blockDim.x + threadIdx.x; p < nnz; p += (long long)gridDim.x * blockDim.x) {
        const int c = col[p];
        bad_col |= (c < 0) | (c >= n_b);
        bad_val |= !isfinite(val[p]);
    }
    if (bad_col) flags[0] = 1;
    if (bad_val) flags[1] = 1;
}

// columns strictly ascending inside every row (one warp per row); a violation raises flags[3]
__global__ void k_validate_rows(const int* __restrict__ row_ptr, const int* __restrict__ col, int n_v, int* flags) {
    const int lane = threadIdx.x & 31;
    int bad = 0;
    for (long long j = (blockIdx.x * (long long)blockDim.x + threadIdx.x) >> 5; j < n_v; j += ((long long)gridDim.x * blockDim.x) >> 5) {
        const int p0 = row_ptr[j], p1 = row_ptr[j + 1];
        for (int p = p0 + 1 + lane; p < p1; p += 32) bad |= col[p] <= col[p - 1];
    }
    if (bad) flags[3] = 1;
}

__global__ void k_iota_keys(const int* __restrict__ col, unsigned int* keys, unsigned int* vals, long long nnz) {
    for (long long p = blockIdx.x * (long long)blockDim.x + threadIdx.x; p < nnz; p += (long long)gridDim.x * blockDim.x) {
        keys[p] = (unsigned int)col[p];
        vals[p] = (unsigned int)p;
    }
}

// rowT_ptr[i] = first position of the sorted column keys that is >= i
__global__ void k_rowT_ptr(const unsigned int* __restrict__ keys, long long nnz, int n_b, int* rowT_ptr) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i > n_b) return;
    long long lo = 0, hi = nnz;
    while (lo < hi) {
        const long long mid = (lo + hi) >> 1;
        if (keys[mid] < (unsigned int)i) lo = mid + 1; else hi = mid;
    }
    rowT_ptr[i] = (int)lo;
}

// entry q of D^T comes from entry p = perm[q] of D: its column is the row of D holding p (upper_bound on row_ptr)
__global__ void k_fill_transpose(const unsigned int* __restrict__ perm, const int* __restrict__ row_ptr, int n_v,
                                 const float* __restrict__ val, long long nnz, int* colT, float* valT) {
    for (long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x; q < nnz; q += (long long)gridDim.x * blockDim.x) {
        const int p = (int)perm[q];
        int lo = 0, hi = n_v;   // largest j with row_ptr[j] <= p
        while (lo < hi) {
            const int mid = (lo + hi + 1) >> 1;
            if (row_ptr[mid] <= p) lo = mid; else hi = mid - 1;
        }
        colT[q] = lo;
        valT[q] = val[p];
    }
}

// Number of distinct columns in every quad (4 consecutive rows) of D: one warp per quad marks the columns in a
// shared-memory bitmap.  Dynamic shared memory: warps x words x 4 bytes, words = ceil(n_b / 32).
__global__ void k_quad_union(const int* __restrict__ row_ptr, const int* __restrict__ col, int n_v, int n_quads, int words, int* U) {
    extern __shared__ uint32_t k_quad_smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nwarp = blockDim.x >> 5;
    uint32_t* bm = k_quad_smem + (size_t)warp * words;
    for (int q = blockIdx.x * nwarp + warp; q < n_quads; q += gridDim.x * nwarp) {
        const int p0 = row_ptr[4 * q], p1 = row_ptr[min(4 * q + 4, n_v)];
        if (p0 == p1) { if (lane == 0) U[q] = 0; continue; }
        for (int w = lane; w < words; w += 32) bm[w] = 0u;
        __syncwarp();
        for (int p = p0 + lane; p < p1; p += 32) { const int c = col[p]; atomicOr(&bm[c >> 5], 1u << (c & 31)); }
        __syncwarp();
        int cnt = 0;
        for (int w = lane; w < words; w += 32) cnt += __popc(bm[w]);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
        if (lane == 0) U[q] = cnt;
        __syncwarp();
    }
}

// Re-pack D into the dose pass's block records: one CTA per record copies the header and table, then
//   row format:  one warp per row copies values and columns (16- or 32-bit) to the row's 16-byte aligned slot range
//                and zero-fills the padding;
//   quad format: one warp per quad marks its columns in a bitmap, ranks them (prefix popcount) and scatters every
//                entry of the 4 rows to (rank of its column, row) -- explicit zeros where a row lacks a column.
// Dynamic shared memory (quad format only): warps x 2 x words x 4 bytes.
template <bool COL16>
__global__ void k_pack_blocks(const int4* __restrict__ pk, const uint32_t* __restrict__ meta, const int* __restrict__ row_ptr,
                              const int* __restrict__ col, const float* __restrict__ val, int n_v, int words, unsigned char* pack) {
    extern __shared__ uint32_t k_pack_smem[];
    const int4 d = pk[blockIdx.x];
    const uint32_t* m = meta + d.x;
    unsigned char* rec = pack + (size_t)(unsigned int)d.z * 128u;
    uint32_t* rec_w = reinterpret_cast<uint32_t*>(rec);
    for (int i = threadIdx.x; i < d.y; i += blockDim.x) rec_w[i] = m[i];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nwarp = blockDim.x >> 5;
    if (d.w == 0) {
        const int nrows = (int)m[0], r0 = (int)m[1], slots = (int)m[3];
        float* val_o = reinterpret_cast<float*>(rec + (size_t)d.y * 4);
        unsigned char* col_o = reinterpret_cast<unsigned char*>(val_o + slots + ZPAD);
        for (int row = warp; row < nrows; row += nwarp) {
            const int so = (int)(m[META_HDR + row] & 0xFFFFu), se = (int)(m[META_HDR + row + 1] & 0xFFFFu);
            const int p0 = row_ptr[r0 + row], len = row_ptr[r0 + row + 1] - p0;
            for (int k = lane; k < se - so; k += 32) {
                const float v = k < len ? val[p0 + k] : 0.0f;
                const int c = k < len ? col[p0 + k] : 0;
                val_o[so + k] = v;
                if (COL16) reinterpret_cast<unsigned short*>(col_o)[so + k] = (unsigned short)c;
                else reinterpret_cast<int*>(col_o)[so + k] = c;
            }
        }
        if (threadIdx.x < ZPAD) {   // the zero slots lanes past a row's end read
            val_o[slots + threadIdx.x] = 0.0f;
            if (COL16) reinterpret_cast<unsigned short*>(col_o)[slots + threadIdx.x] = 0;
            else reinterpret_cast<int*>(col_o)[slots + threadIdx.x] = 0;
        }
    } else {
        const int nq = (int)m[0], r0 = (int)m[1], nbc = (int)m[3];
        float* val_o = reinterpret_cast<float*>(rec + (size_t)d.y * 4);
        unsigned short* col_o = reinterpret_cast<unsigned short*>(val_o + (size_t)(nbc + 1) * 4);
        uint32_t* bm = k_pack_smem + (size_t)warp * 2 * words;
        uint32_t* pre = bm + words;
        for (int qi = warp; qi < nq; qi += nwarp) {
            const int off = (int)(m[META_HDR + 2 * qi] & 0xFFFFu), off_n = (int)(m[META_HDR + 2 * qi + 2] & 0xFFFFu);
            if (off_n == off) continue;
            const int ra = r0 + 4 * qi, rb = min(ra + 4, n_v);
            const int p0 = row_ptr[ra], p1 = row_ptr[rb];
            for (int k = lane; k < (off_n - off) * 4; k += 32) val_o[(size_t)off * 4 + k] = 0.0f;
            for (int k = lane; k < off_n - off; k += 32) col_o[off + k] = 0;
            for (int w = lane; w < words; w += 32) bm[w] = 0u;
            __syncwarp();
            for (int p = p0 + lane; p < p1; p += 32) { const int c = col[p]; atomicOr(&bm[c >> 5], 1u << (c & 31)); }
            __syncwarp();
            int running = 0;
            for (int base = 0; base < words; base += 32) {
                const int w = base + lane;
                const int cnt = w < words ? __popc(bm[w]) : 0;
                int inc = cnt;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) { const int t = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += t; }
                if (w < words) pre[w] = (uint32_t)(running + inc - cnt);
                running += __shfl_sync(0xffffffffu, inc, 31);
            }
            __syncwarp();
            for (int row = ra; row < rb; ++row) {
                const int q0 = row_ptr[row], q1 = row_ptr[row + 1];
                for (int p = q0 + lane; p < q1; p += 32) {
                    const int c = col[p];
                    const int rank = (int)pre[c >> 5] + __popc(bm[c >> 5] & ((1u << (c & 31)) - 1u));     // position inside the quad
                    const int pos = off + rank;
                    // rows rotated by bits 3 and 2 of the position: the dose pass's row-splitting butterfly needs no selects
                    val_o[(size_t)pos * 4 + ((row - ra) ^ (((rank >> 3) & 1) * 2 + ((rank >> 2) & 1)))] = val[p];
                    col_o[pos] = (unsigned short)c;
                }
            }
            __syncwarp();
        }
        if (threadIdx.x < 4) val_o[(size_t)nbc * 4 + threadIdx.x] = 0.0f;   // the zero column
        if (threadIdx.x < 8) col_o[nbc + threadIdx.x] = 0;
    }
}

// The packed D^T stream: one warp per aligned group of 32 entries of the padded stream.  Entries past the end of a row
// repeat its last voxel with value 0.  flags[2] is raised when a group spans more than 65535 voxels (no 16-bit form).
__global__ void k_pack_transpose(const int* __restrict__ rowT_ptr, const int* __restrict__ rowP_ptr, const int* __restrict__ colT,
                                 const float* __restrict__ valT, int n_b, long long n_groups, float* valP, unsigned short* idP,
                                 unsigned int* baseP, int* flags) {
    const int lane = threadIdx.x & 31;
    for (long long t = (blockIdx.x * (long long)blockDim.x + threadIdx.x) >> 5; t < n_groups; t += ((long long)gridDim.x * blockDim.x) >> 5) {
        const int e = (int)(t * 32);
        int lo = 0, hi = n_b;          // the row holding packed position e: largest i with rowP_ptr[i] <= e
        while (lo < hi) {
            const int mid = (lo + hi + 1) >> 1;
            if (rowP_ptr[mid] <= e) lo = mid; else hi = mid - 1;
        }
        const int k = e - rowP_ptr[lo] + lane, len = rowT_ptr[lo + 1] - rowT_ptr[lo];
        const int src = rowT_ptr[lo] + min(k, len - 1);
        const int id = len > 0 ? colT[src] : 0;
        const float v = k < len ? valT[src] : 0.0f;
        const int base = __shfl_sync(0xffffffffu, id, 0);
        if (id - base > 65535) flags[2] = 1;
        valP[e + lane] = v;
        idP[e + lane] = (unsigned short)(id - base);
        if (lane == 0) baseP[t] = (unsigned int)base;
    }
}

struct RPtrs { float* p[R_MAX + 1]; };
// ---- the row-pair stream of D^T: rows 2P and 2P+1 (sorted voxel lists A and B) merged into their union.
__device__ __forceinline__ int lower_bound_dev(const int* __restrict__ a, int n, int v) {
    int lo = 0, hi = n;
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if (a[mid] < v) lo = mid + 1; else hi = mid;
    }
    return lo;
}
// size of the union of every pair (one CTA per pair): |A| + |B| - |A and B|
__global__ void k_pair_count(const int* __restrict__ rowT_ptr, const int* __restrict__ colT, int n_b, int* U) {
    __shared__ int common;
    const int P = blockIdx.x;
    const int a0 = rowT_ptr[2 * P], a1 = rowT_ptr[2 * P + 1], b1 = 2 * P + 2 <= n_b ? rowT_ptr[2 * P + 2] : a1;
    const int* A = colT + a0;
    const int* B = colT + a1;
    const int nA = a1 - a0, nB = b1 - a1;
    if (threadIdx.x == 0) common = 0;
    __syncthreads();
    int c = 0;
    for (int k = threadIdx.x; k < nA; k += blockDim.x) {
        const int rb = lower_bound_dev(B, nB, A[k]);
        c += (rb < nB && B[rb] == A[k]);
    }
    if (c) atomicAdd(&common, c);
    __syncthreads();
    if (threadIdx.x == 0) U[P] = nA + nB - common;
}
// An element v of A or B goes to union position (#A < v) + (#B < v) - (#common < v); the last term is a running count of
// the matches, kept by a block-wide exclusive scan.  val2 is zero beforehand; the padding repeats the pair's last voxel.
__global__ void __launch_bounds__(256) k_pair_fill(const int* __restrict__ rowT_ptr, const int* __restrict__ colT, const float* __restrict__ valT,
                                                   int n_b, const int* __restrict__ pairP_ptr, float2* val2, int* voxU) {
    typedef cub::BlockScan<int, 256> Scan;
    __shared__ typename Scan::TempStorage tmp;
    const int P = blockIdx.x;
    const int a0 = rowT_ptr[2 * P], a1 = rowT_ptr[2 * P + 1], b1 = 2 * P + 2 <= n_b ? rowT_ptr[2 * P + 2] : a1;
    const int nA = a1 - a0, nB = b1 - a1;
    const int base = pairP_ptr[P], end = pairP_ptr[P + 1];
    for (int half = 0; half < 2; ++half) {
        const int* X = colT + (half ? a1 : a0);        // the list being placed
        const int* Y = colT + (half ? a0 : a1);        // the other one
        const float* XV = valT + (half ? a1 : a0);
        const int nX = half ? nB : nA, nY = half ? nA : nB;
        int carry = 0;
        for (int k0 = 0; k0 < nX; k0 += 256) {
            const int k = k0 + threadIdx.x;
            int v = 0, ry = 0, eq = 0;
            if (k < nX) {
                v = X[k];
                ry = lower_bound_dev(Y, nY, v);
                eq = (ry < nY && Y[ry] == v);
            }
            int before, total;
            Scan(tmp).ExclusiveSum(eq, before, total);
            __syncthreads();
            if (k < nX) {
                const int pos = base + k + ry - (carry + before);
                if (half) val2[pos].y = XV[k]; else val2[pos].x = XV[k];
                voxU[pos] = v;
            }
            carry += total;
        }
        __syncthreads();
    }
    const int last = max(nA ? colT[a1 - 1] : 0, nB ? colT[b1 - 1] : 0);
    // the union has nA + nB - common entries; find it as the first unwritten position: the count kernel gave it as U[P]
    // implicitly through pairP_ptr, but the padded end is what is stored, so fill backwards from `end` while untouched
    for (int t = end - 1 - (int)threadIdx.x; t >= base && t >= end - 128; t -= 256) {
        // entries [base + U, end) are padding: they are exactly those never written above; mark them via a sentinel
        if (voxU[t] < 0) voxU[t] = last;
    }
}
// 16-bit offsets of the pair stream: one warp per aligned group of 32 entries; flags[2] is raised when a group is too wide
__global__ void k_pair_tiles(const int* __restrict__ voxU, long long n_groups, unsigned short* idP, unsigned int* baseP, int* flags) {
    const int lane = threadIdx.x & 31;
    for (long long t = (blockIdx.x * (long long)blockDim.x + threadIdx.x) >> 5; t < n_groups; t += ((long long)gridDim.x * blockDim.x) >> 5) {
        const int id = voxU[t * 32 + lane];
        const int base = __shfl_sync(0xffffffffu, id, 0);
        if (id - base > 65535 || id < base) flags[2] = 1;
        idP[t * 32 + lane] = (unsigned short)(id - base);
        if (lane == 0) baseP[t] = (unsigned int)base;
    }
}

// d = 0 and the matching constant residual on every row; the dose pass then overwrites the rows its blocks cover.
__global__ void k_fill_zero_dose_rows(const uint8_t* __restrict__ sid, const float4* __restrict__ table, const State* st, int n_v,
                                      const RPtrs R, float* d) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n_v) return;
    float4 t = table[sid[j]];
    if (st->tvu) t.x = st->tvu[j];
    if (st->tvo) t.y = st->tvo[j];
    const float u = fmaxf(0.0f, t.x), o = fmaxf(0.0f, -t.y);
    const float r = 2.0f * __fmaf_rn(t.w, o, -__fmul_rn(t.z, u));
#pragma unroll
    for (int i = 0; i <= R_MAX; ++i)
        if (R.p[i]) R.p[i][j] = r;
    if (d) d[j] = 0.0f;
}

// The constants of the rows no record covers (dose 0 whatever x is): their objective, State::G_skip, and their residual
// in every residual buffer of the loop.  Runs at plan creation and whenever the per-voxel limits change.  The objective
// is summed in a fixed order: every block adds its rows (thread-strided, warp butterfly, warps in order) into part[block],
// k_skip_final adds the blocks' partials in block order.
constexpr int SKIP_BLOCKS = 128;
__global__ void __launch_bounds__(1024) k_skip_constants(const uint8_t* __restrict__ sid, const unsigned char* __restrict__ covered,
                                                         const float4* __restrict__ table, const State* st, int n_v, const RPtrs R, double* part) {
    __shared__ double red[32];
    double acc = 0.0;
    const int per = (n_v + gridDim.x - 1) / gridDim.x;            // a contiguous chunk of rows per block
    const int j0 = blockIdx.x * per, j1 = min(n_v, j0 + per);
    for (int j = j0 + threadIdx.x; j < j1; j += blockDim.x) {
        if (covered[j]) continue;
        float4 t = table[sid[j]];
        if (st->tvu) t.x = st->tvu[j];
        if (st->tvo) t.y = st->tvo[j];
        const float u = fmaxf(0.0f, t.x), o = fmaxf(0.0f, -t.y);
        const float r = 2.0f * __fmaf_rn(t.w, o, -__fmul_rn(t.z, u));
#pragma unroll
        for (int i = 0; i <= R_MAX; ++i)
            if (R.p[i]) R.p[i][j] = r;
        const double du = (double)u, d_o = (double)o;
        acc = __dadd_rn(acc, __fma_rn((double)t.z, __dmul_rn(du, du), __dmul_rn((double)t.w, __dmul_rn(d_o, d_o))));
    }
    acc = warp_sum(acc);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int w = 0; w < (int)(blockDim.x >> 5); ++w) s += red[w];
        part[blockIdx.x] = s;
    }
}
__global__ void k_skip_final(const double* __restrict__ part, int n, State* st) {
    double s = 0.0;
    for (int b = 0; b < n; ++b) s += part[b];
    st->G_skip = s;
}

__global__ void k_check_x(const float* __restrict__ x, int n_b, State* st) {
    int bad = 0;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n_b; i += gridDim.x * blockDim.x) {
        const float v = x[i];
        bad |= !(v >= 0.0f) | !isfinite(v);
    }
    if (bad) st->bad_x = 1;
}

__global__ void k_reset_state(State* st) {
    st->G_k = 0.0; st->lambda = st->lambda0;
    st->fwd_passes = 0; st->tr_passes = 0;
    st->iter = 0; st->iter_target = 0; st->m = 0; st->stop_reason = STOP_MAX_ITERS;
    st->xi = 0; st->ri = 0;   // the MODE_INIT dose pass reads xbuf[0], writes rbuf[1] and makes it current
    st->cont_outer = 0; st->cont_inner = 0; st->bad_x = 0;
    st->ticket_f = 0u; st->ticket_t = 0u; st->gridbar = 0u; st->clamped = 0; st->fault = 0;
}

__global__ void k_copy_current_x(const DevPlan P, float* x) {
    const float* src = P.xbuf[P.st->xi];
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < P.n_b; i += gridDim.x * blockDim.x) x[i] = src[i];
}

inline int grid_for(long long n, int block) {
    long long g = (n + block - 1) / block;
    return (int)std::max<long long>(1, std::min<long long>(g, 148 * 16));
}

// ------------------------------------------------------------------------------------------------ host builders
// How much a record may hold.  Large matrices get the full sizes; a small one is cut into at least ~TARGET_RECORDS
// records so that every consumer warp of every CTA has several (a record is consumed by one warp).  The layout itself
// (which rows go into which record) is done on the device: layout.cuh.
// ring_est: roughly the bytes the dose pass's ring will have (what the gather array and g leave of shared memory).
static RecordCaps record_caps(int64_t n_v, int64_t nnz, int64_t ring_est, int quad_cap_user) {
    auto clampi = [](int64_t v, int lo, int hi) { return (int)std::max<int64_t>(lo, std::min<int64_t>(hi, v)); };
    RecordCaps c;
    c.chunk_slots = clampi((nnz / TARGET_RECORDS + 3) & ~(int64_t)3, 64, ROW_REC_SLOTS);
    c.max_rows = clampi(n_v / TARGET_RECORDS, 8, MAXROWS_F);
    // quad records: at least one per consumer warp must fit in the ring (18 bytes per union column); measured on the
    // 9- and 15-field phantoms, 384 .. 448 columns (~7 KB) is the sweet spot: 16 records being consumed then hold ~110 KB
    // of the ring and ~60 KB stay in flight (576 columns, best with round 1's heavier quad loop, leave ~30 KB: 3 % slower)
    const int cap = quad_cap_user > 0 ? std::max(32, std::min(quad_cap_user, 4096)) : QUAD_CAP;
    c.quad_cap = clampi(std::min<int64_t>(nnz / 3 / TARGET_RECORDS, ring_est / (W_CONS * 18)), 32, cap);
    // a single quad may exceed quad_cap (it then fills a record by itself), but two such records must fit in the ring
    c.quad_max = clampi((ring_est / 2 - 256) / 18, 0, 65528);
    return c;
}

// Contiguous block ranges of (nearly) equal total cost, one per CTA.
void partition_blocks(const std::vector<double>& cost, int grid, std::vector<int>& cta_blk) {
    const size_t n = cost.size();
    std::vector<double> pre(n + 1, 0.0);
    for (size_t b = 0; b < n; ++b) pre[b + 1] = pre[b] + cost[b];
    cta_blk.assign(grid + 1, 0);
    size_t b = 0;
    for (int c = 0; c < grid; ++c) {
        const double want = pre[n] * c / grid;
        while (b < n && pre[b] < want) ++b;
        cta_blk[c] = (int)b;
    }
    cta_blk[grid] = (int)n;
}

// Equal-nnz ranges of the D^T stream, each spanning at most RL_MAX rows, and the gradient partial slots.
// One contiguous, `align`-aligned share of the D^T stream per CTA -- share[c] of the total, equal shares unless plan
// creation has measured otherwise -- cut into ranges of at most RL_MAX rows, and the gradient partial slots.
void build_ranges(const std::vector<int>& rpT, int n_b, const std::vector<double>& share, int align, std::vector<TrRange>& ranges,
                  std::vector<int>& rowslot_ptr, std::vector<int>& cta_rng) {
    const long long nnz = rpT[n_b];
    const int grid = (int)share.size();
    ranges.clear();
    rowslot_ptr.assign(n_b + 1, 0);
    cta_rng.assign(grid + 1, 0);
    if (nnz == 0) return;
    std::vector<int> cnt(n_b, 0);
    long long e = 0;
    int row = 0, slot = 0;
    double cum = 0.0;
    for (int c = 0; c < grid; ++c) {
        cta_rng[c] = (int)ranges.size();
        cum += share[c];
        long long stop = c == grid - 1 ? nnz : std::min<long long>(nnz, (long long)(cum * (double)nnz / align + 0.5) * align);
        while (e < stop) {
            while (rpT[row + 1] <= e) ++row;
            TrRange R;
            memset(&R, 0, sizeof R);
            R.e_begin = (int)e;
            R.first_row = row;
            const long long e_end = std::min<long long>(stop, rpT[std::min(n_b, row + RL_MAX)]);
            R.e_end = (int)e_end;
            int last = row;
            while (rpT[last + 1] < e_end) ++last;
            R.n_rows = last - row + 1;
            R.slot_base = slot;
            for (int i = row; i <= last; ++i) ++cnt[i];
            slot += R.n_rows;
            ranges.push_back(R);
            e = e_end;
        }
    }
    cta_rng[grid] = (int)ranges.size();
    for (int i = 0; i < n_b; ++i) rowslot_ptr[i + 1] = rowslot_ptr[i] + cnt[i];
}

}  // namespace

// ------------------------------------------------------------------------------------------------ launch helpers
static cudaError_t launch_dose(imrt_plan* pl, const PassArgs& A) {
    k_dose<<<pl->P.grid_f, NTHREADS, pl->smem_bytes, pl->stream>>>(pl->P, A);
    return cudaGetLastError();
}
static cudaError_t launch_transpose(imrt_plan* pl, const PassArgs& A) {
    k_transpose<<<pl->P.grid_t, NTHREADS, pl->smem_bytes, pl->stream>>>(pl->P, A);
    return cudaGetLastError();
}
static cudaError_t launch_persistent(imrt_plan* pl) {
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof cfg);
    cfg.gridDim = dim3(pl->grid_p);
    cfg.blockDim = dim3(NTHREADS);
    cfg.dynamicSmemBytes = pl->smem_bytes;
    cfg.stream = pl->stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeCooperative;
    at[0].val.cooperative = 1;   // co-residency of all CTAs is required by the grid barrier
    cfg.attrs = at;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, k_persistent, pl->P);
}

// A new partition of the dose pass: upload it and lay out every CTA's ring schedule for it.
static imrt_status upload_partition(imrt_plan* pl, const std::vector<int>& cta_blk) {
    cudaStream_t st = pl->stream;
    CUDA_TRY(pl, cudaMemcpyAsync(pl->cta_blk_w, cta_blk.data(), sizeof(int) * cta_blk.size(), cudaMemcpyHostToDevice, st));
    k_ring_layout<<<pl->P.grid_f, 32, 0, st>>>(pl->blk_w, pl->cta_blk_w, pl->P.grid_f, (unsigned int)pl->P.ring_f_bytes);
    CUDA_TRY(pl, cudaGetLastError());
    CUDA_TRY(pl, cudaStreamSynchronize(st));   // cta_blk is a host vector the caller may drop
    pl->cta_blk_h = cta_blk;
    return IMRT_STATUS_OK;
}

// A short run of the device-resident loop from x = whatever xbuf[0] holds (zeros at plan creation), for its per-CTA
// pass timers: inside the loop the passes follow each other without launch gaps and the SMs do not behave quite as
// they do for an isolated launch, so the final rounds of both rebalancings are measured here.
static imrt_status timing_loop_run(imrt_plan* pl) {
    cudaStream_t st = pl->stream;
    k_reset_state<<<1, 1, 0, st>>>(pl->P.st);
    PassArgs A;
    memset(&A, 0, sizeof A);
    A.mode = MODE_INIT;
    CUDA_TRY(pl, launch_dose(pl, A));
    k_set_target<<<1, 1, 0, st>>>(pl->P.st, 3, 0.0);
    CUDA_TRY(pl, launch_persistent(pl));
    k_reset_state<<<1, 1, 0, st>>>(pl->P.st);
    CUDA_TRY(pl, cudaGetLastError());
    return IMRT_STATUS_OK;
}
constexpr int LOOP_MEASUREMENTS = 1;   // 3 gains 0.7 % of loop speed and costs 16 ms of plan creation (cfg3)
static bool can_time_in_loop(const imrt_plan* pl) { return pl->prm.max_iters >= 3 && pl->opt.tune_level >= 2; }

// The same for the transpose pass: equal shares of the D^T stream do not take equal time (the gathers of r hit the L2
// differently from SM to SM), so measure every CTA's pass time and hand out shares in proportion to measured speed.
// Cut the D^T stream into the given per-CTA shares and upload the schedule.  false: the tables would not fit.
static imrt_status upload_shares(imrt_plan* pl, const std::vector<double>& share, bool& fits) {
    const int n_b = pl->n_rows_tr;
    cudaStream_t st = pl->stream;
    std::vector<TrRange> ranges;
    std::vector<int> rowslot, cta_rng;
    build_ranges(pl->rp_tr, n_b, share, pl->tr_align, ranges, rowslot, cta_rng);
    fits = (int64_t)ranges.size() <= pl->max_ranges && rowslot[n_b] + 4 <= pl->max_slots;
    if (!fits) return IMRT_STATUS_OK;
    pl->tr_share = share;
    CUDA_TRY(pl, cudaMemcpyAsync(pl->tr_range_w, ranges.data(), sizeof(TrRange) * ranges.size(), cudaMemcpyHostToDevice, st));
    CUDA_TRY(pl, cudaMemcpyAsync(pl->rowslot_w, rowslot.data(), sizeof(int) * (n_b + 1), cudaMemcpyHostToDevice, st));
    CUDA_TRY(pl, cudaMemcpyAsync(pl->cta_rng_w, cta_rng.data(), sizeof(int) * cta_rng.size(), cudaMemcpyHostToDevice, st));
    CUDA_TRY(pl, cudaStreamSynchronize(st));
    pl->P.n_ranges = (int)ranges.size();
    pl->P.n_slots = rowslot[n_b];
    return IMRT_STATUS_OK;
}

static imrt_status tune_transpose(imrt_plan* pl) {
    const int grid = pl->P.grid_t, n_b = pl->n_rows_tr;
    if (pl->opt.tune_level < 1 || grid < 2 || pl->rp_tr[n_b] < (long long)grid * 8 * CHUNK_T) return IMRT_STATUS_OK;
    cudaStream_t st = pl->stream;
    PassArgs A;
    memset(&A, 0, sizeof A);
    A.mode = MODE_EVAL;
    A.r_in = pl->P.rbuf[0];
    A.g_out = pl->g_scratch;
    std::vector<unsigned long long> t(2 * (size_t)grid);
    const int iso_rounds = 3, rounds = iso_rounds + (can_time_in_loop(pl) ? 5 : 0);
    double best_worst = 1e300;
    std::vector<double> best_share;
    for (int it = 0; it <= rounds; ++it) {
        std::vector<double> durs(grid, 0.0);
        const int n_meas = it < iso_rounds ? 1 : LOOP_MEASUREMENTS;      // pass times inside the loop vary more: average a few
        for (int ms = 0; ms < n_meas; ++ms) {
            if (it < iso_rounds) {
                for (int rep = 0; rep < 2; ++rep) CUDA_TRY(pl, launch_transpose(pl, A));   // the first warms up, the second is read
            } else {
                const imrt_status ls = timing_loop_run(pl);
                if (ls != IMRT_STATUS_OK) return ls;
            }
            CUDA_TRY(pl, cudaMemcpyAsync(t.data(), pl->P.cta_ns + 2048, sizeof(unsigned long long) * t.size(), cudaMemcpyDeviceToHost, st));
            CUDA_TRY(pl, cudaStreamSynchronize(st));
            for (int c = 0; c < grid; ++c) durs[c] += (double)(t[2 * c + 1] - t[2 * c]) / n_meas;
        }
        double sum = 0.0, worst = 0.0;
        std::vector<double> share(grid);
        for (int c = 0; c < grid; ++c) {
            const double dur = durs[c];
            worst = std::max(worst, dur);
            share[c] = dur > 0.0 ? pl->tr_share[c] / dur : pl->tr_share[c];     // share per unit time = speed
            sum += share[c];
        }
        // keep the best schedule seen in the final kind of measurement (in the loop if possible, else isolated)
        if (it >= (rounds > iso_rounds ? iso_rounds : 0) && worst < best_worst) { best_worst = worst; best_share = pl->tr_share; }
        if (it == rounds) break;
        for (int c = 0; c < grid; ++c) share[c] /= sum;
        bool fits = true;
        const imrt_status us = upload_shares(pl, share, fits);
        if (us != IMRT_STATUS_OK) return us;
        if (!fits) break;      // keep the last good schedule
    }
    if (!best_share.empty() && best_share != pl->tr_share) {
        bool fits = true;
        return upload_shares(pl, best_share, fits);
    }
    return IMRT_STATUS_OK;
}

// The static partition of the dose pass is only as good as its cost model, and the model cannot know how the
// instruction-bound blocks (short rows at the field edges) trade against the bandwidth-bound ones on this device.
// So measure: run the pass, read every CTA's streaming time, rescale the cost of each CTA's blocks by its measured
// time per unit of modelled cost, re-partition, and repeat a few times.
static imrt_status tune_partition(imrt_plan* pl) {
    pl->tune_spread[0] = pl->tune_spread[1] = 0.0;
    const int grid = pl->P.grid_f;
    const size_t n_blk = pl->blk_cost.size();
    if (pl->opt.tune_level < 1 || n_blk < (size_t)grid * 8) return IMRT_STATUS_OK;
    cudaStream_t st = pl->stream;
    PassArgs A;              // the loop's own dose pass (R trial points) on x = 0
    memset(&A, 0, sizeof A);
    A.mode = MODE_TIMING;
    std::vector<int> cta_blk;
    partition_blocks(pl->blk_cost, grid, cta_blk);
    std::vector<unsigned long long> t(2 * (size_t)grid);
    std::vector<double> dur(grid);
    const int iso_rounds = 3;
    const int rounds = iso_rounds + (can_time_in_loop(pl) ? 5 : 0);
    double best_worst = 1e300;
    std::vector<int> best_blk;
    for (int it = 0; it <= rounds; ++it) {
        std::fill(dur.begin(), dur.end(), 0.0);
        const int n_meas = it < iso_rounds ? 1 : LOOP_MEASUREMENTS;      // pass times inside the loop vary more: average a few
        for (int ms = 0; ms < n_meas; ++ms) {
            if (it < iso_rounds) {
                for (int rep = 0; rep < 2; ++rep) CUDA_TRY(pl, launch_dose(pl, A));   // the first warms up, the second is read
            } else {
                const imrt_status ls = timing_loop_run(pl);
                if (ls != IMRT_STATUS_OK) return ls;
            }
            CUDA_TRY(pl, cudaMemcpyAsync(t.data(), pl->P.cta_ns, sizeof(unsigned long long) * t.size(), cudaMemcpyDeviceToHost, st));
            CUDA_TRY(pl, cudaStreamSynchronize(st));
            for (int c = 0; c < grid; ++c) dur[c] += (double)(t[2 * c + 1] - t[2 * c]) / n_meas;
        }
        double mean = 0.0, worst = 0.0;
        for (int c = 0; c < grid; ++c) {
            mean += dur[c] / grid;
            worst = std::max(worst, dur[c]);
        }
        if (it == 0) pl->tune_spread[0] = worst / mean;
        // keep the best partition seen in the final kind of measurement (in the loop if possible, else isolated)
        if (it >= (rounds > iso_rounds ? iso_rounds : 0) && worst < best_worst) { best_worst = worst; best_blk = cta_blk; pl->tune_spread[1] = worst / mean; }
        if (it == rounds) break;
        for (int c = 0; c < grid; ++c) {
            double sum = 0.0;
            for (int b = cta_blk[c]; b < cta_blk[c + 1]; ++b) sum += pl->blk_cost[b];
            if (sum <= 0.0 || dur[c] <= 0.0) continue;
            const double f = dur[c] / sum;
            for (int b = cta_blk[c]; b < cta_blk[c + 1]; ++b) pl->blk_cost[b] *= f;
        }
        partition_blocks(pl->blk_cost, grid, cta_blk);
        const imrt_status us = upload_partition(pl, cta_blk);
        if (us != IMRT_STATUS_OK) return us;
    }
    if (!best_blk.empty() && best_blk != cta_blk) return upload_partition(pl, best_blk);
    return IMRT_STATUS_OK;
}

// What imrt_plan_get_tuning hands out: this header, then cta_blk int[grid_f + 1], then tr_share double[grid_t].
constexpr unsigned int TUNING_MAGIC = 0x696d7274u;
struct TuningBlob {
    unsigned int magic;
    int grid_f, grid_t, pad;
    int64_t n_blk, nnz_tr;
};

// graph:  k_begin -> WHILE(outer){ k_transpose -> WHILE(inner){ k_dose } }
static imrt_status build_graph(imrt_plan* pl) {
    CUDA_TRY(pl, cudaGraphCreate(&pl->graph, 0));
    cudaGraphConditionalHandle h_outer, h_inner;
    CUDA_TRY(pl, cudaGraphConditionalHandleCreate(&h_outer, pl->graph, 0, 0));
    CUDA_TRY(pl, cudaGraphConditionalHandleCreate(&h_inner, pl->graph, 0, 0));
    PassArgs A;
    memset(&A, 0, sizeof A);
    A.mode = MODE_TRIAL;
    A.use_handles = 1;
    A.h_outer = h_outer;
    A.h_inner = h_inner;

    cudaGraphNode_t n_begin, n_outer, n_tr, n_inner, n_dose;
    {
        State* st = pl->P.st;
        int use = 1;
        void* args[] = {&st, &use, &h_outer};
        cudaGraphNodeParams np = {};
        np.type = cudaGraphNodeTypeKernel;
        np.kernel.func = (void*)k_begin;
        np.kernel.gridDim = dim3(1);
        np.kernel.blockDim = dim3(1);
        np.kernel.kernelParams = args;
        CUDA_TRY(pl, cudaGraphAddNode(&n_begin, pl->graph, nullptr, 0, &np));
    }
    cudaGraph_t body_outer, body_inner;
    {
        cudaGraphNodeParams np = {};
        np.type = cudaGraphNodeTypeConditional;
        np.conditional.handle = h_outer;
        np.conditional.type = cudaGraphCondTypeWhile;
        np.conditional.size = 1;
        CUDA_TRY(pl, cudaGraphAddNode(&n_outer, pl->graph, &n_begin, 1, &np));
        body_outer = np.conditional.phGraph_out[0];
    }
    {
        void* args[] = {&pl->P, &A};
        cudaGraphNodeParams np = {};
        np.type = cudaGraphNodeTypeKernel;
        np.kernel.func = (void*)k_transpose;
        np.kernel.gridDim = dim3(pl->P.grid_t);
        np.kernel.blockDim = dim3(NTHREADS);
        np.kernel.sharedMemBytes = (unsigned int)pl->smem_bytes;
        np.kernel.kernelParams = args;
        CUDA_TRY(pl, cudaGraphAddNode(&n_tr, body_outer, nullptr, 0, &np));
    }
    {
        cudaGraphNodeParams np = {};
        np.type = cudaGraphNodeTypeConditional;
        np.conditional.handle = h_inner;
        np.conditional.type = cudaGraphCondTypeWhile;
        np.conditional.size = 1;
        CUDA_TRY(pl, cudaGraphAddNode(&n_inner, body_outer, &n_tr, 1, &np));
        body_inner = np.conditional.phGraph_out[0];
    }
    {
        void* args[] = {&pl->P, &A};
        cudaGraphNodeParams np = {};
        np.type = cudaGraphNodeTypeKernel;
        np.kernel.func = (void*)k_dose;
        np.kernel.gridDim = dim3(pl->P.grid_f);
        np.kernel.blockDim = dim3(NTHREADS);
        np.kernel.sharedMemBytes = (unsigned int)pl->smem_bytes;
        np.kernel.kernelParams = args;
        CUDA_TRY(pl, cudaGraphAddNode(&n_dose, body_inner, nullptr, 0, &np));
    }
    CUDA_TRY(pl, cudaGraphInstantiate(&pl->graph_exec, pl->graph, 0));
    return IMRT_STATUS_OK;
}

// Phase timer of plan creation (imrt_options.profile_create: a synchronisation after every phase; the times are read
// with imrt_plan_get_create_times).
struct PhaseTimer {
    std::vector<double>* out;
    cudaStream_t st;
    std::chrono::steady_clock::time_point t0;
    PhaseTimer(std::vector<double>* o, cudaStream_t s) : out(o), st(s), t0(std::chrono::steady_clock::now()) {}
    void mark() {
        if (!out) return;
        cudaStreamSynchronize(st);
        const auto t1 = std::chrono::steady_clock::now();
        out->push_back(std::chrono::duration<double, std::milli>(t1 - t0).count());
        t0 = t1;
    }
};

// ------------------------------------------------------------------------------------------------ C-ABI
extern "C" {

const char* imrt_version(void) { return "imrtgp 0.2 (sm_100a)"; }

const char* imrt_last_error(const imrt_plan* plan) { return plan ? plan->err.c_str() : g_create_error.c_str(); }

imrt_status imrt_workspace_bytes(int64_t n_v, int64_t n_b, int64_t nnz, int32_t n_structures, int32_t max_iters,
                                 size_t* host_bytes) {
    if (!host_bytes || n_v < 1 || n_b < 1 || nnz < 0 || n_structures < 1 || n_structures > MAX_STRUCTURES || max_iters < 0)
        return fail(nullptr, IMRT_STATUS_INVALID_ARG, "imrt_workspace_bytes: bad argument");
    if (nnz >= (1LL << 31) - 16 || n_v >= (1LL << 31) - 16 || n_b >= (1LL << 31) - 16)
        return fail(nullptr, IMRT_STATUS_UNSUPPORTED, "sizes must fit int32");
    *host_bytes = make_layout(nullptr, n_v, n_b, nnz, n_structures, max_iters).total;
    return IMRT_STATUS_OK;
}

imrt_status imrt_plan_create(imrt_plan** out, int64_t n_v, int64_t n_b, int64_t nnz, const int32_t* row_ptr,
                             const int32_t* col_idx, const float* val, const uint8_t* structure_id, int32_t n_structures,
                             const float* host_t_under, const float* host_t_over, const float* host_w_under,
                             const float* host_w_over, const imrt_params* prm, const imrt_options* host_options,
                             void* workspace, size_t workspace_bytes, void* stream) {
    if (out) *out = nullptr;
    if (!out || !row_ptr || !structure_id || !host_t_under || !host_t_over || !host_w_under || !host_w_over || !prm || !workspace)
        return fail(nullptr, IMRT_STATUS_INVALID_ARG, "imrt_plan_create: null argument");
    if ((nnz > 0 && (!col_idx || !val)) || n_v < 1 || n_b < 1 || nnz < 0 || n_structures < 1 || n_structures > MAX_STRUCTURES)
        return fail(nullptr, IMRT_STATUS_INVALID_ARG, "imrt_plan_create: bad size (n_v %lld, n_b %lld, nnz %lld, n_structures %d)",
                    (long long)n_v, (long long)n_b, (long long)nnz, n_structures);
    if (nnz >= (1LL << 31) - 16 || n_v >= (1LL << 31) - 16 || n_b >= (1LL << 31) - 16)
        return fail(nullptr, IMRT_STATUS_UNSUPPORTED, "sizes must fit int32");
    if (!(prm->eps > 0.0 && prm->eps < 1.0) || !(prm->alpha > 1.0) || !(prm->lambda0 > 0.0) || !std::isfinite(prm->lambda0) ||
        prm->max_ls < 0 || prm->max_iters < 0 || prm->driver < 0 || prm->driver > 2 || prm->ls_batch < 0 || prm->ls_batch > R_MAX)
        return fail(nullptr, IMRT_STATUS_INVALID_ARG, "imrt_plan_create: bad imrt_params (need 0<eps<1, alpha>1, lambda0>0, driver in 0..2)");
    if (((uintptr_t)row_ptr | (uintptr_t)col_idx | (uintptr_t)val | (uintptr_t)workspace) & 15)
        return fail(nullptr, IMRT_STATUS_INVALID_ARG, "imrt_plan_create: device arrays must be 16-byte aligned");
    for (int s = 0; s < n_structures; ++s) {
        const float v[4] = {host_t_under[s], host_t_over[s], host_w_under[s], host_w_over[s]};
        for (float f : v)
            if (!std::isfinite(f)) return fail(nullptr, IMRT_STATUS_BAD_STRUCTURE, "structure %d: non-finite limit or weight", s);
        if (v[2] < 0.0f || v[3] < 0.0f) return fail(nullptr, IMRT_STATUS_BAD_STRUCTURE, "structure %d: negative weight", s);
    }
    const Layout L = make_layout(workspace, n_v, n_b, nnz, n_structures, prm->max_iters);
    if (workspace_bytes < L.total)
        return fail(nullptr, IMRT_STATUS_WORKSPACE_TOO_SMALL, "workspace has %zu bytes, %zu needed", workspace_bytes, L.total);

    int dev = 0, cc_major = 0, n_sm = 0, smem_optin = 0;
    CUDA_TRY(nullptr, cudaGetDevice(&dev));
    CUDA_TRY(nullptr, cudaDeviceGetAttribute(&cc_major, cudaDevAttrComputeCapabilityMajor, dev));
    CUDA_TRY(nullptr, cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
    CUDA_TRY(nullptr, cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
    if (cc_major != 10)
        return fail(nullptr, IMRT_STATUS_UNSUPPORTED_DEVICE, "device has compute capability %d.x; libimrtgp is built for sm_100a only", cc_major);
    if (n_sm > 1024) n_sm = 1024;
    const int n_sm_device = n_sm;
    if (host_options && host_options->n_ctas > 0) n_sm = std::min(n_sm, host_options->n_ctas);      // a share of the device

    imrt_options opt;
    memset(&opt, 0, sizeof opt);
    if (host_options) opt = *host_options;
    if (opt.tune_level < 0 || opt.tune_level > 2 || opt.dose_format < 0 || opt.dose_format > 1 || (opt.col_bits != 0 && opt.col_bits != 32) ||
        opt.transpose_format < 0 || opt.transpose_format > 2 || opt.quad_cap < 0 || opt.n_ctas < 0 || opt.spin_timeout_ms < 0 ||
        (opt.host_tuning && opt.host_tuning_bytes < sizeof(int) * 8))
        return fail(nullptr, IMRT_STATUS_INVALID_ARG, "imrt_plan_create: bad imrt_options");
    imrt_plan* pl = new imrt_plan();
    pl->prm = *prm;
    pl->opt = opt;
    pl->stream = (cudaStream_t)stream;
    pl->n_sm = n_sm;
    pl->n_sm_device = n_sm_device;
    pl->has_x = false;
    pl->graph = nullptr;
    pl->graph_exec = nullptr;
    pl->row_ptr = row_ptr;
    pl->sid = structure_id;
    cudaStream_t st = pl->stream;
    // every early return below releases the handle
    struct Guard { imrt_plan* p; ~Guard() { if (p) { g_create_error = p->err; delete p; } } } guard{pl};

    PhaseTimer phase(opt.profile_create ? &pl->create_ms : nullptr, st);
    // ---- validate: column indices and values, the row structure, the structure ids -- all on the device; only a
    // handful of flags come back (the rows must be known to be sane before any kernel walks them)
    DevPlan& P = pl->P;
    memset(&P, 0, sizeof P);
    CUDA_TRY(pl, cudaMemsetAsync(L.flags, 0, 16 * sizeof(int), st));
    CUDA_TRY(pl, cudaMemsetAsync(L.totals, 0, sizeof(LayoutTotals), st));
    if (nnz > 0) k_validate<<<grid_for(nnz, 256), 256, 0, st>>>(col_idx, val, nnz, (int)n_b, L.flags);
    k_validate_structure<<<grid_for(n_v, 256), 256, 0, st>>>(row_ptr, structure_id, (int)n_v, nnz, n_structures, L.totals);
    CUDA_TRY(pl, cudaGetLastError());
    int flags_h[16];
    LayoutTotals tot;
    CUDA_TRY(pl, cudaMemcpyAsync(flags_h, L.flags, sizeof flags_h, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(pl, cudaMemcpyAsync(&tot, L.totals, sizeof tot, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(pl, cudaStreamSynchronize(st));
    if (tot.bad_row_ptr) return fail(pl, IMRT_STATUS_BAD_CSR, "row_ptr is not a valid CSR row pointer (row_ptr[0] != 0, row_ptr[n_v] != nnz = %lld, or it decreases near row %d)", (long long)nnz, tot.bad_row);
    if (flags_h[0]) return fail(pl, IMRT_STATUS_BAD_CSR, "a column index is outside [0, n_b)");
    if (flags_h[1]) return fail(pl, IMRT_STATUS_BAD_CSR, "a value of D is not finite");
    if (tot.bad_sid) return fail(pl, IMRT_STATUS_BAD_STRUCTURE, "structure_id[%d] >= n_structures", tot.bad_sid - 1);
    if (tot.long_row)
        return fail(pl, IMRT_STATUS_UNSUPPORTED, "row %d of D has more than %d entries; this build handles rows up to that", tot.long_row - 1, MAX_CHUNK_SLOTS);

    // ---- penalty table
    std::vector<float4> table_h(MAX_STRUCTURES, make_float4(0, 0, 0, 0));
    for (int s = 0; s < n_structures; ++s) table_h[s] = make_float4(host_t_under[s], host_t_over[s], host_w_under[s], host_w_over[s]);
    CUDA_TRY(pl, cudaMemcpyAsync(L.table, table_h.data(), sizeof(float4) * MAX_STRUCTURES, cudaMemcpyHostToDevice, st));
    if (nnz > 0) {      // row_ptr is sane: the rows can be walked
        k_validate_rows<<<grid_for(n_v * 32, 256), 256, 0, st>>>(row_ptr, col_idx, (int)n_v, L.flags);
        CUDA_TRY(pl, cudaGetLastError());
    }
    phase.mark();

    // ---- dose-pass blocks: 16-bit columns whenever n_b allows (25 % fewer bytes per non-zero)
    const bool col16 = n_b <= 65536 && opt.col_bits != 32;
    const int64_t nb_pad_est = (n_b + 31) & ~31LL;
    const RecordCaps caps = record_caps(n_v, nnz, (int64_t)smem_optin - SMEM_HEADER - 256 - std::max(SMEM_WPART, SMEM_DSC) - nb_pad_est * 4 * (R_MAX + 1), opt.quad_cap);
    // quad format on offer: count the distinct columns of every 4 consecutive rows
    const int bm_words = (int)((n_b + 31) / 32);
    const bool offer_quads = col16 && n_b <= QUAD_MAX_NB && nnz > 0 && opt.dose_format == 0;
    if (offer_quads) {
        const int n_quads = (int)((n_v + 3) / 4);
        k_quad_union<<<std::min(n_quads / 8 + 1, n_sm * 8), 256, 8 * bm_words * sizeof(uint32_t), st>>>(row_ptr, col_idx, (int)n_v, n_quads, bm_words, L.quadU);
        CUDA_TRY(pl, cudaGetLastError());
    }
    phase.mark();
    // ---- record layout on the device (layout.cuh): count per segment, scan, write
    const Bounds B = bounds_for(n_v, n_b, nnz);
    const int n_seg = (int)((n_v + SEG_ROWS - 1) / SEG_ROWS);
    const int col_bytes = col16 ? 2 : 4;
    CUDA_TRY(pl, cudaMemsetAsync(L.covered, 1, (size_t)n_v, st));
    CUDA_TRY(pl, cudaMemsetAsync(L.seg_rec, 0, sizeof(int) * (n_seg + 2), st));
    CUDA_TRY(pl, cudaMemsetAsync(L.seg_meta, 0, sizeof(int) * (n_seg + 2), st));
    CUDA_TRY(pl, cudaMemsetAsync(L.seg_b128, 0, sizeof(int) * (n_seg + 2), st));
    k_layout_count<<<grid_for(n_seg, 64), 64, 0, st>>>(row_ptr, structure_id, offer_quads ? L.quadU : nullptr, (int)n_v, n_seg, caps, col_bytes,
                                                       L.seg_rec, L.seg_meta, L.seg_b128, L.totals);
    for (int* arr : {L.seg_rec, L.seg_meta, L.seg_b128}) {
        size_t temp = 0;
        CUDA_TRY(pl, cub::DeviceScan::ExclusiveSum(nullptr, temp, arr, arr, n_seg + 1, st));
        if (temp > B.sort_temp) return fail(pl, IMRT_STATUS_WORKSPACE_TOO_SMALL, "internal: scan needs %zu temp bytes", temp);
        CUDA_TRY(pl, cub::DeviceScan::ExclusiveSum(L.sort_temp, temp, arr, arr, n_seg + 1, st));
    }
    LayoutOut LO = {L.blk, L.pk, L.rowmeta, L.cost_fx, L.covered};
    k_layout_write<<<grid_for(n_seg, 64), 64, 0, st>>>(row_ptr, structure_id, offer_quads ? L.quadU : nullptr, (int)n_v, n_seg, caps, col_bytes,
                                                       L.seg_rec, L.seg_meta, L.seg_b128, LO, L.totals);
    CUDA_TRY(pl, cudaGetLastError());
    CUDA_TRY(pl, cudaMemcpyAsync(flags_h, L.flags, sizeof flags_h, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(pl, cudaMemcpyAsync(&tot, L.totals, sizeof tot, cudaMemcpyDeviceToHost, st));
    struct Event {             // released on every path out of this function
        cudaEvent_t e = nullptr;
        ~Event() { if (e) cudaEventDestroy(e); }
    } ev_totals;
    CUDA_TRY(pl, cudaEventCreateWithFlags(&ev_totals.e, cudaEventDisableTiming));
    CUDA_TRY(pl, cudaEventRecord(ev_totals.e, st));
    // ---- explicit transpose: stable radix sort of (column, position) pairs, then gather (north star choice 1).
    // Enqueued before the host waits for the layout totals: the device sorts while the host sizes the next launches.
    CUDA_TRY(pl, cudaMemsetAsync(L.colT, 0, sizeof(int) * B.nnz_pad, st));
    CUDA_TRY(pl, cudaMemsetAsync(L.valT, 0, sizeof(float) * B.nnz_pad, st));
    std::vector<int> rpT((size_t)n_b + 1, 0);
    if (nnz > 0) {
        k_iota_keys<<<grid_for(nnz, 256), 256, 0, st>>>(col_idx, L.keysA, L.valsA, nnz);
        cub::DoubleBuffer<unsigned int> dk(L.keysA, L.keysB), dv(L.valsA, L.valsB);
        int end_bit = 1;
        while ((1LL << end_bit) < n_b) ++end_bit;
        size_t temp = 0;
        CUDA_TRY(pl, cub::DeviceRadixSort::SortPairs(nullptr, temp, dk, dv, (int)nnz, 0, end_bit, st));
        if (temp > B.sort_temp) return fail(pl, IMRT_STATUS_WORKSPACE_TOO_SMALL, "internal: radix sort needs %zu temp bytes, %zu reserved", temp, B.sort_temp);
        CUDA_TRY(pl, cub::DeviceRadixSort::SortPairs(L.sort_temp, temp, dk, dv, (int)nnz, 0, end_bit, st));
        k_rowT_ptr<<<(int)((n_b + 1 + 255) / 256), 256, 0, st>>>(dk.Current(), nnz, (int)n_b, L.rowT_ptr);
        k_fill_transpose<<<grid_for(nnz, 256), 256, 0, st>>>(dv.Current(), row_ptr, (int)n_v, val, nnz, L.colT, L.valT);
        CUDA_TRY(pl, cudaGetLastError());
    } else {
        CUDA_TRY(pl, cudaMemsetAsync(L.rowT_ptr, 0, sizeof(int) * (n_b + 1), st));
    }
    {
        const cudaError_t e = cudaEventSynchronize(ev_totals.e);
        if (e != cudaSuccess) { cudaStreamSynchronize(st); return fail(pl, IMRT_STATUS_CUDA_ERROR, "layout: %s", cudaGetErrorString(e)); }
    }
    if (flags_h[3]) { cudaStreamSynchronize(st); return fail(pl, IMRT_STATUS_BAD_CSR, "column indices are not strictly ascending inside a row"); }
    phase.mark();
    const size_t n_blk = (size_t)tot.n_blk;
    const size_t pack_bytes = (size_t)tot.pack128 * 128;
    if ((int64_t)n_blk > B.max_blk || (int64_t)tot.n_meta > B.max_meta || pack_bytes > B.max_pack) {
        cudaStreamSynchronize(st);
        return fail(pl, IMRT_STATUS_WORKSPACE_TOO_SMALL, "internal: block tables exceed their bound (%zu blocks, %d words, %zu bytes)", n_blk, tot.n_meta, pack_bytes);
    }
    pl->n_blk = (int64_t)n_blk;
    pl->pack_bytes = (int64_t)pack_bytes;
    pl->n_skipped = tot.n_skipped; pl->n_nonempty = tot.n_nonempty; pl->n_quad_rows = tot.n_quad_rows;
    const int grid_f = (int)std::max<size_t>(1, std::min<size_t>((size_t)n_sm, n_blk));
    if (n_blk) {
        const size_t pk_smem = offer_quads ? 8 * 2 * bm_words * sizeof(uint32_t) : 0;
        if (col16) k_pack_blocks<true><<<(unsigned int)n_blk, 256, pk_smem, st>>>(L.pk, L.rowmeta, row_ptr, col_idx, val, (int)n_v, bm_words, L.pack);
        else k_pack_blocks<false><<<(unsigned int)n_blk, 256, 0, st>>>(L.pk, L.rowmeta, row_ptr, col_idx, val, (int)n_v, bm_words, L.pack);
        CUDA_TRY(pl, cudaGetLastError());
    }
    // the modelled partition: exclusive scan of the record costs, one binary search per CTA
    std::vector<int> cta_blk((size_t)grid_f + 1, 0);
    {
        CUDA_TRY(pl, cudaMemsetAsync(L.cost_fx + n_blk, 0, sizeof(long long), st));
        size_t temp = 0;
        CUDA_TRY(pl, cub::DeviceScan::ExclusiveSum(nullptr, temp, L.cost_fx, L.cost_pre, (int)(n_blk + 1), st));
        if (temp > B.sort_temp) return fail(pl, IMRT_STATUS_WORKSPACE_TOO_SMALL, "internal: scan needs %zu temp bytes", temp);
        // the radix sort above owns sort_temp until it has run; the stream serialises the two
        CUDA_TRY(pl, cub::DeviceScan::ExclusiveSum(L.sort_temp, temp, L.cost_fx, L.cost_pre, (int)(n_blk + 1), st));
        k_partition<<<(grid_f + 1 + 127) / 128, 128, 0, st>>>(L.cost_pre, (int)n_blk, grid_f, L.cta_blk);
        CUDA_TRY(pl, cudaGetLastError());
        CUDA_TRY(pl, cudaMemcpyAsync(cta_blk.data(), L.cta_blk, sizeof(int) * (grid_f + 1), cudaMemcpyDeviceToHost, st));
        if (opt.tune_level >= 1 && !opt.host_tuning) {      // the measured rebalancing rescales the costs on the host
            std::vector<long long> cfx(n_blk);
            CUDA_TRY(pl, cudaMemcpyAsync(cfx.data(), L.cost_fx, sizeof(long long) * n_blk, cudaMemcpyDeviceToHost, st));
            CUDA_TRY(pl, cudaStreamSynchronize(st));
            pl->blk_cost.resize(n_blk);
            for (size_t b = 0; b < n_blk; ++b) pl->blk_cost[b] = (double)cfx[b] / 1024.0;
        }
    }
    phase.mark();
    // ---- the explicit transpose was enqueued before the record layout: fetch its row pointers
    if (nnz > 0) CUDA_TRY(pl, cudaMemcpyAsync(rpT.data(), L.rowT_ptr, sizeof(int) * (n_b + 1), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(pl, cudaStreamSynchronize(st));      // rpT and cta_blk are on the host now
    phase.mark();
    imrt_status s = IMRT_STATUS_OK;

    // ---- transpose-pass ranges and gradient slots
    std::vector<TrRange> ranges;
    std::vector<int> rowslot, cta_rng_h;
    // ---- the stream the transpose pass reads.  First choice: row pairs with 16-bit voxel offsets, if that is smaller
    // than single rows; second: single rows with 16-bit offsets; last: the plain 32-bit CSR (a group of 32 entries
    // spanning more than 65,535 voxels rules the 16-bit forms out).
    const bool can16 = nnz > 0 && opt.transpose_format != 2 && nnz + 128 * n_b + 128 < (1LL << 31);
    std::vector<int> rpP((size_t)n_b + 1, 0);
    if (can16)
        for (int64_t i = 0; i < n_b; ++i) rpP[i + 1] = rpP[i] + ((rpT[i + 1] - rpT[i] + 127) & ~127);
    const int n_pairs = (int)((n_b + 1) / 2);
    std::vector<int> rpPair((size_t)n_pairs + 1, 0);
    bool pairs = can16 && n_b >= 2 && opt.transpose_format == 0;
    if (pairs) {
        std::vector<int> U((size_t)n_pairs);
        k_pair_count<<<n_pairs, 256, 0, st>>>(L.rowT_ptr, L.colT, (int)n_b, L.pairU);
        CUDA_TRY(pl, cudaGetLastError());
        CUDA_TRY(pl, cudaMemcpyAsync(U.data(), L.pairU, sizeof(int) * n_pairs, cudaMemcpyDeviceToHost, st));
        CUDA_TRY(pl, cudaStreamSynchronize(st));
        for (int i = 0; i < n_pairs; ++i) rpPair[i + 1] = rpPair[i] + ((U[i] + 127) & ~127);
        pairs = (double)rpPair[n_pairs] * 10.125 < (double)rpP[n_b] * 6.125;       // bytes per entry of the two forms
    }
    if (pairs) {
        const long long tot = rpPair[n_pairs];
        CUDA_TRY(pl, cudaMemcpyAsync(L.rowP_ptr, rpPair.data(), sizeof(int) * (n_pairs + 1), cudaMemcpyHostToDevice, st));
        CUDA_TRY(pl, cudaMemsetAsync(L.valP, 0, sizeof(float) * 2 * tot, st));
        CUDA_TRY(pl, cudaMemsetAsync(L.voxU, 0xFF, sizeof(int) * tot, st));
        k_pair_fill<<<n_pairs, 256, 0, st>>>(L.rowT_ptr, L.colT, L.valT, (int)n_b, L.rowP_ptr, reinterpret_cast<float2*>(L.valP), L.voxU);
        if (tot > 0) k_pair_tiles<<<grid_for(tot, 256), 256, 0, st>>>(L.voxU, tot / 32, L.idP, L.baseP, L.flags);
        CUDA_TRY(pl, cudaGetLastError());
        CUDA_TRY(pl, cudaMemcpyAsync(flags_h, L.flags, sizeof flags_h, cudaMemcpyDeviceToHost, st));
        CUDA_TRY(pl, cudaStreamSynchronize(st));
        if (flags_h[2]) {
            pairs = false;
            CUDA_TRY(pl, cudaMemsetAsync(L.flags, 0, 16 * sizeof(int), st));
        }
    }
    bool id16 = can16 && !pairs;
    if (id16) {
        const long long n_groups = rpP[n_b] / 32;
        CUDA_TRY(pl, cudaMemcpyAsync(L.rowP_ptr, rpP.data(), sizeof(int) * (n_b + 1), cudaMemcpyHostToDevice, st));
        if (n_groups > 0) k_pack_transpose<<<grid_for(n_groups * 32, 256), 256, 0, st>>>(L.rowT_ptr, L.rowP_ptr, L.colT, L.valT, (int)n_b, n_groups, L.valP, L.idP, L.baseP, L.flags);
        CUDA_TRY(pl, cudaGetLastError());
        CUDA_TRY(pl, cudaMemcpyAsync(flags_h, L.flags, sizeof flags_h, cudaMemcpyDeviceToHost, st));
        CUDA_TRY(pl, cudaStreamSynchronize(st));
        if (flags_h[2]) id16 = false;
    }
    const int tr_fmt = pairs ? 2 : id16 ? 1 : 0;
    const int n_rows_tr = pairs ? n_pairs : (int)n_b;
    pl->n_rows_tr = n_rows_tr;
    pl->tr_stream_bytes = pairs ? (int64_t)rpPair[n_pairs] * 10 + rpPair[n_pairs] / 8
                          : id16 ? (int64_t)rpP[n_b] * 6 + rpP[n_b] / 8 : (int64_t)nnz * 8;
    pl->rp_tr = pairs ? rpPair : id16 ? rpP : rpT;
    pl->tr_align = tr_fmt ? 128 : 4;
    const int grid_t = (int)std::max<long long>(1, std::min<long long>(n_sm, (long long)pl->rp_tr[n_rows_tr] / (4 * CHUNK_T) + 1));
    pl->tr_share.assign(grid_t, 1.0 / grid_t);
    build_ranges(pl->rp_tr, n_rows_tr, pl->tr_share, pl->tr_align, ranges, rowslot, cta_rng_h);
    if ((int64_t)ranges.size() > B.max_ranges) return fail(pl, IMRT_STATUS_WORKSPACE_TOO_SMALL, "internal: %zu transpose ranges exceed the bound", ranges.size());
    const int n_slots = rowslot[n_rows_tr];
    if (!ranges.empty()) CUDA_TRY(pl, cudaMemcpyAsync(L.tr_range, ranges.data(), sizeof(TrRange) * ranges.size(), cudaMemcpyHostToDevice, st));
    CUDA_TRY(pl, cudaMemcpyAsync(L.rowslot_ptr, rowslot.data(), sizeof(int) * (n_rows_tr + 1), cudaMemcpyHostToDevice, st));
    CUDA_TRY(pl, cudaMemcpyAsync(L.cta_rng, cta_rng_h.data(), sizeof(int) * cta_rng_h.size(), cudaMemcpyHostToDevice, st));
    pl->max_ranges = B.max_ranges; pl->max_slots = B.max_slots;
    pl->tr_range_w = L.tr_range; pl->rowslot_w = L.rowslot_ptr; pl->cta_rng_w = L.cta_rng;

    phase.mark();
    // ---- shared-memory layout (one layout for the three kernels): header, penalty table, transpose partials, dose
    // scratch, the R trial points, g, then the ring (dose pass) / stages (transpose pass).  R = the largest of 4, 2, 1
    // not above the request that leaves the ring room for 16 records of average size (one per consumer warp).
    const int max_rec = std::max(tot.max_rec_bytes, 128);
    const long long avg_rec = n_blk ? (long long)(pack_bytes / n_blk) : 128;
    const int nb_pad = (int)((n_b + 31) & ~31LL);
    int R = prm->ls_batch == 0 ? R_MAX : prm->ls_batch;
    if (R != 1 && R != 2 && R != 4) return fail(pl, IMRT_STATUS_INVALID_ARG, "imrt_params.ls_batch must be 0, 1, 2 or 4");
    const int stage_t = pairs ? CHUNK_T * 10 + CHUNK_T / 8 : id16 ? CHUNK_T * 6 + CHUNK_T / 8 : STAGE_T_BYTES;
    int off = 0, avail = 0, stt = 0;
    for (;; R /= 2) {
        off = SMEM_HEADER + ((n_structures * 16 + 127) & ~127);
        P.wpart_off = off;                    // the transpose pass's partials and the dose pass's row scratch share one
        P.dsc_off = off;                      // region: a CTA is never in both passes at once
        off += SMEM_WPART > SMEM_DSC ? SMEM_WPART : SMEM_DSC;
        P.x_off = off; off += nb_pad * 4 * R;
        P.g_off = off; off += nb_pad * 4;
        off = (off + 127) & ~127;
        P.stage_off = off;
        avail = smem_optin - off;
        avail = (smem_optin - off) & ~127;
        P.tr_stage_off = (P.x_off + 127) & ~127;
        stt = avail > 0 ? std::min(MAX_STAGES_T, (off + avail - P.tr_stage_off) / stage_t) : 0;
        if (R == 1 || (avail >= 2 * max_rec && avail >= (W_CONS / 2) * avg_rec && stt >= 2)) break;
    }
    if (avail < 2 * max_rec || stt < 2)
        return fail(pl, IMRT_STATUS_UNSUPPORTED, "n_b = %lld beamlets and records of up to %d bytes do not fit in shared memory", (long long)n_b, max_rec);
    pl->smem_bytes = (size_t)off + (size_t)avail;
    P.R = R;
    P.ring_f_bytes = avail;
    P.max_rec_bytes = max_rec;

    P.nnz = nnz; P.n_v = (int)n_v; P.n_b = (int)n_b;
    P.pack = L.pack; P.blk = L.blk; P.cta_blk = L.cta_blk; P.grid_f = grid_f;
    P.col16 = col16 ? 1 : 0;
    P.rowT_ptr = tr_fmt ? L.rowP_ptr : L.rowT_ptr; P.colT = L.colT; P.valT = L.valT;
    P.valP = L.valP; P.idP = L.idP; P.baseP = L.baseP; P.id16 = tr_fmt; P.stage_t_bytes = stage_t;
    P.tr_range = L.tr_range; P.rowslot_ptr = L.rowslot_ptr; P.cta_rng = L.cta_rng;
    P.n_ranges = (int)ranges.size(); P.grid_t = grid_t;
    P.n_stages_t = stt; P.n_slots = n_slots;
    P.table = L.table; P.n_structures = n_structures; P.covered = L.covered;
    P.xbuf[0] = L.xbuf[0]; P.xbuf[1] = L.xbuf[1]; P.g = L.g;
    for (int i = 0; i <= R_MAX; ++i) P.rbuf[i] = L.rbuf[i];
    P.Gpart[0] = L.Gpart[0]; P.Gpart[1] = L.Gpart[1]; P.gslot[0] = L.gslot[0]; P.gslot[1] = L.gslot[1];
    P.cta_ns = L.cta_ns;
    P.st = L.st; P.tr_obj = L.tr_obj; P.tr_lambda = L.tr_lambda; P.tr_step_sq = L.tr_step_sq; P.tr_trials = L.tr_trials;
    pl->r_scratch = L.r_scratch; pl->g_scratch = L.g_scratch; pl->d_scratch = L.d_scratch;
    pl->cta_blk_w = L.cta_blk;
    pl->blk_w = L.blk;
    pl->rowT_ptr_w = L.rowT_ptr; pl->colT_w = L.colT; pl->valT_w = L.valT;
    pl->dvh = L.dvh;
    pl->rank_plans_w = L.rank_plans;
    pl->grid_p = n_sm;

    CUDA_TRY(pl, cudaFuncSetAttribute(k_dose, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl->smem_bytes));
    CUDA_TRY(pl, cudaFuncSetAttribute(k_transpose, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl->smem_bytes));
    CUDA_TRY(pl, cudaFuncSetAttribute(k_persistent, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl->smem_bytes));
    CUDA_TRY(pl, cudaFuncSetAttribute(k_stream, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl->smem_bytes));

    // ---- device state, constant residual of the zero-dose rows
    State st_h;
    memset(&st_h, 0, sizeof st_h);
    st_h.eps = prm->eps; st_h.alpha = prm->alpha; st_h.lambda0 = prm->lambda0; st_h.lambda = prm->lambda0;
    st_h.max_ls = prm->max_ls; st_h.trace_cap = prm->max_iters; st_h.xi = 0; st_h.ri = 0;
    st_h.spin_timeout_ns = (unsigned long long)(pl->opt.spin_timeout_ms > 0 ? pl->opt.spin_timeout_ms : 2000) * 1000000ull;
    CUDA_TRY(pl, cudaMemcpyAsync(L.st, &st_h, sizeof st_h, cudaMemcpyHostToDevice, st));
    CUDA_TRY(pl, cudaMemsetAsync(L.gslot[0], 0, sizeof(double) * 2 * B.max_slots, st));
    CUDA_TRY(pl, cudaMemsetAsync(L.gslot[1], 0, sizeof(double) * 2 * B.max_slots, st));
    CUDA_TRY(pl, cudaMemsetAsync(L.Gpart[0], 0, sizeof(double) * 1024 * R_MAX, st));
    CUDA_TRY(pl, cudaMemsetAsync(L.Gpart[1], 0, sizeof(double) * 1024 * R_MAX, st));
    CUDA_TRY(pl, cudaMemsetAsync(L.xbuf[0], 0, sizeof(float) * (n_b + 4), st));
    CUDA_TRY(pl, cudaMemsetAsync(L.xbuf[1], 0, sizeof(float) * (n_b + 4), st));
    CUDA_TRY(pl, cudaMemsetAsync(L.g, 0, sizeof(float) * (n_b + 4), st));
    CUDA_TRY(pl, cudaMemsetAsync(L.cta_ns, 0, sizeof(unsigned long long) * 4096, st));
    {
        RPtrs rp_all;
        for (int i = 0; i <= R_MAX; ++i) rp_all.p[i] = L.rbuf[i];
        k_fill_zero_dose_rows<<<(int)((n_v + 255) / 256), 256, 0, st>>>(structure_id, L.table, L.st, (int)n_v, rp_all, nullptr);
        k_skip_constants<<<SKIP_BLOCKS, 1024, 0, st>>>(structure_id, L.covered, L.table, L.st, (int)n_v, rp_all, L.Gpart[1]);
        k_skip_final<<<1, 1, 0, st>>>(L.Gpart[1], SKIP_BLOCKS, L.st);
    }
    CUDA_TRY(pl, cudaGetLastError());
    CUDA_TRY(pl, cudaStreamSynchronize(st));

    // ---- a caller-supplied partition (imrt_plan_get_tuning of an earlier plan of this problem) replaces the measurements
    const TuningBlob* tb = static_cast<const TuningBlob*>(opt.host_tuning);
    if (tb) {
        if (tb->magic != TUNING_MAGIC || tb->n_blk != (int64_t)n_blk || tb->grid_f != grid_f || tb->grid_t != grid_t || tb->nnz_tr != pl->rp_tr[n_rows_tr] ||
            opt.host_tuning_bytes < sizeof(TuningBlob) + sizeof(int) * (grid_f + 1) + sizeof(double) * grid_t)
            return fail(pl, IMRT_STATUS_INVALID_ARG, "imrt_options.host_tuning does not belong to this problem / these options / this device");
        const int* cb = reinterpret_cast<const int*>(tb + 1);
        cta_blk.assign(cb, cb + grid_f + 1);
        for (int c = 0; c < grid_f; ++c)
            if (cta_blk[c] > cta_blk[c + 1] || cta_blk[0] != 0 || cta_blk[grid_f] != (int)n_blk)
                return fail(pl, IMRT_STATUS_INVALID_ARG, "imrt_options.host_tuning: corrupt partition");
    }
    s = upload_partition(pl, cta_blk);
    if (s != IMRT_STATUS_OK) return s;
    phase.mark();
    if (tb) {
        std::vector<double> share(grid_t);
        memcpy(share.data(), reinterpret_cast<const char*>(tb + 1) + sizeof(int) * (grid_f + 1), sizeof(double) * grid_t);
        bool fits = true;
        s = upload_shares(pl, share, fits);
        if (s != IMRT_STATUS_OK) return s;
        if (!fits) return fail(pl, IMRT_STATUS_INVALID_ARG, "imrt_options.host_tuning: transpose shares do not fit");
        phase.mark();
        phase.mark();
    } else {
        s = tune_partition(pl);
        if (s != IMRT_STATUS_OK) return s;
        phase.mark();
        s = tune_transpose(pl);
        if (s != IMRT_STATUS_OK) return s;
        phase.mark();
    }
    if (prm->driver == 0) {
        s = build_graph(pl);
        if (s != IMRT_STATUS_OK) return s;
    }
    phase.mark();
    guard.p = nullptr;
    *out = pl;
    return IMRT_STATUS_OK;
}

imrt_status imrt_plan_destroy(imrt_plan* pl) {
    if (!pl) return IMRT_STATUS_INVALID_ARG;
    cudaStreamSynchronize(pl->stream);
    if (pl->graph_exec) cudaGraphExecDestroy(pl->graph_exec);
    if (pl->graph) cudaGraphDestroy(pl->graph);
    delete pl;
    return IMRT_STATUS_OK;
}

imrt_status imrt_plan_set_x(imrt_plan* pl, const float* x0) {
    if (!pl || !x0) return fail(pl, IMRT_STATUS_INVALID_ARG, "imrt_plan_set_x: null argument");
    cudaStream_t st = pl->stream;
    k_reset_state<<<1, 1, 0, st>>>(pl->P.st);
    k_check_x<<<grid_for(pl->P.n_b, 256), 256, 0, st>>>(x0, pl->P.n_b, pl->P.st);
    int bad = 0;
    CUDA_TRY(pl, cudaMemcpyAsync(&bad, &pl->P.st->bad_x, sizeof(int), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(pl, cudaStreamSynchronize(st));
    if (bad) { pl->has_x = false; return fail(pl, IMRT_STATUS_BAD_X, "x0 has a negative or non-finite entry"); }
    CUDA_TRY(pl, cudaMemcpyAsync(pl->P.xbuf[0], x0, sizeof(float) * pl->P.n_b, cudaMemcpyDeviceToDevice, st));
    PassArgs A;
    memset(&A, 0, sizeof A);
    A.mode = MODE_INIT;   // G(x_1), r(x_1): reads xbuf[0], writes rbuf[0], flips xi / ri to 0
    CUDA_TRY(pl, launch_dose(pl, A));
    pl->has_x = true;
    return IMRT_STATUS_OK;
}

__global__ void k_set_limits(State* st, const float* tvu, const float* tvo) { st->tvu = tvu; st->tvo = tvo; }

imrt_status imrt_plan_set_voxel_limits(imrt_plan* pl, const float* t_under_v, const float* t_over_v) {
    if (!pl) return IMRT_STATUS_INVALID_ARG;
    if (((uintptr_t)t_under_v | (uintptr_t)t_over_v) & 3) return fail(pl, IMRT_STATUS_INVALID_ARG, "imrt_plan_set_voxel_limits: misaligned array");
    cudaStream_t st = pl->stream;
    k_set_limits<<<1, 1, 0, st>>>(pl->P.st, t_under_v, t_over_v);
    RPtrs rp_all;
    for (int i = 0; i <= R_MAX; ++i) rp_all.p[i] = pl->P.rbuf[i];
    k_skip_constants<<<SKIP_BLOCKS, 1024, 0, st>>>(pl->sid, pl->P.covered, pl->P.table, pl->P.st, pl->P.n_v, rp_all, pl->P.Gpart[1]);
    k_skip_final<<<1, 1, 0, st>>>(pl->P.Gpart[1], SKIP_BLOCKS, pl->P.st);
    CUDA_TRY(pl, cudaGetLastError());
    pl->has_x = false;     // G(x_1), r(x_1) belong to the old limits
    return IMRT_STATUS_OK;
}

static imrt_status run_common(imrt_plan* pl, int32_t n_iters, double delta) {
    if (!pl) return IMRT_STATUS_INVALID_ARG;
    if (!pl->has_x) return fail(pl, IMRT_STATUS_NOT_READY, "call imrt_plan_set_x first");
    if (n_iters < 0 || !(delta >= 0.0)) return fail(pl, IMRT_STATUS_INVALID_ARG, "run: n_iters and delta must be >= 0");
    cudaStream_t st = pl->stream;
    k_set_target<<<1, 1, 0, st>>>(pl->P.st, n_iters, delta);
    CUDA_TRY(pl, cudaGetLastError());
    if (pl->P.world > 1 && pl->prm.driver != 2)
        return fail(pl, IMRT_STATUS_UNSUPPORTED, "a row-sharded plan runs with the persistent driver (imrt_params.driver = 2) only");
    if (pl->prm.driver == 0) {
        CUDA_TRY(pl, cudaGraphLaunch(pl->graph_exec, st));
    } else if (pl->prm.driver == 2) {
        CUDA_TRY(pl, launch_persistent(pl));
    } else {
        // host-driven: the loop conditions come back after every pass (one sync per trial)
        PassArgs A;
        memset(&A, 0, sizeof A);
        A.mode = MODE_TRIAL;
        cudaGraphConditionalHandle none = 0;
        k_begin<<<1, 1, 0, st>>>(pl->P.st, 0, none);
        int cont[2];
        auto fetch = [&]() -> cudaError_t {
            cudaError_t e = cudaMemcpyAsync(cont, &pl->P.st->cont_outer, 2 * sizeof(int), cudaMemcpyDeviceToHost, st);
            return e != cudaSuccess ? e : cudaStreamSynchronize(st);
        };
        CUDA_TRY(pl, fetch());
        while (cont[0]) {
            CUDA_TRY(pl, launch_transpose(pl, A));
            CUDA_TRY(pl, fetch());
            while (cont[1]) {
                CUDA_TRY(pl, launch_dose(pl, A));
                CUDA_TRY(pl, fetch());
            }
        }
    }
    return IMRT_STATUS_OK;
}

imrt_status imrt_plan_run_iters(imrt_plan* pl, int32_t n_iters) { return run_common(pl, n_iters, 0.0); }

// ---------------------------------------------------------------------------------------------- row-sharded plans
imrt_status imrt_shard_inbox_bytes(int64_t n_b, int32_t world, size_t* host_bytes) {
    if (!host_bytes || n_b < 1 || n_b >= (1LL << 31) - 64 || world < 1 || world > MAX_WORLD)
        return fail(nullptr, IMRT_STATUS_INVALID_ARG, "imrt_shard_inbox_bytes: bad argument (1 <= world <= %d)", MAX_WORLD);
    *host_bytes = inbox_bytes((int)n_b, world);
    return IMRT_STATUS_OK;
}

__global__ void k_reset_shard_seq(State* st) { st->seq_g = 0ull; st->seq_G = 0ull; }

imrt_status imrt_plan_set_shard(imrt_plan* pl, int32_t rank, int32_t world, void* const* host_inboxes) {
    if (!pl || world < 1 || world > MAX_WORLD || rank < 0 || rank >= world || (world > 1 && !host_inboxes))
        return fail(pl, IMRT_STATUS_INVALID_ARG, "imrt_plan_set_shard: bad argument (0 <= rank < world <= %d)", MAX_WORLD);
    if (world > 1 && pl->prm.driver != 2)
        return fail(pl, IMRT_STATUS_UNSUPPORTED, "a row-sharded plan runs with the persistent driver (imrt_params.driver = 2) only");
    for (int q = 0; world > 1 && q < world; ++q)             // validate everything first: a refused call changes nothing
        if (!host_inboxes[q] || ((uintptr_t)host_inboxes[q] & 15))
            return fail(pl, IMRT_STATUS_INVALID_ARG, "imrt_plan_set_shard: inbox %d is null or misaligned", q);
    pl->P.rank = rank;
    pl->P.world = world;
    for (int q = 0; q < MAX_WORLD; ++q) pl->P.inbox[q] = (world > 1 && q < world) ? static_cast<unsigned char*>(host_inboxes[q]) : nullptr;
    // the exchange counters restart with the (zero-filled) inboxes: every rank of a group counts from the same number
    k_reset_shard_seq<<<1, 1, 0, pl->stream>>>(pl->P.st);
    CUDA_TRY(pl, cudaGetLastError());
    pl->has_x = false;         // G(x_1) has to be formed again, and summed over the ranks
    return IMRT_STATUS_OK;
}

imrt_status imrt_plan_run_ranks(imrt_plan* const* host_plans, int32_t n_ranks, int32_t n_iters, double delta) {
    if (!host_plans || n_ranks < 1 || n_ranks > MAX_WORLD || n_iters < 0 || !(delta >= 0.0))
        return fail(nullptr, IMRT_STATUS_INVALID_ARG, "imrt_plan_run_ranks: bad argument");
    imrt_plan* p0 = host_plans[0];
    if (!p0) return fail(nullptr, IMRT_STATUS_INVALID_ARG, "imrt_plan_run_ranks: null plan");
    std::vector<DevPlan> plans(n_ranks);
    int total = 0;
    size_t smem = 0;
    for (int q = 0; q < n_ranks; ++q) {
        imrt_plan* pl = host_plans[q];
        if (!pl) return fail(p0, IMRT_STATUS_INVALID_ARG, "imrt_plan_run_ranks: null plan");
        if (!pl->has_x) return fail(p0, IMRT_STATUS_NOT_READY, "rank %d: call imrt_plan_set_x first", q);
        if (pl->prm.driver != 2 || pl->stream != p0->stream || pl->grid_p != p0->grid_p || pl->P.world != n_ranks || pl->P.rank != q)
            return fail(p0, IMRT_STATUS_INVALID_ARG, "imrt_plan_run_ranks: plan %d must be rank %d of %d (imrt_plan_set_shard), use the persistent "
                        "driver, the stream and the number of CTAs (imrt_options.n_ctas) of plan 0", q, q, n_ranks);
        // ranks that disagree on the batch size or on the trace capacity would count their exchanges differently
        if (pl->P.R != p0->P.R || pl->prm.max_iters != p0->prm.max_iters || pl->P.n_b != p0->P.n_b)
            return fail(p0, IMRT_STATUS_INVALID_ARG, "imrt_plan_run_ranks: plan %d differs from plan 0 in ls_batch (%d / %d), max_iters (%d / %d) or "
                        "n_b (%d / %d)", q, pl->P.R, p0->P.R, pl->prm.max_iters, p0->prm.max_iters, pl->P.n_b, p0->P.n_b);
        plans[q] = pl->P;
        total += pl->grid_p;
        smem = std::max(smem, pl->smem_bytes);
    }
    if (total > p0->n_sm_device)
        return fail(p0, IMRT_STATUS_UNSUPPORTED, "%d ranks of %d CTAs do not fit the device's %d SMs at one CTA per SM (imrt_options.n_ctas)", n_ranks, p0->grid_p, p0->n_sm_device);
    cudaStream_t st = p0->stream;
    for (int q = 0; q < n_ranks; ++q) k_set_target<<<1, 1, 0, st>>>(host_plans[q]->P.st, n_iters, delta);
    CUDA_TRY(p0, cudaMemcpyAsync(p0->rank_plans_w, plans.data(), sizeof(DevPlan) * n_ranks, cudaMemcpyHostToDevice, st));
    CUDA_TRY(p0, cudaStreamSynchronize(st));       // `plans` is a host vector
    CUDA_TRY(p0, cudaFuncSetAttribute(k_persistent_ranks, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof cfg);
    cfg.gridDim = dim3(total);
    cfg.blockDim = dim3(NTHREADS);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeCooperative;
    at[0].val.cooperative = 1;      // the ranks wait on one another: all their CTAs must be co-resident
    cfg.attrs = at;
    cfg.numAttrs = 1;
    const DevPlan* dp = p0->rank_plans_w;
    CUDA_TRY(p0, cudaLaunchKernelEx(&cfg, k_persistent_ranks, dp, p0->grid_p));
    return IMRT_STATUS_OK;
}

imrt_status imrt_plan_run_to_tol(imrt_plan* pl, double delta, int32_t max_iters) {
    if (pl && !(delta > 0.0)) return fail(pl, IMRT_STATUS_INVALID_ARG, "imrt_plan_run_to_tol: delta must be > 0");
    return run_common(pl, max_iters, delta);
}

imrt_status imrt_plan_eval(imrt_plan* pl, const float* x, float* d, float* r, float* g, double* host_obj) {
    if (!pl || !x) return fail(pl, IMRT_STATUS_INVALID_ARG, "imrt_plan_eval: null argument");
    cudaStream_t st = pl->stream;
    float* r_used = r ? r : pl->r_scratch;
    const int n_v = pl->P.n_v;
    RPtrs rp1;
    memset(&rp1, 0, sizeof rp1);
    rp1.p[0] = r_used;
    k_fill_zero_dose_rows<<<(n_v + 255) / 256, 256, 0, st>>>(pl->sid, pl->P.table, pl->P.st, n_v, rp1, d);
    PassArgs A;
    memset(&A, 0, sizeof A);
    A.mode = MODE_EVAL;
    A.x_in = x;
    A.r_out = r_used;
    A.d_out = d;
    CUDA_TRY(pl, launch_dose(pl, A));
    if (g) {
        PassArgs T;
        memset(&T, 0, sizeof T);
        T.mode = MODE_EVAL;
        T.r_in = r_used;
        T.g_out = g;
        CUDA_TRY(pl, launch_transpose(pl, T));
    }
    double obj = 0.0;
    CUDA_TRY(pl, cudaMemcpyAsync(&obj, &pl->P.st->eval_obj, sizeof(double), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(pl, cudaStreamSynchronize(st));
    if (host_obj) *host_obj = obj;
    return IMRT_STATUS_OK;
}

imrt_status imrt_plan_eval_batch(imrt_plan* pl, int32_t n_points, const float* x, float* r, double* host_obj) {
    if (!pl || !x || !host_obj) return fail(pl, IMRT_STATUS_INVALID_ARG, "imrt_plan_eval_batch: null argument");
    if (n_points != 1 && n_points != 2 && n_points != 4) return fail(pl, IMRT_STATUS_INVALID_ARG, "imrt_plan_eval_batch: n_points must be 1, 2 or 4");
    if (n_points > pl->P.R)
        return fail(pl, IMRT_STATUS_UNSUPPORTED, "imrt_plan_eval_batch: this plan evaluates %d trial point(s) per pass (imrt_plan_get_info [10])", pl->P.R);
    cudaStream_t st = pl->stream;
    const int n_v = pl->P.n_v;
    if (r) {      // constant residual of the rows no record covers
        RPtrs rp;
        memset(&rp, 0, sizeof rp);
        for (int j = 0; j < n_points; ++j) rp.p[j] = r + (size_t)j * n_v;
        k_fill_zero_dose_rows<<<(n_v + 255) / 256, 256, 0, st>>>(pl->sid, pl->P.table, pl->P.st, n_v, rp, nullptr);
    }
    PassArgs A;
    memset(&A, 0, sizeof A);
    A.mode = MODE_BATCH;
    A.n_points = n_points;
    A.x_in = x;
    A.r_out = r;
    CUDA_TRY(pl, launch_dose(pl, A));
    double objs[4];
    CUDA_TRY(pl, cudaMemcpyAsync(objs, pl->P.st->eval_objs, sizeof objs, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(pl, cudaStreamSynchronize(st));
    for (int j = 0; j < n_points; ++j) host_obj[j] = objs[j];
    return IMRT_STATUS_OK;
}

imrt_status imrt_plan_gradient(imrt_plan* pl, const float* r, float* g) {
    if (!pl || !r || !g) return fail(pl, IMRT_STATUS_INVALID_ARG, "imrt_plan_gradient: null argument");
    PassArgs T;
    memset(&T, 0, sizeof T);
    T.mode = MODE_EVAL;
    T.r_in = r;
    T.g_out = g;
    CUDA_TRY(pl, launch_transpose(pl, T));
    return IMRT_STATUS_OK;
}

// x+ = max(0, x - lambda g), Delta = ||x+ - x||^2 by ONE block, fixed summation order (Eq. (5)).
__global__ void k_trial_point(const float* __restrict__ x, const float* __restrict__ g, double lambda, int n_b, float* x_out, double* step_sq) {
    __shared__ double red[32];
    const float lam = (float)lambda;
    double acc = 0.0;
    for (int i = threadIdx.x; i < n_b; i += blockDim.x) {
        const float xi = x[i];
        const float xn = fmaxf(0.0f, fmaf(-lam, g[i], xi));
        const float dx = xn - xi;
        acc = __fma_rn((double)dx, (double)dx, acc);
        x_out[i] = xn;
    }
    acc = warp_sum(acc);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int w = 0; w < (int)(blockDim.x >> 5); ++w) s += red[w];
        *step_sq = s;
    }
}

imrt_status imrt_trial_point(const float* x, const float* g, double lambda, int64_t n_b, float* x_out, double* step_sq, void* stream) {
    if (!x || !g || !x_out || !step_sq || n_b < 1 || n_b >= (1LL << 31) || !(lambda > 0.0))
        return fail(nullptr, IMRT_STATUS_INVALID_ARG, "imrt_trial_point: bad argument");
    k_trial_point<<<1, 1024, 0, (cudaStream_t)stream>>>(x, g, lambda, (int)n_b, x_out, step_sq);
    CUDA_TRY(nullptr, cudaGetLastError());
    return IMRT_STATUS_OK;
}

int32_t imrt_armijo_accepts(double G_k, double G_new, double step_sq, double eps, double lambda) {
    return G_new < G_k - (eps / lambda) * step_sq ? 1 : 0;        // step 3 with Eq. (5), strict as printed
}

int32_t imrt_stop_test(double G_old, double G_new, double delta) {
    return (delta > 0.0 && (G_new == 0.0 || fabs(G_new - G_old) / G_new < delta)) ? 1 : 0;     // step 5, reading R5
}

imrt_status imrt_plan_get_x(imrt_plan* pl, float* x) {
    if (!pl || !x) return fail(pl, IMRT_STATUS_INVALID_ARG, "imrt_plan_get_x: null argument");
    if (!pl->has_x) return fail(pl, IMRT_STATUS_NOT_READY, "call imrt_plan_set_x first");
    k_copy_current_x<<<grid_for(pl->P.n_b, 256), 256, 0, pl->stream>>>(pl->P, x);
    CUDA_TRY(pl, cudaGetLastError());
    return IMRT_STATUS_OK;
}

static imrt_status dose_of_current_x(imrt_plan* pl, float* d) {
    const int n_v = pl->P.n_v;
    RPtrs rp0;
    memset(&rp0, 0, sizeof rp0);
    k_fill_zero_dose_rows<<<(n_v + 255) / 256, 256, 0, pl->stream>>>(pl->sid, pl->P.table, pl->P.st, n_v, rp0, d);
    PassArgs A;
    memset(&A, 0, sizeof A);
    A.mode = MODE_EVAL;   // x_in NULL: the current iterate
    A.r_out = pl->r_scratch;
    A.d_out = d;
    CUDA_TRY(pl, launch_dose(pl, A));
    return IMRT_STATUS_OK;
}

imrt_status imrt_plan_get_dose(imrt_plan* pl, float* d) {
    if (!pl || !d) return fail(pl, IMRT_STATUS_INVALID_ARG, "imrt_plan_get_dose: null argument");
    if (!pl->has_x) return fail(pl, IMRT_STATUS_NOT_READY, "call imrt_plan_set_x first");
    return dose_of_current_x(pl, d);
}

imrt_status imrt_plan_dvh(imrt_plan* pl, const double* host_pcts, int32_t n_pcts, double* host_dp, double* host_mean) {
    if (!pl || !host_pcts || !host_dp || !host_mean || n_pcts < 1 || n_pcts > DVH_MAX_PCTS)
        return fail(pl, IMRT_STATUS_INVALID_ARG, "imrt_plan_dvh: bad argument (1 <= n_pcts <= %d)", DVH_MAX_PCTS);
    if (!pl->has_x) return fail(pl, IMRT_STATUS_NOT_READY, "call imrt_plan_set_x first");
    imrt_status s = dose_of_current_x(pl, pl->d_scratch);
    if (s != IMRT_STATUS_OK) return s;
    const char* msg = nullptr;
    cudaError_t e = dvh_points(pl->dvh, pl->d_scratch, pl->sid, pl->P.n_v, pl->P.n_structures, host_pcts, n_pcts, host_dp, host_mean,
                               pl->stream, &msg);
    if (e != cudaSuccess) return fail(pl, IMRT_STATUS_CUDA_ERROR, "dvh: %s (%s)", cudaGetErrorString(e), msg ? msg : "");
    return IMRT_STATUS_OK;
}

imrt_status imrt_plan_get_trace(imrt_plan* pl, int32_t* host_n_iters_done, int32_t* host_stop_reason, double* host_obj,
                                double* host_lambda, int32_t* host_n_trials, double* host_step_sq, int32_t capacity) {
    if (!pl || capacity < 0) return fail(pl, IMRT_STATUS_INVALID_ARG, "imrt_plan_get_trace: bad argument");
    if (!pl->has_x) return fail(pl, IMRT_STATUS_NOT_READY, "call imrt_plan_set_x first");
    cudaStream_t st = pl->stream;
    State s;
    CUDA_TRY(pl, cudaMemcpyAsync(&s, pl->P.st, sizeof s, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(pl, cudaStreamSynchronize(st));
    const int n = std::min(s.iter, capacity);
    if (host_n_iters_done) *host_n_iters_done = s.iter;
    if (host_stop_reason)      // the trace filled up before the requested number of iterations was done
        *host_stop_reason = (s.stop_reason == STOP_MAX_ITERS && s.clamped && s.iter >= s.trace_cap) ? STOP_TRACE_FULL : s.stop_reason;
    if (host_obj) CUDA_TRY(pl, cudaMemcpyAsync(host_obj, pl->P.tr_obj, sizeof(double) * (n + 1), cudaMemcpyDeviceToHost, st));
    if (host_lambda && n) CUDA_TRY(pl, cudaMemcpyAsync(host_lambda, pl->P.tr_lambda, sizeof(double) * n, cudaMemcpyDeviceToHost, st));
    if (host_n_trials && n) CUDA_TRY(pl, cudaMemcpyAsync(host_n_trials, pl->P.tr_trials, sizeof(int) * n, cudaMemcpyDeviceToHost, st));
    if (host_step_sq && n) CUDA_TRY(pl, cudaMemcpyAsync(host_step_sq, pl->P.tr_step_sq, sizeof(double) * n, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(pl, cudaStreamSynchronize(st));
    return IMRT_STATUS_OK;
}

imrt_status imrt_plan_get_counters(imrt_plan* pl, int64_t* host_fwd_passes, int64_t* host_tr_passes) {
    if (!pl) return IMRT_STATUS_INVALID_ARG;
    State s;
    CUDA_TRY(pl, cudaMemcpyAsync(&s, pl->P.st, sizeof s, cudaMemcpyDeviceToHost, pl->stream));
    CUDA_TRY(pl, cudaStreamSynchronize(pl->stream));
    if (host_fwd_passes) *host_fwd_passes = s.fwd_passes;
    if (host_tr_passes) *host_tr_passes = s.tr_passes;
    return IMRT_STATUS_OK;
}

imrt_status imrt_plan_get_info(imrt_plan* pl, int64_t* host_info, int32_t n_info, int32_t* d_rowT_ptr, int32_t* d_colT, float* d_valT) {
    if (!pl) return IMRT_STATUS_INVALID_ARG;
    const int64_t info[16] = {(int64_t)pl->P.nnz, pl->n_blk, pl->P.grid_f, pl->P.grid_t, (int64_t)pl->smem_bytes, pl->pack_bytes,
                              pl->P.n_slots, pl->n_nonempty, pl->n_sm, pl->P.col16, pl->P.R, pl->P.ring_f_bytes, pl->P.n_stages_t, pl->n_quad_rows, pl->P.id16, pl->tr_stream_bytes};
    for (int i = 0; i < n_info && i < 16 && host_info; ++i) host_info[i] = info[i];
    cudaStream_t st = pl->stream;
    if (d_rowT_ptr) CUDA_TRY(pl, cudaMemcpyAsync(d_rowT_ptr, pl->rowT_ptr_w, sizeof(int) * (pl->P.n_b + 1), cudaMemcpyDeviceToDevice, st));
    if (d_colT && pl->P.nnz) CUDA_TRY(pl, cudaMemcpyAsync(d_colT, pl->colT_w, sizeof(int) * pl->P.nnz, cudaMemcpyDeviceToDevice, st));
    if (d_valT && pl->P.nnz) CUDA_TRY(pl, cudaMemcpyAsync(d_valT, pl->valT_w, sizeof(float) * pl->P.nnz, cudaMemcpyDeviceToDevice, st));
    CUDA_TRY(pl, cudaStreamSynchronize(st));
    return IMRT_STATUS_OK;
}

// ---------------------------------------------------------------------------------------------- mixed resolution
namespace {
struct MergeLayout {
    unsigned int *keysA, *keysB, *rowsA, *rowsB, *rows;
    int *group_ptr, *cnt, *flags;
    void* temp;
    size_t temp_bytes, total;
};
MergeLayout merge_layout(void* base, int64_t n_v, int64_t n_groups) {
    Bump w{static_cast<unsigned char*>(base), 0};
    MergeLayout M;
    M.keysA = w.take<unsigned int>(n_v + 4);
    M.keysB = w.take<unsigned int>(n_v + 4);
    M.rowsA = w.take<unsigned int>(n_v + 4);
    M.rowsB = w.take<unsigned int>(n_v + 4);
    M.rows = w.take<unsigned int>(n_v + 4);
    M.group_ptr = w.take<int>(n_groups + 2);
    M.cnt = w.take<int>(n_groups + 2);
    M.flags = w.take<int>(16);
    M.temp_bytes = (size_t)(16 << 20) + (size_t)(n_v + n_groups);
    M.temp = w.take<unsigned char>(M.temp_bytes);
    M.total = (w.off + 255) & ~(size_t)255;
    return M;
}
// bitmap words per warp and warps per block that fit the default 48 KB of shared memory (copies: 1 count, 2 fill)
bool merge_shape(int64_t n_b, int copies, int& words, int& warps) {
    words = (int)((n_b + 31) / 32);
    warps = MERGE_WARPS;
    while (warps > 1 && (size_t)warps * copies * words * 4 > 48 * 1024) warps /= 2;
    return (size_t)warps * copies * words * 4 <= 48 * 1024;
}
}  // namespace

imrt_status imrt_merge_rows_workspace_bytes(int64_t n_v, int64_t n_groups, size_t* host_bytes) {
    if (!host_bytes || n_v < 1 || n_groups < 1 || n_v >= (1LL << 31) - 16 || n_groups >= (1LL << 31) - 16)
        return fail(nullptr, IMRT_STATUS_INVALID_ARG, "imrt_merge_rows_workspace_bytes: bad argument");
    *host_bytes = merge_layout(nullptr, n_v, n_groups).total;
    return IMRT_STATUS_OK;
}

imrt_status imrt_merge_rows_count(int64_t n_v, int64_t n_b, const int32_t* row_ptr, const int32_t* col_idx, const int32_t* group_id,
                                  int64_t n_groups, int32_t* out_row_ptr, int64_t* host_nnz_out, void* workspace, size_t workspace_bytes,
                                  void* stream) {
    if (!row_ptr || !group_id || !out_row_ptr || !host_nnz_out || !workspace || n_v < 1 || n_b < 1 || n_groups < 1 ||
        n_v >= (1LL << 31) - 16 || n_groups >= (1LL << 31) - 16)
        return fail(nullptr, IMRT_STATUS_INVALID_ARG, "imrt_merge_rows_count: bad argument");
    const MergeLayout M = merge_layout(workspace, n_v, n_groups);
    if (workspace_bytes < M.total) return fail(nullptr, IMRT_STATUS_WORKSPACE_TOO_SMALL, "workspace has %zu bytes, %zu needed", workspace_bytes, M.total);
    int words, warps;
    if (!merge_shape(n_b, 2, words, warps)) return fail(nullptr, IMRT_STATUS_UNSUPPORTED, "imrt_merge_rows: n_b = %lld is too large for the column bitmap", (long long)n_b);
    cudaStream_t st = (cudaStream_t)stream;
    CUDA_TRY(nullptr, cudaMemsetAsync(M.flags, 0, 16 * sizeof(int), st));
    k_merge_keys<<<grid_for(n_v, 256), 256, 0, st>>>(group_id, (int)n_v, (int)n_groups, M.keysA, M.rowsA, M.flags);
    k_merge_check_row_ptr<<<grid_for(n_v, 256), 256, 0, st>>>(row_ptr, (int)n_v, M.flags);
    if (col_idx) k_merge_check_cols<<<grid_for(n_v * 32, 256), 256, 0, st>>>(row_ptr, col_idx, (int)n_v, (int)n_b, M.flags);
    cub::DoubleBuffer<unsigned int> dk(M.keysA, M.keysB), dv(M.rowsA, M.rowsB);
    int end_bit = 1;
    while ((1LL << end_bit) < n_groups) ++end_bit;
    size_t temp = 0;
    CUDA_TRY(nullptr, cub::DeviceRadixSort::SortPairs(nullptr, temp, dk, dv, (int)n_v, 0, end_bit, st));
    if (temp > M.temp_bytes) return fail(nullptr, IMRT_STATUS_WORKSPACE_TOO_SMALL, "internal: sort needs %zu temp bytes", temp);
    CUDA_TRY(nullptr, cub::DeviceRadixSort::SortPairs(M.temp, temp, dk, dv, (int)n_v, 0, end_bit, st));     // stable: rows stay ascending
    CUDA_TRY(nullptr, cudaMemcpyAsync(M.rows, dv.Current(), sizeof(unsigned int) * n_v, cudaMemcpyDeviceToDevice, st));
    k_merge_group_ptr<<<(int)((n_groups + 1 + 255) / 256), 256, 0, st>>>(dk.Current(), (int)n_v, (int)n_groups, M.group_ptr);
    merge_shape(n_b, 1, words, warps);
    CUDA_TRY(nullptr, cudaMemsetAsync(M.cnt, 0, sizeof(int) * (n_groups + 2), st));
    int flags_h[16];
    CUDA_TRY(nullptr, cudaMemcpyAsync(flags_h, M.flags, sizeof flags_h, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(nullptr, cudaStreamSynchronize(st));
    if (flags_h[0]) return fail(nullptr, IMRT_STATUS_INVALID_ARG, "imrt_merge_rows_count: a group id is outside [0, n_groups)");
    if (flags_h[1]) return fail(nullptr, IMRT_STATUS_BAD_CSR, "imrt_merge_rows_count: row_ptr[0] != 0 or row_ptr decreases");
    if (flags_h[2]) return fail(nullptr, IMRT_STATUS_BAD_CSR, "imrt_merge_rows_count: a column index is outside [0, n_b)");
    k_merge_count<<<(int)std::min<int64_t>((n_groups + warps - 1) / warps, 148 * 8), MERGE_WARPS * 32, (size_t)warps * words * 4, st>>>(
        row_ptr, col_idx, M.rows, M.group_ptr, (int)n_groups, words, warps, M.cnt);
    temp = 0;
    CUDA_TRY(nullptr, cub::DeviceScan::ExclusiveSum(nullptr, temp, M.cnt, out_row_ptr, (int)(n_groups + 1), st));
    if (temp > M.temp_bytes) return fail(nullptr, IMRT_STATUS_WORKSPACE_TOO_SMALL, "internal: scan needs %zu temp bytes", temp);
    CUDA_TRY(nullptr, cub::DeviceScan::ExclusiveSum(M.temp, temp, M.cnt, out_row_ptr, (int)(n_groups + 1), st));
    int32_t total = 0;
    CUDA_TRY(nullptr, cudaMemcpyAsync(&total, out_row_ptr + n_groups, sizeof total, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(nullptr, cudaStreamSynchronize(st));
    *host_nnz_out = total;
    return IMRT_STATUS_OK;
}

imrt_status imrt_merge_rows_fill(int64_t n_v, int64_t n_b, const int32_t* row_ptr, const int32_t* col_idx, const float* val,
                                 int64_t n_groups, const int32_t* out_row_ptr, int32_t* out_col, float* out_val, void* workspace,
                                 size_t workspace_bytes, void* stream) {
    if (!row_ptr || !out_row_ptr || !workspace || n_v < 1 || n_b < 1 || n_groups < 1)
        return fail(nullptr, IMRT_STATUS_INVALID_ARG, "imrt_merge_rows_fill: bad argument");
    const MergeLayout M = merge_layout(workspace, n_v, n_groups);
    if (workspace_bytes < M.total) return fail(nullptr, IMRT_STATUS_WORKSPACE_TOO_SMALL, "workspace has %zu bytes, %zu needed", workspace_bytes, M.total);
    int words, warps;
    if (!merge_shape(n_b, 2, words, warps)) return fail(nullptr, IMRT_STATUS_UNSUPPORTED, "imrt_merge_rows: n_b = %lld is too large for the column bitmap", (long long)n_b);
    if (!out_col || !out_val || !col_idx || !val) return IMRT_STATUS_OK;      // an empty merged matrix
    k_merge_fill<<<(int)std::min<int64_t>((n_groups + warps - 1) / warps, 148 * 8), MERGE_WARPS * 32, (size_t)warps * 2 * words * 4, (cudaStream_t)stream>>>(
        row_ptr, col_idx, val, M.rows, M.group_ptr, (int)n_groups, words, warps, out_row_ptr, out_col, out_val);
    CUDA_TRY(nullptr, cudaGetLastError());
    return IMRT_STATUS_OK;
}

imrt_status imrt_plan_get_tuning(imrt_plan* pl, void* host_buf, size_t capacity, size_t* host_bytes) {
    if (!pl || !host_bytes) return fail(pl, IMRT_STATUS_INVALID_ARG, "imrt_plan_get_tuning: null argument");
    const int gf = pl->P.grid_f, gt = pl->P.grid_t;
    const size_t need = sizeof(TuningBlob) + sizeof(int) * (gf + 1) + sizeof(double) * gt;
    *host_bytes = need;
    if (!host_buf) return IMRT_STATUS_OK;
    if (capacity < need || (int)pl->cta_blk_h.size() != gf + 1 || (int)pl->tr_share.size() != gt)
        return fail(pl, IMRT_STATUS_INVALID_ARG, "imrt_plan_get_tuning: buffer too small (%zu needed)", need);
    TuningBlob tb = {TUNING_MAGIC, gf, gt, 0, pl->n_blk, (int64_t)pl->rp_tr[pl->n_rows_tr]};
    char* o = static_cast<char*>(host_buf);
    memcpy(o, &tb, sizeof tb);
    memcpy(o + sizeof tb, pl->cta_blk_h.data(), sizeof(int) * (gf + 1));
    memcpy(o + sizeof tb + sizeof(int) * (gf + 1), pl->tr_share.data(), sizeof(double) * gt);
    return IMRT_STATUS_OK;
}

imrt_status imrt_plan_get_create_times(imrt_plan* pl, double* host_ms, int32_t capacity, int32_t* host_n) {
    if (!pl || !host_n || capacity < 0) return fail(pl, IMRT_STATUS_INVALID_ARG, "imrt_plan_get_create_times: bad argument");
    const int n = std::min<int>((int)pl->create_ms.size(), capacity);
    for (int i = 0; i < n && host_ms; ++i) host_ms[i] = pl->create_ms[i];
    *host_n = n;
    return IMRT_STATUS_OK;
}

imrt_status imrt_plan_get_pass_timing(imrt_plan* pl, int32_t kind, int64_t* host_start_ns, int64_t* host_end_ns, int32_t capacity,
                                      int32_t* host_n_ctas) {
    if (!pl || kind < 0 || kind > 1 || capacity < 0) return fail(pl, IMRT_STATUS_INVALID_ARG, "imrt_plan_get_pass_timing: bad argument");
    const int n = kind == 0 ? pl->P.grid_f : (pl->prm.driver == 2 ? pl->grid_p : pl->P.grid_t);
    std::vector<unsigned long long> t(2048);
    CUDA_TRY(pl, cudaMemcpyAsync(t.data(), pl->P.cta_ns + 2048 * kind, sizeof(unsigned long long) * 2048, cudaMemcpyDeviceToHost, pl->stream));
    CUDA_TRY(pl, cudaStreamSynchronize(pl->stream));
    if (host_n_ctas) *host_n_ctas = n;
    for (int c = 0; c < n && c < capacity; ++c) {
        if (host_start_ns) host_start_ns[c] = (int64_t)t[2 * c];
        if (host_end_ns) host_end_ns[c] = (int64_t)t[2 * c + 1];
    }
    return IMRT_STATUS_OK;
}

imrt_status imrt_plan_launch_pass(imrt_plan* pl, int32_t kind, int32_t n_repeat) {
    if (!pl || kind < 0 || kind > 3 || n_repeat < 0) return fail(pl, IMRT_STATUS_INVALID_ARG, "imrt_plan_launch_pass: bad argument");
    if (!pl->has_x) return fail(pl, IMRT_STATUS_NOT_READY, "call imrt_plan_set_x first");
    if (kind >= 2) {      // streaming ceilings: the pass's bytes through its ring / stages, no arithmetic
        if (kind == 3 && pl->P.id16 != 2) return fail(pl, IMRT_STATUS_UNSUPPORTED, "the stream-only transpose pass exists for the row-pair stream only");
        for (int i = 0; i < n_repeat; ++i) {
            k_stream<<<kind == 2 ? pl->P.grid_f : pl->P.grid_t, NTHREADS, pl->smem_bytes, pl->stream>>>(pl->P, kind - 2);
            CUDA_TRY(pl, cudaGetLastError());
        }
        return IMRT_STATUS_OK;
    }
    PassArgs A;
    memset(&A, 0, sizeof A);
    A.mode = kind == 0 ? MODE_TIMING : MODE_EVAL;   // dose pass: the line search's pass, residuals to the trial buffers
    A.g_out = pl->g_scratch;                        // transpose pass: on r(x_k), output to scratch
    for (int i = 0; i < n_repeat; ++i) CUDA_TRY(pl, kind == 0 ? launch_dose(pl, A) : launch_transpose(pl, A));
    return IMRT_STATUS_OK;
}

}  // extern "C"

// ------------------------------------------------------------------------------------------------ DVH without a workspace
// imrt_dvh_static (include/imrtgp.h): the dose-volume-histogram kernels of dvh.cuh run on scratch that lives inside the
// library image instead of in memory the caller hands over.  Meant for code that has a dose on the device but may not
// allocate: a planning service whose own pool already owns all of HBM (a raw cudaMalloc would simply fail), or a section
// that must not take the device-wide stall a cudaMalloc / cudaFree brings with it.
//
// g_dvh_static is ONE array per device for the life of the process (every device that loads the library keeps its
// IMRT_DVH_STATIC_BYTES until exit).  In host code the name g_dvh_static is only a handle for the runtime, never an address
// a kernel can use; the address on the current device comes from cudaGetSymbolAddress below, once per device.
#include <mutex>

namespace {

constexpr int DVH_STATIC_MAX_STRUCTURES = 16;                                // part[] and the documented limit
constexpr int DVH_STATIC_MAX_QUERIES = 128;                                  // n_structures * n_pcts: one 2,048-bin histogram each
constexpr size_t DVH_STATIC_HIST = sizeof(unsigned int) * DVH_STATIC_MAX_QUERIES * DVH_BINS;     // 1 MiB
constexpr size_t DVH_STATIC_CNT = sizeof(unsigned int) * 256;                // dvh_points clears 256 counters / sums
constexpr size_t DVH_STATIC_SUM = sizeof(double) * 256;
constexpr size_t DVH_STATIC_PART = sizeof(double) * DVH_SUM_BLOCKS * DVH_STATIC_MAX_STRUCTURES;
constexpr size_t DVH_STATIC_QUERY = sizeof(DvhQuery) * DVH_STATIC_MAX_QUERIES;
constexpr size_t DVH_STATIC_FLAG = 256;                                      // largest structure id seen (input check)
constexpr size_t DVH_STATIC_OFF_CNT = DVH_STATIC_HIST;
constexpr size_t DVH_STATIC_OFF_SUM = DVH_STATIC_OFF_CNT + DVH_STATIC_CNT;
constexpr size_t DVH_STATIC_OFF_PART = DVH_STATIC_OFF_SUM + DVH_STATIC_SUM;
constexpr size_t DVH_STATIC_OFF_QUERY = DVH_STATIC_OFF_PART + DVH_STATIC_PART;
constexpr size_t DVH_STATIC_OFF_FLAG = DVH_STATIC_OFF_QUERY + DVH_STATIC_QUERY;
constexpr size_t DVH_STATIC_BYTES = DVH_STATIC_OFF_FLAG + DVH_STATIC_FLAG;   // 1,128,704 bytes
static_assert(DVH_STATIC_OFF_CNT % 256 == 0 && DVH_STATIC_OFF_SUM % 256 == 0 && DVH_STATIC_OFF_PART % 256 == 0 &&
              DVH_STATIC_OFF_QUERY % 256 == 0 && DVH_STATIC_OFF_FLAG % 256 == 0, "pieces of the static scratch stay 256-byte aligned");

constexpr int DVH_STATIC_MAX_DEVICES = 64;
std::mutex g_dvh_static_lock;                                                // one call at a time: the array is shared
unsigned char* g_dvh_static_addr[DVH_STATIC_MAX_DEVICES] = {nullptr};       // device address of g_dvh_static, per device ordinal

}  // namespace

static __device__ __align__(256) unsigned char g_dvh_static[DVH_STATIC_BYTES];

// Largest structure id among the n_v voxels -> the flag word of the static scratch (device code may name the array).
__global__ void k_dvh_static_max_sid(const uint8_t* __restrict__ sid, int n_v) {
    unsigned int m = 0u;
    for (int j = blockIdx.x * blockDim.x + threadIdx.x; j < n_v; j += gridDim.x * blockDim.x) m = max(m, (unsigned int)sid[j]);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = max(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0 && m) atomicMax(reinterpret_cast<unsigned int*>(g_dvh_static + DVH_STATIC_OFF_FLAG), m);
}

extern "C" imrt_status imrt_dvh_static(const float* dose, const uint8_t* structure_id, int64_t n_v, int32_t n_structures,
                                       const double* host_pcts, int32_t n_pcts, double* host_dp, double* host_mean, void* stream) {
    if (!dose || !structure_id || !host_pcts || !host_dp || !host_mean || n_v < 1 || n_structures < 1 || n_pcts < 1)
        return fail(nullptr, IMRT_STATUS_INVALID_ARG, "imrt_dvh_static: null pointer or non-positive size");
    if (n_structures > DVH_STATIC_MAX_STRUCTURES || n_pcts > DVH_MAX_PCTS || n_structures * n_pcts > DVH_STATIC_MAX_QUERIES || n_v > (1LL << 30))
        return fail(nullptr, IMRT_STATUS_UNSUPPORTED,
                    "imrt_dvh_static: the built-in scratch (%zu bytes) holds at most %d structures, %d percentages per structure, %d "
                    "structure x percentage pairs and 2^30 voxels; got n_structures = %d, n_pcts = %d, n_v = %lld -- use imrt_plan_dvh "
                    "(caller-provided workspace) for more", DVH_STATIC_BYTES, DVH_STATIC_MAX_STRUCTURES, DVH_MAX_PCTS, DVH_STATIC_MAX_QUERIES,
                    (int)n_structures, (int)n_pcts, (long long)n_v);
    cudaStream_t st = (cudaStream_t)stream;
    std::lock_guard<std::mutex> hold(g_dvh_static_lock);      // held until the stream has drained: calls never overlap on the GPU

    // Set-up, once per device, with that device current: ask the runtime where this device keeps the array.
    int dev = -1;
    CUDA_TRY(nullptr, cudaGetDevice(&dev));
    if (dev < 0 || dev >= DVH_STATIC_MAX_DEVICES) return fail(nullptr, IMRT_STATUS_UNSUPPORTED, "imrt_dvh_static: device ordinal %d >= %d", dev, DVH_STATIC_MAX_DEVICES);
    if (!g_dvh_static_addr[dev]) {
        unsigned char* p = nullptr;
        CUDA_TRY(nullptr, cudaGetSymbolAddress((void**)&p, g_dvh_static));
        if (!p) return fail(nullptr, IMRT_STATUS_CUDA_ERROR, "imrt_dvh_static: cudaGetSymbolAddress returned a null address");
        g_dvh_static_addr[dev] = p;
    }
    unsigned char* base = g_dvh_static_addr[dev];

    // The array still holds the previous call's histograms, sums and flag.  dvh_points clears cnt, sum and (per round) hist
    // and overwrites every part / query entry it reads; the flag is cleared here.
    unsigned int* flag = reinterpret_cast<unsigned int*>(base + DVH_STATIC_OFF_FLAG);
    CUDA_TRY(nullptr, cudaMemsetAsync(flag, 0, sizeof(unsigned int), st));
    k_dvh_static_max_sid<<<std::max(1, (int)std::min<int64_t>((n_v + 255) / 256, 148 * 8)), 256, 0, st>>>(structure_id, (int)n_v);
    CUDA_TRY(nullptr, cudaGetLastError());
    unsigned int max_sid = 0u;
    CUDA_TRY(nullptr, cudaMemcpyAsync(&max_sid, flag, sizeof max_sid, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(nullptr, cudaStreamSynchronize(st));
    if (max_sid >= (unsigned int)n_structures)
        return fail(nullptr, IMRT_STATUS_BAD_STRUCTURE, "imrt_dvh_static: structure_id %u >= n_structures %d", max_sid, (int)n_structures);

    DvhWork W;
    W.hist = reinterpret_cast<unsigned int*>(base);
    W.cnt = reinterpret_cast<unsigned int*>(base + DVH_STATIC_OFF_CNT);
    W.sum = reinterpret_cast<double*>(base + DVH_STATIC_OFF_SUM);
    W.part = reinterpret_cast<double*>(base + DVH_STATIC_OFF_PART);
    W.query = reinterpret_cast<DvhQuery*>(base + DVH_STATIC_OFF_QUERY);
    const char* what = nullptr;
    cudaError_t e = dvh_points(W, dose, structure_id, (int)n_v, n_structures, host_pcts, n_pcts, host_dp, host_mean, st, &what);
    if (e != cudaSuccess) {
        cudaStreamSynchronize(st);                            // nothing of this call may still be using the array when the lock drops
        return fail(nullptr, IMRT_STATUS_CUDA_ERROR, "imrt_dvh_static: %s (%s)", cudaGetErrorString(e), what ? what : "");
    }
    return IMRT_STATUS_OK;
}
