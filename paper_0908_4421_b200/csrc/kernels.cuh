// kernels.cuh -- the device side of libimrtgp (sm_100a).
//
// Two streaming passes and the scalar logic between them (PAPER.md = /root/reference/PAPER.md):
//
//   dose pass       d = D x+, penalty, residual r, objective partials      PAPER.md:51-66 Eq. (1)-(2), :128 kernels 1-2
//   transpose pass  g = D^T r on an explicit D^T CSR                       PAPER.md:107 step 1, :128 kernel 3
//   trial point     x+ = max(0, x - lambda g), Delta = ||x+ - x||^2       PAPER.md:90, :109-111, :128 kernel 4
//   Armijo / stop   C = G_k - (eps/lambda) Delta, accept iff G+ < C        PAPER.md:92-95 Eq. (5), :110-114
//
// Both passes are persistent CTAs (one per SM): a producer warp streams the matrix with 1-D bulk async copies
// (cp.async.bulk, the TMA unit) into a ring of shared-memory stages guarded by mbarriers; 16 consumer warps
// gather the vector (x+ from shared memory, r through L1/L2 with an evict-last hint), multiply-add in fp32 and
// reduce with warp shuffles.  Objective and gradient partials are fp64 and are combined in a fixed order, so a run
// is bit-reproducible and no floating-point atomics are used anywhere.
//
// The same pass bodies are driven three ways (imrt_params.driver): by one cooperative persistent kernel that
// holds the whole loop (grid barrier between passes, replicated scalar state), by a CUDA graph with nested
// conditional WHILE nodes (the last CTA of each pass takes the decision and sets the loop conditions), or by
// the host (debugging).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "pipeline.cuh"

namespace imrt {

// ------------------------------------------------------------------------------------------------ constants
constexpr int W_CONS = 16;                    // consumer warps per CTA
constexpr int N_CONS = W_CONS * 32;           // consumer threads
constexpr int NTHREADS = N_CONS + 32;         // + one producer warp
// dose pass: D is re-packed once into self-contained block records (one bulk copy each, see DosePack below)
constexpr int META_HDR = 4;                   // header words {rows, first row, batches dealt before | flags, slots}
constexpr int MIN_CHUNK_SLOTS = 2048;           // smallest slot capacity of a dose-pass stage the host will choose
constexpr int MAXROWS_F = 507;                // rows per block: header + row table fit 2 KB
constexpr int META_F_BYTES = (META_HDR + MAXROWS_F + 1) * 4;
constexpr int CHUNK_T = 4096;                 // nnz per transpose-pass stage (pure streaming)
constexpr int SLICE_T = CHUNK_T / W_CONS;     // contiguous nnz per consumer warp per stage
constexpr int CHUNK_T_PAD = CHUNK_T + 4;            // + alignment shift of a range start (<= 3 entries)
constexpr int STAGE_T_BYTES = CHUNK_T_PAD * 8;
constexpr int RL_MAX = 32;                    // rows of D^T one transpose range may span
constexpr int MAX_STAGES = 12;
constexpr int MAX_STRUCTURES = 256;
constexpr int SMEM_HEADER = 1024;             // barriers, flags, reduction scratch
constexpr int SMEM_WPART = RL_MAX * W_CONS * 8;

enum { MODE_TRIAL = 0, MODE_INIT = 1, MODE_EVAL = 2 };
enum { STOP_MAX_ITERS = 0, STOP_TOLERANCE = 1, STOP_STATIONARY = 2, STOP_LS_STALLED = 3 };

// ------------------------------------------------------------------------------------------------ device data
struct State {                 // lives in the workspace; the single source of truth between launches
    double G_k;                // objective at the current iterate
    double lambda;             // step size of the pending trial
    double step_sq;            // Delta of the pending trial
    double eps, alpha, lambda0, delta_tol;
    double eval_obj;           // output of MODE_EVAL dose passes
    long long fwd_passes, tr_passes;
    int max_ls;
    int iter;                  // accepted iterations since set_x
    int iter_target;           // stop when iter reaches this
    int trace_cap;
    int m;                     // backtracking steps taken in the current line search
    int stop_reason;
    int xi;                    // xbuf[xi] is the current iterate, xbuf[xi^1] the trial point
    int ri;                    // rbuf[ri] is r(x_k), rbuf[ri^1] receives r(x+)
    int cont_outer, cont_inner;  // loop conditions (mirrors of the graph conditionals; read by the host driver)
    int bad_x;                 // set_x validation result
    unsigned int ticket_f, ticket_t;   // last-CTA tickets
    unsigned int gridbar;      // grid barrier counter of the persistent kernel
    int pad;
};

struct TrRange {               // a contiguous piece of the D^T nnz stream, 32 bytes
    int e_begin, e_end;        // element range [e_begin, e_end) of the D^T stream
    int first_row;             // row of D^T holding e_begin
    int n_rows;                // rows spanned (<= RL_MAX)
    int slot_base;             // first gradient partial slot
    int pad[3];
};

struct DevPlan {
    // D (borrowed): CSR, rows = voxels
    const int* col;
    const float* val;
    long long nnz;
    int n_v, n_b;
    // dose pass: D re-packed into block records (owned).  A record is 128-byte aligned and holds, in this order,
    //   header  uint32[4]  {rows, first row, warp batches dealt before this block (mod W_CONS), slots}
    //   rows    uint32[rows + 1]  slot offset of the row (low 16 bits, a multiple of 4) | structure id << 16;
    //                             padded to a multiple of 4 words
    //   val     fp32[slots]       every row padded with zeros to a multiple of 4 slots
    //   col     uint16[slots] (n_b <= 65536) or int32[slots]
    const unsigned char* pack;
    const int2* blk;           // {record offset / 128, record bytes}
    const int* cta_blk;        // [grid_f + 1] block range per CTA
    int grid_f, n_stages_f;
    int stage_f_bytes;         // bytes of one dose-pass stage (largest record, 128-byte multiple)
    int col16;                 // 1: 16-bit column indices in the records
    // D^T (owned): CSR, rows = beamlets, padded with zeros to a multiple of 4 entries
    const int* rowT_ptr;
    const int* colT;
    const float* valT;
    // transpose pass: equal-nnz ranges
    const TrRange* tr_range;
    const int* rowslot_ptr;    // [n_b + 1] slots of row i are [rowslot_ptr[i], rowslot_ptr[i+1])
    int n_ranges, grid_t, n_stages_t, n_slots;
    // penalty table and skipped (matrix-free) rows
    const float4* table;       // (t_under, t_over, w_under, w_over)
    int n_structures;
    int pad0;
    double G_skip;             // objective of the rows no block covers (d = 0 there, constant)
    // vectors
    float* xbuf[2];
    float* g;
    float* rbuf[2];
    double* Gpart[2];          // [grid_f] objective partials, double-buffered by pass parity
    double* gslot[2];          // [n_slots] gradient partials, double-buffered
    State* st;
    unsigned long long* cta_ns;  // [2][1024][2] per-CTA {start, end of streaming} of the last dose / transpose pass, ns
    double* tr_obj;            // trace: [cap + 1]
    double* tr_lambda;         // [cap]
    double* tr_step_sq;        // [cap]
    int* tr_trials;            // [cap]
    int wpart_off;             // byte offsets into dynamic shared memory: transpose per-(row, warp) partials,
    int x_off, g_off;          // the trial point x+ (gathered by the dose pass) and the gradient (persistent kernel)
    int stage_off;             // byte offset of the stage ring
};

struct PassArgs {
    const float* x_in;         // dose pass: where to evaluate (NULL = the trial point xbuf[xi^1]; MODE_EVAL: x_k)
    const float* r_in;         // transpose pass: residual (NULL = rbuf[ri])
    float* r_out;              // dose pass: residual out (NULL = rbuf[ri^1])
    float* d_out;              // dose pass: dose out or NULL
    float* g_out;              // transpose pass MODE_EVAL: gradient out
    int mode;
    int use_handles;           // 1 inside the conditional graph
    cudaGraphConditionalHandle h_outer, h_inner;
};

// ------------------------------------------------------------------------------------------------ shared memory
struct SmemHeader {
    uint64_t full_f[MAX_STAGES], empty_f[MAX_STAGES], full_t[MAX_STAGES], empty_t[MAX_STAGES];
    double red[32];            // block-reduction scratch
    double bcast[4];
    int flag;
};
static_assert(sizeof(SmemHeader) <= SMEM_HEADER, "header");

struct Pipe {                  // running stage counters; identical in producer and consumers
    unsigned int it_f, it_t;
};

__device__ __forceinline__ void cta_init(SmemHeader* h, const DevPlan& P, float4* table_s) {
    if (threadIdx.x == 0) {
        for (int s = 0; s < MAX_STAGES; ++s) {
            mbar_init(&h->full_f[s], 1);
            mbar_init(&h->empty_f[s], W_CONS);
            mbar_init(&h->full_t[s], 1);
            mbar_init(&h->empty_t[s], W_CONS);
        }
        mbar_fence_init();
    }
    for (int s = threadIdx.x; s < P.n_structures; s += NTHREADS) table_s[s] = P.table[s];
    __syncthreads();
}

__device__ __forceinline__ unsigned long long global_ns() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
    return t;
}

// ------------------------------------------------------------------------------------------------ block reduce
// Sum over all NTHREADS threads in a fixed order; result valid in every thread.
__device__ __forceinline__ double block_sum(double v, SmemHeader* h) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    v = warp_sum(v);
    __syncthreads();
    if (lane == 0) h->red[warp] = v;
    __syncthreads();
    double s = 0.0;
#pragma unroll
    for (int w = 0; w < NTHREADS / 32; ++w) s += h->red[w];
    return s;
}

// ------------------------------------------------------------------------------------------------ trial point
// x+ = max(0, x - lambda g), Delta = sum (x+ - x)^2      PAPER.md:90 (projection), :109/:111 (steps 2, 4), Eq. (5).
// fp32 elementwise, fp64 sum.  All NTHREADS threads call it; x is global (read through L2: another CTA may have
// written it), g and x_new may be shared or global memory.
__device__ __forceinline__ double compute_trial(const float* x, const float* g, double lambda, float* x_new, int n_b,
                                                SmemHeader* h) {
    const float lam = (float)lambda;
    double acc = 0.0;
    for (int i = threadIdx.x; i < n_b; i += NTHREADS) {
        const float xi = __ldcg(x + i);
        const float xn = fmaxf(0.0f, fmaf(-lam, g[i], xi));
        const float dx = xn - xi;
        acc += (double)dx * (double)dx;
        x_new[i] = xn;
    }
    return block_sum(acc, h);
}

// ------------------------------------------------------------------------------------------------ dose pass
// VW lanes per row, RB = 32 / VW rows per warp batch, 4 consecutive slots per lane and trip: rows start on 16-byte
// boundaries inside a record and are zero-padded to a multiple of 4 slots, so values and columns come in with one
// 128-bit (64-bit for 16-bit columns) shared-memory load each and nothing has to be masked inside a row.  The row
// groups of a warp run the trip count of their longest row (neighbouring voxels have rows of similar length),
// gather x+ from shared memory, multiply-add in fp32 and reduce with log2(VW) shuffles; lane 0 of each group then
// does its voxel's penalty and residual (Eq. (1) generalised: F = w- u^2 + w+ o^2, r = 2 (w+ o - w- u)).
// Batches are numbered across the CTA's blocks and dealt round-robin to the consumer warps, which never
// synchronise with each other: a warp with nothing to do in this stage moves on to the next one.
constexpr int VW = 8;
constexpr int RB = 32 / VW;

template <bool COL16>
__device__ __forceinline__ void dose_block(const unsigned char* __restrict__ rec, const float* __restrict__ x_s,
                                           const float4* __restrict__ table_s, float* __restrict__ r_out,
                                           float* __restrict__ d_out, int warp, int lane, double& Gacc) {
    const uint4 hdr = *reinterpret_cast<const uint4*>(rec);
    const int nrows = (int)hdr.x;
    const int nbatch = (nrows + RB - 1) / RB;
    const uint32_t* rows = reinterpret_cast<const uint32_t*>(rec) + META_HDR;
    const float* val_s = reinterpret_cast<const float*>(rows + ((nrows + 1 + 3) & ~3));
    const unsigned char* col_s = reinterpret_cast<const unsigned char*>(val_s + hdr.w);
    const int grp = lane / VW, sub = lane % VW;
    for (int q = (warp - (int)hdr.z) & (W_CONS - 1); q < nbatch; q += W_CONS) {
        const int row = q * RB + grp;
        const bool valid = row < nrows;
        uint32_t m0 = 0u, m1 = 0u;
        if (valid) { m0 = rows[row]; m1 = rows[row + 1]; }
        const int s = (int)(m0 & 0xFFFFu), e = (int)(m1 & 0xFFFFu);
        const int len_max = __reduce_max_sync(0xffffffffu, e - s);   // warp-uniform trip count
        float a0 = 0.0f, a1 = 0.0f, a2 = 0.0f, a3 = 0.0f;
        int k = s + 4 * sub;
        for (int kb = 0; kb < len_max; kb += 4 * VW, k += 4 * VW) {
            if (k < e) {
                const float4 v = *reinterpret_cast<const float4*>(val_s + k);
                int c0, c1, c2, c3;
                if (COL16) {
                    const uint2 c = *reinterpret_cast<const uint2*>(col_s + 2 * k);
                    c0 = (int)(c.x & 0xFFFFu); c1 = (int)(c.x >> 16); c2 = (int)(c.y & 0xFFFFu); c3 = (int)(c.y >> 16);
                } else {
                    const int4 c = *reinterpret_cast<const int4*>(col_s + 4 * k);
                    c0 = c.x; c1 = c.y; c2 = c.z; c3 = c.w;
                }
                a0 = fmaf(v.x, x_s[c0], a0);
                a1 = fmaf(v.y, x_s[c1], a1);
                a2 = fmaf(v.z, x_s[c2], a2);
                a3 = fmaf(v.w, x_s[c3], a3);
            }
        }
        const float d = vec_sum<VW>((a0 + a1) + (a2 + a3));
        if (valid && sub == 0) {
            const float4 t = table_s[(m0 >> 16) & 0xFFu];
            const float u = fmaxf(0.0f, t.x - d);
            const float o = fmaxf(0.0f, d - t.y);
            r_out[hdr.y + row] = 2.0f * (t.w * o - t.z * u);
            if (d_out) d_out[hdr.y + row] = d;
            Gacc += (double)t.z * ((double)u * (double)u) + (double)t.w * ((double)o * (double)o);
        }
    }
}

// All NTHREADS threads of the CTA call this.  x_s: the trial point in shared memory.  Writes the CTA's objective
// partial to Gpart[blockIdx.x] (thread 0).  Ends with a CTA-wide barrier.
template <bool COL16>
__device__ __forceinline__ void dose_pass_t(const DevPlan& P, SmemHeader* h, unsigned char* smem, const float4* table_s,
                                            const float* x_s, float* r_out, float* d_out, double* Gpart, Pipe& pipe) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int S = P.n_stages_f;
    const uint32_t SB = (uint32_t)P.stage_f_bytes;
    unsigned char* stages = smem + P.stage_off;
    const int b0 = (blockIdx.x < P.grid_f) ? P.cta_blk[blockIdx.x] : 0;
    const int b1 = (blockIdx.x < P.grid_f) ? P.cta_blk[blockIdx.x + 1] : 0;
    int s = (int)(pipe.it_f % (unsigned int)S);
    unsigned int ph = (pipe.it_f / (unsigned int)S) & 1u;
    double Gacc = 0.0;
    const unsigned long long t_start = global_ns();
    const uint32_t full_a = smem_u32(&h->full_f[0]), empty_a = smem_u32(&h->empty_f[0]), stages_a = smem_u32(stages);

    if (warp == W_CONS) {
        // ---------------- producer warp: lane 0 drives the TMA unit, one bulk copy per block record; the
        // descriptors of the next 32 blocks are requested before the current 32 are issued
        const uint64_t pol = policy_evict_first();   // streamed once per pass: keep it from pushing r / x out of L2
        int2 next = (b0 + lane < b1) ? __ldg(P.blk + b0 + lane) : make_int2(0, 0);
        for (int bb = b0; bb < b1; bb += 32) {
            const int2 mine = next;
            next = (bb + 32 + lane < b1) ? __ldg(P.blk + bb + 32 + lane) : make_int2(0, 0);
            const int nb_here = min(32, b1 - bb);
            for (int j = 0; j < nb_here; ++j) {
                const int off128 = __shfl_sync(0xffffffffu, mine.x, j);
                const int bytes = __shfl_sync(0xffffffffu, mine.y, j);
                if (lane == 0) {
                    mbar_wait_a(empty_a + 8u * s, ph ^ 1u);
                    const uint32_t bar = full_a + 8u * s;
                    mbar_expect_tx_a(bar, (uint32_t)bytes);
                    bulk_g2s_a(stages_a + (uint32_t)s * SB, P.pack + (size_t)(unsigned int)off128 * 128u, (uint32_t)bytes, bar, pol);
                }
                if (++s == S) { s = 0; ph ^= 1u; }
            }
        }
    } else {
        // ---------------- consumer warps
        const unsigned char* st_p = stages + (size_t)s * SB;
        const unsigned char* st_end = stages + (size_t)S * SB;
        uint32_t fb = full_a + 8u * s, eb = empty_a + 8u * s;
        for (int b = b0; b < b1; ++b) {
            mbar_wait_a(fb, ph);
#ifndef IMRT_EXP_SKIP_COMPUTE
            dose_block<COL16>(st_p, x_s, table_s, r_out, d_out, warp, lane, Gacc);
#endif
            __syncwarp();
            if (lane == 0) mbar_arrive_a(eb);
            st_p += SB; fb += 8u; eb += 8u;
            if (st_p == st_end) { st_p = stages; fb = full_a; eb = empty_a; ph ^= 1u; }
        }
    }
    pipe.it_f += (unsigned int)(b1 - b0);
    const double Gcta = block_sum(Gacc, h);   // producer lanes contribute 0
    if (threadIdx.x == 0 && blockIdx.x < P.grid_f) {
        Gpart[blockIdx.x] = Gcta;
        P.cta_ns[2 * blockIdx.x] = t_start;            // when this CTA's share of the pass began and ended: lets the
        P.cta_ns[2 * blockIdx.x + 1] = global_ns();    // host see (and rebalance) the static partition
    }
    __syncthreads();
}

__device__ __forceinline__ void dose_pass(const DevPlan& P, SmemHeader* h, unsigned char* smem, const float4* table_s,
                                          const float* x_s, float* r_out, float* d_out, double* Gpart, Pipe& pipe) {
    if (P.col16) dose_pass_t<true>(P, h, smem, table_s, x_s, r_out, d_out, Gpart, pipe);
    else dose_pass_t<false>(P, h, smem, table_s, x_s, r_out, d_out, Gpart, pipe);
}

// Objective of a finished dose pass: fixed-order sum of the CTA partials + the constant of the skipped rows.
// Every thread of the calling CTA gets the value.
__device__ __forceinline__ double reduce_objective(const DevPlan& P, const double* Gpart, SmemHeader* h) {
    double v = 0.0;
    for (int c = threadIdx.x; c < P.grid_f; c += NTHREADS) v += __ldcg(Gpart + c);
    return block_sum(v, h) + P.G_skip;
}

// ------------------------------------------------------------------------------------------------ transpose pass
// Streams equal-nnz ranges of D^T; every consumer warp owns a contiguous slice of each stage, gathers r, and keeps
// an fp64 running sum per row of D^T; per (warp,row) sums meet in shared memory and leave as one fp64 partial
// per (range,row) slot.  All NTHREADS threads call this.  Ends with a CTA-wide barrier.
__device__ __forceinline__ void transpose_pass(const DevPlan& P, SmemHeader* h, unsigned char* smem, double* wpart,
                                               const float* __restrict__ r_in, double* gslot, Pipe& pipe) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int S = P.n_stages_t;
    unsigned char* stages = smem + P.stage_off;
    unsigned int it = pipe.it_t;
    const unsigned long long t_start = global_ns();
    int s = (int)(it % (unsigned int)S);
    unsigned int ph = (it / (unsigned int)S) & 1u;

    if (warp == W_CONS) {
        const uint64_t pol = policy_evict_first();
        if (lane == 0) {
            for (int rg = blockIdx.x; rg < P.n_ranges; rg += gridDim.x) {
                const int e0 = P.tr_range[rg].e_begin, e1 = P.tr_range[rg].e_end;
                for (int cs = e0; cs < e1; cs += CHUNK_T, ++it) {
                    mbar_wait(&h->empty_t[s], ph ^ 1u);
                    int n = e1 - cs;
                    n = n > CHUNK_T ? CHUNK_T : n;
                    const int shift = e0 & 3;   // 16-byte source alignment: start the copy up to 3 entries early
                    const uint32_t bytes = (uint32_t)((n + shift + 3) & ~3) * 4u;   // D^T is padded: always in bounds
                    int* col_s = reinterpret_cast<int*>(stages + (size_t)s * STAGE_T_BYTES);
                    float* val_s = reinterpret_cast<float*>(col_s + CHUNK_T_PAD);
                    mbar_expect_tx(&h->full_t[s], 2u * bytes);
                    bulk_g2s(col_s, P.colT + (cs - shift), bytes, &h->full_t[s], pol);
                    bulk_g2s(val_s, P.valT + (cs - shift), bytes, &h->full_t[s], pol);
                    if (++s == S) { s = 0; ph ^= 1u; }
                }
            }
        } else {
            for (int rg = blockIdx.x; rg < P.n_ranges; rg += gridDim.x) {
                const int e0 = P.tr_range[rg].e_begin, e1 = P.tr_range[rg].e_end;
                it += (unsigned int)((e1 - e0 + CHUNK_T - 1) / CHUNK_T);
            }
        }
    } else {
        const uint64_t keep = policy_evict_last();
        for (int rg = blockIdx.x; rg < P.n_ranges; rg += gridDim.x) {
            const TrRange R = P.tr_range[rg];
            for (int i = threadIdx.x; i < RL_MAX * W_CONS; i += N_CONS) wpart[i] = 0.0;
            named_bar_sync(1, N_CONS);
            int cur_row = R.first_row;
            int cur_end = __ldg(P.rowT_ptr + cur_row + 1);
            double dacc = 0.0;
            bool touched = false;
            for (int cs = R.e_begin; cs < R.e_end; cs += CHUNK_T, ++it) {
                mbar_wait(&h->full_t[s], ph);
                const int* col_s = reinterpret_cast<const int*>(stages + (size_t)s * STAGE_T_BYTES) + (R.e_begin & 3);
                const float* val_s = reinterpret_cast<const float*>(stages + (size_t)s * STAGE_T_BYTES) + CHUNK_T_PAD + (R.e_begin & 3);
                const int ce = min(cs + CHUNK_T, R.e_end);
                int pos = cs + warp * SLICE_T;
                const int b = min(pos + SLICE_T, ce);
                while (pos < b) {
                    while (cur_end <= pos) {   // the slice moved past the end of the current row (warp-uniform)
                        if (touched) {
                            const double sum = warp_sum(dacc);
                            if (lane == 0) wpart[(cur_row - R.first_row) * W_CONS + warp] = sum;
                            dacc = 0.0;
                            touched = false;
                        }
                        ++cur_row;
                        cur_end = __ldg(P.rowT_ptr + cur_row + 1);
                    }
                    const int seg_end = min(b, cur_end);
                    const int* cp = col_s + (pos - cs);
                    const float* vp = val_s + (pos - cs);
                    float acc = 0.0f;
                    if (seg_end - pos == SLICE_T) {
                        int c[SLICE_T / 32];
                        float rr[SLICE_T / 32];
#pragma unroll
                        for (int u = 0; u < SLICE_T / 32; ++u) c[u] = cp[lane + 32 * u];
#pragma unroll
                        for (int u = 0; u < SLICE_T / 32; ++u) rr[u] = ld_keep(r_in + c[u], keep);
#pragma unroll
                        for (int u = 0; u < SLICE_T / 32; ++u) acc = fmaf(vp[lane + 32 * u], rr[u], acc);
                    } else {
                        for (int k = lane; k < seg_end - pos; k += 32) acc = fmaf(vp[k], ld_keep(r_in + cp[k], keep), acc);
                    }
                    dacc += (double)acc;
                    touched = true;
                    pos = seg_end;
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(&h->empty_t[s]);
                if (++s == S) { s = 0; ph ^= 1u; }
            }
            if (touched) {
                const double sum = warp_sum(dacc);
                if (lane == 0) wpart[(cur_row - R.first_row) * W_CONS + warp] = sum;
            }
            named_bar_sync(1, N_CONS);
            for (int t = threadIdx.x; t < R.n_rows; t += N_CONS) {
                double sum = 0.0;
#pragma unroll
                for (int w = 0; w < W_CONS; ++w) sum += wpart[t * W_CONS + w];
                gslot[R.slot_base + t] = sum;
            }
            named_bar_sync(1, N_CONS);
        }
    }
    pipe.it_t = it;
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) {
        P.cta_ns[2048 + 2 * blockIdx.x] = t_start;
        P.cta_ns[2048 + 2 * blockIdx.x + 1] = global_ns();
    }
}

// g_i = sum of the slots of row i, in slot order (fixed).  All NTHREADS threads; g_out shared or global.
__device__ __forceinline__ void reduce_gradient(const DevPlan& P, const double* gslot, float* g_out) {
    for (int i = threadIdx.x; i < P.n_b; i += NTHREADS) {
        const int s0 = __ldg(P.rowslot_ptr + i), s1 = __ldg(P.rowslot_ptr + i + 1);
        double sum = 0.0;
        for (int s = s0; s < s1; ++s) sum += __ldcg(gslot + s);
        g_out[i] = (float)sum;
    }
}

// ------------------------------------------------------------------------------------------------ scalar logic
struct Loop {                  // the loop's scalar state, replicated in registers by the persistent kernel
    double G_k, lambda, step_sq;
    int iter, m, stop_reason, xi, ri;
    long long fwd, tr;
};

// After a transpose pass of the loop: start the line search (PAPER.md:109 step 2).  Returns true if a trial is pending.
// Called by all threads with identical arguments; x, g, x_trial may be shared or global.
__device__ __forceinline__ bool begin_line_search(const State* st, Loop& L, const float* x, const float* g, float* x_trial,
                                                  int n_b, SmemHeader* h) {
    L.tr += 1;
    if (L.G_k == 0.0) { L.stop_reason = STOP_STATIONARY; return false; }   // reading R4
    L.lambda = st->lambda0;
    L.m = 0;
    L.step_sq = compute_trial(x, g, L.lambda, x_trial, n_b, h);
    if (L.step_sq == 0.0) { L.stop_reason = STOP_STATIONARY; return false; }   // reading R4
    return true;
}

enum { DEC_ACCEPT_CONTINUE = 0, DEC_ACCEPT_STOP = 1, DEC_REJECT_RETRY = 2, DEC_REJECT_STOP = 3 };

// After a dose pass of the loop: Armijo test (PAPER.md:110 step 3, Eq. (5)), step 4 or step 5.  Scalar work only; the
// caller recomputes the trial point on DEC_REJECT_RETRY.  write_trace: only one CTA records.
__device__ __forceinline__ int armijo_decide(const DevPlan& P, const State* st, Loop& L, double G_new, bool write_trace) {
    L.fwd += 1;
    const double C = L.G_k - (st->eps / L.lambda) * L.step_sq;   // Eq. (5)
    if (G_new < C) {                                              // step 3, strict as printed
        const int k = L.iter;
        if (write_trace) {
            P.tr_obj[k + 1] = G_new;
            P.tr_lambda[k] = L.lambda;
            P.tr_step_sq[k] = L.step_sq;
            P.tr_trials[k] = L.m + 1;
        }
        const double G_old = L.G_k;
        L.G_k = G_new;
        L.iter = k + 1;
        L.xi ^= 1;
        L.ri ^= 1;
        if (st->delta_tol > 0.0 && (G_new == 0.0 || fabs(G_new - G_old) / G_new < st->delta_tol)) {   // step 5
            L.stop_reason = STOP_TOLERANCE;
            return DEC_ACCEPT_STOP;
        }
        if (L.iter >= st->iter_target) { L.stop_reason = STOP_MAX_ITERS; return DEC_ACCEPT_STOP; }
        return DEC_ACCEPT_CONTINUE;
    }
    L.m += 1;                                                     // step 4
    if (L.m > st->max_ls) { L.stop_reason = STOP_LS_STALLED; return DEC_REJECT_STOP; }
    L.lambda = L.lambda / st->alpha;
    return DEC_REJECT_RETRY;
}

__device__ __forceinline__ void loop_load(const State* st, Loop& L) {
    L.G_k = st->G_k; L.lambda = st->lambda; L.step_sq = st->step_sq;
    L.iter = st->iter; L.m = st->m; L.stop_reason = st->stop_reason; L.xi = st->xi; L.ri = st->ri;
    L.fwd = st->fwd_passes; L.tr = st->tr_passes;
}
__device__ __forceinline__ void loop_store(State* st, const Loop& L) {
    st->G_k = L.G_k; st->lambda = L.lambda; st->step_sq = L.step_sq;
    st->iter = L.iter; st->m = L.m; st->stop_reason = L.stop_reason; st->xi = L.xi; st->ri = L.ri;
    st->fwd_passes = L.fwd; st->tr_passes = L.tr;
}

// Last-CTA election (threadfence reduction pattern).  Every thread has fenced its global writes before the call.
__device__ __forceinline__ bool cta_is_last(unsigned int* ticket, SmemHeader* h) {
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        const unsigned int t = atomicAdd(ticket, 1u);
        const int last = (t == gridDim.x - 1);
        if (last) { *ticket = 0u; __threadfence(); }
        h->flag = last;
    }
    __syncthreads();
    return h->flag != 0;
}

// ------------------------------------------------------------------------------------------------ kernels
extern __shared__ __align__(128) unsigned char imrt_smem[];

// Dose pass as a kernel of its own (graph / host drivers, set_x, eval, get_dose).
__global__ void __launch_bounds__(NTHREADS, 1) k_dose(const __grid_constant__ DevPlan P, const PassArgs A) {
    SmemHeader* h = reinterpret_cast<SmemHeader*>(imrt_smem);
    float4* table_s = reinterpret_cast<float4*>(imrt_smem + SMEM_HEADER);
    float* x_s = reinterpret_cast<float*>(imrt_smem + P.x_off);
    State* st = P.st;
    cta_init(h, P, table_s);
    const int xi = st->xi, ri = st->ri;
    const float* x_in = A.x_in ? A.x_in : (A.mode == MODE_EVAL ? P.xbuf[xi] : P.xbuf[xi ^ 1]);
    float* r_out = A.r_out ? A.r_out : P.rbuf[ri ^ 1];
    for (int i = threadIdx.x; i < P.n_b; i += NTHREADS) x_s[i] = x_in[i];
    __syncthreads();
    Pipe pipe = {0u, 0u};
    const int par = (int)(st->fwd_passes & 1);
    dose_pass(P, h, imrt_smem, table_s, x_s, r_out, A.d_out, P.Gpart[par], pipe);
    __threadfence();
    if (!cta_is_last(&st->ticket_f, h)) return;

    // ---- the last CTA to finish takes the decision
    const double G_new = reduce_objective(P, P.Gpart[par], h);
    if (A.mode == MODE_EVAL) {
        if (threadIdx.x == 0) st->eval_obj = G_new;   // not counted: fwd_passes / tr_passes count the loop's passes
        return;
    }
    if (A.mode == MODE_INIT) {
        if (threadIdx.x == 0) {
            st->G_k = G_new; st->fwd_passes += 1; st->ri = ri ^ 1; st->xi = xi ^ 1;
            P.tr_obj[0] = G_new;
        }
        return;
    }
    Loop L;
    loop_load(st, L);
    const int dec = armijo_decide(P, st, L, G_new, threadIdx.x == 0);
    if (dec == DEC_REJECT_RETRY)   // x_k is xbuf[xi], the next trial goes to xbuf[xi^1]
        L.step_sq = compute_trial(P.xbuf[xi], P.g, L.lambda, P.xbuf[xi ^ 1], P.n_b, h);
    if (threadIdx.x == 0) {
        loop_store(st, L);
        const int inner = (dec == DEC_REJECT_RETRY);
        const int outer = (dec == DEC_ACCEPT_CONTINUE);
        st->cont_inner = inner;
        st->cont_outer = outer;
        if (A.use_handles) {
            cudaGraphSetConditional(A.h_inner, inner);
            cudaGraphSetConditional(A.h_outer, outer);
        }
    }
}

// Transpose pass as a kernel of its own.
__global__ void __launch_bounds__(NTHREADS, 1) k_transpose(const __grid_constant__ DevPlan P, const PassArgs A) {
    SmemHeader* h = reinterpret_cast<SmemHeader*>(imrt_smem);
    float4* table_s = reinterpret_cast<float4*>(imrt_smem + SMEM_HEADER);
    double* wpart = reinterpret_cast<double*>(imrt_smem + P.wpart_off);
    State* st = P.st;
    cta_init(h, P, table_s);
    const int xi = st->xi, ri = st->ri;
    const float* r_in = A.r_in ? A.r_in : P.rbuf[ri];
    Pipe pipe = {0u, 0u};
    const int par = (int)(st->tr_passes & 1);
    transpose_pass(P, h, imrt_smem, wpart, r_in, P.gslot[par], pipe);
    if (!cta_is_last(&st->ticket_t, h)) return;

    if (A.mode == MODE_EVAL) {
        reduce_gradient(P, P.gslot[par], A.g_out);
        return;
    }
    reduce_gradient(P, P.gslot[par], P.g);
    __syncthreads();
    Loop L;
    loop_load(st, L);
    const bool pending = begin_line_search(st, L, P.xbuf[xi], P.g, P.xbuf[xi ^ 1], P.n_b, h);
    if (threadIdx.x == 0) {
        loop_store(st, L);
        st->cont_inner = pending;
        if (!pending) st->cont_outer = 0;
        if (A.use_handles) {
            cudaGraphSetConditional(A.h_inner, pending);
            if (!pending) cudaGraphSetConditional(A.h_outer, 0);
        }
    }
}

// First node of the conditional graph / first step of the host driver: arm the outer loop.
__global__ void k_begin(State* st, int use_handles, cudaGraphConditionalHandle h_outer) {
    const int go = st->iter < st->iter_target;
    st->stop_reason = STOP_MAX_ITERS;
    st->cont_outer = go;
    st->cont_inner = 0;
    if (use_handles) cudaGraphSetConditional(h_outer, go);
}

// Plain launch before a run: how far to go and with which tolerance.
__global__ void k_set_target(State* st, int n_more, double delta_tol) {
    int target = st->iter + n_more;
    if (target > st->trace_cap) target = st->trace_cap;
    st->iter_target = target;
    st->delta_tol = delta_tol;
    st->gridbar = 0u;
}

// The whole loop in one cooperative launch (driver 2): PAPER.md:99-114 with no host involvement at all.
// Every CTA keeps x_k, g and x+ in shared memory and replays the same scalar decisions from the same fixed-order
// reductions, so CTAs never exchange anything but the pass partials; CTA 0 records the trace.
__global__ void __launch_bounds__(NTHREADS, 1) k_persistent(const __grid_constant__ DevPlan P) {
    SmemHeader* h = reinterpret_cast<SmemHeader*>(imrt_smem);
    float4* table_s = reinterpret_cast<float4*>(imrt_smem + SMEM_HEADER);
    double* wpart = reinterpret_cast<double*>(imrt_smem + P.wpart_off);
    float* xb = reinterpret_cast<float*>(imrt_smem + P.x_off);     // x+ (the dose pass gathers from it)
    float* g_s = reinterpret_cast<float*>(imrt_smem + P.g_off);
    State* st = P.st;
    cta_init(h, P, table_s);
    Loop L;
    loop_load(st, L);
    const int iter_target = st->iter_target;
    L.stop_reason = STOP_MAX_ITERS;
    Pipe pipe = {0u, 0u};
    unsigned int epoch = 0;
    const bool rec = (blockIdx.x == 0) && (threadIdx.x == 0);

    while (L.iter < iter_target) {
        const int tpar = (int)(L.tr & 1);
        transpose_pass(P, h, imrt_smem, wpart, P.rbuf[L.ri], P.gslot[tpar], pipe);
        grid_barrier(&st->gridbar, epoch);
        reduce_gradient(P, P.gslot[tpar], g_s);
        __syncthreads();
        if (!begin_line_search(st, L, P.xbuf[L.xi], g_s, xb, P.n_b, h)) break;   // x_k lives in global memory
        int dec;
        for (;;) {
            const int fpar = (int)(L.fwd & 1);
            dose_pass(P, h, imrt_smem, table_s, xb, P.rbuf[L.ri ^ 1], nullptr, P.Gpart[fpar], pipe);
            grid_barrier(&st->gridbar, epoch);
            const double G_new = reduce_objective(P, P.Gpart[fpar], h);
            dec = armijo_decide(P, st, L, G_new, rec);
            if (dec != DEC_REJECT_RETRY) break;
            L.step_sq = compute_trial(P.xbuf[L.xi], g_s, L.lambda, xb, P.n_b, h);
        }
        if ((dec == DEC_ACCEPT_CONTINUE || dec == DEC_ACCEPT_STOP) && blockIdx.x == 0) {
            // x_{k+1} = x+: publish it (L.xi already points at the new buffer); the other CTAs read it only after the
            // next grid barrier
            float* xg = P.xbuf[L.xi];
            for (int i = threadIdx.x; i < P.n_b; i += NTHREADS) xg[i] = xb[i];
        }
        if (dec != DEC_ACCEPT_CONTINUE) break;
    }
    // every CTA has passed the last grid barrier before CTA 0 gets here with a changed state
    grid_barrier(&st->gridbar, epoch);
    if (blockIdx.x == 0) {
        for (int i = threadIdx.x; i < P.n_b; i += NTHREADS) P.g[i] = g_s[i];
        if (threadIdx.x == 0) {
            loop_store(st, L);
            st->cont_outer = 0;
            st->cont_inner = 0;
        }
    }
}

}  // namespace imrt
