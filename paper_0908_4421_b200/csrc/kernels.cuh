// kernels.cuh -- the device side of libimrtgp (sm_100a).
//
// Two streaming passes and the scalar logic between them (PAPER.md = /root/reference/PAPER.md):
//
//   dose pass       d = D x+, penalty, residual r, objective partials      PAPER.md:51-66 Eq. (1)-(2), :128 kernels 1-2
//   transpose pass  g = D^T r on an explicit D^T CSR                       PAPER.md:107 step 1, :128 kernel 3
//   trial point     x+ = max(0, x - lambda g), Delta = ||x+ - x||^2       PAPER.md:90, :109-111, :128 kernel 4
//   Armijo / stop   C = G_k - (eps/lambda) Delta, accept iff G+ < C        PAPER.md:92-95 Eq. (5), :110-114
//
// Both passes are persistent CTAs (one per SM): producer warps stream the matrix with 1-D bulk async copies
// (cp.async.bulk, the TMA unit) into shared memory guarded by mbarriers; 16 consumer warps gather the vector (the
// trial points x+ from shared memory, r through L1/L2 with an evict-last hint), multiply-add in fp32 and reduce with
// warp shuffles.  The dose pass evaluates R = 1, 2 or 4 line-search trial points per pass over D (one record per
// consumer warp, records travelling through a byte ring whose schedule is laid out at plan creation); the transpose
// pass streams a packed D^T in fixed stages shared by the consumer warps.  Objective and gradient partials are fp64
// and are combined in a fixed order, so a plan's runs are bit-reproducible and no floating-point atomics are used
// anywhere.
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
constexpr int N_PROD = 2;                     // producer warps of the dose pass (the transpose pass uses the first only)
constexpr int NTHREADS = N_CONS + 32 * N_PROD;
// dose pass: D is re-packed once into self-contained block records (one bulk copy each, see DevPlan::pack)
constexpr int META_HDR = 4;                   // header words {rows, first row, 0, slots}
constexpr int ROW_REC_SLOTS = 1024;           // slots per row-format record (fewer for small matrices; one longer row alone)
constexpr int MAX_CHUNK_SLOTS = 8192;         // longest row of D this build handles (slot offsets are 16-bit)
constexpr int MAXROWS_F = 256;                // rows per block
constexpr int QUAD_MAX_NB = 16384;            // quad-format records are offered up to this many beamlets (pack-kernel bitmap)
constexpr int QUAD_CAP = 384;                 // union columns per quad record, at most (see record_caps)
constexpr int QUAD_MAXQ = 64;                 // quads per record
constexpr int SEG_ROWS = 256;                 // rows per format decision
constexpr int TARGET_RECORDS = 8192;          // a small matrix is cut into at least about this many records (imrtgp.cu)
constexpr int ZPAD = 4;                       // zero slots after a block's last row: where lanes past a row's end read
constexpr int R_MAX = 4;                      // line-search trial points evaluated per dose pass (1, 2 or 4)
constexpr int CHUNK_T = 2048;                 // entries per transpose-pass stage: 4 groups x 4 warps x 512-entry slices.  (Stages of
                                              // 4,096 entries for 2 groups of 8 warps hold the same 16 slices but hand the ring back in
                                              // 41 KB steps: 4 % slower; 1,024 entries for 8 groups of 2: 20 % slower.)
constexpr int TGROUPS = 4;                    // the consumer warps take the stages in turns, in this many groups:
constexpr int SLICE_T = CHUNK_T / (W_CONS / TGROUPS);   // contiguous nnz per warp of a stage's group (gathers in flight)
constexpr int CHUNK_T_PAD = CHUNK_T + 4;            // + alignment shift of a range start (<= 3 entries)
constexpr int STAGE_T_BYTES = CHUNK_T_PAD * 8;
constexpr int RL_MAX = 32;                    // rows of D^T one transpose range may span
constexpr int RING_ENTRIES = 64;              // dose-pass records in flight per CTA (a multiple of the team count)
constexpr int MAX_STAGES_T = 16;
constexpr int MAX_STRUCTURES = 256;
constexpr int MAX_WORLD = 16;                 // ranks of a row-sharded problem (one GPU each, or co-resident on one device)
constexpr int SMEM_HEADER = 3072;             // barriers, flags, reduction scratch
constexpr int SMEM_WPART = RL_MAX * W_CONS * 8 * 2;   // transpose pass: per-(row, warp) fp64 partials, two per row pair
constexpr int SMEM_DSC = W_CONS * 32 * R_MAX * 4;   // per-warp scratch: dose of 32 rows x R trial points

enum { MODE_TRIAL = 0, MODE_INIT = 1, MODE_EVAL = 2, MODE_TIMING = 3, MODE_BATCH = 4 };
enum { STOP_MAX_ITERS = 0, STOP_TOLERANCE = 1, STOP_STATIONARY = 2, STOP_LS_STALLED = 3, STOP_TRACE_FULL = 4, STOP_PEER_TIMEOUT = 5 };

// ------------------------------------------------------------------------------------------------ device data
struct State {                 // lives in the workspace; the single source of truth between launches
    double G_k;                // objective at the current iterate
    double lambda;             // step size of the first trial of the pending batch
    double eps, alpha, lambda0, delta_tol;
    double eval_obj;           // output of MODE_EVAL dose passes
    double eval_objs[4];       // outputs of a MODE_BATCH dose pass (imrt_plan_eval_batch)
    double G_skip;             // objective of the rows no block covers (their dose is 0: a constant)
    const float* tvu;          // optional per-voxel limits T-_j / T+_j [n_v] (NULL: the structure's, reading R16)
    const float* tvo;
    long long fwd_passes, tr_passes;
    int max_ls;
    int iter;                  // accepted iterations since set_x
    int iter_target;           // stop when iter reaches this
    int trace_cap;
    int m;                     // backtracking steps taken in the current line search (= index of the batch's first trial)
    int stop_reason;
    int xi;                    // xbuf[xi] is the current iterate
    int ri;                    // rbuf[ri] is r(x_k); trial j of a batch writes rbuf[(ri + 1 + j) % (R + 1)]
    int cont_outer, cont_inner;  // loop conditions (mirrors of the graph conditionals; read by the host driver)
    int bad_x;                 // set_x validation result
    unsigned int ticket_f, ticket_t;   // last-CTA tickets
    unsigned int gridbar;      // grid barrier counter of the persistent kernel
    int clamped;               // the last run's target was cut short by the trace capacity
    unsigned long long seq_g, seq_G;   // row-sharded plans: exchanges of the gradient / of objectives done so far (never reset)
    int G_is_local;            // row-sharded plans: G_k is this slab's share only (after set_x), not yet the sum over the ranks
    int fault;                 // sticky: a wait of the persistent loop timed out (STOP_PEER_TIMEOUT); cleared by imrt_plan_set_x
    unsigned long long spin_timeout_ns;   // bound on every in-kernel wait (grid barrier, inbox flags); imrt_options.spin_timeout_ms
};

struct TrRange {               // a contiguous piece of the D^T nnz stream, 32 bytes
    int e_begin, e_end;        // element range [e_begin, e_end) of the D^T stream
    int first_row;             // row of D^T holding e_begin
    int n_rows;                // rows spanned (<= RL_MAX)
    int slot_base;             // first gradient partial slot
    int pad[3];
};

struct DevPlan {
    long long nnz;
    int n_v, n_b;
    // dose pass: D re-packed into block records (owned).  A record is 128-byte aligned and holds, in this order,
    // ROW format (any matrix):
    //   header  uint32[4]  {rows, first row, 0, slots}
    //   rows    uint32[rows + 1]  slot offset of the row (low 16 bits, a multiple of 4) | structure id << 16;
    //                             padded to a multiple of 4 words
    //   val     fp32[slots + ZPAD]   every row padded with zeros to a multiple of 4 slots; ZPAD zeros at the end
    //   col     uint16[slots + ZPAD] (n_b <= 65536) or int32[slots + ZPAD]
    // QUAD format (chosen per 256-row segment where it is smaller; n_b <= QUAD_MAX_NB):
    //   header  uint32[4]  {quads, first row (a multiple of 4), 1, union columns}
    //   quads   uint32[2 (quads + 1)]  {column offset of the quad (low 16 bits) | row-exists mask << 16,
    //                                   the 4 structure ids}; the last pair holds the total; padded to 4 words
    //   val     fp32[columns + 1][4]   per union column the 4 rows' values, slot j = row j ^ (2 b3 + b2) with b3 b2 = bits 3, 2
    //                                  of the column's position inside its quad (dose_block_quads); one zero column at the end
    //   col     uint16[columns + 8]
    // One record is consumed by ONE warp.
    const unsigned char* pack;
    const int4* blk;           // {record offset / 128, record bytes, ring offset, blocks of the CTA to reclaim first}:
                               // the last two are the ring schedule of the current partition (k_ring_layout)
    const int* cta_blk;        // [grid_f + 1] block range per CTA
    int grid_f;
    int ring_f_bytes;          // bytes of the dose pass's shared-memory ring (records are placed at their own size)
    int max_rec_bytes;         // largest record
    int col16;                 // 1: 16-bit column indices in the records
    int R;                     // trial points per dose pass of the line search (1, 2 or 4)
    int pad1;
    // D^T (owned): CSR, rows = beamlets, padded with zeros to a multiple of 4 entries ...
    const int* rowT_ptr;       // row pointers of the stream the transpose pass reads (the packed one when id16)
    const int* colT;
    const float* valT;
    // ... and, unless a row has neighbouring entries more than 65535 voxels apart, the packed stream the transpose
    // pass reads instead (id16 = 1): every row padded to a multiple of 128 entries (zero values), voxel ids as
    // 16-bit offsets from one 32-bit base per aligned group of 32 entries: 6.1 instead of 8 bytes per non-zero
    const float* valP;         // id16 = 1: fp32 per entry;  id16 = 2: float2 per entry of a ROW PAIR (see below)
    const unsigned short* idP;
    const unsigned int* baseP;
    // id16 = 2 (chosen when smaller): rows 2i and 2i+1 of D^T (neighbouring beamlets, whose voxel lists overlap by ~87 %)
    // share ONE voxel list, the union of theirs, with a float2 of values per voxel (0 where a row lacks it): 10.1 bytes
    // per union entry, one gather of r per TWO multiply-adds.  rowT_ptr then points into the pair stream (one "row" per
    // pair), and a gradient slot holds two sums.
    int id16;
    int stage_t_bytes;         // bytes of one transpose-pass stage
    // transpose pass: equal-nnz ranges
    const TrRange* tr_range;
    const int* rowslot_ptr;    // [n_b + 1] slots of row i are [rowslot_ptr[i], rowslot_ptr[i+1])
    const int* cta_rng;        // [grid_t + 1] ranges of CTA c are [cta_rng[c], cta_rng[c+1])
    int n_ranges, grid_t, n_stages_t, n_slots;
    // penalty table and skipped (matrix-free) rows
    const float4* table;       // (t_under, t_over, w_under, w_over)
    int n_structures;
    int pad0;
    const unsigned char* covered;   // [n_v] 1: the row belongs to a record; 0: dose 0, constant penalty (State::G_skip)
    // vectors
    float* xbuf[2];
    float* g;
    float* rbuf[R_MAX + 1];    // residual buffers: one holds r(x_k), the others receive r of the batch's trial points
    double* Gpart[2];          // [grid_f][R] objective partials, double-buffered by pass parity
    double* gslot[2];          // [n_slots] gradient partials, double-buffered
    State* st;
    unsigned long long* cta_ns;  // [2][1024][2] per-CTA {start, end of streaming} of the last dose / transpose pass, ns
    double* tr_obj;            // trace: [cap + 1]
    double* tr_lambda;         // [cap]
    double* tr_step_sq;        // [cap]
    int* tr_trials;            // [cap]
    // row-sharded problems: this plan holds the rows of rank `rank` of `world`; inbox[q] is rank q's
    // exchange buffer (peer memory over NVLink, or plain device memory when the ranks share one device)
    int rank, world;
    unsigned char* inbox[MAX_WORLD];
    int wpart_off;             // byte offsets into dynamic shared memory: transpose per-(row, warp) partials,
    int dsc_off;               // dose-pass per-warp scratch,
    int x_off, g_off;          // the trial points x+ [n_b][R] (gathered by the dose pass) and the gradient (persistent kernel)
    int stage_off;             // byte offset of the dose pass's ring
    int tr_stage_off;          // byte offset of the transpose pass's stages: they also cover the trial points and g, which are
                               // dead while a transpose pass runs (both are rebuilt right after it)
};

struct PassArgs {
    const float* x_in;         // dose pass, MODE_EVAL / MODE_INIT: where to evaluate (NULL = the current iterate)
    const float* r_in;         // transpose pass: residual (NULL = rbuf[ri])
    float* r_out;              // dose pass, MODE_EVAL: residual out
    float* d_out;              // dose pass, MODE_EVAL: dose out or NULL
    float* g_out;              // transpose pass MODE_EVAL: gradient out
    int mode;
    int n_points;              // MODE_BATCH: points at x_in ([n_points][n_b]); residuals to r_out ([n_points][n_v]) or scratch
    int use_handles;           // 1 inside the conditional graph
    cudaGraphConditionalHandle h_outer, h_inner;
};

// The loop's constants: State fields that do not change during a run.  The persistent kernel keeps a copy in shared
// memory (the scalar phases between the passes are chains of latencies; every global read they do not make is ~0.3 us).
struct LoopConst {
    double eps, alpha, lambda0, delta_tol, G_skip;
    unsigned long long spin_timeout_ns;
    int max_ls, iter_target;
};
__device__ __forceinline__ LoopConst loop_const(const State* st) {
    LoopConst C;
    C.eps = st->eps; C.alpha = st->alpha; C.lambda0 = st->lambda0; C.delta_tol = st->delta_tol; C.G_skip = st->G_skip;
    C.max_ls = st->max_ls; C.iter_target = st->iter_target; C.spin_timeout_ns = st->spin_timeout_ns;
    return C;
}

// ------------------------------------------------------------------------------------------------ shared memory
struct SmemHeader {
    uint64_t full_f[RING_ENTRIES], full_t[MAX_STAGES_T], empty_t[MAX_STAGES_T];
    uint32_t next_blk[W_CONS];        // dose pass: number (over the CTA's life) of the next block each consumer warp will finish
    double red[32 * R_MAX];    // block-reduction scratch
    double bcast[4];
    int flag;
    int fault;                 // persistent kernel: a bounded wait gave up (grid_barrier / shard_wait); 0 at kernel start
    LoopConst lc;              // persistent kernel: the run's constants
    int cta, n_cta;            // this CTA's index among the CTAs of ITS plan and their number: h->cta / gridDim.x, except when
                               // several plans (ranks) share one cooperative launch (k_persistent_ranks)
};
static_assert(sizeof(SmemHeader) <= SMEM_HEADER, "header");

struct Pipe {                  // running stage counters; identical in producer and consumers
    unsigned int it_f, it_t;
};

__device__ __forceinline__ void cta_init(SmemHeader* h, const DevPlan& P, float4* table_s, int cta = (int)blockIdx.x, int n_cta = (int)gridDim.x) {
    if (threadIdx.x == 0) {
        h->cta = cta;
        h->n_cta = n_cta;
        h->fault = 0;
        for (int s = 0; s < RING_ENTRIES; ++s) mbar_init(&h->full_f[s], 1);
        for (int s = 0; s < MAX_STAGES_T; ++s) {
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
// The same for R values at once; every component is summed in exactly the order block_sum uses.
template <int R>
__device__ __forceinline__ void block_sum_vec(double (&v)[R], SmemHeader* h) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int r = 0; r < R; ++r) v[r] = warp_sum(v[r]);
    __syncthreads();
    if (lane == 0) {
#pragma unroll
        for (int r = 0; r < R; ++r) h->red[r * 32 + warp] = v[r];
    }
    __syncthreads();
#pragma unroll
    for (int r = 0; r < R; ++r) {
        double s = 0.0;
#pragma unroll
        for (int w = 0; w < NTHREADS / 32; ++w) s += h->red[r * 32 + w];
        v[r] = s;
    }
}

// ------------------------------------------------------------------------------------------------ trial points
// x+ = max(0, x - lambda g), Delta = sum (x+ - x)^2      PAPER.md:90 (projection), :109/:111 (steps 2, 4), Eq. (5).
// fp32 elementwise, fp64 sum.  A batch holds the next R trial points of the line search: lambda, lambda/alpha, ...
// (the same division chain step 4 performs one trial at a time).  All NTHREADS threads call it; x is global (read
// through L2: another CTA may have written it), g may be shared or global; xs is the shared-memory array the dose
// pass gathers from, [n_b][R].
template <int R>
__device__ __forceinline__ void trial_batch(const float* x, const float* g, double lambda, double alpha, float* xs, int n_b,
                                            SmemHeader* h, double (&step_sq)[R]) {
    float lam[R];
    double l = lambda;
#pragma unroll
    for (int r = 0; r < R; ++r) { lam[r] = (float)l; l = l / alpha; step_sq[r] = 0.0; }
    constexpr int U = 4;         // rows per thread whose loads are issued together (x comes from L2)
    for (int base = threadIdx.x; base < n_b; base += NTHREADS * U) {
        float xv[U], gv[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int i = base + u * NTHREADS;
            xv[u] = i < n_b ? __ldcg(x + i) : 0.0f;
            gv[u] = i < n_b ? g[i] : 0.0f;
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int i = base + u * NTHREADS;
            if (i < n_b) {
                float* o = xs + (size_t)i * R;
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const float xn = fmaxf(0.0f, fmaf(-lam[r], gv[u], xv[u]));
                    const float dx = xn - xv[u];
                    step_sq[r] = __fma_rn((double)dx, (double)dx, step_sq[r]);
                    o[r] = xn;
                }
            }
        }
    }
    block_sum_vec<R>(step_sq, h);
}

// Only Delta of the first trial (the STATIONARY test of reading R4 at the start of a line search).
__device__ __forceinline__ double first_step_sq(const float* x, const float* g, double lambda, int n_b, SmemHeader* h) {
    const float lam = (float)lambda;
    double acc = 0.0;
    for (int i = threadIdx.x; i < n_b; i += NTHREADS) {
        const float xi = __ldcg(x + i);
        const float dx = fmaxf(0.0f, fmaf(-lam, g[i], xi)) - xi;
        acc = __fma_rn((double)dx, (double)dx, acc);
    }
    return block_sum(acc, h);
}

// A single point x (MODE_EVAL / MODE_INIT): copy it to the gather array.
__device__ __forceinline__ void stage_point(const float* x, float* xs, int n_b) {
    for (int i = threadIdx.x; i < n_b; i += NTHREADS) xs[i] = x[i];
    __syncthreads();
}

// ------------------------------------------------------------------------------------------------ dose pass
// One block record is consumed by ONE warp (the CTA's blocks are dealt round-robin to its 16 consumer warps, which
// never synchronise with each other).  Inside a record: VW = 8 lanes per row, 4 rows per warp batch, 4 consecutive
// slots per lane and trip.  Rows start on 16-byte boundaries and are zero-padded to a multiple of 4 slots, so values
// and columns come in with one 128-bit (64-bit for 16-bit columns) shared-memory load each; a lane past the end of
// its row reads the record's zero slots instead, which keeps the trip loop free of divergent branches.  The row
// groups of a batch run the trip count of their longest row (neighbouring voxels have rows of similar length).
// Each lane gathers the R trial values of its 4 beamlets from shared memory ([n_b][R], one vector load per beamlet),
// multiply-adds in fp32 (one accumulator per slot position and trial point, so the sum of a row does not depend on
// R) and the group reduces with 3 shuffles.  Doses of 32 rows are parked in a per-warp scratch; then every lane
// takes one row: penalty and residual per trial point (Eq. (1) generalised: F = w- u^2 + w+ o^2,
// r = 2 (w+ o - w- u)), coalesced stores of r, fp64 accumulation of F.
constexpr int VW = 8;
constexpr int RB = 32 / VW;

struct VoxelLimits {           // optional per-voxel limits (State::tvu / tvo), loaded once per pass
    const float* tu;
    const float* to;
    __device__ __forceinline__ void apply(float4& t, size_t j) const {
        if (tu) t.x = __ldg(tu + j);
        if (to) t.y = __ldg(to + j);
    }
};

template <int R> struct XVec;
template <> struct XVec<1> { float v[1]; __device__ __forceinline__ void load(const unsigned char* p) { v[0] = *reinterpret_cast<const float*>(p); } };
template <> struct XVec<2> { float v[2]; __device__ __forceinline__ void load(const unsigned char* p) { const float2 t = *reinterpret_cast<const float2*>(p); v[0] = t.x; v[1] = t.y; } };
template <> struct XVec<4> { float v[4]; __device__ __forceinline__ void load(const unsigned char* p) { const float4 t = *reinterpret_cast<const float4*>(p); v[0] = t.x; v[1] = t.y; v[2] = t.z; v[3] = t.w; } };

template <bool COL16, int R>
__device__ __forceinline__ void dose_block(const unsigned char* __restrict__ rec, const unsigned char* __restrict__ xs_b,
                                           const float4* __restrict__ table_s, float* __restrict__ dsc,
                                           float* const (&r_out)[R], float* __restrict__ d_out, const VoxelLimits vl, int lane,
                                           double (&Gacc)[R]) {
    const uint4 hdr = *reinterpret_cast<const uint4*>(rec);
    const int nrows = (int)hdr.x, slots = (int)hdr.w;
    const uint32_t* rows = reinterpret_cast<const uint32_t*>(rec) + META_HDR;
    const unsigned char* val_b = reinterpret_cast<const unsigned char*>(rows + ((nrows + 1 + 3) & ~3));
    const unsigned char* col_b = val_b + (size_t)(slots + ZPAD) * 4;
    const int grp = lane / VW, sub = lane % VW;
    constexpr int XB = 4 * R;   // bytes per beamlet in the gather array
    const int nbatch = (nrows + RB - 1) / RB;
    // 8 batches (32 rows) make one penalty step
    for (int q0 = 0; q0 < nbatch; q0 += 8) {
#pragma unroll 1
        for (int kq = 0; kq < 8; ++kq) {
            const int q = q0 + kq;
            if (q >= nbatch) break;
            const int row = q * RB + grp;
            uint32_t m0 = 0u, m1 = 0u;
            if (row < nrows) { m0 = rows[row]; m1 = rows[row + 1]; }
            const int s = (int)(m0 & 0xFFFFu), e = (int)(m1 & 0xFFFFu);
            const int len_max = __reduce_max_sync(0xffffffffu, e - s);   // warp-uniform trip count
            float acc[4][R];
#pragma unroll
            for (int j = 0; j < 4; ++j)
#pragma unroll
                for (int r = 0; r < R; ++r) acc[j][r] = 0.0f;
            int k = s + 4 * sub;
#pragma unroll 2
            for (int kb = 0; kb < len_max; kb += 4 * VW, k += 4 * VW) {
                const int kk = k < e ? k : slots;          // past the row's end: the zero slots
                const float4 v = *reinterpret_cast<const float4*>(val_b + 4 * kk);
                uint32_t o0, o1, o2, o3;                   // byte offsets into the gather array
                if (COL16) {
                    const uint2 c = *reinterpret_cast<const uint2*>(col_b + 2 * kk);
                    o0 = (c.x & 0xFFFFu) * XB; o1 = (c.x >> 16) * XB; o2 = (c.y & 0xFFFFu) * XB; o3 = (c.y >> 16) * XB;
                } else {
                    const uint4 c = *reinterpret_cast<const uint4*>(col_b + 4 * kk);
                    o0 = c.x * XB; o1 = c.y * XB; o2 = c.z * XB; o3 = c.w * XB;
                }
                XVec<R> x0, x1, x2, x3;
                x0.load(xs_b + o0); x1.load(xs_b + o1); x2.load(xs_b + o2); x3.load(xs_b + o3);
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    acc[0][r] = fmaf(v.x, x0.v[r], acc[0][r]);
                    acc[1][r] = fmaf(v.y, x1.v[r], acc[1][r]);
                    acc[2][r] = fmaf(v.z, x2.v[r], acc[2][r]);
                    acc[3][r] = fmaf(v.w, x3.v[r], acc[3][r]);
                }
            }
            float d[R];
#pragma unroll
            for (int r = 0; r < R; ++r) d[r] = vec_sum<VW>((acc[0][r] + acc[1][r]) + (acc[2][r] + acc[3][r]));
            if (sub == 0) {   // rows past the end park a zero nobody reads
                float* o = dsc + (kq * RB + grp) * R;
#pragma unroll
                for (int r = 0; r < R; ++r) o[r] = d[r];
            }
        }
        __syncwarp();
        const int row = (q0 + lane / RB) * RB + (lane % RB);     // the row parked at position `lane`
        if (row < nrows) {
            float4 t = table_s[(rows[row] >> 16) & 0xFFu];
            XVec<R> dv;
            dv.load(reinterpret_cast<const unsigned char*>(dsc + lane * R));
            const size_t j = (size_t)hdr.y + row;
            vl.apply(t, j);
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const float dd = dv.v[r];
                const float u = fmaxf(0.0f, t.x - dd);
                const float o = fmaxf(0.0f, dd - t.y);
                r_out[r][j] = 2.0f * __fmaf_rn(t.w, o, -__fmul_rn(t.z, u));      // explicit roundings: every
                const double du = (double)u, d_o = (double)o;                     // instantiation sums alike
                Gacc[r] = __dadd_rn(Gacc[r], __fma_rn((double)t.z, __dmul_rn(du, du), __dmul_rn((double)t.w, __dmul_rn(d_o, d_o))));
            }
            if (R == 1 && d_out) d_out[j] = dv.v[0];
        }
        __syncwarp();
    }
}

// The same for a record in QUAD format: 4 consecutive rows of D (neighbouring voxels, which see nearly the same
// beamlets) share one sorted list of columns, the union of theirs; per union column the record holds the 4 rows'
// values as one 16-byte vector (explicit zeros where a row has no entry) and one 16-bit column.  A warp takes TWO
// quads at a time, one per half-warp: per trip every lane takes one union column of its quad -- one vector load of 4
// values, one column, ONE gather of the R trial values (16 neighbouring beamlets per half: conflict-free), 4 R
// multiply-adds.  Against the row format this needs a quarter of the gathers and of the column bytes and -- where
// the rows of a quad overlap well -- fewer bytes of HBM traffic per non-zero (18 bytes per union column).  Rows are
// short (a quad has ~130 union columns), so the reduction and the penalty evaluation at the end of a quad cost as
// many instructions as its multiply-adds; two quads per warp halve that share and leave every lane of the warp
// with exactly one (row, trial) sum at R = 4.
// Which trial point of a batch a lane ends up with after the quad reduction, and whether it ends up with a sum at all.
template <int R> __device__ __forceinline__ int quad_trial(int lane) { return R == 4 ? (lane & 3) : R == 2 ? ((lane >> 1) & 1) : 0; }
template <int R> __device__ __forceinline__ bool quad_owner(int lane) { return (lane & (R == 4 ? 0 : R == 2 ? 1 : 3)) == 0; }

// The reduction is one xor butterfly over the 16 lanes of a half-warp for every (row, trial) sum -- the same tree of
// additions whatever R is -- but at each step a lane keeps only half of what it holds: xor 8 splits the rows
// {0,1} | {2,3}, xor 4 leaves one row, xor 2 / xor 1 split the trial points (R = 4; xor 2 only for R = 2).  4 R - 1
// shuffles for two quads, and lane (b4 b3 b2 b1 b0) ends with row 2 b3 + b2 of trial 2 b1 + b0 of quad b4.  The
// packing rotates the rows of every column so that the two row-splitting steps need no selects (see below).
// my_r: the residual buffer of this lane's trial.  Gq: this lane's objective partial (of its own trial).
template <int R>
__device__ __forceinline__ void dose_block_quads(const unsigned char* __restrict__ rec, const unsigned char* __restrict__ xs_b,
                                                 const float4* __restrict__ table_s, float* __restrict__ my_r,
                                                 float* __restrict__ d_out, const VoxelLimits vl, int lane, double& Gq) {
    const uint4 hdr = *reinterpret_cast<const uint4*>(rec);
    const int nq = (int)hdr.x, nbc = (int)hdr.w;
    const uint32_t* qt = reinterpret_cast<const uint32_t*>(rec) + META_HDR;
    const unsigned char* val_b = reinterpret_cast<const unsigned char*>(qt + ((2 * (nq + 1) + 3) & ~3));
    const unsigned char* col_b = val_b + (size_t)(nbc + 1) * 16;
    constexpr int XB = 4 * R;
    const int half = lane >> 4, l16 = lane & 15;
    const bool hi8 = (lane & 8) != 0, hi4 = (lane & 4) != 0, hi2 = (lane & 2) != 0, hi1 = (lane & 1) != 0;
    const int rr = (hi8 ? 2 : 0) + (hi4 ? 1 : 0);          // the row this lane ends up with
    const bool owner = quad_owner<R>(lane);
    for (int q0 = 0; q0 < nq; q0 += 2) {
        // A quad without a partner (the record's only or last one: typically a long quad that fills a record by itself)
        // is split between the halves instead, columns [s, mid) and [mid, e); their sums meet in one more xor step.
        const bool lone = q0 + 1 >= nq;
        const int qi = lone ? q0 : q0 + half;
        const uint2 w = *reinterpret_cast<const uint2*>(qt + 2 * qi);
        int s = (int)(w.x & 0xFFFFu), e = (int)(qt[2 * qi + 2] & 0xFFFFu);
        if (lone) {
            // the cut is a multiple of 16 columns after s: lane l16 then takes the columns at positions = l16 (mod 16) of
            // the quad in BOTH halves, which is what the packed row rotation (below) is keyed to
            const int mid = min(e, s + 16 * ((e - s + 31) >> 5));
            if (half) s = mid; else e = mid;
        }
        const int len = e - s;
        const int olen = __shfl_xor_sync(0xffffffffu, len, 16);
        const int trips = max(len, olen);
        const int n_fast = min(len, olen) >> 4;            // trips in which BOTH halves have a full 16 columns: no clamping
        // rows {0,1} and {2,3} of a trial are kept as register pairs: one packed multiply-add (FFMA2, the trial value as
        // its broadcast operand) does two rows -- 2 R instead of 4 R issue slots per column, each half an IEEE fma
        float2 acc01[R], acc23[R];
#pragma unroll
        for (int r = 0; r < R; ++r) acc01[r] = acc23[r] = make_float2(0.0f, 0.0f);
        {
            const unsigned char* vp = val_b + 16 * (s + l16);
            const unsigned char* cp = col_b + 2 * (s + l16);
#pragma unroll 2
            for (int i = 0; i < n_fast; ++i, vp += 256, cp += 32) {
                const float4 v = *reinterpret_cast<const float4*>(vp);
                const uint32_t c = *reinterpret_cast<const unsigned short*>(cp);
                XVec<R> x;
                x.load(xs_b + c * XB);
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const float2 xr = make_float2(x.v[r], x.v[r]);
                    acc01[r] = __ffma2_rn(make_float2(v.x, v.y), xr, acc01[r]);
                    acc23[r] = __ffma2_rn(make_float2(v.z, v.w), xr, acc23[r]);
                }
            }
        }
        for (int t0 = 16 * n_fast; t0 < trips; t0 += 16) {      // the ragged end: at most a few trips per pair
            const int k = s + t0 + l16;
            const int kk = k < e ? k : nbc;                // past the quad's end: the zero column
            const float4 v = *reinterpret_cast<const float4*>(val_b + 16 * kk);
            const uint32_t c = *reinterpret_cast<const unsigned short*>(col_b + 2 * kk);
            XVec<R> x;
            x.load(xs_b + c * XB);
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const float2 xr = make_float2(x.v[r], x.v[r]);
                acc01[r] = __ffma2_rn(make_float2(v.x, v.y), xr, acc01[r]);
                acc23[r] = __ffma2_rn(make_float2(v.z, v.w), xr, acc23[r]);
            }
        }
        // The record stores the 4 rows' values of the column at position p of its quad ROTATED: slot j holds row
        // j ^ (2 b3 + b2), b3 b2 = bits 3 and 2 of p -- and p = l16 (mod 16) for the lane that takes the column.  So in every
        // lane slot 0 already holds the row the lane ends up with (2 b3 + b2), slot 1 its xor-4 partner's row, slots 2, 3 its
        // xor-8 partner's rows: the row-splitting steps keep the low slots and send the high ones, with no selects.
        float h[R];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const float a0 = acc01[r].x + __shfl_xor_sync(0xffffffffu, acc23[r].x, 8);
            const float a1 = acc01[r].y + __shfl_xor_sync(0xffffffffu, acc23[r].y, 8);
            h[r] = a0 + __shfl_xor_sync(0xffffffffu, a1, 4);
        }
        float d;
        if (R == 4) {
            const float g0 = (hi2 ? h[R > 2 ? 2 : 0] : h[0]) + __shfl_xor_sync(0xffffffffu, hi2 ? h[0] : h[R > 2 ? 2 : 0], 2);
            const float g1 = (hi2 ? h[R > 3 ? 3 : 0] : h[R > 1 ? 1 : 0]) + __shfl_xor_sync(0xffffffffu, hi2 ? h[R > 1 ? 1 : 0] : h[R > 3 ? 3 : 0], 2);
            d = (hi1 ? g1 : g0) + __shfl_xor_sync(0xffffffffu, hi1 ? g0 : g1, 1);
        } else if (R == 2) {
            const float g = (hi2 ? h[R > 1 ? 1 : 0] : h[0]) + __shfl_xor_sync(0xffffffffu, hi2 ? h[0] : h[R > 1 ? 1 : 0], 2);
            d = g + __shfl_xor_sync(0xffffffffu, g, 1);
        } else {
            const float g = h[0] + __shfl_xor_sync(0xffffffffu, h[0], 2);
            d = g + __shfl_xor_sync(0xffffffffu, g, 1);
        }
        if (lone) d += __shfl_xor_sync(0xffffffffu, d, 16);
        if (owner && !(lone && half) && ((w.x >> (16 + rr)) & 1u)) {  // the row exists
            float4 t = table_s[(w.y >> (8 * rr)) & 0xFFu];
            const size_t jrow = (size_t)hdr.y + 4 * qi + rr;
            vl.apply(t, jrow);
            const float u = fmaxf(0.0f, t.x - d);
            const float o = fmaxf(0.0f, d - t.y);
            my_r[jrow] = 2.0f * __fmaf_rn(t.w, o, -__fmul_rn(t.z, u));
            const double du = (double)u, d_o = (double)o;
            Gq = __dadd_rn(Gq, __fma_rn((double)t.z, __dmul_rn(du, du), __dmul_rn((double)t.w, __dmul_rn(d_o, d_o))));
            if (R == 1 && d_out) d_out[jrow] = d;
        }
    }
}

// All NTHREADS threads of the CTA call this.  xs: the R trial points in shared memory.  Writes the CTA's R objective
// partials to Gpart[blockIdx.x * R ..] (thread 0).  Ends with a CTA-wide barrier.
// STREAM: the read-only streaming ceiling of the pass -- the producers move every record through the ring exactly as in
// the real pass, the consumer warps wait for their records and hand them back untouched (imrt_plan_launch_pass kind 2).
template <bool COL16, int R, bool STREAM = false>
__device__ __forceinline__ void dose_pass_t(const DevPlan& P, SmemHeader* h, unsigned char* smem, const float4* table_s,
                                            const float* xs, float* const (&r_out)[R], float* d_out, double* Gpart, Pipe& pipe) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    unsigned char* ring = smem + P.stage_off;
    const int b0 = (h->cta < P.grid_f) ? P.cta_blk[h->cta] : 0;
    const int b1 = (h->cta < P.grid_f) ? P.cta_blk[h->cta + 1] : 0;
    const int nb = b1 - b0;
    double Gacc[R];              // objective partials of the row-format records (every lane, every trial) ...
#pragma unroll
    for (int r = 0; r < R; ++r) Gacc[r] = 0.0;
    double Gq = 0.0;             // ... and of the quad-format records (this lane's trial only)
    const unsigned long long t_start = global_ns();
    const uint32_t full_a = smem_u32(&h->full_f[0]), ring_a = smem_u32(ring);
    volatile uint32_t* next_blk = h->next_blk;
    const unsigned int it0 = pipe.it_f;        // blocks are numbered over the CTA's life: this pass has it0 .. it0 + nb - 1
    if (warp < W_CONS && lane == 0) next_blk[warp] = it0 + (unsigned int)warp;
    __syncthreads();

    // The ring: records keep their own size (128-byte multiples) and are laid end to end in a circular byte buffer;
    // a record that does not fit before the end starts over at 0.  Where each record goes, and how many of the CTA's
    // earlier blocks must have left the ring before its copy may be issued, depends only on the record sizes, so it is
    // computed once per partition (k_ring_layout) and travels with the block descriptors.  Block number `it` uses
    // full barrier it % 64 in phase it / 64; a warp's consecutive blocks are 16 apart, so the previous user of a
    // barrier is always a block the same warps have already finished.  Space is reclaimed in issue order: every
    // consumer warp publishes the number of the next block it will finish, and the minimum over the warps bounds
    // the blocks that are gone.
    if (warp >= W_CONS) {
        // ---------------- producer warps: producer p issues the CTA's blocks p, p + N_PROD, ... (lane 0 drives the TMA
        // unit, one bulk copy per block record); the descriptors of its next 32 blocks are requested before the current
        // 32 are issued
        const int pw = warp - W_CONS;
        const uint64_t pol = policy_evict_first();   // streamed once per pass: keep it from pushing r / x out of L2
        unsigned int gone = it0;                       // every block numbered below this has been consumed
        int4 next = (pw + N_PROD * lane < nb) ? __ldg(P.blk + b0 + pw + N_PROD * lane) : make_int4(0, 0, 0, 0);
        for (int bb = pw; bb < nb; bb += 32 * N_PROD) {
            const int4 mine = next;
            next = (bb + N_PROD * (32 + lane) < nb) ? __ldg(P.blk + b0 + bb + N_PROD * (32 + lane)) : make_int4(0, 0, 0, 0);
            const int nb_here = min(32, (nb - bb + N_PROD - 1) / N_PROD);
            for (int j = 0; j < nb_here; ++j) {
                const int off128 = __shfl_sync(0xffffffffu, mine.x, j);
                const uint32_t bytes = (uint32_t)__shfl_sync(0xffffffffu, mine.y, j);
                const uint32_t at = (uint32_t)__shfl_sync(0xffffffffu, mine.z, j);
                const unsigned int need = it0 + (unsigned int)__shfl_sync(0xffffffffu, mine.w, j);
                if ((int)(need - gone) > 0) {
                    do {
                        const unsigned int v = next_blk[lane & (W_CONS - 1)];
                        gone = __reduce_min_sync(0xffffffffu, v - it0) + it0;     // numbers wrap: compare relative to it0
                    } while ((int)(need - gone) > 0);
                    __threadfence_block();   // the consumers' reads of the space (seen through next_blk) come first
                }
                if (lane == 0) {
                    const uint32_t bar = full_a + 8u * ((it0 + (unsigned int)(bb + N_PROD * j)) & (RING_ENTRIES - 1));
                    mbar_expect_tx_a(bar, bytes);
                    bulk_g2s_a(ring_a + at, P.pack + (size_t)(unsigned int)off128 * 128u, bytes, bar, pol);
                }
            }
        }
    } else {
        // ---------------- consumer warps: warp w takes the CTA's blocks w, w + 16, ...
        float* dsc = reinterpret_cast<float*>(smem + P.dsc_off) + warp * 32 * R_MAX;
        const unsigned char* xs_b = reinterpret_cast<const unsigned char*>(xs);
        float* my_r = r_out[0];
#pragma unroll
        for (int r = 1; r < R; ++r) my_r = quad_trial<R>(lane) == r ? r_out[r] : my_r;
        const VoxelLimits vl = {P.st->tvu, P.st->tvo};
        int at_next = (warp < nb) ? __ldg(&P.blk[b0 + warp].z) : 0;
        for (int i = warp; i < nb; i += W_CONS) {
            const int at = at_next;
            if (i + W_CONS < nb) at_next = __ldg(&P.blk[b0 + i + W_CONS].z);
            const unsigned int it = it0 + (unsigned int)i;
            mbar_wait_a(full_a + 8u * (it & (RING_ENTRIES - 1)), (it / RING_ENTRIES) & 1u);
            const unsigned char* rec = ring + at;
            if (STREAM) {
                // nothing: the record is only waited for
            } else if (COL16 && reinterpret_cast<const uint32_t*>(rec)[2] != 0u)      // header word 2: record format
                dose_block_quads<R>(rec, xs_b, table_s, my_r, d_out, vl, lane, Gq);
            else
                dose_block<COL16, R>(rec, xs_b, table_s, dsc, r_out, d_out, vl, lane, Gacc);
            __syncwarp();
            if (lane == 0) {
                __threadfence_block();
                next_blk[warp] = it + (unsigned int)W_CONS;
            }
        }
        if (lane == 0) next_blk[warp] = it0 + (unsigned int)nb + (unsigned int)W_CONS;   // nothing left: never the minimum
    }
    pipe.it_f += (unsigned int)nb;
    // the two kinds of partials are summed separately (each in an order that does not depend on R) and then added
    double Gqv[R];
#pragma unroll
    for (int r = 0; r < R; ++r) Gqv[r] = (warp < W_CONS && quad_trial<R>(lane) == r) ? Gq : 0.0;
    block_sum_vec<R>(Gacc, h);   // producer lanes contribute 0
    block_sum_vec<R>(Gqv, h);
#pragma unroll
    for (int r = 0; r < R; ++r) Gacc[r] += Gqv[r];
    if (threadIdx.x == 0 && h->cta < P.grid_f) {
#pragma unroll
        for (int r = 0; r < R; ++r) Gpart[h->cta * R + r] = Gacc[r];
        P.cta_ns[2 * h->cta] = t_start;            // when this CTA's share of the pass began and ended: lets the
        P.cta_ns[2 * h->cta + 1] = global_ns();    // host see (and rebalance) the static partition
    }
    __syncthreads();
}

template <int R, bool STREAM = false>
__device__ __forceinline__ void dose_pass(const DevPlan& P, SmemHeader* h, unsigned char* smem, const float4* table_s,
                                          const float* xs, float* const (&r_out)[R], float* d_out, double* Gpart, Pipe& pipe) {
    if (P.col16) dose_pass_t<true, R, STREAM>(P, h, smem, table_s, xs, r_out, d_out, Gpart, pipe);
    else dose_pass_t<false, R, STREAM>(P, h, smem, table_s, xs, r_out, d_out, Gpart, pipe);
}

// Objectives of a finished dose pass: fixed-order sums of the CTA partials + the constant of the skipped rows.
// Every thread of the calling CTA gets the values.
template <int R>
__device__ __forceinline__ void reduce_objective(const DevPlan& P, const double* Gpart, SmemHeader* h, double (&G)[R], double G_skip) {
#pragma unroll
    for (int r = 0; r < R; ++r) G[r] = 0.0;
    for (int c = threadIdx.x; c < P.grid_f; c += NTHREADS) {
#pragma unroll
        for (int r = 0; r < R; ++r) G[r] += __ldcg(Gpart + c * R + r);
    }
    block_sum_vec<R>(G, h);
#pragma unroll
    for (int r = 0; r < R; ++r) G[r] += G_skip;
}

// ------------------------------------------------------------------------------------------------ transpose pass
// g = D^T r (PAPER.md:107 step 1, :128 kernel 3) on the explicit transpose.  One contiguous share of the D^T stream per
// CTA, cut into ranges of at most RL_MAX rows; a producer warp streams fixed-size stages with bulk copies, the consumer
// warps gather r, multiply-add in fp32 over short slices and keep fp64 running sums per row; per-(warp, row) sums meet
// in shared memory and leave as one fp64 partial per (range, row) slot.  All NTHREADS threads call a pass; it ends with
// a CTA-wide barrier.  Every consumer warp observes EVERY stage's full barrier and arrives on its empty barrier
// (count W_CONS), so the producer can never refill a slot before all warps have seen its phase.

// ---- single rows.  ID16 = false: the plain 32-bit CSR (rows are not padded, a slice may span several rows, a range may
// start at any multiple of 4 entries).  ID16 = true: the packed stream -- voxel ids as 16-bit offsets from one 32-bit
// base per aligned group of 32 entries, rows padded to 128 entries.  2,048-entry stages taken in turns by four groups
// of 4 consumer warps (a contiguous 512-entry slice and 16 gathers of r in flight per lane): 4 stages are being
// consumed while the other 4 of the ring are in flight, and the ring is handed back to the producer in 20 KB steps.  A software-pipelined variant (every warp a 128-entry slice of every stage, values
// parked in registers, multiply-adds four stages later) measured no faster in isolation and slower inside the persistent
// kernel (register pressure): the pass is bound by L2 throughput -- the stream plus the r gathers -- not by latency.
template <bool ID16>
__device__ __forceinline__ void transpose_pass_rows(const DevPlan& P, SmemHeader* h, unsigned char* smem, double* wpart,
                                               const float* __restrict__ r_in, double* gslot, Pipe& pipe) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int S = P.n_stages_t;
    unsigned char* stages = smem + P.tr_stage_off;
    unsigned int it = pipe.it_t;
    const int rg0 = (h->cta < P.grid_t) ? P.cta_rng[h->cta] : 0;       // this CTA's ranges
    const int rg1 = (h->cta < P.grid_t) ? P.cta_rng[h->cta + 1] : 0;
    const unsigned long long t_start = global_ns();
    int s = (int)(it % (unsigned int)S);
    unsigned int ph = (it / (unsigned int)S) & 1u;

    if (warp >= W_CONS) {
        const uint64_t pol = policy_evict_first();
        if (warp == W_CONS && lane == 0) {
            for (int rg = rg0; rg < rg1; ++rg) {
                const int e0 = P.tr_range[rg].e_begin, e1 = P.tr_range[rg].e_end;
                for (int cs = e0; cs < e1; cs += CHUNK_T, ++it) {
                    mbar_wait(&h->empty_t[s], ph ^ 1u);
                    int n = e1 - cs;
                    n = n > CHUNK_T ? CHUNK_T : n;
                    unsigned char* st = stages + (size_t)s * (size_t)P.stage_t_bytes;
                    if (ID16) {
                        // packed stream: rows padded to 128 entries, so n is a multiple of 128 and everything is aligned;
                        // stage = values | 16-bit voxel offsets | one 32-bit base per 32 entries
                        mbar_expect_tx(&h->full_t[s], (uint32_t)n * 6u + (uint32_t)n / 8u);
                        bulk_g2s(st, P.valP + cs, (uint32_t)n * 4u, &h->full_t[s], pol);
                        bulk_g2s(st + CHUNK_T * 4, P.idP + cs, (uint32_t)n * 2u, &h->full_t[s], pol);
                        bulk_g2s(st + CHUNK_T * 6, P.baseP + cs / 32, (uint32_t)n / 8u, &h->full_t[s], pol);
                    } else {
                        const int shift = e0 & 3;   // 16-byte source alignment: start the copy up to 3 entries early
                        const uint32_t bytes = (uint32_t)((n + shift + 3) & ~3) * 4u;   // D^T is padded: always in bounds
                        int* col_s = reinterpret_cast<int*>(st);
                        float* val_s = reinterpret_cast<float*>(col_s + CHUNK_T_PAD);
                        mbar_expect_tx(&h->full_t[s], 2u * bytes);
                        bulk_g2s(col_s, P.colT + (cs - shift), bytes, &h->full_t[s], pol);
                        bulk_g2s(val_s, P.valT + (cs - shift), bytes, &h->full_t[s], pol);
                    }
                    if (++s == S) { s = 0; ph ^= 1u; }
                }
            }
        } else {
            for (int rg = rg0; rg < rg1; ++rg) {
                const int e0 = P.tr_range[rg].e_begin, e1 = P.tr_range[rg].e_end;
                it += (unsigned int)((e1 - e0 + CHUNK_T - 1) / CHUNK_T);
            }
        }
    } else {
        const uint64_t keep = policy_evict_last();
        for (int rg = rg0; rg < rg1; ++rg) {
            const TrRange R = P.tr_range[rg];
            for (int i = threadIdx.x; i < RL_MAX * W_CONS; i += N_CONS) wpart[i] = 0.0;
            named_bar_sync(1, N_CONS);
            int cur_row = R.first_row;
            int cur_end = __ldg(P.rowT_ptr + cur_row + 1);
            double dacc = 0.0;
            bool touched = false;
            for (int cs = R.e_begin; cs < R.e_end; cs += CHUNK_T, ++it) {
                if ((int)(it % TGROUPS) != warp / (W_CONS / TGROUPS)) {      // another group's stage: not consumed here, but
                    mbar_wait(&h->full_t[s], ph);      // its phase must be OBSERVED and the observation reported: the empty
                    if (lane == 0) mbar_arrive(&h->empty_t[s]);   // barrier counts all W_CONS warps, so the producer cannot
                    if (++s == S) { s = 0; ph ^= 1u; } // refill a slot before every warp has seen its phase complete
                    continue;
                }
                mbar_wait(&h->full_t[s], ph);
                const unsigned char* st = stages + (size_t)s * (size_t)P.stage_t_bytes;
                const int* col_s = reinterpret_cast<const int*>(st) + (R.e_begin & 3);
                const float* val_s = ID16 ? reinterpret_cast<const float*>(st)
                                          : reinterpret_cast<const float*>(st) + CHUNK_T_PAD + (R.e_begin & 3);
                const unsigned short* id_s = reinterpret_cast<const unsigned short*>(st + CHUNK_T * 4);
                const unsigned int* base_s = reinterpret_cast<const unsigned int*>(st + CHUNK_T * 6);
                const int ce = min(cs + CHUNK_T, R.e_end);
                int pos = cs + (warp % (W_CONS / TGROUPS)) * SLICE_T;
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
                    if (ID16) {
                        // pos and seg_end are multiples of 32 (rows are padded): whole 32-entry tiles, one base each
                        const unsigned short* ip = id_s + (pos - cs);
                        const unsigned int* bp = base_s + (pos - cs) / 32;
                        const int nt = (seg_end - pos) / 32;
                        if (nt == SLICE_T / 32) {
                            unsigned int c[SLICE_T / 32];
                            float rr[SLICE_T / 32];
#pragma unroll
                            for (int u = 0; u < SLICE_T / 32; ++u) c[u] = bp[u] + ip[lane + 32 * u];
#pragma unroll
                            for (int u = 0; u < SLICE_T / 32; ++u) rr[u] = ld_keep(r_in + c[u], keep);
#pragma unroll
                            for (int u = 0; u < SLICE_T / 32; ++u) acc = fmaf(vp[lane + 32 * u], rr[u], acc);
                        } else {
                            for (int u = 0; u < nt; ++u) acc = fmaf(vp[lane + 32 * u], ld_keep(r_in + (bp[u] + ip[lane + 32 * u]), keep), acc);
                        }
                    } else if (seg_end - pos == SLICE_T) {
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
    // (the slots become visible to the other CTAs through the release that follows: the grid barrier's, or the ticket's)
    __syncthreads();
    if (threadIdx.x == 0) {
        P.cta_ns[2048 + 2 * h->cta] = t_start;
        P.cta_ns[2048 + 2 * h->cta + 1] = global_ns();
    }
}

// The same pass over the ROW-PAIR stream (DevPlan::id16 == 2): an entry is one voxel of the union of two rows with a
// float2 of values, so one gather of r feeds two multiply-adds and every sum, partial and slot comes in twos.
template <bool STREAM = false>
__device__ __forceinline__ void transpose_pass_pairs(const DevPlan& P, SmemHeader* h, unsigned char* smem, double* wpart,
                                                     const float* __restrict__ r_in, double* gslot, Pipe& pipe) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int S = P.n_stages_t;
    unsigned char* stages = smem + P.tr_stage_off;
    unsigned int it = pipe.it_t;
    const int rg0 = (h->cta < P.grid_t) ? P.cta_rng[h->cta] : 0;
    const int rg1 = (h->cta < P.grid_t) ? P.cta_rng[h->cta + 1] : 0;
    const unsigned long long t_start = global_ns();
    int s = (int)(it % (unsigned int)S);
    unsigned int ph = (it / (unsigned int)S) & 1u;
    const float2* val2P = reinterpret_cast<const float2*>(P.valP);

    if (warp >= W_CONS) {
        const uint64_t pol = policy_evict_first();
        for (int rg = rg0; rg < rg1; ++rg) {
            const int e0 = P.tr_range[rg].e_begin, e1 = P.tr_range[rg].e_end;
            for (int cs = e0; cs < e1; cs += CHUNK_T, ++it) {
                if (warp == W_CONS && lane == 0) {
                    mbar_wait(&h->empty_t[s], ph ^ 1u);
                    const uint32_t n = (uint32_t)min(CHUNK_T, e1 - cs);    // a multiple of 128: everything stays aligned
                    unsigned char* st = stages + (size_t)s * (size_t)P.stage_t_bytes;
                    mbar_expect_tx(&h->full_t[s], n * 10u + n / 8u);
                    bulk_g2s(st, val2P + cs, n * 8u, &h->full_t[s], pol);
                    bulk_g2s(st + CHUNK_T * 8, P.idP + cs, n * 2u, &h->full_t[s], pol);
                    bulk_g2s(st + CHUNK_T * 10, P.baseP + cs / 32, n / 8u, &h->full_t[s], pol);
                }
                if (++s == S) { s = 0; ph ^= 1u; }
            }
        }
    } else {
        const uint64_t keep = policy_evict_last();
        for (int rg = rg0; rg < rg1; ++rg) {
            const TrRange R = P.tr_range[rg];
            for (int i = threadIdx.x; i < 2 * RL_MAX * W_CONS; i += N_CONS) wpart[i] = 0.0;
            named_bar_sync(1, N_CONS);
            int cur_row = R.first_row;
            int cur_end = __ldg(P.rowT_ptr + cur_row + 1);
            double dacc0 = 0.0, dacc1 = 0.0;
            bool touched = false;
            for (int cs = R.e_begin; cs < R.e_end; cs += CHUNK_T, ++it) {
                if ((int)(it % TGROUPS) != warp / (W_CONS / TGROUPS)) {      // another group's stage: not consumed here, but
                    mbar_wait(&h->full_t[s], ph);      // its phase must be OBSERVED and the observation reported: the empty
                    if (lane == 0) mbar_arrive(&h->empty_t[s]);   // barrier counts all W_CONS warps, so the producer cannot
                    if (++s == S) { s = 0; ph ^= 1u; } // refill a slot before every warp has seen its phase complete
                    continue;
                }
                mbar_wait(&h->full_t[s], ph);
                const unsigned char* st = stages + (size_t)s * (size_t)P.stage_t_bytes;
                const float2* val_s = reinterpret_cast<const float2*>(st);
                const unsigned short* id_s = reinterpret_cast<const unsigned short*>(st + CHUNK_T * 8);
                const unsigned int* base_s = reinterpret_cast<const unsigned int*>(st + CHUNK_T * 10);
                const int ce = min(cs + CHUNK_T, R.e_end);
                int pos = cs + (warp % (W_CONS / TGROUPS)) * SLICE_T;
                const int b = min(pos + SLICE_T, ce);
                while (!STREAM && pos < b) {
                    while (cur_end <= pos) {   // the slice moved past the end of the current row pair (warp-uniform)
                        if (touched) {
                            const double s0 = warp_sum(dacc0), s1 = warp_sum(dacc1);
                            if (lane == 0) {
                                wpart[2 * ((cur_row - R.first_row) * W_CONS + warp)] = s0;
                                wpart[2 * ((cur_row - R.first_row) * W_CONS + warp) + 1] = s1;
                            }
                            dacc0 = dacc1 = 0.0;
                            touched = false;
                        }
                        ++cur_row;
                        cur_end = __ldg(P.rowT_ptr + cur_row + 1);
                    }
                    const int seg_end = min(b, cur_end);
                    const float2* vp = val_s + (pos - cs);
                    const unsigned short* ip = id_s + (pos - cs);
                    const unsigned int* bp = base_s + (pos - cs) / 32;
                    const int nt = (seg_end - pos) / 32;       // whole 32-entry tiles: pairs are padded to 128 entries
                    float acc0 = 0.0f, acc1 = 0.0f;
                    if (nt == SLICE_T / 32) {
                        unsigned int c[SLICE_T / 32];
                        float rr[SLICE_T / 32];
#pragma unroll
                        for (int u = 0; u < SLICE_T / 32; ++u) c[u] = bp[u] + ip[lane + 32 * u];
#pragma unroll
                        for (int u = 0; u < SLICE_T / 32; ++u) rr[u] = ld_keep(r_in + c[u], keep);
#pragma unroll
                        for (int u = 0; u < SLICE_T / 32; ++u) {
                            const float2 v = vp[lane + 32 * u];
                            acc0 = fmaf(v.x, rr[u], acc0);
                            acc1 = fmaf(v.y, rr[u], acc1);
                        }
                    } else {
                        for (int u = 0; u < nt; ++u) {
                            const float rv = ld_keep(r_in + (bp[u] + ip[lane + 32 * u]), keep);
                            const float2 v = vp[lane + 32 * u];
                            acc0 = fmaf(v.x, rv, acc0);
                            acc1 = fmaf(v.y, rv, acc1);
                        }
                    }
                    dacc0 += (double)acc0;
                    dacc1 += (double)acc1;
                    touched = true;
                    pos = seg_end;
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(&h->empty_t[s]);
                if (++s == S) { s = 0; ph ^= 1u; }
            }
            if (touched) {
                const double s0 = warp_sum(dacc0), s1 = warp_sum(dacc1);
                if (lane == 0) {
                    wpart[2 * ((cur_row - R.first_row) * W_CONS + warp)] = s0;
                    wpart[2 * ((cur_row - R.first_row) * W_CONS + warp) + 1] = s1;
                }
            }
            named_bar_sync(1, N_CONS);
            for (int t = threadIdx.x; t < 2 * R.n_rows; t += N_CONS) {     // t = 2 * row + half
                double sum = 0.0;
#pragma unroll
                for (int w = 0; w < W_CONS; ++w) sum += wpart[2 * ((t >> 1) * W_CONS + w) + (t & 1)];
                gslot[2 * (size_t)R.slot_base + t] = sum;
            }
            named_bar_sync(1, N_CONS);
        }
    }
    pipe.it_t = it;
    // (the slots become visible to the other CTAs through the release that follows: the grid barrier's, or the ticket's)
    __syncthreads();
    if (threadIdx.x == 0) {
        P.cta_ns[2048 + 2 * h->cta] = t_start;
        P.cta_ns[2048 + 2 * h->cta + 1] = global_ns();
    }
}

__device__ __forceinline__ void transpose_pass(const DevPlan& P, SmemHeader* h, unsigned char* smem, double* wpart,
                                               const float* __restrict__ r_in, double* gslot, Pipe& pipe) {
    if (P.id16 == 2) transpose_pass_pairs<false>(P, h, smem, wpart, r_in, gslot, pipe);
    else if (P.id16) transpose_pass_rows<true>(P, h, smem, wpart, r_in, gslot, pipe);
    else transpose_pass_rows<false>(P, h, smem, wpart, r_in, gslot, pipe);
}

// g_i = sum of the slots of row i, in slot order (fixed).  All NTHREADS threads; g_out shared or global.
__device__ __forceinline__ void reduce_gradient(const DevPlan& P, const double* gslot, float* g_out) {
    constexpr int U = 4;         // rows per thread whose loads are issued together (the slots come from L2)
    const int pairs = (P.id16 == 2);      // row i of D^T is half `i & 1` of stream row i >> 1; a slot holds two sums
    for (int base = threadIdx.x; base < P.n_b; base += NTHREADS * U) {
        int s0[U], s1[U];
        double sum[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int i = base + u * NTHREADS;
            s0[u] = i < P.n_b ? __ldg(P.rowslot_ptr + (i >> pairs)) : 0;
            s1[u] = i < P.n_b ? __ldg(P.rowslot_ptr + (i >> pairs) + 1) : 0;
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int i = base + u * NTHREADS;
            sum[u] = s0[u] < s1[u] ? __ldcg(gslot + ((size_t)s0[u] << pairs) + (i & pairs)) : 0.0;
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int i = base + u * NTHREADS;
            for (int s = s0[u] + 1; s < s1[u]; ++s) sum[u] += __ldcg(gslot + ((size_t)s << pairs) + (i & pairs));   // slot order
            if (i < P.n_b) g_out[i] = (float)sum[u];
        }
    }
}

// ------------------------------------------------------------------------------------------------ row-sharded exchange
// rank q holds a slab of rows of D, computes a partial gradient over ALL beamlets and a partial
// objective; the path's two exchange steps are the sums of those over the ranks.  Every rank owns an INBOX; a rank
// PUSHES its partial into slot [rank] of every rank's inbox (remote stores over NVLink peer memory), then raises a
// sequence flag there with a system-scope release; every CTA of a rank spins on its OWN inbox's flags (local memory)
// and adds the world's partials in rank order -- the same order on every rank, so all ranks hold the same bits and take
// the same decisions without any broadcast.  Two buffers per exchange kind, selected by the sequence number's parity: a
// rank can be at most one exchange ahead of its slowest peer (it needs that peer's push to finish the current one).
//   inbox: flags_g u64[MAX_WORLD] | flags_G u64[MAX_WORLD] | G double[2][MAX_WORLD][R_MAX] | g float[2][world][nb_pad]
constexpr int INBOX_FLAGS_G = 0, INBOX_FLAGS_BIGG = 8 * MAX_WORLD, INBOX_BIGG = 16 * MAX_WORLD;
constexpr int INBOX_G = INBOX_BIGG + 8 * 2 * MAX_WORLD * R_MAX;
__host__ __device__ inline int inbox_nb_pad(int n_b) { return (n_b + 31) & ~31; }
__host__ __device__ inline size_t inbox_bytes(int n_b, int world) { return (size_t)INBOX_G + (size_t)2 * world * inbox_nb_pad(n_b) * 4; }

__device__ __forceinline__ void st_release_sys(unsigned long long* p, unsigned long long v) {
    asm volatile("st.release.sys.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ unsigned long long ld_acquire_sys(const unsigned long long* p) {
    unsigned long long v;
    asm volatile("ld.acquire.sys.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}

// Failure detection: a peer that never launched, died, or was given a different iteration count
// never raises its flag.  Every wait on an inbox flag is therefore bounded by State::spin_timeout_ns; a rank that gives
// up POISONS the exchange -- SHARD_POISON into its slot of every rank's flags and into all flags of its own inbox, so
// that its peers and its own other CTAs fall out of their waits at once instead of each sitting out the full timeout --
// and sets BAR_FAULT in its grid-barrier counter.  The inboxes must be zero-filled again before they are reused.
constexpr unsigned long long SHARD_POISON = ~0ull;
// true: the flag reached seq in time and is not poisoned
__device__ __forceinline__ bool shard_wait(const unsigned long long* f, unsigned long long seq, unsigned long long timeout_ns) {
    unsigned int polls = 0u;
    unsigned long long t0 = 0ull;
    for (;;) {
        const unsigned long long v = ld_acquire_sys(f);
        if (v >= seq) return v != SHARD_POISON;
        if ((++polls & 63u) == 0u) {
            const unsigned long long now = spin_clock_ns();
            if (t0 == 0ull) t0 = now;
            else if (now - t0 > timeout_ns) return false;
        }
    }
}
// Called by all threads of a CTA whose wait failed (block-uniform): tell everybody, remember it in h->fault.
__device__ __forceinline__ void shard_give_up(const DevPlan& P, SmemHeader* h) {
    if ((int)threadIdx.x < P.world) {
        const int q = threadIdx.x;
        st_release_sys(reinterpret_cast<unsigned long long*>(P.inbox[q] + INBOX_FLAGS_G) + P.rank, SHARD_POISON);
        st_release_sys(reinterpret_cast<unsigned long long*>(P.inbox[q] + INBOX_FLAGS_BIGG) + P.rank, SHARD_POISON);
        st_release_sys(reinterpret_cast<unsigned long long*>(P.inbox[P.rank] + INBOX_FLAGS_G) + q, SHARD_POISON);
        st_release_sys(reinterpret_cast<unsigned long long*>(P.inbox[P.rank] + INBOX_FLAGS_BIGG) + q, SHARD_POISON);
    }
    if (threadIdx.x == 0) {
        atomicOr(&P.st->gridbar, BAR_FAULT);
        h->fault = 1;
    }
    __syncthreads();
}

// g_s: this slab's partial gradient on entry (every CTA of the rank holds the same), the sum over the ranks on exit.
// fp32 partials, added in fp64 in rank order, rounded once.  All NTHREADS threads call it.  false: a peer did not answer.
__device__ __forceinline__ bool shard_sum_gradient(const DevPlan& P, SmemHeader* h, float* g_s, unsigned long long seq,
                                                   unsigned long long timeout_ns) {
    const int nbp = inbox_nb_pad(P.n_b), par = (int)(seq & 1ull);
    if (h->cta == 0) {
        for (int q = 0; q < P.world; ++q) {
            float* dst = reinterpret_cast<float*>(P.inbox[q] + INBOX_G) + (size_t)(par * P.world + P.rank) * nbp;
            for (int i = threadIdx.x; i < P.n_b; i += NTHREADS) dst[i] = g_s[i];
        }
        __threadfence_system();
        __syncthreads();
        if ((int)threadIdx.x < P.world)
            st_release_sys(reinterpret_cast<unsigned long long*>(P.inbox[threadIdx.x] + INBOX_FLAGS_G) + P.rank, seq);
    }
    bool ok = true;
    if ((int)threadIdx.x < P.world) {
        const unsigned long long* f = reinterpret_cast<const unsigned long long*>(P.inbox[P.rank] + INBOX_FLAGS_G) + threadIdx.x;
        ok = shard_wait(f, seq, timeout_ns);
    }
    if (__syncthreads_or(!ok)) { shard_give_up(P, h); return false; }
    const float* src = reinterpret_cast<const float*>(P.inbox[P.rank] + INBOX_G) + (size_t)par * P.world * nbp;
    for (int i = threadIdx.x; i < P.n_b; i += NTHREADS) {
        double sum = 0.0;
        for (int q = 0; q < P.world; ++q) sum += (double)__ldcg(src + (size_t)q * nbp + i);       // rank order
        g_s[i] = (float)sum;
    }
    __syncthreads();
    return true;
}

// G: this slab's R partial objectives on entry (the same in every thread of every CTA of the rank), the sums on exit.
// false: a peer did not answer.
template <int R>
__device__ __forceinline__ bool shard_sum_objective(const DevPlan& P, SmemHeader* h, double (&G)[R], unsigned long long seq,
                                                    unsigned long long timeout_ns) {
    const int par = (int)(seq & 1ull);
    if (h->cta == 0 && (int)threadIdx.x < P.world) {
        const int q = threadIdx.x;
        double* dst = reinterpret_cast<double*>(P.inbox[q] + INBOX_BIGG) + (size_t)(par * MAX_WORLD + P.rank) * R_MAX;
#pragma unroll
        for (int r = 0; r < R; ++r) dst[r] = G[r];
        st_release_sys(reinterpret_cast<unsigned long long*>(P.inbox[q] + INBOX_FLAGS_BIGG) + P.rank, seq);   // the same thread wrote the data
    }
    bool ok = true;
    if ((int)threadIdx.x < P.world) {
        const unsigned long long* f = reinterpret_cast<const unsigned long long*>(P.inbox[P.rank] + INBOX_FLAGS_BIGG) + threadIdx.x;
        ok = shard_wait(f, seq, timeout_ns);
    }
    if (__syncthreads_or(!ok)) { shard_give_up(P, h); return false; }
    const double* src = reinterpret_cast<const double*>(P.inbox[P.rank] + INBOX_BIGG) + (size_t)par * MAX_WORLD * R_MAX;
#pragma unroll
    for (int r = 0; r < R; ++r) {
        double sum = 0.0;
        for (int q = 0; q < P.world; ++q) sum += __ldcg(src + (size_t)q * R_MAX + r);              // rank order
        G[r] = sum;
    }
    return true;
}

// ------------------------------------------------------------------------------------------------ scalar logic
struct Loop {                  // the loop's scalar state, replicated in registers by the persistent kernel
    double G_k, lambda;
    int iter, m, stop_reason, xi, ri;
    long long fwd, tr;
    unsigned long long seq_g, seq_G;
};

// After a transpose pass of the loop: start the line search (PAPER.md:109 step 2).  Returns true if trials are pending.
// Called by all threads with identical arguments; x is global, g may be shared or global.
__device__ __forceinline__ bool begin_line_search(const State* st, Loop& L, const float* x, const float* g, int n_b, SmemHeader* h) {
    L.tr += 1;
    if (L.G_k == 0.0) { L.stop_reason = STOP_STATIONARY; return false; }   // reading R4
    L.lambda = st->lambda0;
    L.m = 0;
    if (first_step_sq(x, g, L.lambda, n_b, h) == 0.0) { L.stop_reason = STOP_STATIONARY; return false; }   // reading R4
    return true;
}

enum { DEC_ACCEPT_CONTINUE = 0, DEC_ACCEPT_STOP = 1, DEC_REJECT_RETRY = 2, DEC_REJECT_STOP = 3 };

// After a dose pass of the loop that evaluated the R trial points lambda, lambda/alpha, ...: steps 3-5 of PAPER.md:110-112
// applied to them IN ORDER, exactly as the one-trial-at-a-time loop would: Armijo test (Eq. (5)) on trial j; the first
// trial that passes is accepted (j_acc) and the later ones are ignored; each failure is one step 4.  Scalar work only.
// write_trace: only one CTA records.
template <int R>
__device__ __forceinline__ int armijo_decide(const DevPlan& P, const LoopConst& st, Loop& L, const double (&G_new)[R],
                                             const double (&step_sq)[R], bool write_trace, int& j_acc) {
    L.fwd += 1;
    j_acc = -1;
    double lam = L.lambda;
#pragma unroll
    for (int j = 0; j < R; ++j) {
        const double C = L.G_k - (st.eps / lam) * step_sq[j];       // Eq. (5)
        if (G_new[j] < C) {                                           // step 3, strict as printed
            const int k = L.iter;
            if (write_trace) {
                P.tr_obj[k + 1] = G_new[j];
                P.tr_lambda[k] = lam;
                P.tr_step_sq[k] = step_sq[j];
                P.tr_trials[k] = L.m + 1;
            }
            const double G_old = L.G_k;
            L.G_k = G_new[j];
            L.iter = k + 1;
            L.xi ^= 1;
            L.ri = (L.ri + 1 + j) % (R + 1);
            j_acc = j;
            if (st.delta_tol > 0.0 && (G_new[j] == 0.0 || fabs(G_new[j] - G_old) / G_new[j] < st.delta_tol)) {   // step 5
                L.stop_reason = STOP_TOLERANCE;
                return DEC_ACCEPT_STOP;
            }
            if (L.iter >= st.iter_target) { L.stop_reason = STOP_MAX_ITERS; return DEC_ACCEPT_STOP; }
            return DEC_ACCEPT_CONTINUE;
        }
        L.m += 1;                                                     // step 4
        if (L.m > st.max_ls) { L.stop_reason = STOP_LS_STALLED; return DEC_REJECT_STOP; }
        lam = lam / st.alpha;
    }
    L.lambda = lam;            // first step size of the next batch
    return DEC_REJECT_RETRY;
}

__device__ __forceinline__ void loop_load(const State* st, Loop& L) {
    L.G_k = st->G_k; L.lambda = st->lambda;
    L.iter = st->iter; L.m = st->m; L.stop_reason = st->stop_reason; L.xi = st->xi; L.ri = st->ri;
    L.fwd = st->fwd_passes; L.tr = st->tr_passes;
    L.seq_g = st->seq_g; L.seq_G = st->seq_G;
}
__device__ __forceinline__ void loop_store(State* st, const Loop& L) {
    st->G_k = L.G_k; st->lambda = L.lambda;
    st->iter = L.iter; st->m = L.m; st->stop_reason = L.stop_reason; st->xi = L.xi; st->ri = L.ri;
    st->fwd_passes = L.fwd; st->tr_passes = L.tr;
    st->seq_g = L.seq_g; st->seq_G = L.seq_G;
}

// Last-CTA election (threadfence reduction pattern).  The CTA's global writes are ordered before thread 0's fence by
// the bar.sync (the fence is cumulative), so no other thread needs a fence of its own; the last CTA's second fence is
// the acquire side (it also invalidates L1) before it reads the other CTAs' partials.
__device__ __forceinline__ bool cta_is_last(unsigned int* ticket, SmemHeader* h) {
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        const unsigned int t = atomicAdd(ticket, 1u);
        const int last = (t == (unsigned int)h->n_cta - 1u);
        if (last) { *ticket = 0u; __threadfence(); }
        h->flag = last;
    }
    __syncthreads();
    return h->flag != 0;
}

// x_{k+1} = trial point j of the batch: copy it from the gather array to global memory.
template <int R>
__device__ __forceinline__ void publish_x(const float* xs, int j, float* x_out, int n_b) {
    for (int i = threadIdx.x; i < n_b; i += NTHREADS) x_out[i] = xs[(size_t)i * R + j];
}

// ------------------------------------------------------------------------------------------------ kernels
extern __shared__ __align__(128) unsigned char imrt_smem[];

// The dose pass's ring schedule for the current partition: CTA c's blocks are walked in order; the walk places every
// record in a circular buffer of ring_bytes (end to end; a record that does not fit before the end starts over at
// 0) and notes how many earlier blocks must have left the ring first (at most RING_ENTRIES in flight).
// One warp per CTA of the dose pass: the lanes fetch the record sizes of 256 blocks at a time and write the results
// back (coalesced); lane 0 does the walk in shared memory.  The tail trails the head by at most RING_ENTRIES blocks,
// so a circular array of that many ring offsets is all the history the walk needs.
constexpr int RING_LAYOUT_CHUNK = 256;
__global__ void __launch_bounds__(32) k_ring_layout(int4* blk, const int* __restrict__ cta_blk, int grid_f, unsigned int ring_bytes) {
    __shared__ unsigned int at_s[RING_ENTRIES];
    __shared__ int bytes_s[RING_LAYOUT_CHUNK], w_s[RING_LAYOUT_CHUNK];
    __shared__ unsigned int z_s[RING_LAYOUT_CHUNK];
    const int c = blockIdx.x, lane = threadIdx.x;
    if (c >= grid_f) return;
    const int b0 = cta_blk[c], b1 = cta_blk[c + 1];
    unsigned int head = 0u;
    int tail = b0;
    for (int base = b0; base < b1; base += RING_LAYOUT_CHUNK) {
        const int n = min(RING_LAYOUT_CHUNK, b1 - base);
        for (int j = lane; j < n; j += 32) bytes_s[j] = blk[base + j].y;
        __syncwarp();
        if (lane == 0) {
            for (int j = 0; j < n; ++j) {
                const int b = base + j;
                const unsigned int bytes = (unsigned int)bytes_s[j];
                unsigned int at;
                for (;;) {
                    bool fits;
                    if (tail == b) { at = 0u; fits = true; }                 // nothing in flight
                    else {
                        const unsigned int t = at_s[(tail - b0) & (RING_ENTRIES - 1)];   // the oldest record in flight
                        if (head > t) {
                            if (head + bytes <= ring_bytes) { at = head; fits = true; }
                            else { at = 0u; fits = bytes <= t; }
                        } else { at = head; fits = head + bytes <= t; }
                    }
                    if (fits && b - tail < RING_ENTRIES) break;
                    ++tail;
                }
                head = at + bytes;
                at_s[(b - b0) & (RING_ENTRIES - 1)] = at;
                z_s[j] = at;
                w_s[j] = tail - b0;
            }
        }
        __syncwarp();
        for (int j = lane; j < n; j += 32) {
            blk[base + j].z = (int)z_s[j];
            blk[base + j].w = w_s[j];
        }
        __syncwarp();
    }
}

// A single-point dose pass (MODE_EVAL: eval / get_dose / timing; MODE_INIT: G(x_1), r(x_1)).  Uses the R = 1 path.
__device__ __forceinline__ void dose_single(const DevPlan& P, const PassArgs& A, SmemHeader* h, const float4* table_s, float* xs) {
    State* st = P.st;
    const int xi = st->xi, ri = st->ri;
    const int r_next = (ri + 1) % (P.R + 1);
    const float* x_in = A.x_in ? A.x_in : P.xbuf[xi];
    float* const r_out[1] = {A.mode == MODE_EVAL ? A.r_out : P.rbuf[r_next]};
    stage_point(x_in, xs, P.n_b);
    Pipe pipe = {0u, 0u};
    const int par = (int)(st->fwd_passes & 1);
    dose_pass<1>(P, h, imrt_smem, table_s, xs, r_out, A.mode == MODE_EVAL ? A.d_out : nullptr, P.Gpart[par], pipe);
    if (!cta_is_last(&st->ticket_f, h)) return;
    double G[1];
    reduce_objective<1>(P, P.Gpart[par], h, G, st->G_skip);
    if (threadIdx.x != 0) return;
    if (A.mode == MODE_EVAL) {
        st->eval_obj = G[0];            // not counted: fwd_passes / tr_passes count the loop's passes
    } else {
        st->G_k = G[0]; st->fwd_passes += 1; st->ri = r_next;   // xbuf[xi] already holds x_1
        st->G_is_local = P.world > 1;
        P.tr_obj[0] = G[0];
    }
}

// One batch of R line-search trials (graph / host drivers): every CTA builds the trial points itself.
template <int R>
__device__ __forceinline__ void dose_trials(const DevPlan& P, const PassArgs& A, SmemHeader* h, const float4* table_s, float* xs) {
    State* st = P.st;
    const int xi = st->xi, ri = st->ri;
    double step_sq[R];
    trial_batch<R>(P.xbuf[xi], P.g, st->lambda, st->alpha, xs, P.n_b, h, step_sq);
    __syncthreads();
    float* r_out[R];
#pragma unroll
    for (int j = 0; j < R; ++j) r_out[j] = P.rbuf[(ri + 1 + j) % (R + 1)];
    Pipe pipe = {0u, 0u};
    const int par = (int)(st->fwd_passes & 1);
    dose_pass<R>(P, h, imrt_smem, table_s, xs, r_out, nullptr, P.Gpart[par], pipe);
    if (!cta_is_last(&st->ticket_f, h)) return;

    // ---- the last CTA to finish takes the decision
    double G_new[R];
    const LoopConst C = loop_const(st);
    reduce_objective<R>(P, P.Gpart[par], h, G_new, C.G_skip);
    Loop L;
    loop_load(st, L);
    int j_acc;
    const int dec = armijo_decide<R>(P, C, L, G_new, step_sq, threadIdx.x == 0, j_acc);
    if (j_acc >= 0) publish_x<R>(xs, j_acc, P.xbuf[xi ^ 1], P.n_b);
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

// The loop's R-point dose pass on R copies of the current iterate, residuals to the trial buffers, no decision and no
// state change: what plan creation times to balance the partition and what imrt_plan_launch_pass launches.
template <int R>
__device__ __forceinline__ void dose_timing(const DevPlan& P, SmemHeader* h, const float4* table_s, float* xs) {
    State* st = P.st;
    const float* x = P.xbuf[st->xi];
    const int ri = st->ri;
    for (int i = threadIdx.x; i < P.n_b; i += NTHREADS) {
        const float v = x[i];
#pragma unroll
        for (int r = 0; r < R; ++r) xs[(size_t)i * R + r] = v;
    }
    __syncthreads();
    float* r_out[R];
#pragma unroll
    for (int j = 0; j < R; ++j) r_out[j] = P.rbuf[(ri + 1 + j) % (R + 1)];
    Pipe pipe = {0u, 0u};
    dose_pass<R>(P, h, imrt_smem, table_s, xs, r_out, nullptr, P.Gpart[(int)(st->fwd_passes & 1)], pipe);
}

// imrt_plan_eval_batch: the loop's R-point dose pass on R GIVEN points (A.x_in, [R][n_b]); residuals to A.r_out
// ([R][n_v]) or to the trial buffers; objectives to State::eval_objs.  No decision, no state change.
template <int R>
__device__ __forceinline__ void dose_batch(const DevPlan& P, const PassArgs& A, SmemHeader* h, const float4* table_s, float* xs) {
    State* st = P.st;
    const int ri = st->ri;
    for (int i = threadIdx.x; i < P.n_b; i += NTHREADS) {
#pragma unroll
        for (int r = 0; r < R; ++r) xs[(size_t)i * R + r] = A.x_in[(size_t)r * P.n_b + i];
    }
    __syncthreads();
    float* r_out[R];
#pragma unroll
    for (int j = 0; j < R; ++j) r_out[j] = A.r_out ? A.r_out + (size_t)j * P.n_v : P.rbuf[(ri + 1 + j) % (P.R + 1)];
    Pipe pipe = {0u, 0u};
    const int par = (int)(st->fwd_passes & 1);
    dose_pass<R>(P, h, imrt_smem, table_s, xs, r_out, nullptr, P.Gpart[par], pipe);
    if (!cta_is_last(&st->ticket_f, h)) return;
    double G[R];
    reduce_objective<R>(P, P.Gpart[par], h, G, st->G_skip);
    if (threadIdx.x == 0) {
#pragma unroll
        for (int r = 0; r < R; ++r) st->eval_objs[r] = G[r];
    }
}

// Dose pass as a kernel of its own (graph / host drivers, set_x, eval, get_dose).
__global__ void __launch_bounds__(NTHREADS, 1) k_dose(const __grid_constant__ DevPlan P, const PassArgs A) {
    SmemHeader* h = reinterpret_cast<SmemHeader*>(imrt_smem);
    float4* table_s = reinterpret_cast<float4*>(imrt_smem + SMEM_HEADER);
    float* xs = reinterpret_cast<float*>(imrt_smem + P.x_off);
    cta_init(h, P, table_s);
    if (A.mode == MODE_TIMING) {
        if (P.R == 4) dose_timing<4>(P, h, table_s, xs);
        else if (P.R == 2) dose_timing<2>(P, h, table_s, xs);
        else dose_timing<1>(P, h, table_s, xs);
    } else if (A.mode == MODE_BATCH) {
        if (A.n_points == 4) dose_batch<4>(P, A, h, table_s, xs);
        else if (A.n_points == 2) dose_batch<2>(P, A, h, table_s, xs);
        else dose_batch<1>(P, A, h, table_s, xs);
    } else if (A.mode != MODE_TRIAL) dose_single(P, A, h, table_s, xs);
    else if (P.R == 4) dose_trials<4>(P, A, h, table_s, xs);
    else if (P.R == 2) dose_trials<2>(P, A, h, table_s, xs);
    else dose_trials<1>(P, A, h, table_s, xs);
}

// The streaming ceilings of the two passes (imrt_plan_launch_pass kinds 2 and 3): every byte a pass reads travels
// through the same ring / stages, nobody computes.  kind 0: the dose pass's records; 1: the row-pair D^T stream.
__global__ void __launch_bounds__(NTHREADS, 1) k_stream(const __grid_constant__ DevPlan P, int kind) {
    SmemHeader* h = reinterpret_cast<SmemHeader*>(imrt_smem);
    float4* table_s = reinterpret_cast<float4*>(imrt_smem + SMEM_HEADER);
    float* xs = reinterpret_cast<float*>(imrt_smem + P.x_off);
    cta_init(h, P, table_s);
    Pipe pipe = {0u, 0u};
    if (kind == 0) {
        float* r_out[1] = {nullptr};
        dose_pass<1, true>(P, h, imrt_smem, table_s, xs, r_out, nullptr, P.Gpart[0], pipe);
    } else if (P.id16 == 2) {
        transpose_pass_pairs<true>(P, h, imrt_smem, reinterpret_cast<double*>(imrt_smem + P.wpart_off), P.rbuf[0], P.gslot[0], pipe);
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
    const bool pending = begin_line_search(st, L, P.xbuf[xi], P.g, P.n_b, h);
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
    st->clamped = target > st->trace_cap;
    if (target > st->trace_cap) target = st->trace_cap;
    st->iter_target = target;
    st->delta_tol = delta_tol;
    st->gridbar = 0u;
}

// The whole loop in one cooperative launch (driver 2): PAPER.md:99-114 with no host involvement at all.
// Every CTA keeps g and the trial points in shared memory and replays the same scalar decisions from the same
// fixed-order reductions, so CTAs never exchange anything but the pass partials; CTA 0 records the trace and
// publishes the accepted iterate.
template <int R>
__device__ __forceinline__ void persistent_loop(const DevPlan& P, int cta, int n_cta) {
    SmemHeader* h = reinterpret_cast<SmemHeader*>(imrt_smem);
    float4* table_s = reinterpret_cast<float4*>(imrt_smem + SMEM_HEADER);
    double* wpart = reinterpret_cast<double*>(imrt_smem + P.wpart_off);
    float* xs = reinterpret_cast<float*>(imrt_smem + P.x_off);     // the R trial points (the dose pass gathers from them)
    float* g_s = reinterpret_cast<float*>(imrt_smem + P.g_off);
    State* st = P.st;
    if (st->fault) return;                 // a wait of an earlier launch gave up: nothing runs until imrt_plan_set_x
    cta_init(h, P, table_s, cta, n_cta);
    if (threadIdx.x == 0) h->lc = loop_const(st);
    __syncthreads();
    const LoopConst& C = h->lc;
    // h->fault (shared, block-uniform after every wait): a bounded wait gave up -- leave without touching another barrier
    Loop L;
    loop_load(st, L);
    const int iter_target = C.iter_target;
    const double alpha = C.alpha;
    L.stop_reason = STOP_MAX_ITERS;
    const bool sharded = P.world > 1;
    if (sharded && st->G_is_local) {       // G(x_1) of imrt_plan_set_x is this slab's share: make it the sum over the ranks
        double G1[1] = {L.G_k};
        const bool ok = shard_sum_objective<1>(P, h, G1, ++L.seq_G, C.spin_timeout_ns);
        L.G_k = G1[0];
        if (ok && h->cta == 0 && threadIdx.x == 0) P.tr_obj[0] = G1[0];
    }
    Pipe pipe = {0u, 0u};
    unsigned int epoch = 0;
    const bool rec = (h->cta == 0) && (threadIdx.x == 0);

    bool g_valid = false;                  // g_s holds the gradient of the current iterate (a transpose pass ran in this launch)
    while (!h->fault && L.iter < iter_target) {
        const int tpar = (int)(L.tr & 1);
        // The transpose stages overlay xs and g_s (DevPlan::tr_stage_off = x_off).  Everybody is done with both -- the
        // publish loop below read xs, trial_batch / reduce_gradient wrote them through the generic proxy -- before the
        // producer warp lets the TMA unit write over them: proxy fence in every thread, then a CTA barrier.
        fence_proxy_async_smem();
        __syncthreads();
        transpose_pass(P, h, imrt_smem, wpart, P.rbuf[L.ri], P.gslot[tpar], pipe);
        if (grid_barrier(&st->gridbar, epoch, h->n_cta, C.spin_timeout_ns, &h->fault)) break;
        reduce_gradient(P, P.gslot[tpar], g_s);
        g_valid = true;
        __syncthreads();
        if (sharded && !shard_sum_gradient(P, h, g_s, ++L.seq_g, C.spin_timeout_ns)) break;   // exchange step 1: g = sum over the row slabs
        // start of the line search (PAPER.md:109 step 2; the same decisions begin_line_search takes, with the first
        // trial's Delta taken from the batch that is built anyway).  x_k lives in global memory.
        L.tr += 1;
        if (L.G_k == 0.0) { L.stop_reason = STOP_STATIONARY; break; }          // reading R4
        L.lambda = C.lambda0;
        L.m = 0;
        int dec, j_acc = -1;
        for (;;) {
            double step_sq[R], G_new[R];
            trial_batch<R>(P.xbuf[L.xi], g_s, L.lambda, alpha, xs, P.n_b, h, step_sq);
            if (L.m == 0 && step_sq[0] == 0.0) { L.stop_reason = STOP_STATIONARY; dec = DEC_REJECT_STOP; break; }   // reading R4
            __syncthreads();
            float* r_out[R];
#pragma unroll
            for (int j = 0; j < R; ++j) r_out[j] = P.rbuf[(L.ri + 1 + j) % (R + 1)];
            const int fpar = (int)(L.fwd & 1);
            dose_pass<R>(P, h, imrt_smem, table_s, xs, r_out, nullptr, P.Gpart[fpar], pipe);
            if (grid_barrier(&st->gridbar, epoch, h->n_cta, C.spin_timeout_ns, &h->fault)) { dec = DEC_REJECT_STOP; break; }
            reduce_objective<R>(P, P.Gpart[fpar], h, G_new, C.G_skip);
            if (sharded && !shard_sum_objective<R>(P, h, G_new, ++L.seq_G, C.spin_timeout_ns)) {      // exchange step 2: G = sum over the row slabs
                dec = DEC_REJECT_STOP; break;
            }
            dec = armijo_decide<R>(P, C, L, G_new, step_sq, rec, j_acc);
            if (dec != DEC_REJECT_RETRY) break;
        }
        if (j_acc >= 0) {
            // x_{k+1}: publish it (L.xi already points at the new buffer).  Every CTA holds all of it and writes one slice,
            // so no CTA enters the next pass late; the others read it only after the next grid barrier.
            const int per = ((P.n_b + h->n_cta - 1) / h->n_cta + 31) & ~31;
            const int i0 = h->cta * per, i1 = min(P.n_b, i0 + per);
            float* x_out = P.xbuf[L.xi];
            for (int i = i0 + (int)threadIdx.x; i < i1; i += NTHREADS) x_out[i] = xs[(size_t)i * R + j_acc];
        }
        if (dec != DEC_ACCEPT_CONTINUE) break;
    }
    // every CTA has passed the last grid barrier before CTA 0 gets here with a changed state
    if (!h->fault) grid_barrier(&st->gridbar, epoch, h->n_cta, C.spin_timeout_ns, &h->fault);
    if (h->fault) {
        // Failure exit: some CTA of this rank, or a peer rank, did not show up within the bound.  The
        // iterate buffers may be half written: the plan refuses to run until the next imrt_plan_set_x (State::fault).
        if (h->cta == 0 && threadIdx.x == 0) {
            st->fault = 1;
            st->stop_reason = STOP_PEER_TIMEOUT;
            st->cont_outer = 0;
            st->cont_inner = 0;
        }
        return;
    }
    if (h->cta == 0) {
        if (g_valid)                       // a launch that did no iteration leaves P.g as it was
            for (int i = threadIdx.x; i < P.n_b; i += NTHREADS) P.g[i] = g_s[i];
        if (threadIdx.x == 0) {
            loop_store(st, L);
            st->cont_outer = 0;
            st->cont_inner = 0;
            st->G_is_local = 0;
        }
    }
}

__global__ void __launch_bounds__(NTHREADS, 1) k_persistent(const __grid_constant__ DevPlan P) {
    if (P.R == 4) persistent_loop<4>(P, (int)blockIdx.x, (int)gridDim.x);
    else if (P.R == 2) persistent_loop<2>(P, (int)blockIdx.x, (int)gridDim.x);
    else persistent_loop<1>(P, (int)blockIdx.x, (int)gridDim.x);
}

// Several ranks of a row-sharded problem CO-RESIDENT on one device: one cooperative launch, rank q = the CTAs
// [q ctas_per_rank, (q + 1) ctas_per_rank), each running the loop of its own plan and exchanging with the others through
// their inboxes exactly as ranks on different GPUs do.  (Ranks that wait on one another must share ONE cooperative
// launch on a single device: separate launches are not guaranteed to run at the same time.)
static_assert(sizeof(SmemHeader) + sizeof(DevPlan) <= SMEM_HEADER, "the header region also holds a plan");
__global__ void __launch_bounds__(NTHREADS, 1) k_persistent_ranks(const DevPlan* __restrict__ plans, int ctas_per_rank) {
    DevPlan* Ps = reinterpret_cast<DevPlan*>(imrt_smem + sizeof(SmemHeader));
    const int rank = (int)blockIdx.x / ctas_per_rank, cta = (int)blockIdx.x % ctas_per_rank;
    {
        const int* src = reinterpret_cast<const int*>(plans + rank);
        int* dst = reinterpret_cast<int*>(Ps);
        for (int i = threadIdx.x; i < (int)(sizeof(DevPlan) / 4); i += NTHREADS) dst[i] = src[i];
        __syncthreads();
    }
    const DevPlan& P = *Ps;
    if (P.R == 4) persistent_loop<4>(P, cta, ctas_per_rank);
    else if (P.R == 2) persistent_loop<2>(P, cta, ctas_per_rank);
    else persistent_loop<1>(P, cta, ctas_per_rank);
}

}  // namespace imrt
