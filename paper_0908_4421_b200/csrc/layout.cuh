// layout.cuh -- plan creation on the device: validation of the row structure and the layout of the dose pass's block
// records (which rows / quads go into which record, record sizes and offsets, headers and row tables).
//
// The layout is decided independently per segment of SEG_ROWS rows (a record never crosses a segment), greedily from
// the first row to the last, so one thread per segment walks its rows twice: a COUNT pass (records, table words, bytes
// per segment), an exclusive scan over the segments, and a WRITE pass that repeats the walk and emits block
// descriptors, pack descriptors, headers, row tables, the covered[] flags and a modelled cost per record.  Nothing but
// a handful of totals ever travels to the host.  (DevPlan::pack in kernels.cuh documents the record formats.)
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "kernels.cuh"

namespace imrt {

struct RecordCaps {
    int chunk_slots;   // row format: slots per record
    int max_rows;      // row format: rows per record
    int quad_cap;      // quad format: union columns per record
    int quad_max;      // quad format: union columns of ONE quad at most (a longer one goes to row-format records)
};

struct LayoutTotals {          // device -> host, once
    int n_blk, n_meta, pack128;           // records, table words, bytes / 128 of the packed stream
    int n_skipped, n_nonempty, n_quad_rows;
    int max_rec_bytes;
    int bad_row_ptr;                      // 1: row_ptr[0] != 0, row_ptr decreases somewhere, or row_ptr[n_v] != nnz
    int bad_row;                          // first row where row_ptr decreases / that is too long (diagnostics)
    int bad_sid;                          // 1 + first row whose structure id is out of range, or 0
    int long_row;                         // 1 + a row with more than MAX_CHUNK_SLOTS entries, or 0
    int max_row_len;
};

// row_ptr monotone, structure ids in range, longest row.  flags -> LayoutTotals.
__global__ void k_validate_structure(const int* __restrict__ row_ptr, const uint8_t* __restrict__ sid, int n_v, long long nnz,
                                     int n_structures, LayoutTotals* T) {
    int max_len = 0;
    for (int j = blockIdx.x * blockDim.x + threadIdx.x; j < n_v; j += gridDim.x * blockDim.x) {
        const int a = row_ptr[j], b = row_ptr[j + 1];
        if (b < a) { T->bad_row_ptr = 1; T->bad_row = j; }
        if ((int)sid[j] >= n_structures) atomicMax(&T->bad_sid, j + 1);
        max_len = max(max_len, b - a);
        if (b - a > MAX_CHUNK_SLOTS) atomicMax(&T->long_row, j + 1);
    }
    if (blockIdx.x == 0 && threadIdx.x == 0 && (row_ptr[0] != 0 || (long long)row_ptr[n_v] != nnz)) T->bad_row_ptr = 1;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) max_len = max(max_len, __shfl_xor_sync(0xffffffffu, max_len, o));
    if ((threadIdx.x & 31) == 0 && max_len > 0) atomicMax(&T->max_row_len, max_len);
}

struct SegCount { int n_rec, n_meta, b128; };

// What the WRITE pass emits per record.
struct LayoutOut {
    int4* blk;                 // {record offset / 128, record bytes, 0, 0}
    int4* pk;                  // {table word offset, table words, record offset / 128, format}
    uint32_t* meta;            // headers + row tables, record after record
    long long* cost_fx;        // modelled cost of every record, fixed point (x 1024)
    unsigned char* covered;
};

__device__ __forceinline__ int pad4i(int n) { return (n + 3) & ~3; }

// The greedy walk over one segment.  WRITE = false: only counts.  Returns the counts; the WRITE pass starts from the
// segment's scanned offsets (rec0, meta0, off128).
template <bool WRITE>
__device__ __forceinline__ SegCount layout_segment(int seg, const int* __restrict__ rp, const uint8_t* __restrict__ sid, const int* __restrict__ quadU,
                                                   int n_v, RecordCaps caps, int col_bytes, int rec0, int meta0, int off128, const LayoutOut& O,
                                                   int& n_skipped, int& n_nonempty, int& n_quad_rows, int& max_rec) {
    const int seg0 = seg * SEG_ROWS, seg1 = min(n_v, seg0 + SEG_ROWS);
    SegCount C = {0, 0, 0};
    int rec = rec0, mo = meta0, off = off128;
    auto skip_row = [&](int j) {
        ++n_skipped;
        if (WRITE) O.covered[j] = 0;
    };
    auto close_record = [&](int mw_used, int payload_bytes, int fmt, int rows, int slots) {
        const int mw = META_HDR + ((mw_used - META_HDR + 3) & ~3);       // the table is padded to a multiple of 4 words
        const int bytes = (mw * 4 + payload_bytes + 127) & ~127;
        if (WRITE) {
            for (int t = mw_used; t < mw; ++t) O.meta[mo + t] = 0u;
            O.blk[rec] = make_int4(off, bytes, 0, 0);
            O.pk[rec] = make_int4(mo, mw, off, fmt);
            // cost of a block in SM cycles: the slower of streaming its bytes at a 1/n_sm share of HBM bandwidth and of
            // issuing its instructions (per-row work dominates where rows are short); refined by tune_partition()
            const double c = fmax(bytes / 22.4, 130.0 + 18.0 * rows + 0.08 * slots);
            O.cost_fx[rec] = (long long)(c * 1024.0 + 0.5);
        }
        max_rec = max(max_rec, bytes);
        ++rec; mo += mw; off += bytes / 128;
        ++C.n_rec; C.n_meta += mw; C.b128 += bytes / 128;
    };
    // ---- which format is smaller on this segment
    long long bytes_rows = 0, bytes_quads = 0;
    for (int j = seg0; j < seg1; ++j) {
        const int len = rp[j + 1] - rp[j];
        if (len > 0) { bytes_rows += (long long)pad4i(len) * (4 + col_bytes) + 4; ++n_nonempty; }
    }
    bool quads = quadU != nullptr && bytes_rows > 0;
    if (quads) {
        bool fits = true;
        for (int q = seg0 / 4; q < (seg1 + 3) / 4; ++q)
            if (quadU[q] > 0) { bytes_quads += (long long)quadU[q] * 18 + 8; fits = fits && quadU[q] <= caps.quad_max; }
        quads = fits && bytes_quads < bytes_rows;
    }
    if (!quads) {
        // ---- row-format records
        int j = seg0;
        while (j < seg1) {
            if (rp[j + 1] == rp[j]) { skip_row(j); ++j; continue; }
            const int r0 = j;
            int slots = pad4i(rp[j + 1] - rp[j]);       // a row longer than the cap gets a record of its own
            int last = j, empties = 0, jj = j + 1;
            while (jj < seg1 && jj - r0 < caps.max_rows) {
                const int len = rp[jj + 1] - rp[jj];
                if (len == 0) {
                    if (++empties > 32) break;
                    ++jj;
                    continue;
                }
                if (slots + pad4i(len) > caps.chunk_slots) break;
                slots += pad4i(len);
                empties = 0;
                last = jj;
                ++jj;
            }
            const int r1 = last + 1, nrows = r1 - r0;
            if (WRITE) {
                uint32_t* m = O.meta + mo;
                m[0] = (uint32_t)nrows; m[1] = (uint32_t)r0; m[2] = 0u; m[3] = (uint32_t)slots;
                int so = 0;
                for (int row = r0; row < r1; ++row) {
                    m[META_HDR + row - r0] = (uint32_t)so | ((uint32_t)sid[row] << 16);
                    so += pad4i(rp[row + 1] - rp[row]);
                }
                m[META_HDR + nrows] = (uint32_t)so;
            }
            close_record(META_HDR + nrows + 1, (slots + ZPAD) * (4 + col_bytes), 0, nrows, slots);
            j = r1;
        }
    } else {
        // ---- quad-format records
        int q = seg0 / 4;
        const int q_end = (seg1 + 3) / 4;
        auto skip_quad = [&](int qq) { for (int j = 4 * qq; j < min(n_v, 4 * qq + 4); ++j) skip_row(j); };
        while (q < q_end) {
            if (quadU[q] == 0) { skip_quad(q); ++q; continue; }
            const int q0 = q;
            int cols = quadU[q];
            int last = q, empties = 0, qq = q + 1;
            while (qq < q_end && qq - q0 < QUAD_MAXQ) {
                if (quadU[qq] == 0) {
                    if (++empties > 8) break;
                    ++qq;
                    continue;
                }
                if (cols + quadU[qq] > caps.quad_cap) break;
                cols += quadU[qq];
                empties = 0;
                last = qq;
                ++qq;
            }
            int q1 = last + 1, nq = q1 - q0;
            if (nq > 2 && (nq & 1)) {             // a warp takes two quads at a time: keep the pairs full
                cols -= quadU[q1 - 1];
                q1 -= 1;
                nq = q1 - q0;
            }
            int rows_here = 0;
            for (int t = q0; t < q1; ++t) rows_here += min(4, n_v - 4 * t);
            if (WRITE) {
                uint32_t* m = O.meta + mo;
                m[0] = (uint32_t)nq; m[1] = (uint32_t)(4 * q0); m[2] = 1u; m[3] = (uint32_t)cols;
                int co = 0;
                for (int t = q0; t < q1; ++t) {
                    uint32_t mask = 0u, sids = 0u;
                    for (int i = 0; i < 4; ++i)
                        if (4 * t + i < n_v) { mask |= 1u << i; sids |= (uint32_t)sid[4 * t + i] << (8 * i); }
                    m[META_HDR + 2 * (t - q0)] = (uint32_t)co | (mask << 16);
                    m[META_HDR + 2 * (t - q0) + 1] = sids;
                    co += quadU[t];
                }
                m[META_HDR + 2 * nq] = (uint32_t)co;
                m[META_HDR + 2 * nq + 1] = 0u;
            }
            close_record(META_HDR + 2 * (nq + 1), (cols + 1) * 16 + (cols + 8) * 2, 1, rows_here, 4 * cols);
            n_quad_rows += rows_here;
            q = q1;
            for (; q < q_end && quadU[q] == 0; ++q) skip_quad(q);   // trailing empties of the run belong to no record
        }
    }
    return C;
}

__global__ void k_layout_count(const int* __restrict__ rp, const uint8_t* __restrict__ sid, const int* __restrict__ quadU, int n_v, int n_seg,
                               RecordCaps caps, int col_bytes, int* seg_rec, int* seg_meta, int* seg_b128, LayoutTotals* T) {
    int n_skipped = 0, n_nonempty = 0, n_quad_rows = 0, max_rec = 0;
    for (int seg = blockIdx.x * blockDim.x + threadIdx.x; seg < n_seg; seg += gridDim.x * blockDim.x) {
        LayoutOut none = {};
        const SegCount C = layout_segment<false>(seg, rp, sid, quadU, n_v, caps, col_bytes, 0, 0, 0, none, n_skipped, n_nonempty, n_quad_rows, max_rec);
        seg_rec[seg] = C.n_rec; seg_meta[seg] = C.n_meta; seg_b128[seg] = C.b128;
    }
    if (n_skipped) atomicAdd(&T->n_skipped, n_skipped);
    if (n_nonempty) atomicAdd(&T->n_nonempty, n_nonempty);
    if (n_quad_rows) atomicAdd(&T->n_quad_rows, n_quad_rows);
    if (max_rec) atomicMax(&T->max_rec_bytes, max_rec);
}

// seg_* hold the EXCLUSIVE scans now ([n_seg + 1], the totals in the last entry)
__global__ void k_layout_write(const int* __restrict__ rp, const uint8_t* __restrict__ sid, const int* __restrict__ quadU, int n_v, int n_seg,
                               RecordCaps caps, int col_bytes, const int* __restrict__ seg_rec, const int* __restrict__ seg_meta,
                               const int* __restrict__ seg_b128, LayoutOut O, LayoutTotals* T) {
    int a = 0, b = 0, c = 0, d = 0;
    for (int seg = blockIdx.x * blockDim.x + threadIdx.x; seg < n_seg; seg += gridDim.x * blockDim.x)
        layout_segment<true>(seg, rp, sid, quadU, n_v, caps, col_bytes, seg_rec[seg], seg_meta[seg], seg_b128[seg], O, a, b, c, d);
    if (blockIdx.x == 0 && threadIdx.x == 0) { T->n_blk = seg_rec[n_seg]; T->n_meta = seg_meta[n_seg]; T->pack128 = seg_b128[n_seg]; }
}

// Contiguous block ranges of (nearly) equal total cost, one per CTA: cta_blk[c] = the first block whose exclusive cost
// prefix reaches c / grid of the total.  pre: EXCLUSIVE scan of cost_fx, [n_blk + 1].
__global__ void k_partition(const long long* __restrict__ pre, int n_blk, int grid, int* cta_blk) {
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c > grid) return;
    if (c == grid) { cta_blk[c] = n_blk; return; }
    const long long total = pre[n_blk];
    // want = total * c / grid without overflow (total < 2^53 in practice; use 128-bit-safe split)
    const long long want = (total / grid) * c + ((total % grid) * c) / grid;
    int lo = 0, hi = n_blk;
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if (pre[mid] < want) lo = mid + 1; else hi = mid;
    }
    cta_blk[c] = lo;
}

}  // namespace imrt
