// frnn_kernels.cuh -- device code of the B200 FRNN path (sm_100a).  Product code: shares nothing
// with oracle/.  Steps S2..S10 of SURVEY.md section 8(a); design notes in DESIGN.md section 6.
//
//   bin_kernel      S2     cell index on a toroidal grid over the first G coordinates + histogram
//   cell_scan_kernel S3    cell starts + list of occupied cells ("segments"); blocks take their base
//                          from one atomic (no inter-block wait), rows of the table are padded so a
//                          run never needs the next block's start
//   scatter_kernel  S4     counting-sort scatter into the cell-ordered copy
//   search_kernel   S5-S7  ONE pass: a warp per occupied cell, neighbour runs flattened across
//                          lanes, whole 8-term FMA chains per lane; hits go to a per-row slot buffer
//   emit_kernel     S8-S10 degree scan (decoupled look-back) fused with the per-row ordering by dst
//                          and the compaction into the (src,dst)-sorted COO; exact K-cap selection
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace frnn {

constexpr int kDim = 8;
constexpr unsigned kFull = 0xffffffffu;

// ------------------------------------------------------------------------------------------------
// Grid geometry.  Cell coordinate of x along a binned dim:  floor(clamp(x * inv_cell)) mod 2^bits.
// inv_cell = 1 / (r * (1 + 2^-7)): the slack makes |x-y| <= r(1+1e-6) imply floor difference <= 1
// even after the fp32 rounding of x*inv_cell for |x*inv_cell| <= 2^15 (R9); clamping is
// monotone, so points beyond +-2^15 cells only pile up in the boundary cells (slower, still exact).
// The modulo (toroidal wrap) only ever ADDS candidates: far-apart points may share a cell, the
// full-D distance test rejects them.
//
// Linear cell id  lin = (((event << bits | c0) << bits | c1) ...) << bits | c_last.
// Table index     pid = lin + (lin >> bits): every row of 2^bits cells along the last coordinate
// is followed by one padding entry whose count is 0, so after the exclusive scan it holds the END
// of the row and  [start[pid(lo)], start[pid(hi) + 1])  is a valid run for any lo <= hi in the row.
// ------------------------------------------------------------------------------------------------
constexpr float kCoordClamp = 32768.0f;

__device__ __forceinline__ uint32_t cell_coord(float x, float inv_cell, uint32_t mask) {
    float a = __fmul_rn(x, inv_cell);
    a = fminf(fmaxf(a, -kCoordClamp), kCoordClamp);   // NaN -> -clamp: never out of bounds
    return static_cast<uint32_t>(__float2int_rd(a)) & mask;
}

template <int G>
__device__ __forceinline__ uint32_t cell_of_point(const float4& a, const float4& b, uint32_t event, float inv_cell, int bits) {
    const uint32_t mask = (1u << bits) - 1u;
    const float x[8] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w};
    uint32_t lin = event;
#pragma unroll
    for (int d = 0; d < G; ++d) lin = (lin << bits) | cell_coord(x[d], inv_cell, mask);
    return lin;
}

__device__ __forceinline__ uint32_t padded(uint32_t lin, int bits) { return lin + (lin >> bits); }

// DESIGN.md R3: the pinned fp32 order.  Explicit rounding intrinsics: nvcc may not contract,
// reassociate or reorder them.  Each lane runs the whole chain for one (query, candidate) pair.
__device__ __forceinline__ float d2_pinned(const float4& qa, const float4& qb, const float4& ca, const float4& cb) {
    float t, acc;
    t = __fsub_rn(qa.x, ca.x); acc = __fmaf_rn(t, t, 0.0f);
    t = __fsub_rn(qa.y, ca.y); acc = __fmaf_rn(t, t, acc);
    t = __fsub_rn(qa.z, ca.z); acc = __fmaf_rn(t, t, acc);
    t = __fsub_rn(qa.w, ca.w); acc = __fmaf_rn(t, t, acc);
    t = __fsub_rn(qb.x, cb.x); acc = __fmaf_rn(t, t, acc);
    t = __fsub_rn(qb.y, cb.y); acc = __fmaf_rn(t, t, acc);
    t = __fsub_rn(qb.z, cb.z); acc = __fmaf_rn(t, t, acc);
    t = __fsub_rn(qb.w, cb.w); acc = __fmaf_rn(t, t, acc);
    return acc;
}

__device__ __forceinline__ int event_of_row(const int64_t* __restrict__ ev_off, int n_events, int64_t row) {
    int lo = 0, hi = n_events;                 // largest e with ev_off[e] <= row
    while (hi - lo > 1) {
        int mid = (lo + hi) >> 1;
        if (ev_off[mid] <= row) lo = mid; else hi = mid;
    }
    return lo;
}

// Host event offsets travel as kernel arguments, kN at a time.
struct OffsetChunk {
    static constexpr int kN = 128;
    int first, count;
    int64_t v[kN];
};
__global__ void set_offsets_kernel(OffsetChunk c, int64_t* __restrict__ ev_off) {
    if (static_cast<int>(threadIdx.x) < c.count) ev_off[c.first + threadIdx.x] = c.v[threadIdx.x];
}

// ------------------------------------------------------------------------------------------------
// S2: cell index + histogram.  The atomicAdd's return value is the point's rank inside its cell,
// which makes the later scatter a pure function of (cell_start, rank): no second atomic pass.
// ------------------------------------------------------------------------------------------------
template <int G>
__global__ void __launch_bounds__(256) bin_kernel(const float4* __restrict__ pts, int64_t n_total,
                                                  const int64_t* __restrict__ ev_off, int n_events,
                                                  float inv_cell, int bits,
                                                  uint32_t* __restrict__ cell_count,
                                                  uint32_t* __restrict__ pcell, uint32_t* __restrict__ prank) {
    const int64_t i = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (i >= n_total) return;
    const float4 a = pts[2 * i];
    float4 b = make_float4(0.f, 0.f, 0.f, 0.f);
    if (G > 4) b = pts[2 * i + 1];
    const uint32_t ev = ev_off ? static_cast<uint32_t>(event_of_row(ev_off, n_events, i)) : 0u;
    const uint32_t pid = padded(cell_of_point<G>(a, b, ev, inv_cell, bits), bits);
    pcell[i] = pid;
    prank[i] = atomicAdd(&cell_count[pid], 1u);
}

// ------------------------------------------------------------------------------------------------
// S4: counting-sort scatter.  Order inside a cell is the (arbitrary) atomic order; the final
// result does not depend on it because every row is ordered by dst at the end.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) scatter_kernel(const float4* __restrict__ pts, int64_t n_total,
                                                      const uint32_t* __restrict__ cell_start,
                                                      const uint32_t* __restrict__ pcell,
                                                      const uint32_t* __restrict__ prank,
                                                      float4* __restrict__ spts, int32_t* __restrict__ sidx) {
    const int64_t i = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (i >= n_total) return;
    const uint32_t s = cell_start[pcell[i]] + prank[i];
    const float4 a = pts[2 * i], b = pts[2 * i + 1];
    spts[2 * static_cast<int64_t>(s)] = a;
    spts[2 * static_cast<int64_t>(s) + 1] = b;
    sidx[s] = static_cast<int32_t>(i);
}

// ------------------------------------------------------------------------------------------------
// S3: cell starts.  Each block owns a few WHOLE padded rows of the table (about 4096 entries),
// computes its total, reserves its range of the cell-ordered copy with ONE 64-bit atomicAdd that
// packs (occupied cells << 32 | points), then scans its rows in strips of 1024.  Blocks land in
// arrival order: no inter-block wait, and since a run only ever reads start[lo] and start[hi+1] of
// one row (the padding entry holds the row's end) nothing depends on the order of the blocks.
// The block also appends its occupied cells to the segment list (same atomic).
// ------------------------------------------------------------------------------------------------
struct Segment {          // one occupied cell: the unit of work of the search kernel
    uint32_t cell;        // linear cell id (event index in the high bits)
    uint32_t start;       // first slot in the cell-ordered copy
    uint32_t len;         // points in the cell
    uint32_t interior;    // 1 if no coordinate of the cell is 0 or 2^bits-1 (no wrap among its neighbours)
};

constexpr int kCellThreads = 1024;
constexpr int kCellTile = 4 * kCellThreads;      // table entries per block (upper bound)

// A block owns `rows_per_block` whole padded rows = rows_per_block * (2^bits + 1) <= kCellTile
// entries (a multiple of 4, so every thread moves one aligned uint4).
template <int G>
__global__ void __launch_bounds__(kCellThreads) cell_scan_kernel(uint32_t* __restrict__ cells, int64_t n_entries, int rows_per_block,
                                                                 int bits, Segment* __restrict__ segs,
                                                                 unsigned long long* __restrict__ cursor) {
    __shared__ uint32_t s_pts[32], s_occ[32];
    __shared__ unsigned long long s_base;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t row_len = (1u << bits) + 1u;
    const uint32_t blk_entries = static_cast<uint32_t>(rows_per_block) * row_len;
    const int64_t blk_base = static_cast<int64_t>(blockIdx.x) * blk_entries;
    const uint32_t local = threadIdx.x * 4u;
    const bool act = local < blk_entries && blk_base + local < n_entries;      // n_entries is a multiple of 4 as well
    uint4 v = make_uint4(0u, 0u, 0u, 0u);
    if (act) v = *reinterpret_cast<const uint4*>(cells + blk_base + local);
    const uint32_t tp = v.x + v.y + v.z + v.w;
    const uint32_t to = (v.x != 0u) + (v.y != 0u) + (v.z != 0u) + (v.w != 0u);
    uint32_t ip = tp, io = to;                                                 // inclusive warp scans
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t a = __shfl_up_sync(kFull, ip, o), b = __shfl_up_sync(kFull, io, o);
        if (lane >= o) { ip += a; io += b; }
    }
    if (lane == 31) { s_pts[warp] = ip; s_occ[warp] = io; }
    __syncthreads();
    if (warp == 0) {
        const uint32_t wp = s_pts[lane], wo = s_occ[lane];
        uint32_t sp = wp, so = wo;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t a = __shfl_up_sync(kFull, sp, o), b = __shfl_up_sync(kFull, so, o);
            if (lane >= o) { sp += a; so += b; }
        }
        s_pts[lane] = sp - wp;                                                 // exclusive warp offsets
        s_occ[lane] = so - wo;
        if (lane == 31) {
            const unsigned long long total = (static_cast<unsigned long long>(so) << 32) | sp;
            s_base = total ? atomicAdd(cursor, total) : 0ull;
        }
    }
    __syncthreads();
    if (!act) return;
    const unsigned long long base = s_base;
    uint32_t p = static_cast<uint32_t>(base) + s_pts[warp] + (ip - tp);
    uint32_t oc = static_cast<uint32_t>(base >> 32) + s_occ[warp] + (io - to);
    const uint32_t cnt[4] = {v.x, v.y, v.z, v.w};
    uint4 out;
    out.x = p; out.y = p + v.x; out.z = out.y + v.y; out.w = out.z + v.z;
    *reinterpret_cast<uint4*>(cells + blk_base + local) = out;
    if (to) {
        const uint32_t mask = (1u << bits) - 1u;
        const float inv_row = 1.0f / static_cast<float>(row_len);
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            if (cnt[k]) {
                // table index -> linear id: drop the padding entries of the rows before this one
                const uint32_t e = local + k;
                const uint32_t row_local = __float2uint_rz((static_cast<float>(e) + 0.5f) * inv_row);     // e / row_len, e < 4096
                const uint32_t lin = static_cast<uint32_t>(blk_base + e) - (blockIdx.x * static_cast<uint32_t>(rows_per_block) + row_local);
                bool interior = true;
#pragma unroll
                for (int d = 0; d < G; ++d) {
                    const uint32_t c = (lin >> (d * bits)) & mask;
                    interior = interior && c != 0u && c != mask;
                }
                segs[oc] = Segment{lin, p, cnt[k], interior ? 1u : 0u};
                ++oc;
            }
            p += cnt[k];
        }
    }
}

// ------------------------------------------------------------------------------------------------
// S5: neighbour-cell enumeration for one occupied cell.  The last binned coordinate is the
// fastest-varying one in the linear cell id, so its three adjacent cells are ONE contiguous run of
// the cell-ordered copy: 3^G cells = 3^(G-1) runs.  Up to 27 runs live in lanes (one per lane);
// G > 4 loops over 3^(G-4) run groups.  Interior cells (the common case) reach a neighbour row by
// adding a per-lane constant to the cell id; cells on a face of the toroidal grid take the general
// path with wrapped coordinates and, for the last coordinate, a second "piece".
//
// Flattening: an inclusive warp scan of the run lengths gives every run its offset E_k in the
// flattened candidate list.  For the chunk [b, b+32) each lane needs the run with the largest
// E_k <= b + lane: (number of non-empty runs with E_k <= b) + popc of the marks of runs starting
// inside (b, b+lane] -- one REDUX.OR, one ballot and two popc instead of a per-lane search.
// f(slot_or_minus1) is called once per chunk with one candidate slot per lane (-1 = no candidate).
// ------------------------------------------------------------------------------------------------
__host__ __device__ constexpr int pow3(int e) { return e <= 0 ? 1 : 3 * pow3(e - 1); }

template <int G>
struct Neigh {
    static constexpr int LD = (G - 1 < 3) ? (G - 1) : 3;     // coordinates enumerated across lanes
    static constexpr int RL = pow3(LD);                      // runs per group (<= 27)
    static constexpr int GD = G - 1 - LD;                    // coordinates enumerated by the group loop
    static constexpr int NG = pow3(GD);
};

// signed cell-id offset of this lane's neighbour row (interior cells only)
template <int G>
__device__ __forceinline__ int lane_row_delta(int lane, int bits) {
    int kk = lane, delta = 0;
#pragma unroll
    for (int d = Neigh<G>::GD; d < G - 1; ++d) {
        const int o = kk % 3 - 1;
        kk /= 3;
        delta += o * (1 << ((G - 1 - d) * bits));
    }
    return delta;
}

template <int G, bool INTERIOR, class F>
__device__ __forceinline__ void for_each_candidate_chunk(uint32_t cell, int bits, int lane_delta,
                                                         const uint32_t* __restrict__ cell_start, int* s_delta,
                                                         int lane, F&& f) {
    using N = Neigh<G>;
    const uint32_t mask = (1u << bits) - 1u;
    const uint32_t c_last = cell & mask;
    const uint32_t lt_mask = (1u << lane) - 1u;
    const bool edge_lo = c_last == 0u, edge_hi = c_last == mask;
    const int n_pieces = (!INTERIOR && (edge_lo || edge_hi)) ? 2 : 1;
    for (int grp = 0; grp < N::NG; ++grp) {
        uint32_t row;                                        // padded table index of the neighbour row's cell 0
        if (INTERIOR) {
            int gdelta = 0, gg = grp;
#pragma unroll
            for (int d = 0; d < N::GD; ++d) { gdelta += (gg % 3 - 1) * (1 << ((G - 1 - d) * bits)); gg /= 3; }
            row = padded((cell & ~mask) + static_cast<uint32_t>(lane_delta + gdelta), bits);
        } else {
            uint32_t base = cell >> (G * bits);
            int kk = lane, gg = grp;
#pragma unroll
            for (int d = 0; d < G - 1; ++d) {
                int o;
                if (d < N::GD) { o = gg % 3 - 1; gg /= 3; } else { o = kk % 3 - 1; kk /= 3; }
                const uint32_t cd = (cell >> ((G - 1 - d) * bits)) & mask;
                base = (base << bits) | ((cd + static_cast<uint32_t>(o)) & mask);
            }
            row = padded(base << bits, bits);
        }
        for (int piece = 0; piece < n_pieces; ++piece) {
            uint32_t lo, hi;
            if (INTERIOR)        { lo = c_last - 1u; hi = c_last + 1u; }
            else if (piece == 0) { lo = edge_lo ? 0u : c_last - 1u; hi = edge_hi ? mask : c_last + 1u; }
            else                 { lo = hi = edge_lo ? mask : 0u; }
            uint32_t s = 0, e = 0;
            if (lane < N::RL) { s = cell_start[row + lo]; e = cell_start[row + hi + 1u]; }
            const int len = static_cast<int>(e - s);
            int incl = len;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int t = __shfl_up_sync(kFull, incl, o);
                if (lane >= o) incl += t;
            }
            const int total = __shfl_sync(kFull, incl, 31);
            if (total == 0) continue;
            const int excl = incl - len;
            const uint32_t nz = __ballot_sync(kFull, len > 0);
            __syncwarp();
            if (len > 0) s_delta[__popc(nz & lt_mask)] = static_cast<int>(s) - excl;   // slot = t + delta within the run
            __syncwarp();
            for (int b = 0; b < total; b += 32) {
                const int rel = excl - b;                                // where this run starts relative to the chunk
                const uint32_t mark = (len > 0 && rel > 0 && rel < 32) ? (1u << rel) : 0u;
                const uint32_t marks = __reduce_or_sync(kFull, mark);
                const int before = __popc(__ballot_sync(kFull, len > 0 && rel <= 0));
                const int ord = before - 1 + __popc(marks & ((2u << lane) - 1u));
                const int t = b + lane;
                const int slot = t < total ? t + s_delta[ord] : -1;
                f(slot);
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------
// S6/S7: the single search pass.  One warp per segment (occupied cell), persistent grid-stride
// over the segment list.  Queries = the cell's points (<= 32 per pass) staged in shared memory and
// read back as broadcasts; candidates = one per lane per chunk (2 x 128-bit loads of the 32-byte
// row).  Lane q keeps the running hit count of query q.  Every hit (j, d2) is appended to the
// query's slot buffer hits[row * kSlot + pos] (pos < kSlot); the count keeps running beyond kSlot,
// which tells emit_kernel to resolve that row by recomputation.
// ------------------------------------------------------------------------------------------------
constexpr int kSearchWarps = 8;
// ptxas caps registers from the launch bounds: 5 resident blocks of 256 threads = 48 registers.
#ifndef FRNN_SEARCH_MIN_BLOCKS
#define FRNN_SEARCH_MIN_BLOCKS 5
#endif
constexpr int kSlot = 32;              // hit slots per row in the scratch buffer
constexpr int kEmitThreads = 512;      // rows per emit tile

struct SearchArgs {
    const float4* spts;
    const int32_t* sidx;          // slot -> global row index
    const uint32_t* cell_start;
    const Segment* segs;
    const unsigned long long* cursor;   // high 32 bits = number of segments
    uint32_t* cnt;                // [n_total] uncapped |S_i| at the global row index
    int2* hits;                   // [n_total * kSlot] (j global, d2 bits)
    unsigned long long* tile_deg; // [ceil(n_total / kEmitThreads)] sum of min(|S_i|, k_max) per emit tile (zeroed)
    float r2;
    int bits;
    uint32_t k_max;
};

template <int G, bool INTERIOR>
__device__ __forceinline__ void search_segment(const SearchArgs& a, const Segment& seg, float4* q, int* s_delta, int lane,
                                               int lane_delta, uint32_t lt_mask) {
    const float inf = __int_as_float(0x7f800000);
    for (uint32_t q0 = 0; q0 < seg.len; q0 += 32) {
        const int nq = min(32u, seg.len - q0);
        const uint32_t first_slot = seg.start + q0;
        const bool has = lane < nq;
        int32_t my_row = 0;
        uint32_t my_cnt = 0;
        __syncwarp();
        if (has) {
            q[2 * lane] = a.spts[2 * static_cast<int64_t>(first_slot + lane)];
            q[2 * lane + 1] = a.spts[2 * static_cast<int64_t>(first_slot + lane) + 1];
            my_row = a.sidx[first_slot + lane];
        }
        __syncwarp();
        for_each_candidate_chunk<G, INTERIOR>(seg.cell, a.bits, lane_delta, a.cell_start, s_delta, lane, [&](int cslot) {
            float4 ca = make_float4(inf, 0.f, 0.f, 0.f), cb = make_float4(0.f, 0.f, 0.f, 0.f);   // no candidate: d2 = inf
            int32_t cj = 0;
            if (cslot >= 0) {
                ca = a.spts[2 * static_cast<int64_t>(cslot)];
                cb = a.spts[2 * static_cast<int64_t>(cslot) + 1];
                cj = a.sidx[cslot];
            }
            const int self_q = cslot - static_cast<int>(first_slot);   // the query this candidate IS (if in [0, nq))
            for (int qi = 0; qi < nq; ++qi) {
                const float d2 = d2_pinned(q[2 * qi], q[2 * qi + 1], ca, cb);
                const bool hit = d2 <= a.r2 && self_q != qi;
                const uint32_t m = __ballot_sync(kFull, hit);
                if (m) {
                    const uint32_t base = __shfl_sync(kFull, my_cnt, qi);
                    const int32_t row = __shfl_sync(kFull, my_row, qi);
                    if (hit) {
                        const uint32_t pos = base + __popc(m & lt_mask);
                        if (pos < kSlot) a.hits[static_cast<int64_t>(row) * kSlot + pos] = make_int2(cj, __float_as_int(d2));
                    }
                    if (lane == qi) my_cnt += __popc(m);
                }
            }
        });
        if (has) {
            a.cnt[my_row] = my_cnt;
            // per-tile degree totals: emit_kernel turns them into its global offsets without any
            // inter-block wait
            if (my_cnt) atomicAdd(&a.tile_deg[my_row / kEmitThreads], static_cast<unsigned long long>(my_cnt < a.k_max ? my_cnt : a.k_max));
        }
    }
}

template <int G>
__global__ void __launch_bounds__(kSearchWarps * 32, FRNN_SEARCH_MIN_BLOCKS) search_kernel(SearchArgs a) {
    __shared__ float4 s_q[kSearchWarps][64];
    __shared__ int s_delta[kSearchWarps][32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t lt_mask = (1u << lane) - 1u;
    const uint32_t n_segs = static_cast<uint32_t>(*a.cursor >> 32);
    const uint32_t stride = gridDim.x * kSearchWarps;
    int lane_delta = lane_row_delta<G>(lane, a.bits);
    asm volatile("" : "+r"(lane_delta));                  // keep it in a register: do not recompute per segment
    uint32_t sg = blockIdx.x * kSearchWarps + warp;
    if (sg >= n_segs) return;
    Segment seg = a.segs[sg];
    while (true) {
        const uint32_t nxt = sg + stride;
        Segment seg_next = seg;
        if (nxt < n_segs) seg_next = a.segs[nxt];         // prefetch: the load overlaps this segment's work
        if (seg.interior) search_segment<G, true>(a, seg, s_q[warp], s_delta[warp], lane, lane_delta, lt_mask);
        else              search_segment<G, false>(a, seg, s_q[warp], s_delta[warp], lane, lane_delta, lt_mask);
        if (nxt >= n_segs) break;
        sg = nxt;
        seg = seg_next;
    }
}

// ------------------------------------------------------------------------------------------------
// S8-S10: emit.  Thread per row in ORIGINAL order.  The search pass left sum(min(|S_i|, k_max)) per
// 512-row tile in tile_deg, so a block gets its global edge offset by summing the totals of the
// tiles before it (no inter-block wait), scans its own capped degrees -> CSR row_ptr, and every row
// places its hits at row_ptr[i] + (rank of dst among the row's hits): no sort, the COO comes out
// (src,dst)-sorted.  Rows whose hits did not fit the slot buffer, or with more than k_max hits, are
// recomputed by the whole warp: exact K-smallest by (d2, j) through bisection on the bit pattern of
// d2 and then on j among ties (storage-free), hits written unsorted, ordered by a bitonic network.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void cmp_swap(int32_t* dst, float* d2, int64_t lo, int64_t hi) {
    const int32_t x = dst[lo], y = dst[hi];
    if (x > y) {
        dst[lo] = y; dst[hi] = x;
        const float t = d2[lo]; d2[lo] = d2[hi]; d2[hi] = t;
    }
}

// in-place ascending sort of (dst, d2)[0..len) by dst, whole warp, any len: bitonic network whose
// comparators all point upwards, so virtual +inf padding above the row never moves
__device__ __forceinline__ void warp_sort_rows(int32_t* dst, float* d2, int64_t len, int lane) {
    int64_t p2 = 1;
    while (p2 < len) p2 <<= 1;
    for (int64_t k = 2; k <= p2; k <<= 1) {
        const int64_t hk = k >> 1;
        for (int64_t t = lane; t < (p2 >> 1); t += 32) {              // flip stage: i <-> i ^ (k-1)
            const int64_t lo = (t / hk) * k + (t % hk);
            const int64_t hi = lo ^ (k - 1);
            if (hi < len) cmp_swap(dst, d2, lo, hi);
        }
        __syncwarp();
        for (int64_t j = k >> 2; j >= 1; j >>= 1) {
            for (int64_t t = lane; t < (p2 >> 1); t += 32) {
                const int64_t lo = (t / j) * (2 * j) + (t % j);
                const int64_t hi = lo + j;
                if (hi < len) cmp_swap(dst, d2, lo, hi);
            }
            __syncwarp();
        }
    }
}

struct EmitArgs {
    const float4* pts;            // original points (to recompute the cell of a big row)
    const float4* spts;
    const int32_t* sidx;
    const uint32_t* cell_start;
    const uint32_t* cnt;
    const int2* hits;
    const unsigned long long* tile_deg;
    const int64_t* ev_off;        // device event offsets (n_events + 1) or NULL for one event
    int n_events;
    int64_t n_total;
    int64_t* row_ptr;             // optional [n_total + 1]
    int32_t* out_src;
    int32_t* out_dst;
    float* out_d2;
    int64_t capacity;
    int64_t* out_count;           // optional
    int64_t* out_edge_offsets;    // optional [n_events + 1]
    int32_t* out_status;
    float r2, inv_cell;
    int bits;
    uint32_t k_max;
};

template <int G, bool INTERIOR>
__device__ __forceinline__ void emit_big_row(const EmitArgs& a, int64_t row, int64_t row_rp, int64_t row_ev, uint32_t row_cnt,
                                             uint32_t cell, const float4& qa, const float4& qb, int* s_delta, int lane,
                                             int lane_delta, uint32_t lt_mask) {
    const float inf = __int_as_float(0x7f800000);
    // visit(g): g(in_radius, j, d2) once per chunk, one candidate per lane
    auto visit = [&](auto&& g) {
        for_each_candidate_chunk<G, INTERIOR>(cell, a.bits, lane_delta, a.cell_start, s_delta, lane, [&](int cslot) {
            float4 ca = make_float4(inf, 0.f, 0.f, 0.f), cb = make_float4(0.f, 0.f, 0.f, 0.f);
            int32_t cj = -1;
            if (cslot >= 0) {
                ca = a.spts[2 * static_cast<int64_t>(cslot)];
                cb = a.spts[2 * static_cast<int64_t>(cslot) + 1];
                cj = a.sidx[cslot];
            }
            const float d2 = d2_pinned(qa, qb, ca, cb);
            g(d2 <= a.r2 && cj != static_cast<int32_t>(row), cj, d2);
        });
    };
    // threshold key (dthr, jthr): keep hits with (d2 bits, j) <= it.  d2 >= +0 always (the chain
    // starts at +0 and adds squares), so bit patterns order like values.
    uint32_t dthr = __float_as_uint(a.r2);
    int32_t jthr = 0x7fffffff;
    if (row_cnt > a.k_max) {
        auto count_le = [&](uint32_t dkey, int32_t jkey) -> uint32_t {
            uint32_t n = 0;
            visit([&](bool in, int32_t cj, float d2) {
                const uint32_t db = __float_as_uint(d2);
                n += __popc(__ballot_sync(kFull, in && (db < dkey || (db == dkey && cj <= jkey))));
            });
            return n;
        };
        uint32_t dlo = 0, dhi = dthr;
        while (dlo < dhi) {
            const uint32_t mid = dlo + ((dhi - dlo) >> 1);
            if (count_le(mid, 0x7fffffff) >= a.k_max) dhi = mid; else dlo = mid + 1;
        }
        int32_t jlo = 0, jhi = 0x7fffffff;
        while (jlo < jhi) {
            const int32_t mid = jlo + ((jhi - jlo) >> 1);
            if (count_le(dlo, mid) >= a.k_max) jhi = mid; else jlo = mid + 1;
        }
        dthr = dlo;
        jthr = jlo;
    }
    const int32_t src = static_cast<int32_t>(row - row_ev);
    uint32_t off = 0;
    visit([&](bool in, int32_t cj, float d2) {
        const uint32_t db = __float_as_uint(d2);
        const bool keep = in && (db < dthr || (db == dthr && cj <= jthr));
        const uint32_t m = __ballot_sync(kFull, keep);
        if (keep) {
            const int64_t pos = row_rp + off + __popc(m & lt_mask);
            if (pos < a.capacity) { a.out_src[pos] = src; a.out_dst[pos] = cj - static_cast<int32_t>(row_ev); a.out_d2[pos] = d2; }
        }
        off += __popc(m);
    });
    __syncwarp();
    const int64_t kept = row_cnt < a.k_max ? row_cnt : a.k_max;
    if (row_rp + kept <= a.capacity)                       // rows cut by the capacity stay unsorted
        warp_sort_rows(a.out_dst + row_rp, a.out_d2 + row_rp, kept, lane);
    __syncwarp();
}

template <int G>
__global__ void __launch_bounds__(kEmitThreads, 2) emit_kernel(EmitArgs a) {
    __shared__ unsigned long long s_warp[kEmitThreads / 32];
    __shared__ unsigned long long s_prefix;
    __shared__ int s_delta[kEmitThreads / 32][32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t lt_mask = (1u << lane) - 1u;
    const uint32_t tile = blockIdx.x;
    const int64_t i = static_cast<int64_t>(tile) * kEmitThreads + threadIdx.x;
    const bool has = i < a.n_total;
    const uint32_t c = has ? a.cnt[i] : 0u;
    const uint32_t deg = c < a.k_max ? c : a.k_max;
    // first hits of the row: issued early so the loads overlap the offset computation
    const int2* h = a.hits + i * kSlot;
    int4 h01 = make_int4(0, 0, 0, 0), h23 = h01;
    if (c > 0) h01 = *reinterpret_cast<const int4*>(h);
    if (c > 2) h23 = *reinterpret_cast<const int4*>(h + 2);
    // ---- global offset of the tile = sum of the totals of the tiles before it
    unsigned long long before = 0;
    for (uint32_t t = threadIdx.x; t < tile; t += kEmitThreads) before += a.tile_deg[t];
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) before += __shfl_xor_sync(kFull, before, o);
    // ---- block scan of deg
    uint32_t incl = deg;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t t = __shfl_up_sync(kFull, incl, o);
        if (lane >= o) incl += t;
    }
    if (lane == 0) s_warp[warp] = before;
    __syncthreads();
    if (warp == 0) {
        unsigned long long b = lane < kEmitThreads / 32 ? s_warp[lane] : 0ull;
#pragma unroll
        for (int o = 8; o >= 1; o >>= 1) b += __shfl_xor_sync(kFull, b, o);
        if (lane == 0) s_prefix = b;
    }
    __syncthreads();
    if (lane == 31) s_warp[warp] = incl;                   // warp totals of deg (fits: <= 32 * k_max... use 64-bit)
    __syncthreads();
    unsigned long long wexcl = 0;
#pragma unroll
    for (int w = 0; w < kEmitThreads / 32; ++w) wexcl += (w < warp) ? s_warp[w] : 0ull;
    const int64_t rp = static_cast<int64_t>(s_prefix + wexcl + (incl - deg));      // row_ptr[i]
    // ---- CSR offsets, count, status, per-event edge offsets
    int64_t ev_base = 0;
    if (has) {
        if (a.row_ptr) a.row_ptr[i] = rp;
        if (a.ev_off) {
            int e = event_of_row(a.ev_off, a.n_events, i);
            ev_base = a.ev_off[e];
            if (a.out_edge_offsets)
                for (; e >= 0 && a.ev_off[e] == i; --e) a.out_edge_offsets[e] = rp;    // event starts (and empty events) at row i
        }
        if (i == a.n_total - 1) {
            const int64_t total = rp + deg;
            if (a.row_ptr) a.row_ptr[a.n_total] = total;
            if (a.out_count) *a.out_count = total;
            if (a.out_edge_offsets)
                for (int e = a.n_events; e >= 0 && a.ev_off[e] == a.n_total; --e) a.out_edge_offsets[e] = total;
            *a.out_status = total > a.capacity ? -3 /* FRNN_ERR_CAPACITY */ : 0;
        }
    }
    // ---- rows that fit their slot buffer: rank by dst, place directly
    const bool big = has && (c > kSlot || c > a.k_max);
    if (has && !big && c > 0) {
        const int32_t src = static_cast<int32_t>(i - ev_base);
        const int32_t eb = static_cast<int32_t>(ev_base);
        auto put = [&](uint32_t rank, int32_t j, int32_t d2bits) {
            const int64_t pos = rp + rank;
            if (pos < a.capacity) { a.out_src[pos] = src; a.out_dst[pos] = j - eb; a.out_d2[pos] = __int_as_float(d2bits); }
        };
        if (c <= 4) {                                      // the common case: everything is already in registers
            const int32_t j0 = h01.x, j1 = c > 1 ? h01.z : 0x7fffffff, j2 = c > 2 ? h23.x : 0x7fffffff, j3 = c > 3 ? h23.z : 0x7fffffff;
            put((j1 < j0) + (j2 < j0) + (j3 < j0), j0, h01.y);
            if (c > 1) put((j0 < j1) + (j2 < j1) + (j3 < j1), j1, h01.w);
            if (c > 2) put((j0 < j2) + (j1 < j2) + (j3 < j2), j2, h23.y);
            if (c > 3) put((j0 < j3) + (j1 < j3) + (j2 < j3), j3, h23.w);
        } else {
            for (uint32_t m = 0; m < c; ++m) {
                const int2 mine = h[m];
                uint32_t rank = 0;
                for (uint32_t u = 0; u < c; ++u) rank += h[u].x < mine.x;
                put(rank, mine.x, mine.y);
            }
        }
    }
    // ---- big rows: recompute with the whole warp
    uint32_t bigs = __ballot_sync(kFull, big);
    if (bigs == 0) return;
    int lane_delta = lane_row_delta<G>(lane, a.bits);
    const uint32_t mask = (1u << a.bits) - 1u;
    for (; bigs; bigs &= bigs - 1) {
        const int bl = __ffs(bigs) - 1;
        const int64_t row = __shfl_sync(kFull, i, bl);
        const int64_t row_rp = __shfl_sync(kFull, rp, bl);
        const int64_t row_ev = __shfl_sync(kFull, ev_base, bl);
        const uint32_t row_cnt = __shfl_sync(kFull, c, bl);
        const float4 qa = a.pts[2 * row], qb = a.pts[2 * row + 1];
        uint32_t ev = 0;
        if (a.ev_off) ev = static_cast<uint32_t>(event_of_row(a.ev_off, a.n_events, row));
        const uint32_t cell = cell_of_point<G>(qa, qb, ev, a.inv_cell, a.bits);
        bool interior = true;
#pragma unroll
        for (int d = 0; d < G; ++d) {
            const uint32_t cd = (cell >> (d * a.bits)) & mask;
            interior = interior && cd != 0u && cd != mask;
        }
        if (interior) emit_big_row<G, true>(a, row, row_rp, row_ev, row_cnt, cell, qa, qb, s_delta[warp], lane, lane_delta, lt_mask);
        else          emit_big_row<G, false>(a, row, row_rp, row_ev, row_cnt, cell, qa, qb, s_delta[warp], lane, lane_delta, lt_mask);
    }
}

}  // namespace frnn
