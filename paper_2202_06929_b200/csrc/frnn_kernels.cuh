// frnn_kernels.cuh -- device code of the B200 FRNN path (sm_100a).  Product code: shares nothing
// with oracle/.  Steps S2..S10 of SURVEY.md section 8(a); design notes in DESIGN.md section 6.
//
//   bin_kernel       S2     cell index on a toroidal grid over the first G coordinates + histogram
//   cell_scan_kernel S3     cell starts; blocks take their base from one atomic (no inter-block wait), rows of the
//                           table are padded so a run never needs the next block's start
//   scatter_kernel   S4     counting-sort scatter into the cell-ordered copy (256-bit row moves) + filter keys
//   search_kernel    S5-S7  ONE pass, thread per query in cell order: 4-byte key filter on the unbinned coordinates,
//                           every unordered pair evaluated once with whole 8-term FMA chains, hits appended to
//                           per-row slot buffers of both end points
//   tile_prefix_kernel S9   (only for calls with many emit tiles) exclusive prefix of the per-tile degree totals
//   emit_kernel      S8-S10 block scan of the capped degrees, one thread per output edge (rank by dst): the
//                           (src,dst)-sorted COO without a sort; exact K-cap selection for the rare big rows
//   dense_search_kernel     SURVEY 8(f) f1: the brute-force variant, shares emit_kernel
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace frnn {

constexpr int kDim = 8;                 // floats of an internal row (and of the fast path's input rows)
constexpr int kDimMax = 16;            // dim 9..16: a second internal row holds coordinates 8..15 (zero padded)
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
    // + half the extent: data centred on the origin sits in the middle of [0, 2^bits), so the seam of
    // the torus (cells 0 and 2^bits-1 are neighbours) is met only by points beyond +-2^(bits-1) cells
    return static_cast<uint32_t>(__float2int_rd(a) + static_cast<int>((mask + 1u) >> 1)) & mask;
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

// Filter key of a point: the cell coordinate (same side, modulo 64) of up to four coordinates that
// are NOT binned (dims G..G+3), one per byte.  Two points within r of each other differ by at most
// one cell in every coordinate (same argument as for the grid), so  |q_a - q_c| mod 64 in {0, 1, 63}
// per field is a NECESSARY condition for an edge: candidates failing it are dropped without touching
// their coordinates.  With A = key(query) + 0x81818181 the bytewise difference A - key(candidate)
// never borrows across bytes (129 + q_a - q_c is in [66, 192]) and its low six bits per byte are
// (q_a - q_c + 1) mod 64: the pair passes iff these are all <= 3 (3 is a harmless false positive).
constexpr uint32_t kKeyBias = 0x81818181u;
constexpr uint32_t kKeyReject = 0x3c3c3c3cu;

template <int G>
__device__ __forceinline__ uint32_t key_of_point(const float4& a, const float4& b, float inv_cell) {
    const float x[8] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w};
    uint32_t key = 0;
#pragma unroll
    for (int f = 0; f < 4; ++f)
        if (G + f < kDim) key |= cell_coord(x[G + f], inv_cell, 63u) << (8 * f);
    return key;
}

// Caller-chosen coordinates (frnn_set_bin_order): p[0..G-1] are the binned coordinates, p[G..G+3]
// the key coordinates.  ANY choice is exact (each binned or keyed coordinate is a necessary condition on its own,
// DESIGN.md R8); the choice only decides how much the grid and the filter prune.  The coordinates are read from the
// caller's row (n x dim, coordinates >= dim read as 0); the internal rows keep the original order, so d2 is untouched.
struct BinOrder {
    int on;                       // 0: the first G coordinates are binned, the next four keyed (the default fast path)
    unsigned char p[8];
};
template <int G>
__device__ __forceinline__ uint32_t cell_ordered(const float* __restrict__ row, int dim, uint32_t event, float inv_cell, int bits,
                                                 const BinOrder& o) {
    const uint32_t mask = (1u << bits) - 1u;
    uint32_t lin = event;
#pragma unroll
    for (int d = 0; d < G; ++d) {
        const int c = o.p[d];
        lin = (lin << bits) | cell_coord(c < dim ? row[c] : 0.0f, inv_cell, mask);
    }
    return lin;
}
template <int G>
__device__ __forceinline__ uint32_t key_ordered(const float* __restrict__ row, int dim, float inv_cell, const BinOrder& o) {
    uint32_t key = 0;
#pragma unroll
    for (int f = 0; f < 4; ++f)
        if (G + f < kDim) {
            const int c = o.p[G + f];
            key |= cell_coord(c < dim ? row[c] : 0.0f, inv_cell, 63u) << (8 * f);
        }
    return key;
}

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

// One 32-byte row = one 256-bit transaction (LDG.E.ENL2.256 / STG.E.ENL2.256 on sm_100a).  The .nc form is
// only used on arrays that no thread writes during the kernel.
__device__ __forceinline__ void load_row_nc(const float4* p, float4& a, float4& b) {
    asm("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
        : "=f"(a.x), "=f"(a.y), "=f"(a.z), "=f"(a.w), "=f"(b.x), "=f"(b.y), "=f"(b.z), "=f"(b.w) : "l"(p));
}
__device__ __forceinline__ void store_row(float4* p, const float4& a, const float4& b) {
    asm volatile("st.global.v8.f32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};"
                 :: "l"(p), "f"(a.x), "f"(a.y), "f"(a.z), "f"(a.w), "f"(b.x), "f"(b.y), "f"(b.z), "f"(b.w) : "memory");
}

// A point of the caller's array as an 8-float row (coordinates 0..7).  dim == 8: one 256-bit load (rows are 32-byte
// aligned).  Other dims: the row is read float by float and padded with zeros: every padded term
// of the R3 chain is t = 0 - 0 = +0, fma(+0, +0, acc) = acc, so d2 over the padded row equals d2 over dim terms bit
// for bit.  load_point_hi: coordinates 8..15 of a point with dim > 8, same padding.
__device__ __forceinline__ void load_point(const float* __restrict__ pts, int64_t i, int dim, float4& a, float4& b) {
    if (dim == kDim) {
        load_row_nc(reinterpret_cast<const float4*>(pts) + 2 * i, a, b);
    } else {
        float x[kDim];
        const float* p = pts + i * dim;
#pragma unroll
        for (int d = 0; d < kDim; ++d) x[d] = d < dim ? p[d] : 0.0f;
        a = make_float4(x[0], x[1], x[2], x[3]);
        b = make_float4(x[4], x[5], x[6], x[7]);
    }
}
__device__ __forceinline__ void load_point_hi(const float* __restrict__ pts, int64_t i, int dim, float4& c, float4& d) {
    float x[kDim];
    const float* p = pts + i * dim + kDim;
#pragma unroll
    for (int k = 0; k < kDim; ++k) x[k] = kDim + k < dim ? p[k] : 0.0f;
    c = make_float4(x[0], x[1], x[2], x[3]);
    d = make_float4(x[4], x[5], x[6], x[7]);
}

// Optional in-graph timeline (frnn_set_profiling(2)): every kernel leaves min(start) and max(end) of the
// %globaltimer readings of thread 0 of its blocks (every 16th block for the start) in stamps[2*phase], stamps[2*phase+1] (start stored complemented so that
// one atomicMax serves both; the buffer is zeroed with the rest of the workspace head).  stamps == NULL
// (the normal case) costs one predictable branch per warp.
__device__ __forceinline__ unsigned long long global_ns() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}
__device__ __forceinline__ void stamp_begin(unsigned long long* stamps, int phase) {
    if (stamps && threadIdx.x == 0 && (blockIdx.x & 15) == 0) atomicMax(&stamps[2 * phase], ~global_ns());
}
__device__ __forceinline__ void stamp_end(unsigned long long* stamps, int phase) {
    if (stamps && threadIdx.x == 0) atomicMax(&stamps[2 * phase + 1], global_ns());
}

// The same for kernels whose threads finish at very different times (search, the warp loops of emit): the LAST thread of
// the block to arrive stamps the end (a shared-memory counter; only touched when the timeline is being recorded).
__device__ __forceinline__ void stamp_end_last(unsigned long long* stamps, int phase, unsigned int* s_done) {
    if (stamps && atomicAdd(s_done, 1u) == blockDim.x - 1u) atomicMax(&stamps[2 * phase + 1], global_ns());
}

// dims 8..15 of a pair: the chain simply goes on (R3: one fp32 chain over d = 0..dim-1 in index order)
__device__ __forceinline__ float d2_continue(float acc, const float4& qc, const float4& qd, const float4& cc, const float4& cd) {
    float t;
    t = __fsub_rn(qc.x, cc.x); acc = __fmaf_rn(t, t, acc);
    t = __fsub_rn(qc.y, cc.y); acc = __fmaf_rn(t, t, acc);
    t = __fsub_rn(qc.z, cc.z); acc = __fmaf_rn(t, t, acc);
    t = __fsub_rn(qc.w, cc.w); acc = __fmaf_rn(t, t, acc);
    t = __fsub_rn(qd.x, cd.x); acc = __fmaf_rn(t, t, acc);
    t = __fsub_rn(qd.y, cd.y); acc = __fmaf_rn(t, t, acc);
    t = __fsub_rn(qd.z, cd.z); acc = __fmaf_rn(t, t, acc);
    t = __fsub_rn(qd.w, cd.w); acc = __fmaf_rn(t, t, acc);
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
    int64_t* ev_off;
    int first, count;
    int64_t v[kN];
};
__global__ void set_offsets_kernel(OffsetChunk c) {
    if (static_cast<int>(threadIdx.x) < c.count) c.ev_off[c.first + threadIdx.x] = c.v[threadIdx.x];
}

// ------------------------------------------------------------------------------------------------
// S2: cell index + histogram.  The atomicAdd's return value is the point's rank inside its cell,
// which makes the later scatter a pure function of (cell_start, rank): no second atomic pass.
// ------------------------------------------------------------------------------------------------
// Every kernel of the path takes ONE by-value argument struct: a call is then a list of (function, grid, struct)
// records, which the host either launches one by one or writes into the kernel nodes of a cached CUDA graph
// (cudaGraphExecKernelNodeSetParams) -- the graph does not depend on n, the pointers or the parameters of a call.
struct BinArgs {
    const float* pts;
    int dim;
    int64_t n_total;
    const int64_t* ev_off;
    int n_events;
    float inv_cell;
    int bits;
    uint32_t* cell_count;
    uint32_t* pcell;
    uint32_t* prank;
    BinOrder order;
    unsigned long long* stamps;
};
template <int G>
__global__ void __launch_bounds__(256) bin_kernel(BinArgs k) {
    stamp_begin(k.stamps, 0);
    const int64_t i = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (i < k.n_total) {
        float4 a, b;
        load_point(k.pts, i, k.dim, a, b);
        const uint32_t ev = k.ev_off ? static_cast<uint32_t>(event_of_row(k.ev_off, k.n_events, i)) : 0u;
        const uint32_t lin = k.order.on ? cell_ordered<G>(k.pts + i * k.dim, k.dim, ev, k.inv_cell, k.bits, k.order)
                                        : cell_of_point<G>(a, b, ev, k.inv_cell, k.bits);
        k.pcell[i] = lin;
        k.prank[i] = atomicAdd(&k.cell_count[padded(lin, k.bits)], 1u);
    }
    stamp_end(k.stamps, 0);
}

// ------------------------------------------------------------------------------------------------
// S4: counting-sort scatter.  Order inside a cell is the (arbitrary) atomic order; the final
// result does not depend on it because every row is ordered by dst at the end.
// ------------------------------------------------------------------------------------------------
struct ScatterArgs {
    const float* pts;
    int dim;
    int64_t n_total;
    int bits;
    float inv_cell;
    const uint32_t* cell_start;
    const uint32_t* pcell;
    const uint32_t* prank;
    float4* spts;
    int32_t* sidx;
    uint32_t* skey;
    float4* spts_hi;
    uint32_t* scell;
    BinOrder order;
    unsigned long long* stamps;
};
template <int G>
__global__ void __launch_bounds__(256) scatter_kernel(ScatterArgs k) {
    stamp_begin(k.stamps, 2);
    const int64_t i = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (i < k.n_total) {
        const uint32_t lin = k.pcell[i];
        const uint32_t s = k.cell_start[padded(lin, k.bits)] + k.prank[i];
        if (k.scell) k.scell[s] = lin;                             // a bin order is set: the search cannot recompute the cell from the row
        float4 a, b;
        load_point(k.pts, i, k.dim, a, b);
        store_row(k.spts + 2 * static_cast<int64_t>(s), a, b);    // one 32-byte sector, one transaction
        k.sidx[s] = static_cast<int32_t>(i);
        k.skey[s] = k.order.on ? key_ordered<G>(k.pts + i * k.dim, k.dim, k.inv_cell, k.order) : key_of_point<G>(a, b, k.inv_cell);
        if (k.spts_hi) {                                           // dim > 8: coordinates 8..15 travel in a second row
            float4 c, d;
            load_point_hi(k.pts, i, k.dim, c, d);
            store_row(k.spts_hi + 2 * static_cast<int64_t>(s), c, d);
        }
    }
    stamp_end(k.stamps, 2);
}

// ------------------------------------------------------------------------------------------------
// S3: cell starts.  Each block owns a few WHOLE padded rows of the table (about 4096 entries),
// computes its total, reserves its range of the cell-ordered copy with ONE atomicAdd, then writes the
// exclusive scan of its entries.  Blocks land in arrival order: no inter-block wait, and since a run
// only ever reads start[lo] and start[hi+1] of one row (the padding entry holds the row's end)
// nothing depends on the order of the blocks.
// ------------------------------------------------------------------------------------------------
constexpr int kCellThreads = 1024;
constexpr int kCellTile = 4 * kCellThreads;      // table entries per block (upper bound)

// A block owns `rows_per_block` whole padded rows = rows_per_block * (2^bits + 1) <= kCellTile
// entries (a multiple of 4, so every thread moves one aligned uint4).
struct ScanArgs {
    uint32_t* cells;
    int64_t n_entries;
    int rows_per_block;
    int bits;
    unsigned int* cursor;
    unsigned long long* stamps;
};
__global__ void __launch_bounds__(kCellThreads) cell_scan_kernel(ScanArgs k) {
    uint32_t* __restrict__ cells = k.cells;
    const int64_t n_entries = k.n_entries;
    const int rows_per_block = k.rows_per_block, bits = k.bits;
    unsigned int* __restrict__ cursor = k.cursor;
    unsigned long long* stamps = k.stamps;
    stamp_begin(stamps, 1);
    __shared__ uint32_t s_pts[32];
    __shared__ uint32_t s_base;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t row_len = (1u << bits) + 1u;
    const uint32_t blk_entries = static_cast<uint32_t>(rows_per_block) * row_len;
    const int64_t blk_base = static_cast<int64_t>(blockIdx.x) * blk_entries;
    const uint32_t local = threadIdx.x * 4u;
    const bool act = local < blk_entries && blk_base + local < n_entries;      // n_entries is a multiple of 4 as well
    uint4 v = make_uint4(0u, 0u, 0u, 0u);
    if (act) v = *reinterpret_cast<const uint4*>(cells + blk_base + local);
    const uint32_t tp = v.x + v.y + v.z + v.w;
    uint32_t ip = tp;                                                          // inclusive warp scan
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t t = __shfl_up_sync(kFull, ip, o);
        if (lane >= o) ip += t;
    }
    if (lane == 31) s_pts[warp] = ip;
    __syncthreads();
    if (warp == 0) {
        const uint32_t wp = s_pts[lane];
        uint32_t sp = wp;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t t = __shfl_up_sync(kFull, sp, o);
            if (lane >= o) sp += t;
        }
        s_pts[lane] = sp - wp;                                                 // exclusive warp offsets
        if (lane == 31) s_base = sp ? atomicAdd(cursor, sp) : 0u;
    }
    __syncthreads();
    if (act) {
        const uint32_t p = s_base + s_pts[warp] + (ip - tp);
        uint4 out;
        out.x = p; out.y = p + v.x; out.z = out.y + v.y; out.w = out.z + v.z;
        *reinterpret_cast<uint4*>(cells + blk_base + local) = out;
    }
    stamp_end(stamps, 1);
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
// S5-S7: the single search pass, ONE THREAD PER QUERY in cell order (thread = slot of the
// cell-ordered copy), so the lanes of a warp sit in the same or adjacent cells and their loads of
// the table, the keys and the candidate rows fall into the same few cache lines.
//
// Every unordered pair is evaluated ONCE.  d2 is bitwise symmetric (x - y = -(y - x) exactly, the
// squares and the FMA chain are identical), so a query only visits the "forward" half of its
// neighbourhood: cell offsets (o_0 .. o_{G-1}) that are lexicographically positive, plus the slots
// after its own in its own cell -- 13.5 of the 27 runs at G = 4 -- and a hit is appended to BOTH
// rows' slot buffers (position from an atomic counter per row).
//
// Phase 1 (filter).  Neighbour rows are visited in sub-batches of 3 rows (the offsets of coordinate
// G-2, unrolled).  A run is [start[row+lo], start[row+hi+1]); its first kBatch candidates are tested
// straight-line -- 3 x kBatch independent 4-byte key loads in flight per thread -- and longer runs
// finish in batches of kBatch.  Only the filter key of a candidate is read here (see key_of_point):
// ~85 % of the candidates of a tracking event are rejected with 3 integer instructions and 4 bytes
// of traffic.  Survivors go on the thread's queue (its own column of a shared-memory array; the
// store is unconditional, the queue pointer advances only for survivors: no branch).
// Phase 2 (evaluate) drains the queue: 32-byte row + index loads (next row in flight while the
// current one is evaluated), the whole R3 chain per lane.  Hit (i, j, d2): pos = cnt[i]++ and
// hits[i * kSlot + pos] = (j, d2) if pos < kSlot, the same for j; the counts keep running beyond
// kSlot, which tells emit_kernel to resolve that row by recomputation.  min(cnt, k_max) is the
// number of increments that found a value < k_max, so the per-tile capped degree totals emit_kernel
// needs are accumulated exactly by the same increments.
// Lanes whose cell touches the seam of the torus in the last coordinate (only points beyond
// +-2^(bits-1) cells from the origin) also filter the wrapped cell.
// ------------------------------------------------------------------------------------------------
constexpr int kSearchThreads = 128;
#ifndef FRNN_SEARCH_MIN_BLOCKS
#define FRNN_SEARCH_MIN_BLOCKS 7       // 7 x 128 threads: 72 registers per thread; 7 x 148 blocks >= one 120k-point event
#endif
#ifndef FRNN_KBATCH
#define FRNN_KBATCH 4
#endif
constexpr int kBatch = FRNN_KBATCH;    // candidates of a run tested per batch
constexpr int kQueue = 32;             // survivor queue entries per thread (>= 2 * 3 * kBatch)
constexpr int kLeft = 15;              // leftover-run entries per thread (the runs of 5 sub-batches)
constexpr int kSlot = 32;              // hit slots per row in the scratch buffer: 256 B per row reserved, one 32-byte sector touched per 4
                                       // hits.  Smaller layouts were built and measured in round 2 (profiles/r02_summary.md): 16 slots cost
                                       // 3 us per event (the 10 rows in 120,000 with more hits are recomputed by a warp, ~3 us each, at the
                                       // end of emit); 4 inline slots + a per-tile overflow pool cost 9 us (same-address returning atomics)
#ifndef FRNN_EMIT_THREADS
#define FRNN_EMIT_THREADS 256
#endif
constexpr int kEmitThreads = FRNN_EMIT_THREADS;   // rows per emit tile
#ifndef FRNN_DEG_SLICES
#define FRNN_DEG_SLICES 8
#endif
constexpr int kDegSlices = FRNN_DEG_SLICES;   // copies of every per-tile degree counter, slice-major: the copies of a tile sit in different sectors

struct SearchArgs {
    const float4* spts;
    const float4* spts_hi;        // coordinates 8..15 of the slots (dim > 8), else NULL
    const int32_t* sidx;          // slot -> global row index
    const uint32_t* skey;         // slot -> filter key
    const uint32_t* cell_start;
    uint32_t* cnt;                // [n_total] uncapped |S_i| at the global row index (zeroed)
    int2* hits;                   // [n_total * kSlot] (j global, d2 bits)
    unsigned long long* tile_deg; // [kDegSlices][n_tiles] partial sums of min(|S_i|, k_max) per emit tile (zeroed)
    uint32_t n_tiles;             // ceil(n_total / kEmitThreads)
    const int64_t* ev_off;        // device event offsets or NULL for one event
    unsigned long long* stamps;   // NULL unless the timeline is being recorded
    const uint32_t* scell;        // slot -> linear cell id, stored by scatter_kernel only when a bin order is set, else NULL
    int64_t n_total;
    int n_events;
    float r2, inv_cell;
    int bits;
    uint32_t k_max;
};

// Filter test + push of one candidate slot j: if the key passes, j is stored at the thread's queue address
// and the address advances by one entry -- four SASS instructions (IADD, LOP3 to a predicate, predicated
// STS and IADD), no branch, no 64-bit pointer arithmetic.
__device__ __forceinline__ void filter_push(uint32_t& qaddr, uint32_t key_a, uint32_t key_c, uint32_t j) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t.reg .u32 t;\n\t"
        "sub.u32 t, %1, %2;\n\t"
        "and.b32 t, t, %4;\n\t"
        "setp.eq.u32 p, t, 0;\n\t"
        "@p st.shared.u32 [%0], %3;\n\t"
        "@p add.u32 %0, %0, %5;\n\t}"
        : "+r"(qaddr)
        : "r"(key_a), "r"(key_c), "r"(j), "n"(kKeyReject), "n"(kSearchThreads * 4)
        : "memory");
}

// The part of a run beyond its first kBatch candidates, (first slot, length), goes on the thread's leftover
// list if it is not empty: predicated 64-bit store and pointer bump, no branch.
__device__ __forceinline__ void leftover_push(uint32_t& laddr, uint32_t j0, uint32_t len) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t.reg .u32 j, n;\n\t"
        "setp.gt.u32 p, %2, %3;\n\t"
        "add.u32 j, %1, %3;\n\t"
        "sub.u32 n, %2, %3;\n\t"
        "@p st.shared.v2.u32 [%0], {j, n};\n\t"
        "@p add.u32 %0, %0, %4;\n\t}"
        : "+r"(laddr)
        : "r"(j0), "r"(len), "n"(kBatch), "n"(kSearchThreads * 8)
        : "memory");
}

template <int G, bool HI>
__global__ void __launch_bounds__(kSearchThreads, FRNN_SEARCH_MIN_BLOCKS) search_kernel(SearchArgs a) {
    constexpr int NU = G >= 2 ? 3 : 1;                    // unrolled offsets of coordinate G-2
    constexpr int NB = pow3(G >= 2 ? G - 2 : 0);          // sub-batches: offsets of coordinates 0..G-3 (dim 0 most significant)
    constexpr int MID = (NB - 1) / 2;                     // the sub-batch with all-zero offsets
    constexpr int kWide = 4;                              // survivors evaluated together (rows in flight per thread)
    __shared__ uint32_t s_queue[kQueue][kSearchThreads];
    __shared__ __align__(8) uint2 s_left[kLeft][kSearchThreads];      // leftover runs (first slot, length), one column per thread
    __shared__ unsigned int s_done;                                   // timeline only: threads of the block that have finished
    stamp_begin(a.stamps, 3);
    const int tid = threadIdx.x;
    if (a.stamps) {                                                   // (kernel argument: uniform)
        if (tid == 0) s_done = 0u;
        __syncthreads();
    }
    const int64_t s64 = static_cast<int64_t>(blockIdx.x) * kSearchThreads + tid;
    if (s64 >= a.n_total) { stamp_end_last(a.stamps, 3, &s_done); return; }      // no block-wide barrier below
    const uint32_t s = static_cast<uint32_t>(s64);
    float4 qa, qb;
    load_row_nc(a.spts + 2 * s64, qa, qb);
    const int32_t my_row = a.sidx[s];
    const uint32_t key_a = a.skey[s] + kKeyBias;
    const uint32_t key_fail = key_a - 4u;                 // a candidate key that never passes: (key_a - key_fail) & reject = 4
    const int bits = a.bits;
    const uint32_t mask = (1u << bits) - 1u;
    // the slot's cell, recomputed from its coordinates (the event from the row index: blocks of the cell-ordered
    // copy land in arrival order, so slots are not ordered by event)
    const uint32_t ev = a.ev_off ? static_cast<uint32_t>(event_of_row(a.ev_off, a.n_events, my_row)) : 0u;
    const uint32_t cell = a.scell ? a.scell[s] : cell_of_point<G>(qa, qb, ev, a.inv_cell, bits);
    const uint32_t c_last = cell & mask;
    const uint32_t lo = c_last ? c_last - 1u : 0u, hi = c_last < mask ? c_last + 1u : mask;
    unsigned long long* const my_tile_deg = a.tile_deg + static_cast<size_t>(blockIdx.x & (kDegSlices - 1)) * a.n_tiles;
    // interior in the coordinates 0..G-2: a neighbour row is the own row plus a constant (no wrap)
    bool interior = true;
#pragma unroll
    for (int d = 0; d < G - 1; ++d) {
        const uint32_t cd = (cell >> ((G - 1 - d) * bits)) & mask;
        interior = interior && cd != 0u && cd != mask;
    }
    const uint32_t own_rowid = cell >> bits;
    uint32_t own_deg = 0;                                 // increments of cnt[my_row] made here that found a value < k_max
    const uint32_t q_base = static_cast<uint32_t>(__cvta_generic_to_shared(&s_queue[0][tid]));
    uint32_t qaddr = q_base;                              // shared-memory address of the next free queue entry
    constexpr uint32_t kQBytes = kSearchThreads * 4;      // one queue entry further down the thread's column
    const uint32_t l_base = static_cast<uint32_t>(__cvta_generic_to_shared(&s_left[0][tid]));
    uint32_t laddr = l_base;                              // shared-memory address of the next free leftover entry
    constexpr uint32_t kLBytes = kSearchThreads * 8;

    // phase 2: evaluate the queued survivors (never the query itself), kWide at a time: kWide 256-bit row
    // loads in flight, then the R3 chains, then -- for the hits (i, j, d2) -- ONE returning atomic on cnt[i]
    // for all hits of the group and one per partner row j, all in flight together, then the stores
    // hits[row * kSlot + pos] = (other, d2) for pos < kSlot on both rows.  The counts keep running beyond kSlot,
    // which tells emit_kernel to resolve that row by recomputation; min(cnt, k_max) is the number of increments
    // that found a value < k_max, so the per-tile capped degree totals are accumulated by the same increments.
    auto drain = [&](bool stash = false) {
        const int qn = static_cast<int>((qaddr - q_base) / kQBytes);
        qaddr = q_base;
        uint32_t hs = 0;                                                 // hits noted in the (by now free) leftover list
        for (int i = 0; i < qn; i += kWide) {
            float4 ca[kWide], cb[kWide];
            int32_t cj[kWide];
            uint32_t js[kWide];
            bool ok[kWide];
#pragma unroll
            for (int v = 0; v < kWide; ++v) {
                ok[v] = i + v < qn;
                js[v] = ok[v] ? s_queue[i + v][tid] : s;                 // padding: my own row (a valid address, masked below)
                load_row_nc(a.spts + 2 * static_cast<int64_t>(js[v]), ca[v], cb[v]);
                cj[v] = a.sidx[js[v]];
            }
            float d2[kWide];
#pragma unroll
            for (int v = 0; v < kWide; ++v) d2[v] = d2_pinned(qa, qb, ca[v], cb[v]);
            if (HI) {                                                    // dim > 8: the chain goes on over coordinates 8..15
                float4 qc, qd;
                load_row_nc(a.spts_hi + 2 * s64, qc, qd);
#pragma unroll
                for (int v = 0; v < kWide; ++v) load_row_nc(a.spts_hi + 2 * static_cast<int64_t>(js[v]), ca[v], cb[v]);
#pragma unroll
                for (int v = 0; v < kWide; ++v) d2[v] = d2_continue(d2[v], qc, qd, ca[v], cb[v]);
            }
            uint32_t nh = 0;
#pragma unroll
            for (int v = 0; v < kWide; ++v) {
                ok[v] = ok[v] && d2[v] <= a.r2;
                nh += ok[v];
            }
            if (nh == 0) continue;
            if (stash && hs + nh <= static_cast<uint32_t>(kLeft)) {      // final drain: only note the hits, commit them all at the end
#pragma unroll
                for (int v = 0; v < kWide; ++v)
                    if (ok[v]) { s_left[hs][tid] = make_uint2(static_cast<uint32_t>(cj[v]), __float_as_uint(d2[v])); ++hs; }
                continue;
            }
            uint32_t pos = atomicAdd(&a.cnt[my_row], nh);
            uint32_t pq[kWide];
#pragma unroll
            for (int v = 0; v < kWide; ++v)
                if (ok[v]) pq[v] = atomicAdd(&a.cnt[cj[v]], 1u);
#pragma unroll
            for (int v = 0; v < kWide; ++v)
                if (ok[v]) {
                    const int d2b = __float_as_int(d2[v]);
                    if (pos < kSlot) a.hits[static_cast<int64_t>(my_row) * kSlot + pos] = make_int2(cj[v], d2b);
                    if (pq[v] < kSlot) a.hits[static_cast<int64_t>(cj[v]) * kSlot + pq[v]] = make_int2(my_row, d2b);
                    own_deg += pos < a.k_max;
                    if (pq[v] < a.k_max) atomicAdd(&my_tile_deg[cj[v] / kEmitThreads], 1ull);
                    ++pos;
                }
        }
        if (hs) {                                                        // the noted hits: ONE atomic on my row, the partners' in flight by four
            uint32_t pos = atomicAdd(&a.cnt[my_row], hs);
            for (uint32_t i = 0; i < hs; i += kWide) {
                uint2 e[kWide];
                uint32_t pq[kWide];
#pragma unroll
                for (int v = 0; v < kWide; ++v)
                    if (i + v < hs) { e[v] = s_left[i + v][tid]; pq[v] = atomicAdd(&a.cnt[e[v].x], 1u); }
#pragma unroll
                for (int v = 0; v < kWide; ++v)
                    if (i + v < hs) {
                        const int32_t cjv = static_cast<int32_t>(e[v].x);
                        if (pos < kSlot) a.hits[static_cast<int64_t>(my_row) * kSlot + pos] = make_int2(cjv, static_cast<int>(e[v].y));
                        if (pq[v] < kSlot) a.hits[static_cast<int64_t>(cjv) * kSlot + pq[v]] = make_int2(my_row, static_cast<int>(e[v].y));
                        own_deg += pos < a.k_max;
                        if (pq[v] < a.k_max) atomicAdd(&my_tile_deg[cjv / kEmitThreads], 1ull);
                        ++pos;
                    }
            }
        }
    };
    // a run of candidate slots [j0, j1), kBatch keys in flight
    auto scan_run = [&](uint32_t j0, uint32_t j1) {
        for (; j0 < j1; j0 += kBatch) {
            if (qaddr - q_base > (kQueue - kBatch) * kQBytes) drain();
            const uint32_t* kp = a.skey + j0;
            const uint32_t len = j1 - j0;
            uint32_t kr[kBatch];
#pragma unroll
            for (int v = 0; v < kBatch; ++v) {
                kr[v] = key_fail;
                if (static_cast<uint32_t>(v) < len) kr[v] = kp[v];
            }
#pragma unroll
            for (int v = 0; v < kBatch; ++v) filter_push(qaddr, key_a, kr[v], j0 + v);
        }
    };
    // the merged loop over the listed leftovers: every iteration each lane with work left tests kBatch candidates
    auto scan_leftovers = [&]() {
        uint32_t la = l_base, cj0 = 0, cn = 0;
        while (true) {
            if (cn == 0u) {
                if (la == laddr) break;
                uint32_t x, y;
                asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(x), "=r"(y) : "r"(la));
                cj0 = x; cn = y;
                la += kLBytes;
            }
            if (qaddr - q_base > (kQueue - kBatch) * kQBytes) drain();
            const uint32_t* kp = a.skey + cj0;
            uint32_t kr[kBatch];
#pragma unroll
            for (int v = 0; v < kBatch; ++v) {
                kr[v] = key_fail;
                if (static_cast<uint32_t>(v) < cn) kr[v] = kp[v];
            }
#pragma unroll
            for (int v = 0; v < kBatch; ++v) filter_push(qaddr, key_a, kr[v], cj0 + v);
            cj0 += kBatch;
            cn = cn > kBatch ? cn - kBatch : 0u;
        }
        laddr = l_base;
    };
    // general form: padded table index of cell 0 of the neighbour row with coordinates 0..G-3 offset by the
    // base-3 digits of b (coordinate 0 most significant) and coordinate G-2 by u - 1, all wrapped
    auto row_of = [&](int b, int u) -> uint32_t {
        uint32_t base = cell >> (G * bits);               // event index
#pragma unroll
        for (int d = 0; d < G - 1; ++d) {
            int o;
            if (d < G - 2) o = (b / pow3(G - 3 - d)) % 3 - 1; else o = u - 1;
            const uint32_t cd = (cell >> ((G - 1 - d) * bits)) & mask;
            base = (base << bits) | ((cd + static_cast<uint32_t>(o)) & mask);
        }
        return (base << bits) + base;                     // padded(base << bits)
    };

    for (int b = MID; b < NB; ++b) {
        const bool zero = b == MID;                       // row offsets 0 in coordinates 0..G-3
        uint32_t row[NU];
        if (interior) {
            int delta = 0, bb = b;                        // neighbour row id - own row id for u = 1
#pragma unroll
            for (int d = G - 3; d >= 0; --d) { delta += (bb % 3 - 1) * (1 << ((G - 2 - d) * bits)); bb /= 3; }
            const uint32_t mid_row = own_rowid + static_cast<uint32_t>(delta);
#pragma unroll
            for (int u = 0; u < NU; ++u) {
                const uint32_t rid = mid_row + static_cast<uint32_t>((G >= 2 ? u : 1) - 1);
                row[u] = (rid << bits) + rid;
            }
        } else {
#pragma unroll
            for (int u = 0; u < NU; ++u) row[u] = row_of(b, G >= 2 ? u : 1);
        }
        uint32_t rs[NU], re[NU];
#pragma unroll
        for (int u = 0; u < NU; ++u) {
            const int uu = G >= 2 ? u : 1;
            rs[u] = a.cell_start[row[u] + lo];
            re[u] = a.cell_start[row[u] + hi + 1u];
            if (zero && uu == 1) rs[u] = s + 1u;          // own row: the slots after mine (my cell and the next one)
            if (zero && uu == 0) re[u] = rs[u];           // backward row: its queries come to me
        }
        if (qaddr - q_base > (kQueue - NU * kBatch) * kQBytes) drain();
        uint32_t kc[NU][kBatch];
#pragma unroll
        for (int u = 0; u < NU; ++u) {
            const uint32_t* kp = a.skey + rs[u];          // one 64-bit base per run, immediate offsets
            const uint32_t len = re[u] - rs[u];
#pragma unroll
            for (int v = 0; v < kBatch; ++v) {
                kc[u][v] = key_fail;
                if (static_cast<uint32_t>(v) < len) kc[u][v] = kp[v];
            }
        }
#pragma unroll
        for (int u = 0; u < NU; ++u)
#pragma unroll
            for (int v = 0; v < kBatch; ++v) filter_push(qaddr, key_a, kc[u][v], rs[u] + v);
        // what is left of runs longer than kBatch is listed now and filtered later, in ONE loop for all the rows
        // (the lanes of a warp have their long runs in different rows: merged, they iterate together)
#pragma unroll
        for (int u = 0; u < NU; ++u) leftover_push(laddr, rs[u], re[u] - rs[u]);
        if (laddr - l_base > (kLeft - NU) * kLBytes) scan_leftovers();
    }
    scan_leftovers();
    // Slots whose cell touches the seam of the torus in the last coordinate (only points beyond +-2^(bits-1)
    // cells from the origin) also visit the wrapped cell of every forward row: cold code.
    if (c_last == 0u || c_last == mask) {
        const uint32_t wrap_cell = c_last == 0u ? mask : 0u;
        for (int b = MID; b < NB; ++b)
            for (int u = 0; u < NU; ++u) {
                const int uu = G >= 2 ? u : 1;
                // own row: only the cell after mine is forward; backward row: nothing
                if (b == MID && (uu == 0 || (uu == 1 && c_last != mask))) continue;
                const uint32_t r = row_of(b, uu);
                scan_run(a.cell_start[r + wrap_cell], a.cell_start[r + wrap_cell + 1u]);
            }
    }
    drain(true);
    // per-tile degree totals: emit_kernel turns them into its global offsets without any inter-block wait
    if (own_deg) atomicAdd(&my_tile_deg[my_row / kEmitThreads], static_cast<unsigned long long>(own_deg));
    stamp_end_last(a.stamps, 3, &s_done);
}

// ------------------------------------------------------------------------------------------------
// the brute-force variant (section 3.1: flat-index nearest neighbours followed by
// the radius cut; "brute force ... quadratic").  Every unordered pair of the event is evaluated once
// with the same R3 chain; block (I, J), J >= I, holds 128 queries in registers and 128 candidate rows in shared
// memory (read back as broadcasts).  Hits go through the same slot buffers, counters and per-tile totals as the
// grid path, so emit_kernel (K cap, ordering, compaction) is shared.
// ------------------------------------------------------------------------------------------------
constexpr int kDenseTile = 128;
struct DenseArgs {
    const float* pts;
    int dim;
    uint32_t* cnt;
    int2* hits;
    unsigned long long* tile_deg;
    uint32_t n_tiles;
    int64_t n;
    float r2;
    uint32_t k_max;
};

// Register tiling: a thread holds kDenseQ queries (kDenseQ x 8 floats) and runs their chains against every candidate row
// it reads from shared memory, so the two 128-bit shared loads of a candidate (broadcasts: all lanes read the same row) are
// paid once per kDenseQ pairs -- 16 kDenseQ FP32 instructions per 2 loads instead of 16.  Block (I, J): queries
// [I * kDenseQ * 128, +kDenseQ * 128) x candidates [J * 128, +128); blocks entirely below the diagonal leave at once, blocks
// on it test j > i per pair.
#ifndef FRNN_DENSE_Q
#define FRNN_DENSE_Q 4
#endif
template <bool HI> struct DenseCfg { static constexpr int Q = HI ? 2 : FRNN_DENSE_Q; };

// a hit of the brute-force search (rare: kept out of line so that the pair loop stays tight)
__device__ __noinline__ void dense_hit(const DenseArgs& a, unsigned long long* my_tile_deg, int32_t row, int32_t cj, float d2) {
    const int d2b = __float_as_int(d2);
    const uint32_t p0 = atomicAdd(&a.cnt[row], 1u);
    const uint32_t p1 = atomicAdd(&a.cnt[cj], 1u);
    if (p0 < kSlot) a.hits[static_cast<int64_t>(row) * kSlot + p0] = make_int2(cj, d2b);
    if (p1 < kSlot) a.hits[static_cast<int64_t>(cj) * kSlot + p1] = make_int2(row, d2b);
    if (p0 < a.k_max) atomicAdd(&my_tile_deg[row / kEmitThreads], 1ull);
    if (p1 < a.k_max) atomicAdd(&my_tile_deg[cj / kEmitThreads], 1ull);
}

// kDenseStep candidate rows per step: Q x kDenseStep chains run, ONE predicate collects "some pair is within r" (an FSETP
// per pair that ORs into it, no branch), and only a step that has a hit goes through its pairs again to commit them --
// a branch per step instead of one per pair (hits are rare: 2.3e-5 of the pairs of a tracking event).
#ifndef FRNN_DENSE_STEP
#define FRNN_DENSE_STEP 4
#endif
constexpr int kDenseStep = FRNN_DENSE_STEP;
template <bool HI, bool DIAG, int Q>
__device__ __forceinline__ void dense_pairs(const DenseArgs& a, const float4 (*s_c)[HI ? 4 : 2], const float4* qa, const float4* qb,
                                            const float4* qc, const float4* qd, const int* qrel, int64_t q_lo, int64_t c_lo,
                                            unsigned long long* my_tile_deg, int tid) {
#pragma unroll 1
    for (int k0 = 0; k0 < kDenseTile; k0 += kDenseStep) {
        float d2[kDenseStep][Q];
#pragma unroll
        for (int s = 0; s < kDenseStep; ++s) {
            const float4 ka = s_c[k0 + s][0], kb = s_c[k0 + s][1];
#pragma unroll
            for (int q = 0; q < Q; ++q) d2[s][q] = d2_pinned(qa[q], qb[q], ka, kb);
            if (HI) {
                const float4 kc = s_c[k0 + s][2], kd = s_c[k0 + s][3];
#pragma unroll
                for (int q = 0; q < Q; ++q) d2[s][q] = d2_continue(d2[s][q], qc[q], qd[q], kc, kd);
            }
        }
        bool any = false;
#pragma unroll
        for (int s = 0; s < kDenseStep; ++s)
#pragma unroll
            for (int q = 0; q < Q; ++q) any = any || d2[s][q] <= a.r2;
        if (any) {
#pragma unroll
            for (int s = 0; s < kDenseStep; ++s)
#pragma unroll
                for (int q = 0; q < Q; ++q)
                    if (d2[s][q] <= a.r2 && (!DIAG || k0 + s > qrel[q]))
                        dense_hit(a, my_tile_deg, static_cast<int32_t>(q_lo + q * kDenseTile + tid), static_cast<int32_t>(c_lo + k0 + s), d2[s][q]);
        }
    }
}

template <bool HI>
__global__ void __launch_bounds__(kDenseTile) dense_search_kernel(DenseArgs a) {
    constexpr int Q = DenseCfg<HI>::Q;
    const uint32_t I = blockIdx.y, J = blockIdx.x;
    const int64_t q_lo = static_cast<int64_t>(I) * Q * kDenseTile;            // first query of the block
    const int64_t c_lo = static_cast<int64_t>(J) * kDenseTile;                // first candidate of the block
    if (c_lo + kDenseTile - 1 <= q_lo) return;                                // every candidate <= every query: nothing forward
    __shared__ float4 s_c[kDenseTile][HI ? 4 : 2];
    const int tid = threadIdx.x;
    const float inf = __int_as_float(0x7f800000);
    float4 qa[Q], qb[Q], qc[Q], qd[Q];
    int qrel[Q];                                                              // query index relative to the first candidate (diagonal blocks)
#pragma unroll
    for (int q = 0; q < Q; ++q) {
        const int64_t qi = q_lo + q * kDenseTile + tid;
        const int64_t rel = qi - c_lo;
        qrel[q] = rel < -1 ? -1 : (rel > kDenseTile ? kDenseTile : static_cast<int>(rel));
        qa[q] = make_float4(-inf, 0.f, 0.f, 0.f);                             // queries beyond the event: -inf, never within r of anything
        qb[q] = make_float4(0.f, 0.f, 0.f, 0.f); qc[q] = qb[q]; qd[q] = qb[q];
        if (qi < a.n) {
            load_point(a.pts, qi, a.dim, qa[q], qb[q]);
            if (HI) load_point_hi(a.pts, qi, a.dim, qc[q], qd[q]);
        }
    }
    const int64_t jr = c_lo + tid;
    float4 ca = make_float4(inf, 0.f, 0.f, 0.f), cb = make_float4(0.f, 0.f, 0.f, 0.f), cc = cb, cd = cb;
    if (jr < a.n) {                                                     // rows beyond the event: +inf, never within r
        load_point(a.pts, jr, a.dim, ca, cb);
        if (HI) load_point_hi(a.pts, jr, a.dim, cc, cd);
    }
    s_c[tid][0] = ca; s_c[tid][1] = cb;
    if (HI) { s_c[tid][2] = cc; s_c[tid][3] = cd; }
    __syncthreads();
    unsigned long long* const my_tile_deg = a.tile_deg + static_cast<size_t>(J & (kDegSlices - 1)) * a.n_tiles;
    if (c_lo < q_lo + Q * kDenseTile)                                         // some candidate index <= some query index: test j > i per pair
        dense_pairs<HI, true, Q>(a, s_c, qa, qb, qc, qd, qrel, q_lo, c_lo, my_tile_deg, tid);
    else
        dense_pairs<HI, false, Q>(a, s_c, qa, qb, qc, qd, qrel, q_lo, c_lo, my_tile_deg, tid);
}

// ------------------------------------------------------------------------------------------------
// S9 for calls with many emit tiles (batches, million-point events): exclusive prefix of the per-tile totals in
// ONE block, so that emit_kernel reads one value per block instead of summing all earlier tiles itself (which is
// quadratic in the number of tiles).  Calls with few tiles skip this kernel: one dependent launch less.
// ------------------------------------------------------------------------------------------------
constexpr int kPrefixThreads = 1024;
struct PrefixArgs {
    const unsigned long long* tile_deg;
    uint32_t n_tiles;
    unsigned long long* tile_prefix;
};
__global__ void __launch_bounds__(kPrefixThreads) tile_prefix_kernel(PrefixArgs k) {
    const unsigned long long* __restrict__ tile_deg = k.tile_deg;
    const uint32_t n_tiles = k.n_tiles;
    unsigned long long* __restrict__ tile_prefix = k.tile_prefix;
    __shared__ unsigned long long s_w[kPrefixThreads / 32];
    __shared__ unsigned long long s_carry;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (threadIdx.x == 0) s_carry = 0;
    __syncthreads();
    for (uint32_t c0 = 0; c0 < n_tiles; c0 += kPrefixThreads) {          // chunks of 1024 tiles, coalesced loads
        const uint32_t t = c0 + threadIdx.x;
        unsigned long long part[kDegSlices], mine = 0;
#pragma unroll
        for (int sl = 0; sl < kDegSlices; ++sl) part[sl] = t < n_tiles ? tile_deg[static_cast<size_t>(sl) * n_tiles + t] : 0ull;
#pragma unroll
        for (int sl = 0; sl < kDegSlices; ++sl) mine += part[sl];
        unsigned long long incl = mine;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const unsigned long long x = __shfl_up_sync(kFull, incl, o);
            if (lane >= o) incl += x;
        }
        if (lane == 31) s_w[warp] = incl;
        __syncthreads();
        unsigned long long wsum = lane < kPrefixThreads / 32 ? s_w[lane] : 0ull;   // scan of the 32 warp totals in every warp
        unsigned long long wincl = wsum;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const unsigned long long x = __shfl_up_sync(kFull, wincl, o);
            if (lane >= o) wincl += x;
        }
        const unsigned long long before_warp = __shfl_sync(kFull, wincl - wsum, warp);
        const unsigned long long total = __shfl_sync(kFull, wincl, 31);
        const unsigned long long carry = s_carry;
        if (t < n_tiles) tile_prefix[t] = carry + before_warp + (incl - mine);
        __syncthreads();
        if (threadIdx.x == 0) s_carry = carry + total;
        __syncthreads();
    }
}

// ------------------------------------------------------------------------------------------------
// S8-S10: emit.  Thread per row in ORIGINAL order.  The search pass left sum(min(|S_i|, k_max)) per
// 256-row tile in tile_deg, so a block gets its global edge offset by summing the totals of the
// tiles before it (no inter-block wait), scans its own capped degrees -> CSR row_ptr, and then
// resolves its rows by class (c = |S_i|, the uncapped count; K = k_max; kSlot = 32 hit slots per row):
//   small   c <= K, c <= kSlot   one thread per OUTPUT EDGE: position = rank of dst among the row's stored hits
//   medium  K < c <= kSlot       (S8 from the slot buffer, no recomputation) one thread per STORED HIT: its rank
//                                under (d2, j) among the row's hits decides whether it is kept (rank < K); a second
//                                sweep places the kept hits by dst among the kept
//   big     c > kSlot            the slot buffer overflowed: the row is recomputed by a whole warp, ONE pass over
//                                its neighbourhood; in-radius hits below the current threshold go as 64-bit keys
//                                (d2 bits, j) into the warp's staging buffer in shared memory (kStage entries).
//                                When the buffer fills up (c > kStage) and at the end (c > K) it is pruned to the K
//                                smallest keys by warp_select_keys -- north_star (3): warp-level top-K on (d2, index)
//                                with index tie-break -- and the K-th key becomes the threshold: a streaming top-K
//                                that serves any count as long as K <= kStage / 2.  A bitonic network then orders
//                                the kept keys by dst.
//   huge    c > kStage and K > kStage / 2: threshold by storage-free bisection on the bit pattern of d2 and then on
//                                j among ties (one neighbourhood pass per step), hits written unsorted and ordered
//                                in place by a bitonic network in global memory
// ------------------------------------------------------------------------------------------------
constexpr int kStage = 512;            // staging entries per warp for recomputed rows (K <= 512: 16 keys per lane)
constexpr int kRankMax = 192;          // up to this many kept hits are ordered by rank counting, more by the bitonic network
template <int V> struct IntTag { static constexpr int value = V; };

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

// ascending bitonic sort of the 64-bit keys k[0..p2) in shared memory by one warp; p2 a power of two >= 2, entries
// beyond the data preset to ~0 (keys are < 2^63, so the padding stays at the top)
__device__ __forceinline__ void warp_sort_keys(unsigned long long* k, int p2, int lane) {
    for (int size = 2; size <= p2; size <<= 1) {
        for (int stride = size >> 1; stride >= 1; stride >>= 1) {
            for (int t = lane; t < (p2 >> 1); t += 32) {
                const int lo = ((t & ~(stride - 1)) << 1) | (t & (stride - 1));
                const int hi = lo | stride;
                const unsigned long long x = k[lo], y = k[hi];
                const bool up = (lo & size) == 0;
                if ((x > y) == up) { k[lo] = y; k[hi] = x; }
            }
            __syncwarp();
        }
    }
}

// Warp top-K on staged keys (north_star (3): per-query K-cap selection on (d2, index) with index tie-break): the k
// smallest of the n distinct 64-bit keys key[0..n) (d2 bits << 32 | j, d2 bits <= hi_max) are moved to key[0..k), in no
// particular order, and the k-th smallest key is returned.  Radix select on the bit pattern of d2 (four passes of one byte,
// each a shared-memory histogram over the staged keys that match the bytes fixed so far), then -- only if several keys
// share the k-th d2 and not all of them are wanted -- a bisection on j among those; then a stable in-place compaction.
// n <= kStage, 1 <= k < n; hist: 256 words of the warp.  All lanes must call it; the staged keys are visible (__syncwarp).
__device__ __forceinline__ unsigned long long warp_select_keys(unsigned long long* key, uint32_t n, uint32_t k, uint32_t* hist,
                                                               int lane, uint32_t lt_mask) {
    const uint32_t* w = reinterpret_cast<const uint32_t*>(key);       // w[2t] = j, w[2t+1] = d2 bits (little endian)
    // the k-th smallest d2 by a radix select, one byte per pass from the top: histogram (256 bins of the warp, shared memory)
    // of that byte over the keys that match the bytes fixed so far, then the bin that holds the kk-th of them
    uint32_t prefix = 0, fixed = 0, kk = k, c_eq = 0;
#pragma unroll 1
    for (int shift = 24; shift >= 0; shift -= 8) {
        // (128-bit accesses: zeroing and reading the lane's 8 bins word by word put the 32 lanes on 4 banks -- an 8-way
        // conflict on each of 16 instructions per pass, which was most of the kernel's shared-memory wavefronts)
        uint4* hist4 = reinterpret_cast<uint4*>(hist);
        hist4[lane] = make_uint4(0u, 0u, 0u, 0u);
        hist4[lane + 32] = make_uint4(0u, 0u, 0u, 0u);
        __syncwarp();
        for (uint32_t t = lane; t < n; t += 32) {
            const uint32_t d = w[2 * t + 1];
            if ((d & fixed) == prefix) atomicAdd(&hist[(d >> shift) & 255u], 1u);
        }
        __syncwarp();
        uint32_t loc[8], sum = 0;
        {
            const uint4 lo4 = hist4[2 * lane], hi4 = hist4[2 * lane + 1];
            loc[0] = lo4.x; loc[1] = lo4.y; loc[2] = lo4.z; loc[3] = lo4.w;
            loc[4] = hi4.x; loc[5] = hi4.y; loc[6] = hi4.z; loc[7] = hi4.w;
        }
#pragma unroll
        for (int b = 0; b < 8; ++b) sum += loc[b];
        uint32_t incl = sum;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t x = __shfl_up_sync(kFull, incl, o);
            if (lane >= o) incl += x;
        }
        const uint32_t excl = incl - sum;
        const bool mine = excl < kk && kk <= incl;                    // exactly one lane holds the kk-th key
        uint32_t bin = 0, before = excl, inbin = 0;
        if (mine) {
#pragma unroll
            for (int b = 0; b < 8; ++b) {
                if (before < kk && kk <= before + loc[b]) { bin = static_cast<uint32_t>(lane * 8 + b); inbin = loc[b]; break; }
                before += loc[b];
            }
        }
        const int src = __ffs(__ballot_sync(kFull, mine)) - 1;
        bin = __shfl_sync(kFull, bin, src);
        before = __shfl_sync(kFull, before, src);
        c_eq = __shfl_sync(kFull, inbin, src);
        prefix |= bin << shift;
        fixed |= 255u << shift;
        kk -= before;
        __syncwarp();
    }
    const uint32_t dk = prefix;                                       // the k-th smallest d2; c_eq keys share it
    const uint32_t need = kk;                                         // how many of those are wanted (>= 1)
    uint32_t jk = 0x7fffffffu;
    if (need < c_eq) {                                                // ties at the k-th d2: the smallest indices win
        uint32_t jlo = 0, jhi = 0x7fffffffu;
        while (jlo < jhi) {
            const uint32_t mid = jlo + ((jhi - jlo) >> 1);
            uint32_t c = 0;
            for (uint32_t t = lane; t < n; t += 32) c += (w[2 * t + 1] == dk) && (w[2 * t] <= mid);
            c = __reduce_add_sync(kFull, c);
            if (c >= need) jhi = mid; else jlo = mid + 1;
        }
        jk = jlo;
    }
    const unsigned long long thr = (static_cast<unsigned long long>(dk) << 32) | jk;
    // compaction, 32 keys at a time in index order: everything a chunk writes lies at or before the chunk itself
    uint32_t out = 0;
    for (uint32_t t0 = 0; t0 < n; t0 += 32) {
        const uint32_t t = t0 + lane;
        const unsigned long long v = t < n ? key[t] : ~0ull;
        const bool keep = v <= thr;
        const uint32_t m = __ballot_sync(kFull, keep);
        __syncwarp();
        if (keep) key[out + __popc(m & lt_mask)] = v;
        out += __popc(m);
        __syncwarp();
    }
    return thr;
}

struct EmitArgs {
    const float* pts;             // original points (to recompute the cell of a big row), n x dim
    int dim;
    const float4* spts;
    const float4* spts_hi;        // coordinates 8..15 of the slots (dim > 8), else NULL
    const int32_t* sidx;
    const uint32_t* cell_start;
    const uint32_t* cnt;
    const int2* hits;
    const unsigned long long* tile_deg;
    const unsigned long long* tile_prefix;   // exclusive prefix of the tile totals (tile_prefix_kernel), or NULL: sum in the block
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
    unsigned long long* stamps;   // NULL unless the timeline is being recorded
    float r2, inv_cell;
    int bits;
    uint32_t k_max;
    uint32_t n_tiles;             // number of emit tiles (= the launch grid unless the grid was rounded up)
    int dense;                    // 1: no grid exists (frnn_build_dense_ex): recomputed rows scan their whole event
    BinOrder order;
};

template <int G, bool INTERIOR>
__device__ __forceinline__ void emit_big_row(const EmitArgs& a, int64_t row, int64_t row_rp, int64_t row_ev, uint32_t row_cnt,
                                          uint32_t cell, const float4& qa, const float4& qb, int* s_delta,
                                          unsigned long long* stage, uint32_t* hist, int lane, int lane_delta, uint32_t lt_mask) {
    const float inf = __int_as_float(0x7f800000);
    const bool hi = a.dim > kDim;                         // coordinates 8..15 exist: the chain goes on over them
    float4 qc = make_float4(0.f, 0.f, 0.f, 0.f), qd = qc;
    if (hi) load_point_hi(a.pts, row, a.dim, qc, qd);
    // visit(g): g(in_radius, j, d2) once per chunk, one candidate per lane
    auto visit = [&](auto&& g) {
        if (a.dense) {                                    // every row of the event, 32 at a time, in original order
            const int64_t ev_end = a.ev_off ? a.ev_off[event_of_row(a.ev_off, a.n_events, row) + 1] : a.n_total;
            for (int64_t j0 = row_ev; j0 < ev_end; j0 += 32) {
                const int64_t j = j0 + lane;
                float4 ca = make_float4(inf, 0.f, 0.f, 0.f), cb = make_float4(0.f, 0.f, 0.f, 0.f);
                if (j < ev_end) load_point(a.pts, j, a.dim, ca, cb);
                float d2 = d2_pinned(qa, qb, ca, cb);
                if (hi) {
                    float4 cc = make_float4(0.f, 0.f, 0.f, 0.f), cd = cc;
                    if (j < ev_end) load_point_hi(a.pts, j, a.dim, cc, cd);
                    d2 = d2_continue(d2, qc, qd, cc, cd);
                }
                g(j < ev_end && d2 <= a.r2 && j != row, static_cast<int32_t>(j), d2);
            }
            return;
        }
        for_each_candidate_chunk<G, INTERIOR>(cell, a.bits, lane_delta, a.cell_start, s_delta, lane, [&](int cslot) {
            float4 ca = make_float4(inf, 0.f, 0.f, 0.f), cb = make_float4(0.f, 0.f, 0.f, 0.f);
            int32_t cj = -1;
            if (cslot >= 0) {
                ca = a.spts[2 * static_cast<int64_t>(cslot)];
                cb = a.spts[2 * static_cast<int64_t>(cslot) + 1];
                cj = a.sidx[cslot];
            }
            float d2 = d2_pinned(qa, qb, ca, cb);
            if (hi) {
                float4 cc = make_float4(0.f, 0.f, 0.f, 0.f), cd = cc;
                if (cslot >= 0) { cc = a.spts_hi[2 * static_cast<int64_t>(cslot)]; cd = a.spts_hi[2 * static_cast<int64_t>(cslot) + 1]; }
                d2 = d2_continue(d2, qc, qd, cc, cd);
            }
            g(d2 <= a.r2 && cj != static_cast<int32_t>(row), cj, d2);
        });
    };
    const int32_t src = static_cast<int32_t>(row - row_ev);
    const uint32_t kept = row_cnt < a.k_max ? row_cnt : a.k_max;

    if (row_cnt <= static_cast<uint32_t>(kStage) || a.k_max <= static_cast<uint32_t>(kStage / 2)) {
        // ---- ONE pass: an in-radius hit becomes a key (d2 bits << 32 | j) in the staging buffer if it is below the current
        // threshold (initially none).  d2 >= +0 always (the chain starts at +0 and adds squares), so bit patterns order
        // like values and the key order IS (d2, j); keys are distinct (j is).  When the buffer is about to fill up, it is
        // pruned to the K smallest keys (warp_select_keys) and the K-th becomes the threshold: a streaming top-K, any count.
        uint32_t fill = 0;
        unsigned long long thr = ~0ull;
        visit([&](bool in, int32_t cj, float d2) {
            const unsigned long long key = (static_cast<unsigned long long>(__float_as_uint(d2)) << 32) | static_cast<uint32_t>(cj);
            const bool take = in && key < thr;
            const uint32_t m = __ballot_sync(kFull, take);
            if (take) {
                const uint32_t at = fill + __popc(m & lt_mask);
                if (at < static_cast<uint32_t>(kStage)) stage[at] = key;
            }
            fill += __popc(m);
            if (fill > static_cast<uint32_t>(kStage - 32) && fill > a.k_max) {       // (K <= kStage / 2 here, or the row would fit)
                __syncwarp();
                thr = warp_select_keys(stage, fill < static_cast<uint32_t>(kStage) ? fill : static_cast<uint32_t>(kStage), a.k_max,
                                       hist, lane, lt_mask);
                fill = a.k_max;
            }
        });
        __syncwarp();
        if (fill > static_cast<uint32_t>(kStage)) fill = kStage;                     // (cannot happen: see the prune condition)
        if (fill > a.k_max) {                             // S8: the K smallest keys
            warp_select_keys(stage, fill, a.k_max, hist, lane, lt_mask);
            fill = a.k_max;
        }
        const uint32_t len = fill;
        // ---- order the kept hits by dst.  Up to kRankMax of them: every lane ranks its (at most kRankMax / 32) hits by counting
        // the kept hits with a smaller j -- one broadcast shared load per kept hit, no dependent chain -- and stores each at
        // its rank (the stores of a row fall into one window of a few hundred bytes).  More: keys (j << 32 | d2 bits) through
        // the bitonic network, coalesced stores.
        if (len <= static_cast<uint32_t>(kRankMax)) {
            const uint32_t* w = reinterpret_cast<const uint32_t*>(stage);   // w[2t] = j, w[2t+1] = d2 bits
            auto rank_and_store = [&](auto e_tag) {
                constexpr int E = decltype(e_tag)::value;                   // kept hits per lane
                uint32_t myj[E], rank[E];
#pragma unroll
                for (int e = 0; e < E; ++e) {
                    const uint32_t t = lane + 32u * e;
                    myj[e] = t < len ? w[2 * t] : 0xffffffffu;
                    rank[e] = 0u;
                }
#pragma unroll 4
                for (uint32_t u = 0; u < len; ++u) {
                    const uint32_t ju = w[2 * u];
#pragma unroll
                    for (int e = 0; e < E; ++e) rank[e] += ju < myj[e];
                }
#pragma unroll
                for (int e = 0; e < E; ++e) {
                    const uint32_t t = lane + 32u * e;
                    const int64_t pos = row_rp + rank[e];
                    if (t < len && pos < a.capacity) {
                        a.out_src[pos] = src;
                        a.out_dst[pos] = static_cast<int32_t>(myj[e]) - static_cast<int32_t>(row_ev);
                        a.out_d2[pos] = __uint_as_float(w[2 * t + 1]);
                    }
                }
            };
            if (len <= 64u) rank_and_store(IntTag<2>{});
            else            rank_and_store(IntTag<kRankMax / 32>{});
            __syncwarp();
            return;
        }
        int p2 = 2;
        while (static_cast<uint32_t>(p2) < len) p2 <<= 1;
        for (int t = lane; t < p2; t += 32) {
            const unsigned long long v = stage[t];
            stage[t] = static_cast<uint32_t>(t) < len ? ((v << 32) | (v >> 32)) : ~0ull;
        }
        __syncwarp();
        warp_sort_keys(stage, p2, lane);
        for (uint32_t t = lane; t < len; t += 32) {       // coalesced stores
            const unsigned long long v = stage[t];
            const int64_t pos = row_rp + t;
            if (pos < a.capacity) {
                a.out_src[pos] = src;
                a.out_dst[pos] = static_cast<int32_t>(v >> 32) - static_cast<int32_t>(row_ev);
                a.out_d2[pos] = __uint_as_float(static_cast<uint32_t>(v));
            }
        }
        __syncwarp();
        return;
    }

    // ---- beyond the staging capacity.  Threshold key (dthr, jthr): keep hits with (d2 bits, j) <= it.
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
    if (row_rp + static_cast<int64_t>(kept) <= a.capacity)   // rows cut by the capacity stay unsorted
        warp_sort_rows(a.out_dst + row_rp, a.out_d2 + row_rp, kept, lane);
    __syncwarp();
}

template <int G>
__global__ void __launch_bounds__(kEmitThreads, 1024 / kEmitThreads) emit_kernel(EmitArgs a) {
    __shared__ unsigned long long s_rp[kEmitThreads + 1];  // offsets of the tile's rows inside the tile (capped degrees)
    __shared__ unsigned long long s_warp[kEmitThreads / 32];
    __shared__ unsigned long long s_prefix;
    __shared__ int32_t s_evb[kEmitThreads];                // first row of the event of every row (batched calls)
    __shared__ uint32_t s_bigmask[kEmitThreads / 32];      // rows that the edge-parallel sweep skips (medium, big, huge)
    __shared__ int s_delta[kEmitThreads / 32][32];
    __shared__ uint32_t s_mp[kEmitThreads + 1];            // medium rows: offsets of their STORED hits inside the tile
    __shared__ uint32_t s_kept[kEmitThreads];              // medium rows: bit h set = stored hit h is among the K nearest
    __shared__ uint32_t s_mwarp[kEmitThreads / 32];
    __shared__ unsigned long long s_stage[kEmitThreads / 32][kStage];   // big rows: per-warp staging of (d2, j) keys
    __shared__ __align__(16) uint32_t s_hist[kEmitThreads / 32][256];                 // big rows: per-warp histogram of the radix select
    __shared__ unsigned int s_done;                        // timeline only: threads of the block that have finished
    if (threadIdx.x == 0) s_done = 0u;                     // (made visible by the barriers below)
    stamp_begin(a.stamps, 4);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t lt_mask = (1u << lane) - 1u;
    const uint32_t tile = blockIdx.x;
    if (tile >= a.n_tiles) return;
    const int64_t tile_row0 = static_cast<int64_t>(tile) * kEmitThreads;
    const int64_t i = tile_row0 + threadIdx.x;
    const bool has = i < a.n_total;
    const uint32_t c = has ? a.cnt[i] : 0u;
    const uint32_t deg = c < a.k_max ? c : a.k_max;
    // ---- global offset of the tile = sum of the totals of the tiles before it
    unsigned long long before = (a.tile_prefix && threadIdx.x == 0) ? a.tile_prefix[tile] : 0ull;
    for (uint32_t t = threadIdx.x; t < (a.tile_prefix ? 0u : tile); t += kEmitThreads) {
        unsigned long long part[kDegSlices];
#pragma unroll
        for (int sl = 0; sl < kDegSlices; ++sl) part[sl] = a.tile_deg[static_cast<size_t>(sl) * a.n_tiles + t];      // all in flight
#pragma unroll
        for (int sl = 0; sl < kDegSlices; ++sl) before += part[sl];
    }
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
        for (int o = 16; o >= 1; o >>= 1) b += __shfl_xor_sync(kFull, b, o);
        if (lane == 0) s_prefix = b;
    }
    __syncthreads();
    if (lane == 31) s_warp[warp] = incl;                   // warp totals of deg
    __syncthreads();
    unsigned long long wexcl = 0;
#pragma unroll
    for (int w = 0; w < kEmitThreads / 32; ++w) wexcl += (w < warp) ? s_warp[w] : 0ull;
    const unsigned long long local_rp = wexcl + (incl - deg);
    const unsigned long long tile_base = s_prefix;
    const int64_t rp = static_cast<int64_t>(tile_base + local_rp);                 // row_ptr[i]
    const bool big = has && c > kSlot;                     // recomputed by a whole warp
    const bool medium = has && c > a.k_max && c <= kSlot;  // K-cap selection from the slot buffer
    s_rp[threadIdx.x] = local_rp;
    if (threadIdx.x == kEmitThreads - 1) s_rp[kEmitThreads] = local_rp + deg;
    const uint32_t bigs_warp = __ballot_sync(kFull, big);
    const uint32_t skip_warp = __ballot_sync(kFull, big || medium);
    if (lane == 0) s_bigmask[warp] = skip_warp;
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
    s_evb[threadIdx.x] = static_cast<int32_t>(ev_base);
    // medium rows exist only when K < kSlot (block-uniform test first: the usual K costs nothing here)
    const bool any_medium = a.k_max < static_cast<uint32_t>(kSlot) && __syncthreads_or(medium ? 1 : 0) != 0;
    if (any_medium) {                                      // block scan of the stored-hit counts of the medium rows
        const uint32_t mc = medium ? c : 0u;
        uint32_t mi = mc;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t t = __shfl_up_sync(kFull, mi, o);
            if (lane >= o) mi += t;
        }
        if (lane == 31) s_mwarp[warp] = mi;
        s_kept[threadIdx.x] = 0u;
        __syncthreads();
        uint32_t mexcl = 0;
#pragma unroll
        for (int w = 0; w < kEmitThreads / 32; ++w) mexcl += (w < warp) ? s_mwarp[w] : 0u;
        s_mp[threadIdx.x] = mexcl + (mi - mc);
        if (threadIdx.x == kEmitThreads - 1) s_mp[kEmitThreads] = mexcl + mi;
    }
    __syncthreads();
    // ---- rows that fit their slot buffer, ONE THREAD PER OUTPUT EDGE: edge p of the tile belongs to the row r
    // with s_rp[r] <= p < s_rp[r+1] (binary search in shared memory), is the row's hit number m = p - s_rp[r],
    // and goes to position rank(dst among the row's hits): no sort, coalesced work, the COO comes out sorted.
    const unsigned long long tile_edges = s_rp[kEmitThreads];
    for (unsigned long long p = threadIdx.x; p < tile_edges; p += kEmitThreads) {
        int r = 0;
#pragma unroll
        for (int step = kEmitThreads / 2; step >= 1; step >>= 1)
            if (s_rp[r + step] <= p) r += step;
        if ((s_bigmask[r >> 5] >> (r & 31)) & 1u) continue;            // medium / big: resolved below
        const unsigned long long r0 = s_rp[r];
        const uint32_t cr = static_cast<uint32_t>(s_rp[r + 1] - r0);   // = uncapped count (the row is small)
        const uint32_t m = static_cast<uint32_t>(p - r0);
        const int64_t row = tile_row0 + r;
        const int2* h = a.hits + row * kSlot;
        const int4 v0 = *reinterpret_cast<const int4*>(h);             // hits 0..3 and mine: three loads in flight (the
        const int4 v1 = *reinterpret_cast<const int4*>(h + 2);         // slot buffer is padded, unused slots are masked)
        const int2 mine = h[m];
        uint32_t rank = (v0.x < mine.x) + (1u < cr && v0.z < mine.x) + (2u < cr && v1.x < mine.x) + (3u < cr && v1.z < mine.x);
        for (uint32_t u = 4; u < cr; u += 2) {                         // two hits per 16-byte load
            const int4 v = *reinterpret_cast<const int4*>(h + u);
            rank += (v.x < mine.x) + (u + 1 < cr && v.z < mine.x);
        }
        const int64_t pos = static_cast<int64_t>(tile_base + r0) + rank;
        if (pos < a.capacity) {
            const int32_t eb = s_evb[r];
            a.out_src[pos] = static_cast<int32_t>(row) - eb;
            a.out_dst[pos] = mine.x - eb;
            a.out_d2[pos] = __int_as_float(mine.y);
        }
    }
    // ---- medium rows (K < c <= kSlot): S8 from the slot buffer, ONE THREAD PER STORED HIT.  Sweep 1: the rank of my hit
    // under (d2 bits, j) among the row's c hits (keys are distinct: j is); rank < K = kept, noted as a bit of the row's
    // word.  Sweep 2: a kept hit goes to position (number of kept hits of the row with a smaller dst).
    if (any_medium) {
        const uint32_t med_total = s_mp[kEmitThreads];
        for (int sweep = 0; sweep < 2; ++sweep) {
            for (uint32_t q = threadIdx.x; q < med_total; q += kEmitThreads) {
                int r = 0;
#pragma unroll
                for (int step = kEmitThreads / 2; step >= 1; step >>= 1)
                    if (s_mp[r + step] <= q) r += step;
                const uint32_t hnum = q - s_mp[r];
                const uint32_t cr = s_mp[r + 1] - s_mp[r];
                const int64_t row = tile_row0 + r;
                const int2* h = a.hits + row * kSlot;
                const int2 mine = h[hnum];
                if (sweep == 0) {
                    const unsigned long long mykey = (static_cast<unsigned long long>(static_cast<uint32_t>(mine.y)) << 32) | static_cast<uint32_t>(mine.x);
                    uint32_t rank = 0;
                    for (uint32_t u = 0; u < cr; u += 2) {             // two hits per 16-byte load (slot buffer padded to kSlot)
                        const int4 v = *reinterpret_cast<const int4*>(h + u);
                        const unsigned long long k0 = (static_cast<unsigned long long>(static_cast<uint32_t>(v.y)) << 32) | static_cast<uint32_t>(v.x);
                        const unsigned long long k1 = (static_cast<unsigned long long>(static_cast<uint32_t>(v.w)) << 32) | static_cast<uint32_t>(v.z);
                        rank += (k0 < mykey) + (u + 1 < cr && k1 < mykey);
                    }
                    if (rank < a.k_max) atomicOr(&s_kept[r], 1u << hnum);
                } else {
                    const uint32_t kept = s_kept[r];
                    if (!((kept >> hnum) & 1u)) continue;
                    uint32_t rank = 0;
                    for (uint32_t u = 0; u < cr; u += 2) {
                        const int4 v = *reinterpret_cast<const int4*>(h + u);
                        rank += (((kept >> u) & 1u) && v.x < mine.x) + (((kept >> (u + 1)) & 1u) && v.z < mine.x);
                    }
                    const int64_t pos = static_cast<int64_t>(tile_base + s_rp[r]) + rank;
                    if (pos < a.capacity) {
                        const int32_t eb = s_evb[r];
                        a.out_src[pos] = static_cast<int32_t>(row) - eb;
                        a.out_dst[pos] = mine.x - eb;
                        a.out_d2[pos] = __int_as_float(mine.y);
                    }
                }
            }
            __syncthreads();
        }
    }
    // ---- big rows: recompute with the whole warp
    uint32_t bigs = bigs_warp;
    if (bigs != 0) {
        int lane_delta = lane_row_delta<G>(lane, a.bits);
        const uint32_t mask = (1u << a.bits) - 1u;
        for (; bigs; bigs &= bigs - 1) {
            const int bl = __ffs(bigs) - 1;
            const int64_t row = __shfl_sync(kFull, i, bl);
            const int64_t row_rp = __shfl_sync(kFull, rp, bl);
            const int64_t row_ev = __shfl_sync(kFull, ev_base, bl);
            const uint32_t row_cnt = __shfl_sync(kFull, c, bl);
            float4 qa, qb;
            load_point(a.pts, row, a.dim, qa, qb);
            uint32_t ev = 0;
            if (a.ev_off) ev = static_cast<uint32_t>(event_of_row(a.ev_off, a.n_events, row));
            const uint32_t cell = a.order.on ? cell_ordered<G>(a.pts + row * a.dim, a.dim, ev, a.inv_cell, a.bits, a.order)
                                             : cell_of_point<G>(qa, qb, ev, a.inv_cell, a.bits);
            bool interior = true;
#pragma unroll
            for (int d = 0; d < G; ++d) {
                const uint32_t cd = (cell >> (d * a.bits)) & mask;
                interior = interior && cd != 0u && cd != mask;
            }
            if (interior) emit_big_row<G, true>(a, row, row_rp, row_ev, row_cnt, cell, qa, qb, s_delta[warp], s_stage[warp], s_hist[warp], lane, lane_delta, lt_mask);
            else          emit_big_row<G, false>(a, row, row_rp, row_ev, row_cnt, cell, qa, qb, s_delta[warp], s_stage[warp], s_hist[warp], lane, lane_delta, lt_mask);
        }
    }
    stamp_end_last(a.stamps, 4, &s_done);
}

}  // namespace frnn
