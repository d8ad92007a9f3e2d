// frnn_kernels.cuh -- device code of the B200 FRNN path (sm_100a).  Product code: shares nothing
// with oracle/.  Steps S2..S10 of SURVEY.md section 8(a); design notes in DESIGN.md section 6.
//
//   bin_kernel      S2  cell index on a toroidal grid over the first G coordinates + histogram
//   scan_kernel     S3/S9 single-pass decoupled look-back scan (cells -> cell_start + segment list;
//                   capped degrees -> CSR row_ptr)
//   scatter_kernel  S4  counting-sort scatter into the cell-ordered copy
//   search_kernel   S5..S8,S10 one warp per occupied cell ("segment"): neighbour runs are
//                   flattened across lanes, every lane evaluates whole 8-term FMA chains
//   sort_rows_kernel S10 per-row ordering by dst + call epilogue (count, status, edge offsets)
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
// ------------------------------------------------------------------------------------------------
constexpr float kCoordClamp = 32768.0f;

__device__ __forceinline__ uint32_t cell_coord(float x, float inv_cell, uint32_t mask) {
    float a = __fmul_rn(x, inv_cell);
    a = fminf(fmaxf(a, -kCoordClamp), kCoordClamp);   // NaN -> -clamp: never out of bounds
    return static_cast<uint32_t>(__float2int_rd(a)) & mask;
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
    const uint32_t mask = (1u << bits) - 1u;
    const float4 a = pts[2 * i];
    float4 b = make_float4(0.f, 0.f, 0.f, 0.f);
    if (G > 4) b = pts[2 * i + 1];
    const float x[8] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w};
    uint32_t lin = ev_off ? static_cast<uint32_t>(event_of_row(ev_off, n_events, i)) : 0u;
#pragma unroll
    for (int d = 0; d < G; ++d) lin = (lin << bits) | cell_coord(x[d], inv_cell, mask);
    pcell[i] = lin;
    prank[i] = atomicAdd(&cell_count[lin], 1u);
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
// S3 / S9: single-pass exclusive scan with decoupled look-back.  One 64-bit descriptor per tile:
// [63:62] flag (0 = not ready, 1 = tile aggregate, 2 = inclusive prefix), [61:0] value.
// Tiles take their index from an atomic ticket, so a tile only ever waits on tiles that have
// already started (no dependence on block scheduling order).
// ------------------------------------------------------------------------------------------------
constexpr int kScanThreads = 512;
constexpr int kScanItems = 8;
constexpr int kScanTile = kScanThreads * kScanItems;
constexpr uint64_t kFlagA = 1ull << 62, kFlagP = 2ull << 62, kValMask = (1ull << 62) - 1;

__device__ __forceinline__ uint64_t ld_volatile_u64(const uint64_t* p) {
    uint64_t v;
    asm volatile("ld.volatile.global.u64 %0, [%1];" : "=l"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ void st_volatile_u64(uint64_t* p, uint64_t v) {
    asm volatile("st.volatile.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

struct Segment {          // one occupied cell: the unit of work of the search kernels
    uint32_t cell;        // linear cell id (event index in the high bits)
    uint32_t start;       // first slot in the cell-ordered copy
    uint32_t len;         // points in the cell
    uint32_t pad;
};

// Policy A: cell histogram -> cell_start (in place) + compacted list of occupied cells.
// Value packs (occupied cells so far) << 32 | (points so far).
struct CellScan {
    uint32_t* cells;          // in: counts, out: exclusive starts; [n] = total
    Segment* segs;
    uint32_t* n_segs;
    __device__ __forceinline__ uint64_t value(uint32_t v) const { return (static_cast<uint64_t>(v != 0) << 32) | v; }
    __device__ __forceinline__ uint32_t load(int64_t i) const { return cells[i]; }
    __device__ __forceinline__ void store(int64_t i, uint32_t v, uint64_t excl) const {
        cells[i] = static_cast<uint32_t>(excl);
        if (v) segs[excl >> 32] = Segment{static_cast<uint32_t>(i), static_cast<uint32_t>(excl), v, 0u};
    }
    __device__ __forceinline__ void finish(int64_t n, uint64_t total) const {
        cells[n] = static_cast<uint32_t>(total);
        *n_segs = static_cast<uint32_t>(total >> 32);
    }
};

// Policy B: uncapped per-row counts -> CSR row_ptr of min(count, k_max)  (S9).
struct DegreeScan {
    const uint32_t* cnt;
    int64_t* row_ptr;         // [n+1]
    uint32_t k_max;
    __device__ __forceinline__ uint64_t value(uint32_t v) const { return v < k_max ? v : k_max; }
    __device__ __forceinline__ uint32_t load(int64_t i) const { return cnt[i]; }
    __device__ __forceinline__ void store(int64_t i, uint32_t, uint64_t excl) const { row_ptr[i] = static_cast<int64_t>(excl); }
    __device__ __forceinline__ void finish(int64_t n, uint64_t total) const { row_ptr[n] = static_cast<int64_t>(total); }
};

template <class Policy>
__global__ void __launch_bounds__(kScanThreads) scan_kernel(Policy p, int64_t n, uint64_t* tile_state, uint32_t* ticket) {
    __shared__ uint64_t s_warp[kScanThreads / 32];
    __shared__ uint64_t s_prefix;
    __shared__ uint32_t s_tile;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (threadIdx.x == 0) s_tile = atomicAdd(ticket, 1u);
    __syncthreads();
    const uint32_t tile = s_tile;
    const int64_t base = static_cast<int64_t>(tile) * kScanTile + static_cast<int64_t>(threadIdx.x) * kScanItems;
    uint32_t v[kScanItems];
    uint64_t tsum = 0;
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) {
        v[k] = (base + k < n) ? p.load(base + k) : 0u;
        tsum += p.value(v[k]);
    }
    uint64_t incl = tsum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        uint64_t t = __shfl_up_sync(kFull, incl, o);
        if (lane >= o) incl += t;
    }
    if (lane == 31) s_warp[warp] = incl;
    __syncthreads();
    uint64_t wexcl = 0, btotal = 0;
#pragma unroll
    for (int w = 0; w < kScanThreads / 32; ++w) {
        uint64_t t = s_warp[w];
        if (w < warp) wexcl += t;
        btotal += t;
    }
    if (warp == 0) {
        uint64_t excl = 0;
        if (lane == 0) st_volatile_u64(&tile_state[tile], (tile == 0 ? kFlagP : kFlagA) | btotal);
        if (tile > 0) {
            int look = static_cast<int>(tile) - 1;
            while (true) {
                const int t = look - lane;
                uint64_t st = kFlagP;                                  // virtual tile -1: prefix 0
                if (t >= 0) {
                    do { st = ld_volatile_u64(&tile_state[t]); } while ((st >> 62) == 0);
                }
                const uint32_t pmask = __ballot_sync(kFull, (st >> 62) == 2);
                const int first_p = pmask ? (__ffs(pmask) - 1) : 31;
                uint64_t val = (lane <= first_p) ? (st & kValMask) : 0ull;
#pragma unroll
                for (int o = 16; o >= 1; o >>= 1) val += __shfl_xor_sync(kFull, val, o);
                excl += val;
                if (pmask) break;
                look -= 32;
            }
            if (lane == 0) st_volatile_u64(&tile_state[tile], kFlagP | (excl + btotal));
        }
        if (lane == 0) s_prefix = excl;
    }
    __syncthreads();
    uint64_t run = s_prefix + wexcl + (incl - tsum);
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) {
        if (base + k < n) {
            p.store(base + k, v[k], run);
            run += p.value(v[k]);
            if (base + k == n - 1) p.finish(n, run);
        }
    }
}

// ------------------------------------------------------------------------------------------------
// S5: neighbour-cell enumeration for one occupied cell.  The last binned coordinate is the
// fastest-varying one in the linear cell id, so its three adjacent cells are ONE contiguous run of
// the cell-ordered copy: 3^G cells = 3^(G-1) runs.  Up to 27 runs live in lanes (one per lane);
// G > 4 loops over 3^(G-4) run groups.  Runs of a group are flattened: an inclusive warp scan of
// the run lengths, then each lane finds "its" candidate of the current 32-chunk by a 5-step
// shuffle search.  f(valid, slot) is called once per chunk with one candidate slot per lane.
// A cell on the 0 / 2^bits-1 face of the last coordinate has its wrapped neighbour in a second
// pass ("piece 1").
// ------------------------------------------------------------------------------------------------
__host__ __device__ constexpr int pow3(int e) { return e <= 0 ? 1 : 3 * pow3(e - 1); }

template <int G, class F>
__device__ __forceinline__ void for_each_candidate_chunk(uint32_t cell, int bits, const uint32_t* __restrict__ cell_start,
                                                         int lane, F&& f) {
    constexpr int LD = (G - 1 < 3) ? (G - 1) : 3;     // coordinates enumerated across lanes
    constexpr int RL = pow3(LD);                      // runs per group (<= 27)
    constexpr int GD = G - 1 - LD;                    // coordinates enumerated by the group loop
    constexpr int NG = pow3(GD);
    const uint32_t mask = (1u << bits) - 1u;
    const uint32_t c_last = cell & mask;
    const bool edge_lo = c_last == 0u, edge_hi = c_last == mask;
    const int n_pieces = (edge_lo || edge_hi) ? 2 : 1;
    const uint32_t ev = cell >> (G * bits);
    for (int grp = 0; grp < NG; ++grp) {
        uint32_t base = ev;
        {
            int kk = lane, gg = grp;
#pragma unroll
            for (int d = 0; d < G - 1; ++d) {
                int o;
                if (d < GD) { o = gg % 3 - 1; gg /= 3; } else { o = kk % 3 - 1; kk /= 3; }
                const uint32_t cd = (cell >> ((G - 1 - d) * bits)) & mask;
                base = (base << bits) | ((cd + static_cast<uint32_t>(o)) & mask);
            }
            base <<= bits;
        }
        for (int piece = 0; piece < n_pieces; ++piece) {
            uint32_t lo, hi;
            if (piece == 0) { lo = edge_lo ? 0u : c_last - 1u; hi = edge_hi ? mask : c_last + 1u; }
            else            { lo = hi = edge_lo ? mask : 0u; }
            uint32_t s = 0, e = 0;
            if (lane < RL) { s = cell_start[base + lo]; e = cell_start[base + hi + 1u]; }
            const int len = static_cast<int>(e - s);
            int incl = len;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                int t = __shfl_up_sync(kFull, incl, o);
                if (lane >= o) incl += t;
            }
            const int total = __shfl_sync(kFull, incl, 31);
            const int delta = static_cast<int>(s) - (incl - len);     // slot = t + delta for t in this run
            for (int b = 0; b < total; b += 32) {
                const int t = b + lane;
                int k = 0;
#pragma unroll
                for (int step = 16; step >= 1; step >>= 1) {
                    const int pk = __shfl_sync(kFull, incl, (k + step - 1) & 31);
                    if (pk <= t) k += step;
                }
                const int slot = t + __shfl_sync(kFull, delta, k & 31);
                f(t < total, slot);
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------
// S6..S8, S10: search.  One warp per segment (occupied cell), persistent grid-stride over the
// segment list.  Queries = the cell's points (<= 32 per pass), staged once in shared memory and
// read back as broadcasts; candidates = one per lane per chunk.  PASS 0 counts |S_i| (uncapped);
// PASS 1 writes the kept hits of every row with |S_i| <= k_max unsorted at row_ptr[i] (the row is
// ordered by dst in sort_rows_kernel) and resolves overflowing rows with a storage-free exact
// selection: bisection on the bit pattern of d2, then on j among ties (S8).
// ------------------------------------------------------------------------------------------------
constexpr int kSearchWarps = 8;

struct SearchArgs {
    const float4* spts;
    const int32_t* sidx;          // slot -> global row index
    const uint32_t* cell_start;
    const Segment* segs;
    const uint32_t* n_segs;
    const int64_t* ev_off;        // device copy of the event offsets (n_events + 1); NULL = one event
    uint32_t* cnt;                // [n_total] uncapped |S_i| at the global row index
    const int64_t* row_ptr;
    int32_t* out_src;
    int32_t* out_dst;
    float* out_d2;
    int64_t capacity;
    float r2;
    int bits;
    uint32_t k_max;
};

template <int G, int PASS>
__global__ void __launch_bounds__(kSearchWarps * 32) search_kernel(SearchArgs a) {
    __shared__ float4 s_q[kSearchWarps][64];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t lt_mask = (1u << lane) - 1u;
    const uint32_t n_segs = *a.n_segs;
    const uint32_t stride = gridDim.x * kSearchWarps;
    float4* q = s_q[warp];
    for (uint32_t sg = blockIdx.x * kSearchWarps + warp; sg < n_segs; sg += stride) {
        const Segment seg = a.segs[sg];
        const int64_t ev_base = a.ev_off ? a.ev_off[seg.cell >> (G * a.bits)] : 0;
        for (uint32_t q0 = 0; q0 < seg.len; q0 += 32) {
            const int nq = min(32u, seg.len - q0);
            const uint32_t my_slot = seg.start + q0 + lane;
            const bool has = lane < nq;
            int32_t my_row = -1;
            __syncwarp();
            if (has) {
                q[2 * lane] = a.spts[2 * static_cast<int64_t>(my_slot)];
                q[2 * lane + 1] = a.spts[2 * static_cast<int64_t>(my_slot) + 1];
                my_row = a.sidx[my_slot];
            }
            __syncwarp();
            if (PASS == 0) {
                uint32_t my_cnt = 0;
                for_each_candidate_chunk<G>(seg.cell, a.bits, a.cell_start, lane, [&](bool valid, int cslot) {
                    float4 ca = make_float4(0.f, 0.f, 0.f, 0.f), cb = ca;
                    if (valid) { ca = a.spts[2 * static_cast<int64_t>(cslot)]; cb = a.spts[2 * static_cast<int64_t>(cslot) + 1]; }
                    for (int qi = 0; qi < nq; ++qi) {
                        const float d2 = d2_pinned(q[2 * qi], q[2 * qi + 1], ca, cb);
                        const bool hit = valid && d2 <= a.r2 && static_cast<uint32_t>(cslot) != seg.start + q0 + qi;
                        const uint32_t m = __ballot_sync(kFull, hit);
                        if (lane == qi) my_cnt += __popc(m);
                    }
                });
                if (has) a.cnt[my_row] = my_cnt;
            } else {
                const uint32_t my_cnt = has ? a.cnt[my_row] : 0u;
                const int64_t my_rp = has ? a.row_ptr[my_row] : 0;
                const int32_t my_src = my_row - static_cast<int32_t>(ev_base);
                uint32_t my_off = 0;
                const uint32_t normal = __ballot_sync(kFull, has && my_cnt > 0 && my_cnt <= a.k_max);
                uint32_t over = __ballot_sync(kFull, has && my_cnt > a.k_max);
                if (normal) {
                    for_each_candidate_chunk<G>(seg.cell, a.bits, a.cell_start, lane, [&](bool valid, int cslot) {
                        float4 ca = make_float4(0.f, 0.f, 0.f, 0.f), cb = ca;
                        int32_t cj = 0;
                        if (valid) {
                            ca = a.spts[2 * static_cast<int64_t>(cslot)]; cb = a.spts[2 * static_cast<int64_t>(cslot) + 1];
                            cj = a.sidx[cslot] - static_cast<int32_t>(ev_base);
                        }
                        for (uint32_t rem = normal; rem; rem &= rem - 1) {
                            const int qi = __ffs(rem) - 1;
                            const float d2 = d2_pinned(q[2 * qi], q[2 * qi + 1], ca, cb);
                            const bool hit = valid && d2 <= a.r2 && static_cast<uint32_t>(cslot) != seg.start + q0 + qi;
                            const uint32_t m = __ballot_sync(kFull, hit);
                            if (m) {
                                const int64_t rp = __shfl_sync(kFull, my_rp, qi);
                                const uint32_t off = __shfl_sync(kFull, my_off, qi);
                                const int32_t src = __shfl_sync(kFull, my_src, qi);
                                if (hit) {
                                    const int64_t pos = rp + off + __popc(m & lt_mask);
                                    if (pos < a.capacity) { a.out_src[pos] = src; a.out_dst[pos] = cj; a.out_d2[pos] = d2; }
                                }
                                if (lane == qi) my_off += __popc(m);
                            }
                        }
                    });
                }
                // S8: rows with more than k_max in-radius neighbours.  Exact K-smallest by (d2, j)
                // without storage: find the threshold key by bisection (every probe re-scans the
                // candidates), then emit the rows' hits with key <= threshold.
                for (; over; over &= over - 1) {
                    const int qi = __ffs(over) - 1;
                    const float4 qa = q[2 * qi], qb = q[2 * qi + 1];
                    const uint32_t self_slot = seg.start + q0 + qi;
                    auto count_le = [&](uint32_t dkey, int32_t jkey) -> uint32_t {   // #{(d2,j) <= (dkey,jkey)}
                        uint32_t c = 0;
                        for_each_candidate_chunk<G>(seg.cell, a.bits, a.cell_start, lane, [&](bool valid, int cslot) {
                            float4 ca = make_float4(0.f, 0.f, 0.f, 0.f), cb = ca;
                            int32_t cj = 0;
                            if (valid) {
                                ca = a.spts[2 * static_cast<int64_t>(cslot)]; cb = a.spts[2 * static_cast<int64_t>(cslot) + 1];
                                cj = a.sidx[cslot];
                            }
                            const float d2 = d2_pinned(qa, qb, ca, cb);
                            const uint32_t db = __float_as_uint(d2);
                            const bool hit = valid && d2 <= a.r2 && static_cast<uint32_t>(cslot) != self_slot &&
                                             (db < dkey || (db == dkey && cj <= jkey));
                            c += __popc(__ballot_sync(kFull, hit));
                        });
                        return c;
                    };
                    // d2 >= +0 always (acc starts at +0 and only adds squares): bit patterns order like values
                    uint32_t dlo = 0, dhi = __float_as_uint(a.r2);
                    while (dlo < dhi) {
                        const uint32_t mid = dlo + ((dhi - dlo) >> 1);
                        if (count_le(mid, 0x7fffffff) >= a.k_max) dhi = mid; else dlo = mid + 1;
                    }
                    int32_t jlo = 0, jhi = 0x7fffffff;
                    while (jlo < jhi) {
                        const int32_t mid = jlo + ((jhi - jlo) >> 1);
                        if (count_le(dlo, mid) >= a.k_max) jhi = mid; else jlo = mid + 1;
                    }
                    const uint32_t dthr = dlo;
                    const int32_t jthr = jlo;
                    const int64_t rp = __shfl_sync(kFull, my_rp, qi);
                    const int32_t src = __shfl_sync(kFull, my_src, qi);
                    uint32_t off = 0;
                    for_each_candidate_chunk<G>(seg.cell, a.bits, a.cell_start, lane, [&](bool valid, int cslot) {
                        float4 ca = make_float4(0.f, 0.f, 0.f, 0.f), cb = ca;
                        int32_t cj = 0;
                        if (valid) {
                            ca = a.spts[2 * static_cast<int64_t>(cslot)]; cb = a.spts[2 * static_cast<int64_t>(cslot) + 1];
                            cj = a.sidx[cslot];
                        }
                        const float d2 = d2_pinned(qa, qb, ca, cb);
                        const uint32_t db = __float_as_uint(d2);
                        const bool hit = valid && d2 <= a.r2 && static_cast<uint32_t>(cslot) != self_slot &&
                                         (db < dthr || (db == dthr && cj <= jthr));
                        const uint32_t m = __ballot_sync(kFull, hit);
                        if (hit) {
                            const int64_t pos = rp + off + __popc(m & lt_mask);
                            if (pos < a.capacity) { a.out_src[pos] = src; a.out_dst[pos] = cj - static_cast<int32_t>(ev_base); a.out_d2[pos] = d2; }
                        }
                        off += __popc(m);
                    });
                }
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------
// S10 (ordering) + call epilogue.  Thread per row: insertion sort of short rows directly in the
// output arrays; longer rows are sorted by the whole warp with a bitonic network whose comparators
// all point upwards, so virtual +inf padding above the row never moves (any row length works).
// Block 0 also publishes count / status / per-event edge offsets.
// ------------------------------------------------------------------------------------------------
constexpr int kSmallRow = 12;

__device__ __forceinline__ void cmp_swap(int32_t* dst, float* d2, int64_t lo, int64_t hi) {
    const int32_t a = dst[lo], b = dst[hi];
    if (a > b) {
        dst[lo] = b; dst[hi] = a;
        const float x = d2[lo]; d2[lo] = d2[hi]; d2[hi] = x;
    }
}

__global__ void __launch_bounds__(256) sort_rows_kernel(const int64_t* row_ptr, int64_t n_total, int64_t capacity,
                                                        int32_t* dst, float* d2,
                                                        const int64_t* ev_off, int n_events,
                                                        int64_t* out_count, int64_t* out_edge_offsets, int32_t* out_status) {
    const int lane = threadIdx.x & 31;
    const int64_t i = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (blockIdx.x == 0) {
        const int64_t total = row_ptr[n_total];
        if (threadIdx.x == 0) {
            if (out_count) *out_count = total;
            *out_status = total > capacity ? -3 /* FRNN_ERR_CAPACITY */ : 0;
        }
        if (out_edge_offsets)
            for (int e = threadIdx.x; e <= n_events; e += blockDim.x) out_edge_offsets[e] = row_ptr[ev_off[e]];
    }
    int64_t b = 0, len = 0;
    if (i < n_total) {
        b = row_ptr[i];
        const int64_t e = row_ptr[i + 1];
        len = e <= capacity ? e - b : 0;          // rows cut by the capacity are left as they are
    }
    if (len >= 2 && len <= kSmallRow) {
        for (int64_t u = b + 1; u < b + len; ++u) {
            const int32_t kj = dst[u];
            const float kd = d2[u];
            int64_t v = u - 1;
            while (v >= b && dst[v] > kj) { dst[v + 1] = dst[v]; d2[v + 1] = d2[v]; --v; }
            dst[v + 1] = kj; d2[v + 1] = kd;
        }
    }
    uint32_t big = __ballot_sync(kFull, len > kSmallRow);
    for (; big; big &= big - 1) {
        const int src_lane = __ffs(big) - 1;
        const int64_t rb = __shfl_sync(kFull, b, src_lane);
        const int64_t rl = __shfl_sync(kFull, len, src_lane);
        int64_t p2 = 1;
        while (p2 < rl) p2 <<= 1;
        for (int64_t k = 2; k <= p2; k <<= 1) {
            const int64_t hk = k >> 1;
            for (int64_t t = lane; t < (p2 >> 1); t += 32) {          // flip stage: i <-> i ^ (k-1)
                const int64_t lo = (t / hk) * k + (t % hk);
                const int64_t hi = lo ^ (k - 1);
                if (hi < rl) cmp_swap(dst + rb, d2 + rb, lo, hi);
            }
            __syncwarp();
            for (int64_t j = k >> 2; j >= 1; j >>= 1) {
                for (int64_t t = lane; t < (p2 >> 1); t += 32) {
                    const int64_t lo = (t / j) * (2 * j) + (t % j);
                    const int64_t hi = lo + j;
                    if (hi < rl) cmp_swap(dst + rb, d2 + rb, lo, hi);
                }
                __syncwarp();
            }
        }
    }
}

}  // namespace frnn
