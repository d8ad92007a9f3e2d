// frnn.cu -- host side of the C ABI declared in include/frnn.h (argument checks, workspace layout,
// launch sequence, CUDA-graph cache).  No CPU fallback: every compute entry point needs a CUDA device.
#include "frnn_kernels.cuh"

#include <math.h>
#include <stdio.h>
#include <string.h>

#include <mutex>
#include <new>
#include <vector>

#include "../../include/frnn.h"

namespace {

using namespace frnn;

constexpr float kCellSlack = 1.0078125f;   // 1 + 2^-7, see cell_coord()
constexpr size_t kAlign = 256;
constexpr int64_t kPrefixTilesMin = 1024;   // above this many emit tiles the tile offsets come from tile_prefix_kernel

int g_force_dims = 0, g_force_bits = 0;
int g_use_graph = 1;
BinOrder g_order = {0, {0, 1, 2, 3, 4, 5, 6, 7}};   // frnn_set_bin_order
bool g_timeline = false;                    // frnn_set_profiling(2): kernels leave %globaltimer stamps in the workspace
constexpr int kTimelinePhases = 5;
const char* const kTimelineNames[kTimelinePhases] = {"bin", "scan_cells", "scatter", "search", "emit"};
thread_local int t_launches = 0;

// Optional per-phase CUDA-event timing (frnn_set_profiling): one event after every phase.
constexpr int kPhases = 6;
const char* const kPhaseNames[kPhases] = {"memset", "bin", "scan_cells", "scatter", "search", "emit"};
bool g_profiling = false;
cudaEvent_t g_ev[kPhases + 1] = {};
bool g_ev_valid = false;
void mark(int phase_done, cudaStream_t st) {        // phase_done = -1: start of the call
    if (g_profiling && g_ev_valid) cudaEventRecord(g_ev[phase_done + 1], st);
}

struct GridChoice { int dims, bits; };

// Grid heuristic: cells per event = 2^(dims*bits).  Finer grids cut candidate rows per query
// (3^dims cells of side ~r are visited) but cost table size and run bookkeeping; the switch points
// come from the sweep recorded in DESIGN.md section 7.
GridChoice choose_grid(int64_t n_total, int n_events, int dim = kDim) {
    const int64_t per_event = n_events > 0 ? (n_total + n_events - 1) / n_events : n_total;
    GridChoice g;
    g.bits = g_force_bits ? g_force_bits : 5;
    if (g_force_dims) g.dims = g_force_dims;
    else if (per_event < 16384) g.dims = 3;
    else if (per_event < 400000) g.dims = 4;
    else g.dims = 5;
    if (!g_force_dims && g.dims > dim) g.dims = dim;          // binning a padded (all-zero) coordinate prunes nothing
    int ev_bits = 0;
    while ((1ll << ev_bits) < n_events) ++ev_bits;
    while (g.dims * g.bits + ev_bits > 30 && g.dims > 1) --g.dims;     // padded table index stays below 2^31
    while (g.dims * g.bits + ev_bits > 30 && g.bits > 2) --g.bits;
    return g;
}

size_t align_up(size_t v) { return (v + kAlign - 1) / kAlign * kAlign; }

struct Layout {
    int64_t n_cells, n_entries, emit_tiles;
    int rows_per_block;
    int64_t scan_blocks;
    size_t off_cells, off_tiles, off_counters, zero_bytes;
    size_t off_pcell, off_prank, off_spts, off_spts_hi, off_scell, off_sidx, off_skey, off_cnt, off_evoff, off_hits, off_tprefix;
    size_t total;
};

Layout make_layout(int64_t n_total, int n_events, GridChoice g, int dim = kDim, bool ordered = false) {
    Layout L;
    L.n_cells = static_cast<int64_t>(n_events) << (g.dims * g.bits);
    const int64_t row_len = (1ll << g.bits) + 1;
    const int64_t n_rows = L.n_cells >> g.bits;
    L.n_entries = n_rows * row_len;
    L.rows_per_block = static_cast<int>((kCellTile / row_len) & ~3ll);      // multiple of 4: every block starts 16-byte aligned
    if (L.rows_per_block < 4) L.rows_per_block = 4;
    L.scan_blocks = (n_rows + L.rows_per_block - 1) / L.rows_per_block;
    L.emit_tiles = (n_total + kEmitThreads - 1) / kEmitThreads;
    size_t o = 0;
    L.off_cells = o;    o = align_up(o + static_cast<size_t>(L.n_entries + 8) * 4);
    L.off_tiles = o;    o = align_up(o + static_cast<size_t>(L.emit_tiles > 0 ? L.emit_tiles : 1) * 8 * kDegSlices);
    L.off_counters = o; o = align_up(o + 256);         // [0..3] cursor of the cell scan (u32); [64..) timeline stamps (u64 x 2 x kTimelinePhases)
    const size_t n = static_cast<size_t>(n_total > 0 ? n_total : 1);
    L.off_cnt = o;      o = align_up(o + n * 4);       // zeroed: the search pass counts with atomics
    L.zero_bytes = o;
    L.off_pcell = o;  o = align_up(o + n * 4);
    L.off_prank = o;  o = align_up(o + n * 4);
    L.off_spts = o;   o = align_up(o + n * 32);
    L.off_spts_hi = o; if (dim > kDim) o = align_up(o + n * 32);      // coordinates 8..15 of the cell-ordered copy
    L.off_scell = o;   if (ordered) o = align_up(o + n * 4);           // slot -> cell id (only with a caller-chosen bin order)
    L.off_sidx = o;   o = align_up(o + n * 4);
    L.off_skey = o;   o = align_up(o + n * 4);
    L.off_evoff = o;  o = align_up(o + static_cast<size_t>(n_events + 1) * 8);
    L.off_tprefix = o; o = align_up(o + static_cast<size_t>(L.emit_tiles > 0 ? L.emit_tiles : 1) * 8);
    L.off_hits = o;   o = align_up(o + n * kSlot * sizeof(int2));
    L.total = o;
    return L;
}

#define FRNN_DISPATCH_G(G_, EXPR)          \
    switch (G_) {                          \
        case 1: { constexpr int GG = 1; EXPR; } break; \
        case 2: { constexpr int GG = 2; EXPR; } break; \
        case 3: { constexpr int GG = 3; EXPR; } break; \
        case 4: { constexpr int GG = 4; EXPR; } break; \
        case 5: { constexpr int GG = 5; EXPR; } break; \
        default: { constexpr int GG = 6; EXPR; } break; \
    }

#define CK(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return FRNN_ERR_CUDA; } while (0)

int check_common(const float* points, int64_t n, int dim, float r, int k_max, const void* out_src, const void* out_dst,
                 const void* out_d2, int64_t capacity) {
    if (n < 0 || k_max < 1 || capacity < 0) return FRNN_ERR_INVALID_ARG;
    if (!(r >= 0.0f) || !isfinite(r)) return FRNN_ERR_INVALID_ARG;
    if (n > 0 && !points) return FRNN_ERR_INVALID_ARG;
    if (dim < 1 || dim > kDimMax) return FRNN_ERR_UNSUPPORTED;
    if (reinterpret_cast<uintptr_t>(points) % (dim == kDim ? 32 : 4)) return FRNN_ERR_INVALID_ARG;   // 8-float rows move as 256-bit transactions
    if (capacity > 0 && (!out_src || !out_dst || !out_d2)) return FRNN_ERR_INVALID_ARG;
    if (n > 0x7fffffffll) return FRNN_ERR_UNSUPPORTED;
    return FRNN_OK;
}

struct Call {                 // everything that determines the enqueued work (also the graph-cache key)
    const float* points;
    int dim = kDim;
    int n_events;
    float r;
    int k_max;
    int32_t* out_src;
    int32_t* out_dst;
    float* out_d2;
    int64_t capacity;
    int64_t* out_count;
    int64_t* out_edge_offsets;
    int32_t* out_status;
    int64_t* out_row_ptr;
    void* workspace;
    int grid_dims, grid_bits;
    std::vector<int64_t> ev_off;
    bool timeline = false;
    bool dense = false;           // frnn_build_dense_ex: brute force instead of the grid
    BinOrder order = {0, {0, 1, 2, 3, 4, 5, 6, 7}};
    bool operator==(const Call& o) const {
        return points == o.points && dim == o.dim && n_events == o.n_events && r == o.r && k_max == o.k_max && out_src == o.out_src &&
               out_dst == o.out_dst && out_d2 == o.out_d2 && capacity == o.capacity && out_count == o.out_count &&
               out_edge_offsets == o.out_edge_offsets && out_status == o.out_status && out_row_ptr == o.out_row_ptr &&
               workspace == o.workspace && grid_dims == o.grid_dims && grid_bits == o.grid_bits && ev_off == o.ev_off && timeline == o.timeline && dense == o.dense &&
               order.on == o.order.on && memcmp(order.p, o.order.p, 8) == 0;
    }
};

// The whole path, enqueued kernel by kernel on `st`.
int enqueue(const Call& c, const Layout& L, cudaStream_t st) {
    const int64_t n_total = c.ev_off[c.n_events];
    char* ws = static_cast<char*>(c.workspace);
    uint32_t* cells = reinterpret_cast<uint32_t*>(ws + L.off_cells);
    unsigned long long* tile_deg = reinterpret_cast<unsigned long long*>(ws + L.off_tiles);
    unsigned int* cursor = reinterpret_cast<unsigned int*>(ws + L.off_counters);
    unsigned long long* stamps = c.timeline ? reinterpret_cast<unsigned long long*>(ws + L.off_counters + 64) : nullptr;
    uint32_t* pcell = reinterpret_cast<uint32_t*>(ws + L.off_pcell);
    uint32_t* prank = reinterpret_cast<uint32_t*>(ws + L.off_prank);
    float4* spts = reinterpret_cast<float4*>(ws + L.off_spts);
    float4* spts_hi = c.dim > kDim ? reinterpret_cast<float4*>(ws + L.off_spts_hi) : nullptr;
    uint32_t* scell = c.order.on ? reinterpret_cast<uint32_t*>(ws + L.off_scell) : nullptr;
    int32_t* sidx = reinterpret_cast<int32_t*>(ws + L.off_sidx);
    uint32_t* skey = reinterpret_cast<uint32_t*>(ws + L.off_skey);
    uint32_t* cnt = reinterpret_cast<uint32_t*>(ws + L.off_cnt);
    int64_t* ev_off = reinterpret_cast<int64_t*>(ws + L.off_evoff);
    int2* hits = reinterpret_cast<int2*>(ws + L.off_hits);
    const float* pts = c.points;
    const int G = c.grid_dims, bits = c.grid_bits;

    const float r2 = c.r * c.r;                               // R2: fl32(r*r), once, on the host
    const float cell_side = fmaxf(c.r * kCellSlack, 1e-30f);
    const float inv_cell = 1.0f / cell_side;

    mark(-1, st);
    if (c.dense) {                                             // brute force: no table, no sort (single event)
        CK(cudaMemsetAsync(ws + L.off_tiles, 0, L.zero_bytes - L.off_tiles, st)); ++t_launches;
        DenseArgs da;
        da.pts = pts; da.dim = c.dim; da.cnt = cnt; da.hits = hits; da.tile_deg = tile_deg; da.n_tiles = static_cast<uint32_t>(L.emit_tiles);
        da.n = n_total; da.r2 = r2; da.k_max = static_cast<uint32_t>(c.k_max);
        const unsigned T = static_cast<unsigned>((n_total + kDenseTile - 1) / kDenseTile);
        if (c.dim > kDim) dense_search_kernel<true><<<dim3(T, T), kDenseTile, 0, st>>>(da);
        else              dense_search_kernel<false><<<dim3(T, T), kDenseTile, 0, st>>>(da);
        ++t_launches; CK(cudaGetLastError());
        EmitArgs ea;
        ea.pts = pts; ea.dim = c.dim; ea.spts = nullptr; ea.spts_hi = nullptr; ea.sidx = nullptr; ea.cell_start = nullptr; ea.cnt = cnt; ea.hits = hits; ea.ev_off = nullptr;
        ea.tile_deg = tile_deg; ea.tile_prefix = nullptr; ea.n_events = 1; ea.n_total = n_total; ea.row_ptr = c.out_row_ptr;
        ea.out_src = c.out_src; ea.out_dst = c.out_dst; ea.out_d2 = c.out_d2; ea.capacity = c.capacity; ea.out_count = c.out_count;
        ea.out_edge_offsets = nullptr; ea.out_status = c.out_status; ea.r2 = r2; ea.inv_cell = inv_cell; ea.bits = bits;
        ea.k_max = static_cast<uint32_t>(c.k_max); ea.stamps = nullptr; ea.dense = 1; ea.order = c.order;
        if (L.emit_tiles > kPrefixTilesMin) {
            unsigned long long* tprefix = reinterpret_cast<unsigned long long*>(ws + L.off_tprefix);
            tile_prefix_kernel<<<1, kPrefixThreads, 0, st>>>(tile_deg, static_cast<uint32_t>(L.emit_tiles), tprefix);
            ++t_launches; CK(cudaGetLastError());
            ea.tile_prefix = tprefix;
        }
        emit_kernel<1><<<static_cast<unsigned>(L.emit_tiles), kEmitThreads, 0, st>>>(ea);
        ++t_launches; CK(cudaGetLastError());
        return FRNN_OK;
    }
    CK(cudaMemsetAsync(ws, 0, L.zero_bytes, st)); ++t_launches;
    // Event offsets reach the device as kernel arguments (no pageable-memory copy, which would
    // synchronise the host with the stream); a single event needs none (base 0).
    if (c.n_events > 1) {
        for (int first = 0; first <= c.n_events; first += OffsetChunk::kN) {
            OffsetChunk ch;
            ch.first = first;
            ch.count = (c.n_events + 1 - first) < OffsetChunk::kN ? (c.n_events + 1 - first) : OffsetChunk::kN;
            for (int k = 0; k < ch.count; ++k) ch.v[k] = c.ev_off[first + k];
            set_offsets_kernel<<<1, OffsetChunk::kN, 0, st>>>(ch, ev_off);
            ++t_launches; CK(cudaGetLastError());
        }
    } else {
        ev_off = nullptr;
    }
    mark(0, st);
    const unsigned row_blocks = static_cast<unsigned>((n_total + 255) / 256);
    FRNN_DISPATCH_G(G, (bin_kernel<GG><<<row_blocks, 256, 0, st>>>(pts, c.dim, n_total, ev_off, c.n_events, inv_cell, bits, cells, pcell, prank, c.order, stamps)));
    ++t_launches; CK(cudaGetLastError());
    mark(1, st);
    cell_scan_kernel<<<static_cast<unsigned>(L.scan_blocks), kCellThreads, 0, st>>>(cells, L.n_entries, L.rows_per_block, bits, cursor, stamps);
    ++t_launches; CK(cudaGetLastError());
    mark(2, st);
    FRNN_DISPATCH_G(G, (scatter_kernel<GG><<<row_blocks, 256, 0, st>>>(pts, c.dim, n_total, bits, inv_cell, cells, pcell, prank, spts, sidx, skey, spts_hi, scell, c.order, stamps)));
    ++t_launches; CK(cudaGetLastError());
    mark(3, st);

    SearchArgs sa;
    sa.scell = scell;
    sa.spts = spts; sa.spts_hi = spts_hi; sa.sidx = sidx; sa.skey = skey; sa.cell_start = cells; sa.cnt = cnt; sa.hits = hits;
    sa.tile_deg = tile_deg; sa.n_tiles = static_cast<uint32_t>(L.emit_tiles); sa.ev_off = ev_off; sa.stamps = stamps; sa.n_total = n_total; sa.n_events = c.n_events; sa.r2 = r2;
    sa.inv_cell = inv_cell; sa.bits = bits; sa.k_max = static_cast<uint32_t>(c.k_max);
    const unsigned search_blocks = static_cast<unsigned>((n_total + kSearchThreads - 1) / kSearchThreads);
    if (spts_hi) { FRNN_DISPATCH_G(G, (search_kernel<GG, true><<<search_blocks, kSearchThreads, 0, st>>>(sa))); }
    else         { FRNN_DISPATCH_G(G, (search_kernel<GG, false><<<search_blocks, kSearchThreads, 0, st>>>(sa))); }
    ++t_launches; CK(cudaGetLastError());
    mark(4, st);

    EmitArgs ea;
    ea.pts = pts; ea.dim = c.dim; ea.spts = spts; ea.spts_hi = spts_hi; ea.sidx = sidx; ea.cell_start = cells; ea.cnt = cnt; ea.hits = hits; ea.ev_off = ev_off;
    ea.tile_deg = tile_deg; ea.tile_prefix = nullptr; ea.n_events = c.n_events; ea.n_total = n_total; ea.row_ptr = c.out_row_ptr;
    ea.out_src = c.out_src; ea.out_dst = c.out_dst; ea.out_d2 = c.out_d2; ea.capacity = c.capacity; ea.out_count = c.out_count;
    ea.out_edge_offsets = c.out_edge_offsets; ea.out_status = c.out_status; ea.r2 = r2; ea.inv_cell = inv_cell; ea.bits = bits;
    ea.k_max = static_cast<uint32_t>(c.k_max); ea.stamps = stamps; ea.dense = 0; ea.order = c.order;
    if (L.emit_tiles > kPrefixTilesMin) {                      // many tiles: their prefix in one small kernel (see tile_prefix_kernel)
        unsigned long long* tprefix = reinterpret_cast<unsigned long long*>(ws + L.off_tprefix);
        tile_prefix_kernel<<<1, kPrefixThreads, 0, st>>>(tile_deg, static_cast<uint32_t>(L.emit_tiles), tprefix);
        ++t_launches; CK(cudaGetLastError());
        ea.tile_prefix = tprefix;
    }
    FRNN_DISPATCH_G(G, (emit_kernel<GG><<<static_cast<unsigned>(L.emit_tiles), kEmitThreads, 0, st>>>(ea)));
    ++t_launches; CK(cudaGetLastError());
    mark(5, st);
    return FRNN_OK;
}

// ---- CUDA-graph cache: the same call (same pointers, sizes, parameters) replays one instantiated
// graph, which costs ~1 us per kernel boundary instead of ~3 us per stream launch (profiles/).
struct CachedGraph { Call key; cudaGraphExec_t exec; int launches; uint64_t stamp; };
std::vector<CachedGraph> g_graphs;
std::mutex g_graph_mutex;
uint64_t g_stamp = 0;
constexpr size_t kMaxGraphs = 128;

int run_call(const Call& c, cudaStream_t st) {
    t_launches = 0;
    const int64_t n_total = c.ev_off[c.n_events];
    if (n_total == 0) {                       // nothing to search: zero the outputs and leave
        if (c.out_count) { CK(cudaMemsetAsync(c.out_count, 0, 8, st)); ++t_launches; }
        if (c.out_edge_offsets) { CK(cudaMemsetAsync(c.out_edge_offsets, 0, 8 * static_cast<size_t>(c.n_events + 1), st)); ++t_launches; }
        if (c.out_row_ptr) { CK(cudaMemsetAsync(c.out_row_ptr, 0, 8, st)); ++t_launches; }
        CK(cudaMemsetAsync(c.out_status, 0, 4, st)); ++t_launches;
        return FRNN_OK;
    }
    const Layout L = make_layout(n_total, c.n_events, GridChoice{c.grid_dims, c.grid_bits}, c.dim, c.order.on != 0);
    bool graph_ok = g_use_graph && !g_profiling && st != nullptr && st != cudaStreamLegacy;
    if (graph_ok) {
        cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
        if (cudaStreamIsCapturing(st, &cs) != cudaSuccess || cs != cudaStreamCaptureStatusNone) graph_ok = false;   // caller is capturing: just enqueue
    }
    if (!graph_ok) return enqueue(c, L, st);

    std::lock_guard<std::mutex> lock(g_graph_mutex);
    for (auto& g : g_graphs) {
        if (g.key == c) {
            g.stamp = ++g_stamp;
            t_launches = g.launches;
            CK(cudaGraphLaunch(g.exec, st));
            return FRNN_OK;
        }
    }
    cudaGraph_t graph = nullptr;
    if (cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal) != cudaSuccess) { cudaGetLastError(); return enqueue(c, L, st); }
    const int rc = enqueue(c, L, st);
    const cudaError_t ce = cudaStreamEndCapture(st, &graph);
    if (rc != FRNN_OK || ce != cudaSuccess || !graph) {
        if (graph) cudaGraphDestroy(graph);
        cudaGetLastError();
        return rc != FRNN_OK ? rc : FRNN_ERR_CUDA;
    }
    cudaGraphExec_t exec = nullptr;
    const cudaError_t ie = cudaGraphInstantiate(&exec, graph, 0);
    cudaGraphDestroy(graph);
    if (ie != cudaSuccess) { cudaGetLastError(); return FRNN_ERR_CUDA; }
    if (g_graphs.size() >= kMaxGraphs) {      // evict the least recently used
        size_t victim = 0;
        for (size_t k = 1; k < g_graphs.size(); ++k)
            if (g_graphs[k].stamp < g_graphs[victim].stamp) victim = k;
        cudaGraphExecDestroy(g_graphs[victim].exec);
        g_graphs.erase(g_graphs.begin() + victim);
    }
    g_graphs.push_back(CachedGraph{c, exec, t_launches, ++g_stamp});
    CK(cudaGraphLaunch(exec, st));
    return FRNN_OK;
}

int prepare(Call& c, size_t workspace_bytes) {
    const int64_t n_total = c.ev_off[c.n_events];
    const GridChoice g = choose_grid(n_total, c.n_events, c.dim);
    c.grid_dims = g.dims;
    c.grid_bits = g.bits;
    c.timeline = g_timeline;
    c.order = g_order;
    if (n_total == 0) return FRNN_OK;
    const Layout L = make_layout(n_total, c.n_events, g, c.dim, c.order.on != 0);
    if (!c.workspace || workspace_bytes < L.total) return FRNN_ERR_WORKSPACE;
    if (reinterpret_cast<uintptr_t>(c.workspace) % kAlign) return FRNN_ERR_INVALID_ARG;
    return FRNN_OK;
}

// cached device buffers for the synchronous convenience entry points
struct Cache {
    void* ws = nullptr; size_t ws_bytes = 0;
    void* misc = nullptr;                       // count (8) + status (4)
    void* pts = nullptr; size_t pts_bytes = 0;
    void* edges = nullptr; size_t edge_cap = 0; // src | dst | d2, edge_cap each
    cudaStream_t stream = nullptr;              // non-default stream so the graph path applies
} g_cache;

int ensure(void** p, size_t* have, size_t need) {
    if (*have >= need && *p) return FRNN_OK;
    if (*p) cudaFree(*p);
    *p = nullptr; *have = 0;
    if (cudaMalloc(p, need) != cudaSuccess) return FRNN_ERR_CUDA;
    *have = need;
    return FRNN_OK;
}

int ensure_stream() {
    if (!g_cache.stream && cudaStreamCreateWithFlags(&g_cache.stream, cudaStreamNonBlocking) != cudaSuccess) return FRNN_ERR_CUDA;
    return FRNN_OK;
}

}  // namespace

extern "C" {

int frnn_version(void) { return 300; }   // 0.3.0

const char* frnn_status_string(int status) {
    switch (status) {
        case FRNN_OK: return "ok";
        case FRNN_ERR_INVALID_ARG: return "invalid argument";
        case FRNN_ERR_UNSUPPORTED: return "unsupported (dim outside 1..16 or too many rows)";
        case FRNN_ERR_CAPACITY: return "edge capacity exceeded";
        case FRNN_ERR_WORKSPACE: return "workspace too small";
        case FRNN_ERR_CUDA: return "CUDA error";
        default: return "unknown status";
    }
}

size_t frnn_workspace_bytes(int64_t n_total, int n_events, int dim, int k_max) {
    if (n_total < 0 || n_events < 1 || dim < 1 || dim > kDimMax || k_max < 1 || n_total > 0x7fffffffll) return 0;
    return make_layout(n_total, n_events, choose_grid(n_total, n_events, dim), dim, g_order.on != 0).total;
}

int frnn_set_grid(int grid_dims, int grid_bits) {
    if (grid_dims < 0 || grid_dims > 6 || (grid_bits != 0 && (grid_bits < 2 || grid_bits > 8))) return FRNN_ERR_INVALID_ARG;
    g_force_dims = grid_dims;
    g_force_bits = grid_bits;
    return FRNN_OK;
}

void frnn_get_grid(int64_t n_total, int n_events, int* grid_dims, int* grid_bits) {
    const GridChoice g = choose_grid(n_total, n_events < 1 ? 1 : n_events);
    if (grid_dims) *grid_dims = g.dims;
    if (grid_bits) *grid_bits = g.bits;
}

int frnn_set_bin_order(const int* order, int count) {
    if (count < 0 || count > 8 || (count > 0 && !order)) return FRNN_ERR_INVALID_ARG;
    BinOrder o = {count > 0 ? 1 : 0, {0, 1, 2, 3, 4, 5, 6, 7}};
    bool used[kDimMax] = {};
    for (int k = 0; k < count; ++k) {
        if (order[k] < 0 || order[k] >= kDimMax || used[order[k]]) return FRNN_ERR_INVALID_ARG;
        used[order[k]] = true;
        o.p[k] = static_cast<unsigned char>(order[k]);
    }
    int next = 0;
    for (int k = count; k < 8; ++k) {                  // the rest: the unused coordinates in ascending order
        while (used[next]) ++next;
        used[next] = true;
        o.p[k] = static_cast<unsigned char>(next);
    }
    g_order = o;
    return FRNN_OK;
}

namespace {
// Per coordinate: the probability that two random points of the sample fall within one cell of each other
// (cells of side r, modulo 64) = sum_c p_c (p_{c-1} + p_c + p_{c+1}).  The smaller, the more that coordinate prunes.
constexpr int kSuggestBins = 64;
__global__ void __launch_bounds__(1024) suggest_kernel(const float* __restrict__ pts, int64_t n, int dim, float inv_cell,
                                                       int64_t stride, float* __restrict__ out /* kDimMax */) {
    __shared__ unsigned int s_h[kDimMax][kSuggestBins];
    for (int k = threadIdx.x; k < kDimMax * kSuggestBins; k += blockDim.x) (&s_h[0][0])[k] = 0u;
    __syncthreads();
    unsigned int mine = 0;
    for (int64_t i = static_cast<int64_t>(threadIdx.x) * stride; i < n; i += static_cast<int64_t>(blockDim.x) * stride) {
        for (int d = 0; d < dim; ++d) atomicAdd(&s_h[d][cell_coord(pts[i * dim + d], inv_cell, kSuggestBins - 1)], 1u);
        ++mine;
    }
    __shared__ unsigned int s_total;
    if (threadIdx.x == 0) s_total = 0;
    __syncthreads();
    atomicAdd(&s_total, mine);
    __syncthreads();
    if (threadIdx.x < kDimMax) {
        const int d = threadIdx.x;
        double acc = 0.0;
        const double tot = s_total ? static_cast<double>(s_total) : 1.0;
        for (int c = 0; c < kSuggestBins; ++c) {
            const double pc = s_h[d][c] / tot;
            const double nb = (s_h[d][(c + kSuggestBins - 1) % kSuggestBins] + s_h[d][c] + s_h[d][(c + 1) % kSuggestBins]) / tot;
            acc += pc * nb;
        }
        out[d] = d < dim ? static_cast<float>(acc) : 2.0f;          // absent coordinates prune nothing: last
    }
}
}  // namespace

int frnn_suggest_bin_order(const float* points, int64_t n, int dim, float r, int* order, float* score, void* cuda_stream) {
    if (!points || !order || n < 1 || !(r >= 0.0f) || !isfinite(r)) return FRNN_ERR_INVALID_ARG;
    if (dim < 1 || dim > kDimMax) return FRNN_ERR_UNSUPPORTED;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    float* d_out = nullptr;
    if (cudaMalloc(reinterpret_cast<void**>(&d_out), kDimMax * sizeof(float)) != cudaSuccess) return FRNN_ERR_CUDA;
    const int64_t stride = n > 65536 ? n / 65536 : 1;              // a sample of at most ~65k points
    const float inv_cell = 1.0f / fmaxf(r * kCellSlack, 1e-30f);
    suggest_kernel<<<1, 1024, 0, st>>>(points, n, dim, inv_cell, stride, d_out);
    float h[kDimMax];
    const cudaError_t e = cudaMemcpyAsync(h, d_out, sizeof(h), cudaMemcpyDeviceToHost, st);
    const cudaError_t e2 = cudaStreamSynchronize(st);
    cudaFree(d_out);
    if (e != cudaSuccess || e2 != cudaSuccess) return FRNN_ERR_CUDA;
    int idx[kDimMax];
    for (int d = 0; d < kDimMax; ++d) idx[d] = d;
    for (int a = 1; a < kDimMax; ++a)                               // stable insertion sort by score
        for (int b = a; b > 0 && h[idx[b]] < h[idx[b - 1]]; --b) { const int t = idx[b]; idx[b] = idx[b - 1]; idx[b - 1] = t; }
    for (int k = 0; k < 8; ++k) order[k] = idx[k];
    if (score) for (int d = 0; d < kDimMax; ++d) score[d] = h[d];
    return FRNN_OK;
}

int frnn_set_graph_mode(int enabled) {
    g_use_graph = enabled != 0;
    return FRNN_OK;
}

int frnn_build_ex(const float* points, int64_t n, int dim, float r, int k_max,
                  int32_t* out_src, int32_t* out_dst, float* out_d2, int64_t edge_capacity,
                  int64_t* out_count, int32_t* out_status, int64_t* out_row_ptr,
                  void* workspace, size_t workspace_bytes, void* cuda_stream) {
    int rc = check_common(points, n, dim, r, k_max, out_src, out_dst, out_d2, edge_capacity);
    if (rc != FRNN_OK) return rc;
    if (!out_count || !out_status) return FRNN_ERR_INVALID_ARG;
    Call c{points, dim, 1, r, k_max, out_src, out_dst, out_d2, edge_capacity, out_count, nullptr, out_status, out_row_ptr, workspace, 0, 0, {0, n}};
    if ((rc = prepare(c, workspace_bytes)) != FRNN_OK) return rc;
    return run_call(c, static_cast<cudaStream_t>(cuda_stream));
}

int frnn_build_dense_ex(const float* points, int64_t n, int dim, float r, int k_max,
                        int32_t* out_src, int32_t* out_dst, float* out_d2, int64_t edge_capacity,
                        int64_t* out_count, int32_t* out_status, int64_t* out_row_ptr,
                        void* workspace, size_t workspace_bytes, void* cuda_stream) {
    int rc = check_common(points, n, dim, r, k_max, out_src, out_dst, out_d2, edge_capacity);
    if (rc != FRNN_OK) return rc;
    if (!out_count || !out_status) return FRNN_ERR_INVALID_ARG;
    if (n > 65535ll * kDenseTile) return FRNN_ERR_UNSUPPORTED;                 // grid.y limit (8.3 M rows)
    Call c{points, dim, 1, r, k_max, out_src, out_dst, out_d2, edge_capacity, out_count, nullptr, out_status, out_row_ptr, workspace, 0, 0, {0, n}};
    c.dense = true;
    if ((rc = prepare(c, workspace_bytes)) != FRNN_OK) return rc;
    return run_call(c, static_cast<cudaStream_t>(cuda_stream));
}

int frnn_build_batched(const float* points, const int64_t* event_offsets, int n_events, int dim, float r, int k_max,
                       int32_t* out_src, int32_t* out_dst, float* out_d2, int64_t edge_capacity,
                       int64_t* out_edge_offsets, int32_t* out_status, int64_t* out_row_ptr,
                       void* workspace, size_t workspace_bytes, void* cuda_stream) {
    if (n_events < 1 || !event_offsets || event_offsets[0] != 0) return FRNN_ERR_INVALID_ARG;
    for (int e = 0; e < n_events; ++e)
        if (event_offsets[e + 1] < event_offsets[e]) return FRNN_ERR_INVALID_ARG;
    int rc = check_common(points, event_offsets[n_events], dim, r, k_max, out_src, out_dst, out_d2, edge_capacity);
    if (rc != FRNN_OK) return rc;
    if (!out_edge_offsets || !out_status) return FRNN_ERR_INVALID_ARG;
    Call c{points, dim, n_events, r, k_max, out_src, out_dst, out_d2, edge_capacity, nullptr, out_edge_offsets, out_status, out_row_ptr,
           workspace, 0, 0, std::vector<int64_t>(event_offsets, event_offsets + n_events + 1)};
    if ((rc = prepare(c, workspace_bytes)) != FRNN_OK) return rc;
    return run_call(c, static_cast<cudaStream_t>(cuda_stream));
}

int frnn_build(const float* points, int64_t n, int dim, float r, int k_max,
               int32_t* out_src, int32_t* out_dst, float* out_d2, int64_t* out_count) {
    if (!out_count) return FRNN_ERR_INVALID_ARG;
    const int64_t cap = n > 0 ? n * static_cast<int64_t>(k_max > 0 ? k_max : 0) : 0;
    int rc = check_common(points, n, dim, r, k_max, out_src, out_dst, out_d2, cap);
    if (rc != FRNN_OK) return rc;
    const size_t need = frnn_workspace_bytes(n, 1, dim, k_max);
    size_t misc_have = g_cache.misc ? 64 : 0;
    if ((rc = ensure(&g_cache.ws, &g_cache.ws_bytes, need)) != FRNN_OK) return rc;
    if ((rc = ensure(&g_cache.misc, &misc_have, 64)) != FRNN_OK) return rc;
    int64_t* d_count = static_cast<int64_t*>(g_cache.misc);
    int32_t* d_status = reinterpret_cast<int32_t*>(static_cast<char*>(g_cache.misc) + 8);
    rc = frnn_build_ex(points, n, dim, r, k_max, out_src, out_dst, out_d2, cap, d_count, d_status, nullptr, g_cache.ws,
                       g_cache.ws_bytes, nullptr);       // legacy default stream, as documented
    if (rc != FRNN_OK) return rc;
    int32_t h_status = 0;
    CK(cudaMemcpy(out_count, d_count, 8, cudaMemcpyDeviceToHost));
    CK(cudaMemcpy(&h_status, d_status, 4, cudaMemcpyDeviceToHost));
    return h_status;
}

int frnn_build_host(const float* points, int64_t n, int dim, float r, int k_max,
                    int32_t* out_src, int32_t* out_dst, float* out_d2, int64_t edge_capacity, int64_t* out_count) {
    if (!out_count) return FRNN_ERR_INVALID_ARG;
    int rc = check_common(points, n, dim, r, k_max, out_src, out_dst, out_d2, edge_capacity);
    if (rc != FRNN_OK) return rc;
    const size_t need = frnn_workspace_bytes(n, 1, dim, k_max);
    size_t misc_have = g_cache.misc ? 64 : 0;
    size_t edge_bytes = g_cache.edge_cap * 12;
    if ((rc = ensure_stream()) != FRNN_OK) return rc;
    if ((rc = ensure(&g_cache.ws, &g_cache.ws_bytes, need)) != FRNN_OK) return rc;
    if ((rc = ensure(&g_cache.misc, &misc_have, 64)) != FRNN_OK) return rc;
    if ((rc = ensure(&g_cache.pts, &g_cache.pts_bytes, static_cast<size_t>(n > 0 ? n : 1) * 64)) != FRNN_OK) return rc;   // room for 16 floats per row whatever dim is
    if (g_cache.edge_cap < static_cast<size_t>(edge_capacity) || !g_cache.edges) {
        if ((rc = ensure(&g_cache.edges, &edge_bytes, static_cast<size_t>(edge_capacity > 0 ? edge_capacity : 1) * 12)) != FRNN_OK) return rc;
        g_cache.edge_cap = static_cast<size_t>(edge_capacity > 0 ? edge_capacity : 1);
    }
    cudaStream_t st = g_cache.stream;
    int32_t* d_src = static_cast<int32_t*>(g_cache.edges);
    int32_t* d_dst = d_src + g_cache.edge_cap;
    float* d_d2 = reinterpret_cast<float*>(d_dst + g_cache.edge_cap);
    int64_t* d_count = static_cast<int64_t*>(g_cache.misc);
    int32_t* d_status = reinterpret_cast<int32_t*>(static_cast<char*>(g_cache.misc) + 8);
    if (n > 0) CK(cudaMemcpyAsync(g_cache.pts, points, static_cast<size_t>(n) * dim * 4, cudaMemcpyHostToDevice, st));
    rc = frnn_build_ex(static_cast<const float*>(g_cache.pts), n, dim, r, k_max, d_src, d_dst, d_d2, edge_capacity, d_count, d_status,
                       nullptr, g_cache.ws, g_cache.ws_bytes, st);
    if (rc != FRNN_OK) return rc;
    CK(cudaMemcpyAsync(out_count, d_count, 8, cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    if (*out_count > edge_capacity) return FRNN_ERR_CAPACITY;
    const size_t e = static_cast<size_t>(*out_count);
    if (e) {
        CK(cudaMemcpyAsync(out_src, d_src, e * 4, cudaMemcpyDeviceToHost, st));
        CK(cudaMemcpyAsync(out_dst, d_dst, e * 4, cudaMemcpyDeviceToHost, st));
        CK(cudaMemcpyAsync(out_d2, d_d2, e * 4, cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
    }
    return FRNN_OK;
}

// ---- host pipeline: H2D of event i+1, build of event i and D2H of event i-1 overlap (one stream per slot); the edge
// copies are DMA transfers of exactly `count` edges, started by the host as soon as it sees a build completed
struct frnn_host_pipeline {
    enum State { FREE, BUILDING, COPYING };
    struct Slot {
        cudaStream_t stream = nullptr;
        cudaEvent_t built = nullptr, done = nullptr;
        void* ws = nullptr;
        float* pts = nullptr;
        int32_t* src = nullptr; int32_t* dst = nullptr; float* d2 = nullptr;
        int64_t* count = nullptr;                                 // device: count (8 bytes) followed by status (4 bytes)
        int64_t* pinned = nullptr;                                // page-locked mirror of the two words above
        int32_t* h_src = nullptr; int32_t* h_dst = nullptr; float* h_d2 = nullptr; int64_t* h_count = nullptr;   // the caller's
        State state = FREE;
    };
    std::vector<Slot> slots;
    int64_t n_max = 0, cap = 0;
    int k_max = 0, next = 0;
    size_t ws_bytes = 0;
};

namespace {
void pipeline_free(frnn_host_pipeline* p) {
    for (auto& s : p->slots) {
        if (s.stream) cudaStreamSynchronize(s.stream);
        if (s.ws) cudaFree(s.ws);
        if (s.pts) cudaFree(s.pts);
        if (s.src) cudaFree(s.src);
        if (s.count) cudaFree(s.count);
        if (s.pinned) cudaFreeHost(s.pinned);
        if (s.built) cudaEventDestroy(s.built);
        if (s.done) cudaEventDestroy(s.done);
        if (s.stream) cudaStreamDestroy(s.stream);
    }
    delete p;
}

// The build of this slot has completed: its edge count is on the host, so the copy of exactly that many edges can be
// handed to the copy engine (it then runs beside the builds and the H2D copies of the other slots).
int pipeline_start_copy(frnn_host_pipeline* p, frnn_host_pipeline::Slot& s) {
    const int64_t c = s.pinned[0];
    const int32_t status = *reinterpret_cast<const int32_t*>(s.pinned + 1);
    *s.h_count = status == 0 ? c : -c - 1;                       // negative: capacity exceeded, -(needed) - 1
    const size_t e = static_cast<size_t>(c < p->cap ? c : p->cap);
    if (e) {
        CK(cudaMemcpyAsync(s.h_src, s.src, e * 4, cudaMemcpyDeviceToHost, s.stream));
        CK(cudaMemcpyAsync(s.h_dst, s.dst, e * 4, cudaMemcpyDeviceToHost, s.stream));
        CK(cudaMemcpyAsync(s.h_d2, s.d2, e * 4, cudaMemcpyDeviceToHost, s.stream));
    }
    CK(cudaEventRecord(s.done, s.stream));
    s.state = frnn_host_pipeline::COPYING;
    return FRNN_OK;
}

int pipeline_retire(frnn_host_pipeline* p, frnn_host_pipeline::Slot& s) {
    if (s.state == frnn_host_pipeline::BUILDING) {
        CK(cudaEventSynchronize(s.built));
        const int rc = pipeline_start_copy(p, s);
        if (rc != FRNN_OK) return rc;
    }
    if (s.state == frnn_host_pipeline::COPYING) {
        CK(cudaEventSynchronize(s.done));
        s.state = frnn_host_pipeline::FREE;
    }
    return FRNN_OK;
}

// builds that have finished in the meantime get their edge copies started (never blocks)
int pipeline_poll(frnn_host_pipeline* p) {
    for (auto& s : p->slots)
        if (s.state == frnn_host_pipeline::BUILDING && cudaEventQuery(s.built) == cudaSuccess) {
            const int rc = pipeline_start_copy(p, s);
            if (rc != FRNN_OK) return rc;
        }
    cudaGetLastError();                                          // cudaErrorNotReady of the queries is not an error
    return FRNN_OK;
}
}  // namespace

int frnn_host_pipeline_create(int64_t n_max, int dim, int k_max, int64_t edge_capacity, int depth, frnn_host_pipeline** out) {
    if (!out || n_max < 1 || k_max < 1 || edge_capacity < 1 || depth < 1 || depth > 16) return FRNN_ERR_INVALID_ARG;
    if (dim != kDim) return FRNN_ERR_UNSUPPORTED;
    frnn_host_pipeline* p = new (std::nothrow) frnn_host_pipeline;
    if (!p) return FRNN_ERR_CUDA;
    p->n_max = n_max; p->k_max = k_max;
    p->cap = edge_capacity;
    p->ws_bytes = frnn_workspace_bytes(n_max, 1, dim, k_max);
    p->slots.resize(static_cast<size_t>(depth));
    for (auto& s : p->slots) {
        bool ok = cudaStreamCreateWithFlags(&s.stream, cudaStreamNonBlocking) == cudaSuccess &&
                  cudaEventCreateWithFlags(&s.built, cudaEventDisableTiming) == cudaSuccess &&
                  cudaEventCreateWithFlags(&s.done, cudaEventDisableTiming) == cudaSuccess &&
                  cudaMalloc(&s.ws, p->ws_bytes) == cudaSuccess &&
                  cudaMalloc(reinterpret_cast<void**>(&s.pts), static_cast<size_t>(n_max) * 32) == cudaSuccess &&
                  cudaMalloc(reinterpret_cast<void**>(&s.src), static_cast<size_t>(p->cap) * 12) == cudaSuccess &&
                  cudaMalloc(reinterpret_cast<void**>(&s.count), 64) == cudaSuccess &&
                  cudaMallocHost(reinterpret_cast<void**>(&s.pinned), 64) == cudaSuccess;
        if (!ok) { cudaGetLastError(); pipeline_free(p); return FRNN_ERR_CUDA; }
        s.dst = s.src + p->cap;
        s.d2 = reinterpret_cast<float*>(s.dst + p->cap);
    }
    *out = p;
    return FRNN_OK;
}

int frnn_host_pipeline_submit(frnn_host_pipeline* p, const float* points, int64_t n, float r,
                              int32_t* out_src, int32_t* out_dst, float* out_d2, int64_t* out_count) {
    if (!p || !points || !out_src || !out_dst || !out_d2 || !out_count || n < 1 || n > p->n_max) return FRNN_ERR_INVALID_ARG;
    auto& s = p->slots[static_cast<size_t>(p->next)];
    int rc = pipeline_retire(p, s);                              // the oldest event in flight: wait for it if it is still there
    if (rc != FRNN_OK) return rc;
    if ((rc = pipeline_poll(p)) != FRNN_OK) return rc;
    CK(cudaMemcpyAsync(s.pts, points, static_cast<size_t>(n) * 32, cudaMemcpyHostToDevice, s.stream));
    int32_t* d_status = reinterpret_cast<int32_t*>(s.count + 1);
    rc = frnn_build_ex(s.pts, n, kDim, r, p->k_max, s.src, s.dst, s.d2, p->cap, s.count, d_status, nullptr, s.ws, p->ws_bytes, s.stream);
    if (rc != FRNN_OK) return rc;
    CK(cudaMemcpyAsync(s.pinned, s.count, 12, cudaMemcpyDeviceToHost, s.stream));
    CK(cudaEventRecord(s.built, s.stream));
    s.h_src = out_src; s.h_dst = out_dst; s.h_d2 = out_d2; s.h_count = out_count;
    s.state = frnn_host_pipeline::BUILDING;
    p->next = (p->next + 1) % static_cast<int>(p->slots.size());
    return FRNN_OK;
}

int frnn_host_pipeline_wait(frnn_host_pipeline* p) {
    if (!p) return FRNN_ERR_INVALID_ARG;
    const int n = static_cast<int>(p->slots.size());
    int rc = pipeline_poll(p);
    for (int k = 0; k < n && rc == FRNN_OK; ++k) rc = pipeline_retire(p, p->slots[static_cast<size_t>((p->next + k) % n)]);   // oldest first
    return rc;
}

void frnn_host_pipeline_destroy(frnn_host_pipeline* p) {
    if (p) pipeline_free(p);
}

int frnn_last_launch_count(void) { return t_launches; }

int frnn_set_profiling(int enabled) {
    g_timeline = enabled == 2;
    if (enabled == 2) enabled = 0;
    if (enabled && !g_ev_valid) {
        for (int i = 0; i <= kPhases; ++i)
            if (cudaEventCreate(&g_ev[i]) != cudaSuccess) return FRNN_ERR_CUDA;
        g_ev_valid = true;
    }
    g_profiling = enabled != 0;
    return FRNN_OK;
}

int frnn_get_profile(float* phase_ms, int max_phases) {
    if (!g_ev_valid || !phase_ms) return FRNN_ERR_INVALID_ARG;
    if (cudaEventSynchronize(g_ev[kPhases]) != cudaSuccess) return FRNN_ERR_CUDA;
    const int n = max_phases < kPhases ? max_phases : kPhases;
    for (int i = 0; i < n; ++i)
        if (cudaEventElapsedTime(&phase_ms[i], g_ev[i], g_ev[i + 1]) != cudaSuccess) return FRNN_ERR_CUDA;
    return n;
}

int frnn_get_timeline(const void* workspace, int64_t n_total, int n_events, int dim, double* begin_us, double* end_us, int max_phases) {
    if (!workspace || !begin_us || !end_us || n_total <= 0 || n_events < 1 || dim < 1 || dim > kDimMax) return FRNN_ERR_INVALID_ARG;
    const Layout L = make_layout(n_total, n_events, choose_grid(n_total, n_events, dim), dim, g_order.on != 0);
    unsigned long long h[2 * kTimelinePhases];
    if (cudaMemcpy(h, static_cast<const char*>(workspace) + L.off_counters + 64, sizeof(h), cudaMemcpyDeviceToHost) != cudaSuccess)
        return FRNN_ERR_CUDA;
    const int n = max_phases < kTimelinePhases ? max_phases : kTimelinePhases;
    const unsigned long long t0 = ~h[0];                   // start of the first kernel
    for (int i = 0; i < n; ++i) {
        begin_us[i] = 1e-3 * static_cast<double>(static_cast<long long>(~h[2 * i] - t0));
        end_us[i] = 1e-3 * static_cast<double>(static_cast<long long>(h[2 * i + 1] - t0));
    }
    return n;
}

const char* frnn_timeline_name(int phase) { return (phase >= 0 && phase < kTimelinePhases) ? kTimelineNames[phase] : ""; }

const char* frnn_phase_name(int phase) { return (phase >= 0 && phase < kPhases) ? kPhaseNames[phase] : ""; }

void frnn_release_cached(void) {
    {
        std::lock_guard<std::mutex> lock(g_graph_mutex);
        for (auto& g : g_graphs) cudaGraphExecDestroy(g.exec);
        g_graphs.clear();
    }
    if (g_cache.ws) cudaFree(g_cache.ws);
    if (g_cache.misc) cudaFree(g_cache.misc);
    if (g_cache.pts) cudaFree(g_cache.pts);
    if (g_cache.edges) cudaFree(g_cache.edges);
    if (g_cache.stream) cudaStreamDestroy(g_cache.stream);
    g_cache = Cache{};
}

}  // extern "C"
