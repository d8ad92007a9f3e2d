// frnn.cu -- host side of the C ABI declared in include/frnn.h (argument checks, workspace layout, launch plan,
// per-workspace CUDA-graph executables).  No CPU fallback: every compute entry point needs a CUDA device.
//
// A call is turned into a PLAN: one optional memset + a list of (kernel function, grid, by-value argument struct).
// The plan is either launched node by node on the caller's stream, or -- the default on a non-default stream --
// written into the nodes of an instantiated CUDA graph that belongs to the call's WORKSPACE and to the plan's shape
// (the list of kernel functions): cudaGraphExecKernelNodeSetParams / cudaGraphExecMemsetNodeSetParams per node whose
// grid or arguments changed since the last call, then one cudaGraphLaunch.  Nothing of the executable depends on n,
// the pointers, r, k_max or the capacity, so a stream of events of different sizes replays ONE graph
// (section 3: the latency "depends almost linearly on the number of spacepoints" -- events differ in size).
#include "frnn_kernels.cuh"
#include "launch_plan.h"

#include <math.h>
#include <stdio.h>
#include <string.h>

#include <atomic>
#include <memory>
#include <mutex>
#include <new>
#include <utility>
#include <vector>

#include "../../include/frnn.h"

namespace {

using namespace frnn;

constexpr float kCellSlack = 1.0078125f;   // 1 + 2^-7, see cell_coord()
constexpr size_t kAlign = 256;
constexpr int64_t kPrefixTilesMin = 1024;   // above this many emit tiles the tile offsets come from tile_prefix_kernel
constexpr int kTimelinePhases = 5;
constexpr size_t kCountersBytes = 256;      // head of every workspace (see make_layout)
constexpr size_t kStampsOffset = 64;        // of the timeline stamps inside it
const char* const kTimelineNames[kTimelinePhases] = {"bin", "scan_cells", "scatter", "search", "emit"};
constexpr int kPhases = 6;
const char* const kPhaseNames[kPhases] = {"memset", "bin", "scan_cells", "scatter", "search", "emit"};

// ---- last CUDA error of this thread (frnn_last_error_string)
thread_local char t_error[256] = "";
int cuda_fail(cudaError_t e, const char* what) {
    snprintf(t_error, sizeof(t_error), "%s: %s (%s)", what, cudaGetErrorString(e), cudaGetErrorName(e));
    cudaGetLastError();                     // do not leave a non-sticky error behind for the caller's next check
    return FRNN_ERR_CUDA;
}
#define CK(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return cuda_fail(e_, #call); } while (0)

// ---- per-call options; the process-wide defaults (frnn_set_grid / _bin_order / _graph_mode / _profiling(2)) are
// snapshotted once per call under a mutex, so concurrent calls never see a half-written default
struct Opts {
    int grid_dims = 0, grid_bits = 0;       // 0 = from the event size
    bool auto_grid = false;                 // FRNN_GRID_AUTO: the call looks at its own event first (one stream synchronise)
    BinOrder order = {0, {0, 1, 2, 3, 4, 5, 6, 7}};
    bool use_graph = true;
    bool timeline = false;
};
std::mutex g_defaults_mutex;
Opts g_defaults;
Opts default_opts() {
    std::lock_guard<std::mutex> lock(g_defaults_mutex);
    return g_defaults;
}

int make_order(const int* order, int count, BinOrder* out) {
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
    bool identity = true;                              // the default order written out: take the fast path
    for (int k = 0; k < 8; ++k) identity = identity && o.p[k] == k;
    if (identity) o.on = 0;
    *out = o;
    return FRNN_OK;
}

int opts_from(const frnn_options* in, Opts* out) {
    Opts o = default_opts();
    if (in) {
        if (in->struct_bytes < sizeof(frnn_options)) return FRNN_ERR_INVALID_ARG;
        if (in->grid_dims < FRNN_GRID_AUTO || in->grid_dims > 6 || (in->grid_bits != 0 && (in->grid_bits < 2 || in->grid_bits > 8))) return FRNN_ERR_INVALID_ARG;
        if (in->launch_mode < 0 || in->launch_mode > 2) return FRNN_ERR_INVALID_ARG;
        o.auto_grid = in->grid_dims == FRNN_GRID_AUTO;
        o.grid_dims = o.auto_grid ? 0 : in->grid_dims;
        o.grid_bits = o.auto_grid ? 0 : in->grid_bits;
        const int rc = make_order(in->order, in->order_count, &o.order);
        if (rc != FRNN_OK) return rc;
        if (in->launch_mode == FRNN_LAUNCH_GRAPH) o.use_graph = true;
        if (in->launch_mode == FRNN_LAUNCH_PLAIN) o.use_graph = false;
        if (in->timeline != 0) o.timeline = true;            // 0 keeps the process-wide setting (frnn_set_profiling(2))
    }
    *out = o;
    return FRNN_OK;
}

thread_local int t_launches = 0;

// Optional per-phase CUDA-event timing (frnn_set_profiling(1)): one event after every phase.  Bench instrumentation,
// process-global, not thread safe (documented).
bool g_profiling = false;
cudaEvent_t g_ev[kPhases + 1] = {};
bool g_ev_valid = false;

struct GridChoice { int dims, bits; };

// Grid: cells per event = 2^(dims*bits).  Finer grids cut candidate rows per query (3^dims cells of side ~r are
// visited) but cost table size and run bookkeeping.  Without a caller's choice (frnn_options, from frnn_suggest_grid or
// by hand) the grid follows the event size alone; the switch points come from the sweep in DESIGN.md section 7.
GridChoice choose_grid(const Opts& o, int64_t n_total, int n_events, int dim) {
    const int64_t per_event = n_events > 0 ? (n_total + n_events - 1) / n_events : n_total;
    GridChoice g;
    g.bits = o.grid_bits ? o.grid_bits : 5;
    if (o.grid_dims) g.dims = o.grid_dims;
    else if (per_event < 16384) g.dims = 3;
    else if (per_event < 400000) g.dims = 4;
    else g.dims = 5;
    if (!o.grid_dims && g.dims > dim) g.dims = dim;          // binning a padded (all-zero) coordinate prunes nothing
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

Layout make_layout(int64_t n_total, int n_events, GridChoice g, int dim, bool ordered) {
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
    // the counters block is the HEAD of the workspace: its offset depends on nothing (not on the grid, the options or n), so
    // frnn_get_timeline finds the stamps of a call whatever options that call was made with (FRNN_GRID_AUTO included)
    L.off_counters = o; o = align_up(o + kCountersBytes);   // [0..3] cursor of the cell scan (u32); [64..) timeline stamps (u64 x 2 x kTimelinePhases)
    L.off_cells = o;    o = align_up(o + static_cast<size_t>(L.n_entries + 8) * 4);
    L.off_tiles = o;    o = align_up(o + static_cast<size_t>(L.emit_tiles > 0 ? L.emit_tiles : 1) * 8 * kDegSlices);
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

// host_points: the pointer is only the source of a copy (frnn_build_host), so the 32-byte row alignment of the device
// fast path does not apply to it
int check_common(const float* points, int64_t n, int dim, float r, int k_max, const void* out_src, const void* out_dst,
                 const void* out_d2, int64_t capacity, bool host_points = false) {
    if (n < 0 || k_max < 1 || capacity < 0) return FRNN_ERR_INVALID_ARG;
    if (!(r >= 0.0f) || !isfinite(r)) return FRNN_ERR_INVALID_ARG;
    if (n > 0 && !points) return FRNN_ERR_INVALID_ARG;
    if (dim < 1 || dim > kDimMax) return FRNN_ERR_UNSUPPORTED;
    if (reinterpret_cast<uintptr_t>(points) % ((dim == kDim && !host_points) ? 32 : 4)) return FRNN_ERR_INVALID_ARG;   // 8-float rows move as 256-bit transactions
    if (capacity > 0 && (!out_src || !out_dst || !out_d2)) return FRNN_ERR_INVALID_ARG;
    if (n > 0x7fffffffll) return FRNN_ERR_UNSUPPORTED;
    return FRNN_OK;
}

struct Call {                 // everything that determines the enqueued work
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
    const int64_t* ev_off;        // HOST, n_events + 1
    bool dense = false;           // frnn_build_dense_ex: brute force instead of the grid
    Opts opts;
};

thread_local Plan t_plan;         // reused: a call allocates nothing once the vectors have grown

// The whole path as a plan.
void make_plan(const Call& c, const Layout& L, Plan& P) {
    P.clear();
    const int64_t n_total = c.ev_off[c.n_events];
    char* ws = static_cast<char*>(c.workspace);
    uint32_t* cells = reinterpret_cast<uint32_t*>(ws + L.off_cells);
    unsigned long long* tile_deg = reinterpret_cast<unsigned long long*>(ws + L.off_tiles);
    unsigned int* cursor = reinterpret_cast<unsigned int*>(ws + L.off_counters);
    unsigned long long* stamps = c.opts.timeline ? reinterpret_cast<unsigned long long*>(ws + L.off_counters + kStampsOffset) : nullptr;
    uint32_t* pcell = reinterpret_cast<uint32_t*>(ws + L.off_pcell);
    uint32_t* prank = reinterpret_cast<uint32_t*>(ws + L.off_prank);
    float4* spts = reinterpret_cast<float4*>(ws + L.off_spts);
    float4* spts_hi = c.dim > kDim ? reinterpret_cast<float4*>(ws + L.off_spts_hi) : nullptr;
    uint32_t* scell = c.opts.order.on ? reinterpret_cast<uint32_t*>(ws + L.off_scell) : nullptr;
    int32_t* sidx = reinterpret_cast<int32_t*>(ws + L.off_sidx);
    uint32_t* skey = reinterpret_cast<uint32_t*>(ws + L.off_skey);
    uint32_t* cnt = reinterpret_cast<uint32_t*>(ws + L.off_cnt);
    int64_t* ev_off = reinterpret_cast<int64_t*>(ws + L.off_evoff);
    int2* hits = reinterpret_cast<int2*>(ws + L.off_hits);
    unsigned long long* tprefix = reinterpret_cast<unsigned long long*>(ws + L.off_tprefix);
    const float* pts = c.points;
    const int G = c.grid_dims, bits = c.grid_bits;
    const BinOrder order = c.opts.order;

    const float r2 = c.r * c.r;                               // R2: fl32(r*r), once, on the host
    const float cell_side = fmaxf(c.r * kCellSlack, 1e-30f);
    const float inv_cell = 1.0f / cell_side;
    const unsigned emit_tiles = static_cast<unsigned>(L.emit_tiles);

    EmitArgs ea;
    ea.pts = pts; ea.dim = c.dim; ea.cnt = cnt; ea.hits = hits; ea.tile_deg = tile_deg; ea.tile_prefix = nullptr;
    ea.n_total = n_total; ea.row_ptr = c.out_row_ptr; ea.out_src = c.out_src; ea.out_dst = c.out_dst; ea.out_d2 = c.out_d2;
    ea.capacity = c.capacity; ea.out_count = c.out_count; ea.out_status = c.out_status; ea.r2 = r2; ea.inv_cell = inv_cell; ea.bits = bits;
    ea.k_max = static_cast<uint32_t>(c.k_max); ea.n_tiles = emit_tiles; ea.order = order;

    if (c.dense) {                                             // brute force: no table, no sort (single event)
        P.ms_dst = ws + L.off_tiles;
        P.ms_bytes = L.zero_bytes - L.off_tiles;
        DenseArgs da;
        da.pts = pts; da.dim = c.dim; da.cnt = cnt; da.hits = hits; da.tile_deg = tile_deg; da.n_tiles = emit_tiles;
        da.n = n_total; da.r2 = r2; da.k_max = static_cast<uint32_t>(c.k_max);
        const unsigned T = static_cast<unsigned>((n_total + kDenseTile - 1) / kDenseTile);              // candidate tiles (x)
        const int qrows = (c.dim > kDim ? DenseCfg<true>::Q : DenseCfg<false>::Q) * kDenseTile;          // queries per block (y)
        const unsigned TQ = static_cast<unsigned>((n_total + qrows - 1) / qrows);
        P.add(c.dim > kDim ? fptr(dense_search_kernel<true>) : fptr(dense_search_kernel<false>), T, TQ, kDenseTile, 4, da);
        ea.spts = nullptr; ea.spts_hi = nullptr; ea.sidx = nullptr; ea.cell_start = nullptr; ea.ev_off = nullptr; ea.n_events = 1;
        ea.out_edge_offsets = nullptr; ea.stamps = nullptr; ea.dense = 1;
        if (L.emit_tiles > kPrefixTilesMin) {
            P.add(fptr(tile_prefix_kernel), 1, 1, kPrefixThreads, 5, PrefixArgs{tile_deg, emit_tiles, tprefix});
            ea.tile_prefix = tprefix;
        }
        P.add(fptr(emit_kernel<1>), emit_tiles, 1, kEmitThreads, 5, ea);
        return;
    }
    P.ms_dst = ws;
    P.ms_bytes = L.zero_bytes;
    // Event offsets reach the device as kernel arguments (no pageable-memory copy, which would
    // synchronise the host with the stream); a single event needs none (base 0).
    if (c.n_events > 1) {
        for (int first = 0; first <= c.n_events; first += OffsetChunk::kN) {
            OffsetChunk ch;
            ch.ev_off = ev_off;
            ch.first = first;
            ch.count = (c.n_events + 1 - first) < OffsetChunk::kN ? (c.n_events + 1 - first) : OffsetChunk::kN;
            for (int k = 0; k < ch.count; ++k) ch.v[k] = c.ev_off[first + k];
            for (int k = ch.count; k < OffsetChunk::kN; ++k) ch.v[k] = 0;
            P.add(fptr(set_offsets_kernel), 1, 1, OffsetChunk::kN, 0, ch);
        }
    } else {
        ev_off = nullptr;
    }
    const unsigned row_blocks = static_cast<unsigned>((n_total + 255) / 256);
    BinArgs ba{pts, c.dim, n_total, ev_off, c.n_events, inv_cell, bits, cells, pcell, prank, order, stamps};
    FRNN_DISPATCH_G(G, (P.add(fptr(bin_kernel<GG>), row_blocks, 1, 256, 1, ba)));
    P.add(fptr(cell_scan_kernel), static_cast<unsigned>(L.scan_blocks), 1, kCellThreads, 2,
          ScanArgs{cells, L.n_entries, L.rows_per_block, bits, cursor, stamps});
    ScatterArgs sc{pts, c.dim, n_total, bits, inv_cell, cells, pcell, prank, spts, sidx, skey, spts_hi, scell, order, stamps};
    FRNN_DISPATCH_G(G, (P.add(fptr(scatter_kernel<GG>), row_blocks, 1, 256, 3, sc)));

    SearchArgs sa;
    sa.scell = scell;
    sa.spts = spts; sa.spts_hi = spts_hi; sa.sidx = sidx; sa.skey = skey; sa.cell_start = cells; sa.cnt = cnt; sa.hits = hits;
    sa.tile_deg = tile_deg; sa.n_tiles = emit_tiles; sa.ev_off = ev_off; sa.stamps = stamps; sa.n_total = n_total; sa.n_events = c.n_events; sa.r2 = r2;
    sa.inv_cell = inv_cell; sa.bits = bits; sa.k_max = static_cast<uint32_t>(c.k_max);
    const unsigned search_blocks = static_cast<unsigned>((n_total + kSearchThreads - 1) / kSearchThreads);
    if (spts_hi) { FRNN_DISPATCH_G(G, (P.add(fptr(search_kernel<GG, true>), search_blocks, 1, kSearchThreads, 4, sa))); }
    else         { FRNN_DISPATCH_G(G, (P.add(fptr(search_kernel<GG, false>), search_blocks, 1, kSearchThreads, 4, sa))); }

    ea.spts = spts; ea.spts_hi = spts_hi; ea.sidx = sidx; ea.cell_start = cells; ea.ev_off = ev_off; ea.n_events = c.n_events;
    ea.out_edge_offsets = c.out_edge_offsets; ea.stamps = stamps; ea.dense = 0;
    if (L.emit_tiles > kPrefixTilesMin) {                      // many tiles: their prefix in one small kernel (see tile_prefix_kernel)
        P.add(fptr(tile_prefix_kernel), 1, 1, kPrefixThreads, 5, PrefixArgs{tile_deg, emit_tiles, tprefix});
        ea.tile_prefix = tprefix;
    }
    FRNN_DISPATCH_G(G, (P.add(fptr(emit_kernel<GG>), emit_tiles, 1, kEmitThreads, 5, ea)));
}

// ---- the plan launched node by node (legacy default stream, a capturing caller, graph mode off, per-phase events)
int launch_plain(const Plan& P, cudaStream_t st) {
    const bool prof = g_profiling && g_ev_valid;
    int cur = 0;                                              // events recorded so far = cur + 1
    if (prof) cudaEventRecord(g_ev[0], st);
    if (P.ms_bytes) { CK(cudaMemsetAsync(P.ms_dst, 0, P.ms_bytes, st)); ++t_launches; }
    for (const Node& nd : P.nodes) {
        if (prof) for (; cur < nd.phase; ++cur) cudaEventRecord(g_ev[cur + 1], st);
        void* argp = const_cast<unsigned char*>(P.args.data() + nd.arg_off);
        CK(cudaLaunchKernel(nd.func, dim3(nd.grid_x, nd.grid_y), dim3(nd.block), &argp, 0, st));
        ++t_launches;
    }
    if (prof) for (; cur < kPhases; ++cur) cudaEventRecord(g_ev[cur + 1], st);
    return FRNN_OK;
}

// ------------------------------------------------------------------------------------------------
// Per-workspace graph executables.  An entry belongs to (workspace pointer, shape = list of kernel functions); a
// workspace sees few shapes (the grid changes with the event-size class, dense vs grid, batched chunk count), so a
// handful of entries per workspace and kMaxExecs in total (least recently used evicted) are plenty.  The global mutex
// covers only the lookup; update + launch run under the entry's own mutex, so threads that use distinct workspaces
// (the contract of include/frnn.h) never wait for each other.
// ------------------------------------------------------------------------------------------------
struct ExecEntry {
    void* workspace = nullptr;
    std::vector<const void*> funcs;
    bool has_memset = true;
    cudaGraph_t graph = nullptr;  // kept alive: its node handles address the executable's nodes in the update calls
    cudaGraphExec_t exec = nullptr;
    cudaGraphNode_t ms_node = nullptr;
    std::vector<cudaGraphNode_t> knodes;
    Plan held;                    // the parameters the executable currently holds
    uint64_t stamp = 0;
    std::mutex mu;
    ~ExecEntry() {
        if (exec) cudaGraphExecDestroy(exec);
        if (graph) cudaGraphDestroy(graph);
    }
};
std::vector<std::shared_ptr<ExecEntry>> g_execs;
std::mutex g_exec_mutex;
uint64_t g_stamp = 0;
constexpr size_t kMaxExecs = 64;
std::atomic<long long> g_graph_builds{0};     // frnn_graph_builds(): a stream of calls of one shape must not move it

bool same_shape(const ExecEntry& e, const Plan& P) {
    if (e.funcs.size() != P.nodes.size() || e.has_memset != (P.ms_bytes != 0)) return false;
    for (size_t k = 0; k < P.nodes.size(); ++k)
        if (e.funcs[k] != P.nodes[k].func) return false;
    return true;
}

cudaKernelNodeParams node_params(const Node& nd, void** argp) {
    cudaKernelNodeParams kp = {};
    kp.func = const_cast<void*>(nd.func);
    kp.gridDim = dim3(nd.grid_x, nd.grid_y);
    kp.blockDim = dim3(nd.block);
    kp.sharedMemBytes = 0;
    kp.kernelParams = argp;
    kp.extra = nullptr;
    return kp;
}
cudaMemsetParams memset_params(const Plan& P) {
    cudaMemsetParams mp = {};
    mp.dst = P.ms_dst;
    mp.pitch = 0;
    mp.value = 0;
    mp.elementSize = 1;
    mp.width = P.ms_bytes;
    mp.height = 1;
    return mp;
}

// build the executable of entry e from plan P (explicit nodes, a linear chain)
int build_exec(ExecEntry& e, const Plan& P) {
    if (e.exec) { cudaGraphExecDestroy(e.exec); e.exec = nullptr; }
    if (e.graph) { cudaGraphDestroy(e.graph); e.graph = nullptr; }
    e.knodes.clear();
    cudaGraph_t graph = nullptr;
    CK(cudaGraphCreate(&graph, 0));
    cudaError_t err = cudaSuccess;
    cudaGraphNode_t prev = nullptr;
    if (P.ms_bytes) {
        const cudaMemsetParams mp = memset_params(P);
        err = cudaGraphAddMemsetNode(&e.ms_node, graph, nullptr, 0, &mp);
        prev = e.ms_node;
    }
    for (size_t k = 0; err == cudaSuccess && k < P.nodes.size(); ++k) {
        void* argp = const_cast<unsigned char*>(P.args.data() + P.nodes[k].arg_off);
        const cudaKernelNodeParams kp = node_params(P.nodes[k], &argp);
        cudaGraphNode_t node = nullptr;
        err = cudaGraphAddKernelNode(&node, graph, prev ? &prev : nullptr, prev ? 1 : 0, &kp);
        e.knodes.push_back(node);
        prev = node;
    }
    if (err == cudaSuccess) err = cudaGraphInstantiate(&e.exec, graph, 0);
    if (err != cudaSuccess) { cudaGraphDestroy(graph); e.exec = nullptr; return cuda_fail(err, "building the CUDA graph"); }
    e.graph = graph;
    g_graph_builds.fetch_add(1, std::memory_order_relaxed);
    e.held = P;                                                // (e.funcs, the identity of the entry, was set at creation)
    return FRNN_OK;
}

// write what changed since the last launch into the executable's nodes
int update_exec(ExecEntry& e, const Plan& P) {
    if (P.ms_bytes && (e.held.ms_dst != P.ms_dst || e.held.ms_bytes != P.ms_bytes)) {
        const cudaMemsetParams mp = memset_params(P);
        const cudaError_t err = cudaGraphExecMemsetNodeSetParams(e.exec, e.ms_node, &mp);
        if (err != cudaSuccess) return cuda_fail(err, "cudaGraphExecMemsetNodeSetParams");
        e.held.ms_dst = P.ms_dst;
        e.held.ms_bytes = P.ms_bytes;
    }
    if (e.held.args.size() != P.args.size()) e.held.args.assign(P.args.size(), 0);     // (same shape: same sizes, in fact)
    for (size_t k = 0; k < P.nodes.size(); ++k) {
        const Node& nd = P.nodes[k];
        Node& old = e.held.nodes[k];
        const unsigned char* src = P.args.data() + nd.arg_off;
        unsigned char* dst = e.held.args.data() + nd.arg_off;
        if (old.grid_x == nd.grid_x && old.grid_y == nd.grid_y && old.block == nd.block && memcmp(src, dst, nd.arg_bytes) == 0) continue;
        void* argp = const_cast<unsigned char*>(src);
        const cudaKernelNodeParams kp = node_params(nd, &argp);
        const cudaError_t err = cudaGraphExecKernelNodeSetParams(e.exec, e.knodes[k], &kp);
        if (err != cudaSuccess) return cuda_fail(err, "cudaGraphExecKernelNodeSetParams");
        memcpy(dst, src, nd.arg_bytes);
        old = nd;
    }
    return FRNN_OK;
}

int launch_graph(const Plan& P, void* workspace, cudaStream_t st) {
    std::shared_ptr<ExecEntry> e;
    {
        std::lock_guard<std::mutex> lock(g_exec_mutex);
        for (auto& x : g_execs)
            if (x->workspace == workspace && same_shape(*x, P)) { e = x; break; }
        if (!e) {
            if (g_execs.size() >= kMaxExecs) {                 // evict the least recently used
                size_t victim = 0;
                for (size_t k = 1; k < g_execs.size(); ++k)
                    if (g_execs[k]->stamp < g_execs[victim]->stamp) victim = k;
                g_execs.erase(g_execs.begin() + victim);       // destroyed when its last user lets go
            }
            e = std::make_shared<ExecEntry>();
            e->workspace = workspace;
            e->has_memset = P.ms_bytes != 0;
            for (const Node& nd : P.nodes) e->funcs.push_back(nd.func);
            g_execs.push_back(e);
        }
        e->stamp = ++g_stamp;
    }
    std::lock_guard<std::mutex> lock(e->mu);
    int rc = FRNN_OK;
    if (!e->exec) rc = build_exec(*e, P);
    else if ((rc = update_exec(*e, P)) != FRNN_OK) rc = build_exec(*e, P);     // an update the driver refuses: start over (counted, see frnn_graph_builds)
    if (rc != FRNN_OK) return rc;
    CK(cudaGraphLaunch(e->exec, st));
    t_launches = static_cast<int>(P.nodes.size()) + (P.ms_bytes ? 1 : 0);
    return FRNN_OK;
}

}  // namespace

namespace frnn {
int run_plan(const Plan& P, void* key, cudaStream_t st, bool want_graph) {
    t_launches = 0;
    bool graph_ok = want_graph && !g_profiling && st != nullptr && st != cudaStreamLegacy;
    if (graph_ok) {
        cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
        if (cudaStreamIsCapturing(st, &cs) != cudaSuccess || cs != cudaStreamCaptureStatusNone) { cudaGetLastError(); graph_ok = false; }   // caller is capturing: just enqueue
    }
    if (!graph_ok) return launch_plain(P, st);
    return launch_graph(P, key, st);
}
bool default_use_graph() { return default_opts().use_graph; }
}  // namespace frnn

namespace {

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
    const Layout L = make_layout(n_total, c.n_events, GridChoice{c.grid_dims, c.grid_bits}, c.dim, c.opts.order.on != 0);
    Plan& P = t_plan;
    make_plan(c, L, P);
    return frnn::run_plan(P, c.workspace, st, c.opts.use_graph);
}

int prepare(Call& c, size_t workspace_bytes) {
    const int64_t n_total = c.ev_off[c.n_events];
    const GridChoice g = choose_grid(c.opts, n_total, c.n_events, c.dim);
    c.grid_dims = g.dims;
    c.grid_bits = g.bits;
    if (n_total == 0) return FRNN_OK;
    const Layout L = make_layout(n_total, c.n_events, g, c.dim, c.opts.order.on != 0);
    if (!c.workspace || workspace_bytes < L.total) return FRNN_ERR_WORKSPACE;
    if (reinterpret_cast<uintptr_t>(c.workspace) % kAlign) return FRNN_ERR_INVALID_ARG;
    return FRNN_OK;
}

// table budget of the data-driven choices: 64 cells per point of an event (a finer table costs more to zero and scan than
// it saves), 2^26 cells in all, and a linear cell id that fits 30 bits
bool grid_within_budget(int g, int bits, double n_event, int n_events) {
    int ev_bits = 0;
    while ((1ll << ev_bits) < n_events) ++ev_bits;
    const double budget = fmin(fmax(65536.0, 64.0 * n_event), 67108864.0 / n_events);
    return g * bits + ev_bits <= 30 && pow(2.0, g * bits) <= budget;
}
int auto_grid(const float* points, int64_t n, int n_events, int dim, float r, cudaStream_t st, int* g, int* bits);   // below

int build_single(const Opts& o, bool dense, const float* points, int64_t n, int dim, float r, int k_max,
                 int32_t* out_src, int32_t* out_dst, float* out_d2, int64_t edge_capacity,
                 int64_t* out_count, int32_t* out_status, int64_t* out_row_ptr,
                 void* workspace, size_t workspace_bytes, void* cuda_stream) {
    int rc = check_common(points, n, dim, r, k_max, out_src, out_dst, out_d2, edge_capacity);
    if (rc != FRNN_OK) return rc;
    if (!out_count || !out_status) return FRNN_ERR_INVALID_ARG;
    if (dense && n > 65535ll * kDenseTile) return FRNN_ERR_UNSUPPORTED;       // grid.y limit (8.3 M rows)
    const int64_t ev_off[2] = {0, n};
    Call c{points, dim, 1, r, k_max, out_src, out_dst, out_d2, edge_capacity, out_count, nullptr, out_status, out_row_ptr, workspace, 0, 0, ev_off};
    c.dense = dense;
    c.opts = o;
    if (o.auto_grid && !dense && n > 0) {                                     // S1 from this very event (synchronises the stream once)
        c.opts.auto_grid = false;
        if ((rc = auto_grid(points, n, 1, dim, r, static_cast<cudaStream_t>(cuda_stream), &c.opts.grid_dims, &c.opts.grid_bits)) != FRNN_OK) return rc;
    }
    if ((rc = prepare(c, workspace_bytes)) != FRNN_OK) return rc;
    return run_call(c, static_cast<cudaStream_t>(cuda_stream));
}

int build_batched(const Opts& o, const float* points, const int64_t* event_offsets, int n_events, int dim, float r, int k_max,
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
           workspace, 0, 0, event_offsets};
    c.opts = o;
    if (o.auto_grid && event_offsets[n_events] > 0) {
        c.opts.auto_grid = false;
        if ((rc = auto_grid(points, event_offsets[n_events], n_events, dim, r, static_cast<cudaStream_t>(cuda_stream), &c.opts.grid_dims,
                            &c.opts.grid_bits)) != FRNN_OK) return rc;
    }
    if ((rc = prepare(c, workspace_bytes)) != FRNN_OK) return rc;
    return run_call(c, static_cast<cudaStream_t>(cuda_stream));
}

size_t workspace_bytes_for(const Opts& o, int64_t n_total, int n_events, int dim, int k_max) {
    if (n_total < 0 || n_events < 1 || dim < 1 || dim > kDimMax || k_max < 1 || n_total > 0x7fffffffll) return 0;
    if (o.auto_grid) {                                                        // room for whichever grid the call may pick
        size_t need = 0;
        Opts t = o;
        t.auto_grid = false;
        for (t.grid_dims = 1; t.grid_dims <= 6 && t.grid_dims <= dim; ++t.grid_dims)
            for (t.grid_bits = 2; t.grid_bits <= 8; ++t.grid_bits) {
                if (!grid_within_budget(t.grid_dims, t.grid_bits, static_cast<double>(n_total) / n_events, n_events)) continue;
                const size_t b = make_layout(n_total, n_events, GridChoice{t.grid_dims, t.grid_bits}, dim, o.order.on != 0).total;
                if (b > need) need = b;
            }
        return need;
    }
    return make_layout(n_total, n_events, choose_grid(o, n_total, n_events, dim), dim, o.order.on != 0).total;
}

// The three edge arrays to the host.  On the device they sit one capacity apart; when the caller's three host arrays are
// equally spaced too (one block holding src | dst | d2, the natural way to allocate them) they travel as ONE 2-D copy of
// three rows -- a DMA set-up costs about 6 us, and three copies per event instead of one cost 17 us of a 100 us event
// (profiles/r02_summary.md); otherwise as three copies.
// (Equally spaced arrays that are SEPARATE page-locked allocations make the runtime refuse the 2-D copy; *refused remembers
// the base pointer for which that happened, so that it is not tried again for the same buffers.)
int copy_edges_to_host(int32_t* h_src, int32_t* h_dst, float* h_d2, const int32_t* d_src, size_t d_cap, size_t e, cudaStream_t st,
                       const void** refused) {
    if (!e) return FRNN_OK;
    const ptrdiff_t p1 = reinterpret_cast<char*>(h_dst) - reinterpret_cast<char*>(h_src);
    const ptrdiff_t p2 = reinterpret_cast<char*>(h_d2) - reinterpret_cast<char*>(h_dst);
    if (p1 == p2 && p1 >= static_cast<ptrdiff_t>(e * 4) && *refused != h_src) {
        if (cudaMemcpy2DAsync(h_src, static_cast<size_t>(p1), d_src, d_cap * 4, e * 4, 3, cudaMemcpyDeviceToHost, st) == cudaSuccess) return FRNN_OK;
        cudaGetLastError();
        *refused = h_src;
    }
    CK(cudaMemcpyAsync(h_src, d_src, e * 4, cudaMemcpyDeviceToHost, st));
    CK(cudaMemcpyAsync(h_dst, d_src + d_cap, e * 4, cudaMemcpyDeviceToHost, st));
    CK(cudaMemcpyAsync(h_d2, d_src + 2 * d_cap, e * 4, cudaMemcpyDeviceToHost, st));
    return FRNN_OK;
}

// cached device buffers for the synchronous convenience entry points (one user at a time: g_cache_mutex)
struct Cache {
    void* ws = nullptr; size_t ws_bytes = 0;
    void* misc = nullptr;                       // count (8) + status (4)
    void* pts = nullptr; size_t pts_bytes = 0;
    void* edges = nullptr; size_t edge_cap = 0; // src | dst | d2, edge_cap each
    cudaStream_t stream = nullptr;              // non-default stream so the graph path applies
} g_cache;
std::mutex g_cache_mutex;

int ensure(void** p, size_t* have, size_t need) {
    if (*have >= need && *p) return FRNN_OK;
    if (*p) cudaFree(*p);
    *p = nullptr; *have = 0;
    CK(cudaMalloc(p, need));
    *have = need;
    return FRNN_OK;
}

int ensure_stream() {
    if (!g_cache.stream) CK(cudaStreamCreateWithFlags(&g_cache.stream, cudaStreamNonBlocking));
    return FRNN_OK;
}

// ------------------------------------------------------------------------------------------------
// S1 from the data: per coordinate, the histogram of the cell coordinate (cells of side
// r (1 + 2^-7), modulo 256) over a sample of the points, and the coordinate's minimum and maximum.  Folded to
// 2^bits cells on the host, a histogram p gives  s(bits) = sum_c p_c (p_(c-1) + p_c + p_(c+1)),  the probability
// that two random points fall within one cell of each other along that coordinate on a torus of 2^bits cells: the
// factor by which binning (or keying) that coordinate cuts the candidates.  PAPER.md:69 (section 3.4): the cost of
// the cells grows as O(3^k k n) in the number k of binned coordinates, which is why the paper stops at three; the
// choice below weighs exactly that against the candidates saved.
// ------------------------------------------------------------------------------------------------
constexpr int kSugBins = 256;
struct SuggestOut {
    unsigned int hist[kDimMax][kSugBins];
    float lo[kDimMax], hi[kDimMax];
    unsigned int sampled;
};
struct SuggestArgs {
    const float* pts;
    int64_t n;
    int dim;
    float inv_cell;
    int64_t stride;
    SuggestOut* out;
};
__global__ void __launch_bounds__(1024) suggest_kernel(SuggestArgs k) {
    __shared__ unsigned int s_h[kDimMax][kSugBins];
    __shared__ float s_lo[kDimMax][32], s_hi[kDimMax][32];
    for (int t = threadIdx.x; t < kDimMax * kSugBins; t += blockDim.x) (&s_h[0][0])[t] = 0u;
    __syncthreads();
    const float inf = __int_as_float(0x7f800000);
    float lo[kDimMax], hi[kDimMax];
#pragma unroll
    for (int d = 0; d < kDimMax; ++d) { lo[d] = inf; hi[d] = -inf; }
    unsigned int mine = 0;
    for (int64_t i = static_cast<int64_t>(threadIdx.x) * k.stride; i < k.n; i += static_cast<int64_t>(blockDim.x) * k.stride) {
#pragma unroll
        for (int d = 0; d < kDimMax; ++d)
            if (d < k.dim) {
                const float x = k.pts[i * k.dim + d];
                atomicAdd(&s_h[d][cell_coord(x, k.inv_cell, kSugBins - 1)], 1u);
                lo[d] = fminf(lo[d], x);
                hi[d] = fmaxf(hi[d], x);
            }
        ++mine;
    }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int d = 0; d < kDimMax; ++d) {
#pragma unroll
        for (int o = 16; o >= 1; o >>= 1) {
            lo[d] = fminf(lo[d], __shfl_xor_sync(kFull, lo[d], o));
            hi[d] = fmaxf(hi[d], __shfl_xor_sync(kFull, hi[d], o));
        }
        if (lane == 0) { s_lo[d][warp] = lo[d]; s_hi[d][warp] = hi[d]; }
    }
    __shared__ unsigned int s_total;
    if (threadIdx.x == 0) s_total = 0;
    __syncthreads();
    atomicAdd(&s_total, mine);
    __syncthreads();
    for (int t = threadIdx.x; t < kDimMax * kSugBins; t += blockDim.x) (&k.out->hist[0][0])[t] = (&s_h[0][0])[t];
    if (threadIdx.x < kDimMax) {
        float a = inf, b = -inf;
        for (int w = 0; w < static_cast<int>(blockDim.x >> 5); ++w) { a = fminf(a, s_lo[threadIdx.x][w]); b = fmaxf(b, s_hi[threadIdx.x][w]); }
        k.out->lo[threadIdx.x] = a;
        k.out->hi[threadIdx.x] = b;
    }
    if (threadIdx.x == 0) k.out->sampled = s_total;
}

// One page-locked result block per HOST THREAD (the kernel writes it through its device alias; 17 KB, allocated by the
// thread's first call and kept): calls from different threads share nothing, so they wait only for their own stream,
// as include/frnn.h promises for calls on distinct workspaces.
thread_local SuggestOut* t_suggest_host = nullptr;

int run_suggest(const float* points, int64_t n, int dim, float r, cudaStream_t st, SuggestOut* result) {
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;       // the estimate synchronises the stream: not while it is being captured
    if (cudaStreamIsCapturing(st, &cs) != cudaSuccess) { cudaGetLastError(); cs = cudaStreamCaptureStatusNone; }
    if (cs != cudaStreamCaptureStatusNone) return FRNN_ERR_UNSUPPORTED;
    if (!t_suggest_host) CK(cudaHostAlloc(reinterpret_cast<void**>(&t_suggest_host), sizeof(SuggestOut), cudaHostAllocMapped));
    SuggestOut* dev = nullptr;
    CK(cudaHostGetDevicePointer(reinterpret_cast<void**>(&dev), t_suggest_host, 0));
    SuggestArgs a;
    a.pts = points; a.n = n; a.dim = dim;
    a.inv_cell = 1.0f / fmaxf(r * kCellSlack, 1e-30f);
    a.stride = (n + 65535) / 65536;                                // every stride-th row: at most 65,536 rows
    if (a.stride < 1) a.stride = 1;
    a.out = dev;
    suggest_kernel<<<1, 1024, 0, st>>>(a);
    CK(cudaGetLastError());
    CK(cudaStreamSynchronize(st));
    *result = *t_suggest_host;
    return FRNN_OK;
}

// s(bits) of one coordinate from its 256-bin histogram
double pair_probability(const unsigned int* h256, int bits, double total) {
    const int m = 1 << bits;
    double p[kSugBins];
    for (int c = 0; c < m; ++c) p[c] = 0.0;
    for (int c = 0; c < kSugBins; ++c) p[c & (m - 1)] += h256[c] / total;
    if (m <= 2) return 1.0;
    double acc = 0.0;
    for (int c = 0; c < m; ++c) acc += p[c] * (p[(c + m - 1) & (m - 1)] + p[c] + p[(c + 1) & (m - 1)]);
    return acc;
}

// Cost model of one call on the grid (g, bits) in microseconds of device time, fitted to the sweeps recorded in
// DESIGN.md section 7 (B200): a fixed part (launch and dependency latency of the six graph nodes), the table entries to
// zero and scan, per query the neighbour rows (the 3^(g-1) term of PAPER.md:69: two table reads and bookkeeping per row,
// with a latency term of its own for g >= 4 because a thread walks its rows one sub-batch after the other) and the
// candidate keys tested, dearer beyond the first four of a run (they take the merged leftover loop).  The model only
// has to RANK the alternatives well enough for the true best to make the shortlist that is then measured.
struct GridCost { double us, cand, surv; };
GridCost grid_cost(const double s[kDimMax][9], const unsigned char* order, int dim, int g, int bits, double n_event, int n_events) {
    static const double kRowLatency[7] = {0, 0, 0, 0.5, 4.7, 46.0, 90.0};          // us, whatever n is
    static const double kRowsPer100k[7] = {0, 0, 0, 1.2, 13.9, 37.4, 110.0};       // us per 100,000 queries
    double cand = n_event;
    for (int d = 0; d < g; ++d) cand *= order[d] < dim ? s[order[d]][bits] : 1.0;
    double surv = cand;
    for (int f = 0; f < 4; ++f)
        if (g + f < kDim && order[g + f] < dim) surv *= s[order[g + f]][6];
    double runs = 1.0;
    for (int d = 0; d + 1 < g; ++d) runs *= 3.0;
    const double entries = static_cast<double>(n_events) * pow(2.0, g * bits) * (1.0 + pow(2.0, -bits));
    const double n_all = n_event * n_events;
    const double beyond = fmax(0.0, cand - 4.0 * runs);                            // candidates past the first four of their run
    GridCost c;
    c.cand = cand;
    c.surv = surv;
    c.us = 23.0 + kRowLatency[g] + 2.0e-6 * entries + n_all * (1e-5 * kRowsPer100k[g] + 0.35e-6 * cand + 1.2e-6 * beyond + 6.0e-6 * surv);
    return c;
}

struct GridTry { int g, bits, order; GridCost c; float measured_us; };

// FRNN_GRID_AUTO: the model's best grid (default coordinate order) for this call's own rows
int auto_grid(const float* points, int64_t n, int n_events, int dim, float r, cudaStream_t st, int* g_out, int* bits_out) {
    SuggestOut so;
    const int rc = run_suggest(points, n, dim, r, st, &so);
    if (rc != FRNN_OK) return rc;
    const double tot = so.sampled ? static_cast<double>(so.sampled) : 1.0;
    double s[kDimMax][9];
    for (int d = 0; d < kDimMax; ++d)
        for (int b = 0; b <= 8; ++b) s[d][b] = (d < dim && b >= 2) ? pair_probability(so.hist[d], b, tot) : 1.0;
    const unsigned char ident[8] = {0, 1, 2, 3, 4, 5, 6, 7};
    const double n_event = static_cast<double>(n) / n_events;
    double best = 0.0;
    *g_out = 0;
    for (int g = 1; g <= 6 && g <= dim; ++g)
        for (int bits = 2; bits <= 8; ++bits) {
            if (!grid_within_budget(g, bits, n_event, n_events)) continue;
            const double us = grid_cost(s, ident, dim, g, bits, n_event, n_events).us;
            if (*g_out == 0 || us < best) { best = us; *g_out = g; *bits_out = bits; }
        }
    return *g_out ? FRNN_OK : FRNN_ERR_UNSUPPORTED;
}

}  // namespace

// ------------------------------------------------------------------------------------------------
// Scratch of frnn_build_static (include/frnn.h): the workspace of one small single-event build, reserved inside the
// library image itself so that the entry point never has to ask the CUDA runtime for device memory.  Every device
// that loads the library carries its own copy of these bytes from the moment the module is loaded until the process
// exits, which is why the limit is kept small (FRNN_STATIC_MAX_ROWS rows).
// The NAME below means two different things.  In device code it is the array.  In host code it is only a handle the
// runtime knows the array by -- it is NOT a device address, and a kernel handed `g_static_scratch` from the host
// would read and write the wrong memory.  Host code therefore asks the runtime for the real address, once per
// device and with that device current (static_scratch_for_current_device), and passes that to the kernels.
// ------------------------------------------------------------------------------------------------
constexpr size_t kStaticScratchBytes = 3u << 20;          // 3 MiB: the 8192-row, dim 9..16 layout needs 2,923,776 bytes
static __device__ __align__(256) unsigned char g_static_scratch[kStaticScratchBytes];

namespace {

constexpr int kStaticMaxDevices = 64;
void* g_static_ptr[kStaticMaxDevices] = {};                // device address of g_static_scratch, per device ordinal
std::mutex g_static_mutex;

// Device address of the current device's copy of g_static_scratch.  The first call on a device asks the runtime for it
// (that may load the module: it must not happen while a stream is being captured); later calls read the cached value.
int static_scratch_for_current_device(void** out) {
    int dev = -1;
    CK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kStaticMaxDevices) {
        snprintf(t_error, sizeof(t_error), "frnn_build_static: device ordinal %d outside 0..%d", dev, kStaticMaxDevices - 1);
        return FRNN_ERR_UNSUPPORTED;
    }
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_ptr[dev]) {
        void* p = nullptr;
        CK(cudaGetSymbolAddress(&p, g_static_scratch));
        if (!p || reinterpret_cast<uintptr_t>(p) % kAlign) {
            snprintf(t_error, sizeof(t_error), "frnn_build_static: cudaGetSymbolAddress returned an unusable address %p", p);
            return FRNN_ERR_CUDA;
        }
        g_static_ptr[dev] = p;
    }
    *out = g_static_ptr[dev];
    return FRNN_OK;
}

}  // namespace

extern "C" {

int frnn_version(void) { return 500; }   // 0.5.0: frnn_build_static, frnn_static_scratch_bytes, frnn_get_grid_opt; counters block at the workspace head

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

const char* frnn_last_error_string(void) { return t_error; }

void frnn_options_init(frnn_options* opt) {
    if (!opt) return;
    memset(opt, 0, sizeof(*opt));
    opt->struct_bytes = static_cast<uint32_t>(sizeof(frnn_options));
}

size_t frnn_workspace_bytes(int64_t n_total, int n_events, int dim, int k_max) {
    return workspace_bytes_for(default_opts(), n_total, n_events, dim, k_max);
}

size_t frnn_workspace_bytes_opt(const frnn_options* opt, int64_t n_total, int n_events, int dim, int k_max) {
    Opts o;
    if (opts_from(opt, &o) != FRNN_OK) return 0;
    return workspace_bytes_for(o, n_total, n_events, dim, k_max);
}

int frnn_set_grid(int grid_dims, int grid_bits) {
    if (grid_dims < 0 || grid_dims > 6 || (grid_bits != 0 && (grid_bits < 2 || grid_bits > 8))) return FRNN_ERR_INVALID_ARG;
    std::lock_guard<std::mutex> lock(g_defaults_mutex);
    g_defaults.grid_dims = grid_dims;
    g_defaults.grid_bits = grid_bits;
    return FRNN_OK;
}

void frnn_get_grid(int64_t n_total, int n_events, int dim, int* grid_dims, int* grid_bits) {
    const GridChoice g = choose_grid(default_opts(), n_total, n_events < 1 ? 1 : n_events, (dim < 1 || dim > kDimMax) ? kDim : dim);
    if (grid_dims) *grid_dims = g.dims;
    if (grid_bits) *grid_bits = g.bits;
}

void frnn_get_grid_opt(const frnn_options* opt, int64_t n_total, int n_events, int dim, int* grid_dims, int* grid_bits) {
    Opts o;
    GridChoice g{0, 0};
    if (opts_from(opt, &o) == FRNN_OK && !o.auto_grid)
        g = choose_grid(o, n_total, n_events < 1 ? 1 : n_events, (dim < 1 || dim > kDimMax) ? kDim : dim);
    if (grid_dims) *grid_dims = g.dims;
    if (grid_bits) *grid_bits = g.bits;
}

int frnn_set_bin_order(const int* order, int count) {
    BinOrder o;
    const int rc = make_order(order, count, &o);
    if (rc != FRNN_OK) return rc;
    std::lock_guard<std::mutex> lock(g_defaults_mutex);
    g_defaults.order = o;
    return FRNN_OK;
}

int frnn_suggest_bin_order(const float* points, int64_t n, int dim, float r, int* order, float* score, void* cuda_stream) {
    if (!points || !order || n < 1 || !(r >= 0.0f) || !isfinite(r)) return FRNN_ERR_INVALID_ARG;
    if (dim < 1 || dim > kDimMax) return FRNN_ERR_UNSUPPORTED;
    SuggestOut so;
    const int rc = run_suggest(points, n, dim, r, static_cast<cudaStream_t>(cuda_stream), &so);
    if (rc != FRNN_OK) return rc;
    float h[kDimMax];
    const double tot = so.sampled ? static_cast<double>(so.sampled) : 1.0;
    for (int d = 0; d < kDimMax; ++d) h[d] = d < dim ? static_cast<float>(pair_probability(so.hist[d], 6, tot)) : 2.0f;   // absent coordinates prune nothing: last
    int idx[kDimMax];
    for (int d = 0; d < kDimMax; ++d) idx[d] = d;
    for (int a = 1; a < kDimMax; ++a)                               // stable insertion sort by score
        for (int b = a; b > 0 && h[idx[b]] < h[idx[b - 1]]; --b) { const int t = idx[b]; idx[b] = idx[b - 1]; idx[b - 1] = t; }
    for (int k = 0; k < 8; ++k) order[k] = idx[k];
    if (score) for (int d = 0; d < kDimMax; ++d) score[d] = h[d];
    return FRNN_OK;
}

int frnn_suggest_grid(const float* points, int64_t n, int n_events, int dim, float r, int measure, frnn_options* opt,
                      frnn_grid_report* report, void* cuda_stream) {
    if (!points || !opt || n < 1 || n_events < 1 || !(r >= 0.0f) || !isfinite(r)) return FRNN_ERR_INVALID_ARG;
    if (dim < 1 || dim > kDimMax) return FRNN_ERR_UNSUPPORTED;
    if (opt->struct_bytes < sizeof(frnn_options)) return FRNN_ERR_INVALID_ARG;
    if (dim == kDim && reinterpret_cast<uintptr_t>(points) % 32) return FRNN_ERR_INVALID_ARG;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    SuggestOut so;
    int rc = run_suggest(points, n, dim, r, st, &so);
    if (rc != FRNN_OK) return rc;
    const double tot = so.sampled ? static_cast<double>(so.sampled) : 1.0;
    double s[kDimMax][9];
    for (int d = 0; d < kDimMax; ++d)
        for (int b = 0; b <= 8; ++b) s[d][b] = (d < dim && b >= 2) ? pair_probability(so.hist[d], b, tot) : 1.0;
    // two candidate orders: the default one and the coordinates ranked by how much they prune (at the key's 64 cells)
    unsigned char orders[2][8] = {{0, 1, 2, 3, 4, 5, 6, 7}, {0, 1, 2, 3, 4, 5, 6, 7}};
    {
        int idx[kDimMax];
        for (int d = 0; d < kDimMax; ++d) idx[d] = d;
        for (int a = 1; a < kDimMax; ++a)
            for (int b = a; b > 0 && s[idx[b]][6] < s[idx[b - 1]][6]; --b) { const int t = idx[b]; idx[b] = idx[b - 1]; idx[b - 1] = t; }
        for (int k = 0; k < 8; ++k) orders[1][k] = static_cast<unsigned char>(idx[k]);
    }
    const int64_t n_first = n / n_events > 0 ? n / n_events : n;                  // rows of the sample event that is measured
    const double n_event = static_cast<double>(n) / n_events;
    std::vector<GridTry> all;
    const bool same_order = memcmp(orders[0], orders[1], 8) == 0;
    for (int g = 1; g <= 6 && g <= dim; ++g)
        for (int bits = 2; bits <= 8; ++bits) {
            if (!grid_within_budget(g, bits, n_event, n_events)) continue;
            GridTry t{g, bits, 0, grid_cost(s, orders[0], dim, g, bits, n_event, n_events), 0.0f};
            if (!same_order) {                     // reorder only for a clear predicted gain: the default order is the fast path
                const GridCost c1 = grid_cost(s, orders[1], dim, g, bits, n_event, n_events);
                if (c1.us < 0.9 * t.c.us) { t.order = 1; t.c = c1; }
            }
            all.push_back(t);
        }
    if (all.empty()) return FRNN_ERR_UNSUPPORTED;
    for (size_t a = 1; a < all.size(); ++a)                                        // by predicted cost
        for (size_t b = a; b > 0 && all[b].c.us < all[b - 1].c.us; --b) std::swap(all[b], all[b - 1]);
    size_t pick = 0, n_tried = 0;
    if (measure) {
        // the shortlist, run for real on the first event of the sample: capacity 0 (no output is written, everything else
        // runs), plain launches (no graph is left behind), 1 warm-up + 3 timed calls each, CUDA events on the stream
        std::vector<size_t> shortlist;
        for (size_t k = 0; k < all.size() && shortlist.size() < static_cast<size_t>(FRNN_GRID_REPORT_TRIES); ++k) {
            if (all[k].c.us > 2.5 * all[0].c.us) break;
            shortlist.push_back(k);
        }
        size_t ws_bytes = 0;
        std::vector<Opts> so_opts(shortlist.size());
        for (size_t k = 0; k < shortlist.size(); ++k) {
            Opts& o = so_opts[k];
            o.grid_dims = all[shortlist[k]].g;
            o.grid_bits = all[shortlist[k]].bits;
            int ord[8];
            for (int q = 0; q < 8; ++q) ord[q] = orders[all[shortlist[k]].order][q];
            make_order(ord, all[shortlist[k]].order ? 8 : 0, &o.order);
            o.use_graph = false;
            const size_t b = workspace_bytes_for(o, n_first, 1, dim, 1 << 20);
            if (b > ws_bytes) ws_bytes = b;
        }
        void* ws = nullptr;
        int64_t* d_misc = nullptr;
        cudaEvent_t e0 = nullptr, e1 = nullptr;
        cudaError_t ce = cudaMalloc(&ws, ws_bytes);
        if (ce == cudaSuccess) ce = cudaMalloc(reinterpret_cast<void**>(&d_misc), 64);
        if (ce == cudaSuccess) ce = cudaEventCreate(&e0);
        if (ce == cudaSuccess) ce = cudaEventCreate(&e1);
        rc = ce == cudaSuccess ? FRNN_OK : cuda_fail(ce, "frnn_suggest_grid: scratch for the measured shortlist");
        float best_us = 0.0f;
        for (size_t k = 0; rc == FRNN_OK && k < shortlist.size(); ++k) {
            for (int rep = 0; rep < 4 && rc == FRNN_OK; ++rep) {
                if (rep == 1) cudaEventRecord(e0, st);
                rc = build_single(so_opts[k], false, points, n_first, dim, r, 1 << 20, nullptr, nullptr, nullptr, 0, d_misc,
                                  reinterpret_cast<int32_t*>(d_misc + 1), nullptr, ws, ws_bytes, st);
            }
            if (rc != FRNN_OK) break;
            cudaEventRecord(e1, st);
            ce = cudaEventSynchronize(e1);
            float ms = 0.0f;
            if (ce == cudaSuccess) ce = cudaEventElapsedTime(&ms, e0, e1);
            if (ce != cudaSuccess) { rc = cuda_fail(ce, "frnn_suggest_grid: timing"); break; }
            all[shortlist[k]].measured_us = 1e3f * ms / 3.0f;
            if (k == 0 || all[shortlist[k]].measured_us < best_us) { best_us = all[shortlist[k]].measured_us; pick = shortlist[k]; }
        }
        if (e0) cudaEventDestroy(e0);
        if (e1) cudaEventDestroy(e1);
        if (d_misc) cudaFree(d_misc);
        if (ws) cudaFree(ws);
        if (rc != FRNN_OK) return rc;
        n_tried = shortlist.size();
        if (report) {
            memset(report, 0, sizeof(*report));
            for (size_t k = 0; k < shortlist.size(); ++k) {
                const GridTry& t = all[shortlist[k]];
                report->tried_dims[k] = t.g; report->tried_bits[k] = t.bits; report->tried_reordered[k] = t.order;
                report->tried_predicted_us[k] = static_cast<float>(t.c.us);
                report->tried_measured_us[k] = t.measured_us;
            }
        }
    } else if (report) {
        memset(report, 0, sizeof(*report));
    }
    const GridTry& best = all[pick];
    opt->grid_dims = best.g;
    opt->grid_bits = best.bits;
    opt->order_count = best.order ? 8 : 0;
    for (int k = 0; k < 8; ++k) opt->order[k] = best.order ? orders[1][k] : k;
    if (report) {
        report->grid_dims = best.g;
        report->grid_bits = best.bits;
        report->reordered = best.order;
        report->n_tried = static_cast<int32_t>(n_tried);
        report->sampled = static_cast<int64_t>(so.sampled);
        report->predicted_candidates = static_cast<float>(best.c.cand);
        report->predicted_survivors = static_cast<float>(best.c.surv);
        report->predicted_us = static_cast<float>(best.c.us);
        report->measured_us = best.measured_us;
        const float side = fmaxf(r * kCellSlack, 1e-30f);
        for (int d = 0; d < kDimMax; ++d) {
            report->extent_cells[d] = d < dim ? (so.hi[d] - so.lo[d]) / side : 0.0f;
            report->pair_probability[d] = d < dim ? static_cast<float>(s[d][best.bits]) : 1.0f;
            report->key_probability[d] = d < dim ? static_cast<float>(s[d][6]) : 1.0f;
        }
    }
    return FRNN_OK;
}

int frnn_set_graph_mode(int enabled) {
    std::lock_guard<std::mutex> lock(g_defaults_mutex);
    g_defaults.use_graph = enabled != 0;
    return FRNN_OK;
}

int frnn_build_ex(const float* points, int64_t n, int dim, float r, int k_max,
                  int32_t* out_src, int32_t* out_dst, float* out_d2, int64_t edge_capacity,
                  int64_t* out_count, int32_t* out_status, int64_t* out_row_ptr,
                  void* workspace, size_t workspace_bytes, void* cuda_stream) {
    return build_single(default_opts(), false, points, n, dim, r, k_max, out_src, out_dst, out_d2, edge_capacity, out_count, out_status,
                        out_row_ptr, workspace, workspace_bytes, cuda_stream);
}

int frnn_build_opt(const frnn_options* opt, const float* points, int64_t n, int dim, float r, int k_max,
                   int32_t* out_src, int32_t* out_dst, float* out_d2, int64_t edge_capacity,
                   int64_t* out_count, int32_t* out_status, int64_t* out_row_ptr,
                   void* workspace, size_t workspace_bytes, void* cuda_stream) {
    Opts o;
    const int rc = opts_from(opt, &o);
    if (rc != FRNN_OK) return rc;
    return build_single(o, false, points, n, dim, r, k_max, out_src, out_dst, out_d2, edge_capacity, out_count, out_status,
                        out_row_ptr, workspace, workspace_bytes, cuda_stream);
}

int frnn_build_dense_ex(const float* points, int64_t n, int dim, float r, int k_max,
                        int32_t* out_src, int32_t* out_dst, float* out_d2, int64_t edge_capacity,
                        int64_t* out_count, int32_t* out_status, int64_t* out_row_ptr,
                        void* workspace, size_t workspace_bytes, void* cuda_stream) {
    return build_single(default_opts(), true, points, n, dim, r, k_max, out_src, out_dst, out_d2, edge_capacity, out_count, out_status,
                        out_row_ptr, workspace, workspace_bytes, cuda_stream);
}

// The build of frnn_build_ex for callers that cannot allocate device memory (see include/frnn.h): same kernels, same
// result, but the workspace is g_static_scratch and the kernels are enqueued one by one (building a graph executable
// would allocate).  Nothing here, and nothing it calls, uses cudaMalloc, cudaFree or a library routine that allocates
// device memory.  The memset at the head of the enqueued work zeroes the part of the scratch that must start at zero
// (cell table, tile totals, counters, per-row counts), so what the previous call left behind does no harm.
size_t frnn_static_scratch_bytes(void) { return kStaticScratchBytes; }

int frnn_build_static(const float* points, int64_t n, int dim, float r, int k_max,
                      int32_t* out_src, int32_t* out_dst, float* out_d2, int64_t edge_capacity,
                      int64_t* out_count, int32_t* out_status, int64_t* out_row_ptr, void* cuda_stream) {
    if (n > FRNN_STATIC_MAX_ROWS) {
        snprintf(t_error, sizeof(t_error), "frnn_build_static: n = %lld exceeds FRNN_STATIC_MAX_ROWS = %d (use frnn_build_ex with a caller-owned workspace)",
                 static_cast<long long>(n), FRNN_STATIC_MAX_ROWS);
        return FRNN_ERR_UNSUPPORTED;
    }
    Opts o;                                    // the automatic grid and the default order whatever the process-wide setters say:
    o.use_graph = false;                       // the scratch is sized for exactly that layout; plain launches (no graph objects)
    if (n > 0 && dim >= 1 && dim <= kDimMax && k_max >= 1 &&
        workspace_bytes_for(o, n, 1, dim, k_max) > kStaticScratchBytes) {          // cannot happen within the row limit; kept as a guard
        snprintf(t_error, sizeof(t_error), "frnn_build_static: the layout of n = %lld rows needs more than the %zu scratch bytes",
                 static_cast<long long>(n), kStaticScratchBytes);
        return FRNN_ERR_UNSUPPORTED;
    }
    void* scratch = nullptr;
    const int rc = static_scratch_for_current_device(&scratch);
    if (rc != FRNN_OK) return rc;
    return build_single(o, false, points, n, dim, r, k_max, out_src, out_dst, out_d2, edge_capacity, out_count, out_status,
                        out_row_ptr, scratch, kStaticScratchBytes, cuda_stream);
}

int frnn_build_batched(const float* points, const int64_t* event_offsets, int n_events, int dim, float r, int k_max,
                       int32_t* out_src, int32_t* out_dst, float* out_d2, int64_t edge_capacity,
                       int64_t* out_edge_offsets, int32_t* out_status, int64_t* out_row_ptr,
                       void* workspace, size_t workspace_bytes, void* cuda_stream) {
    return build_batched(default_opts(), points, event_offsets, n_events, dim, r, k_max, out_src, out_dst, out_d2, edge_capacity,
                         out_edge_offsets, out_status, out_row_ptr, workspace, workspace_bytes, cuda_stream);
}

int frnn_build_batched_opt(const frnn_options* opt, const float* points, const int64_t* event_offsets, int n_events, int dim, float r,
                           int k_max, int32_t* out_src, int32_t* out_dst, float* out_d2, int64_t edge_capacity,
                           int64_t* out_edge_offsets, int32_t* out_status, int64_t* out_row_ptr,
                           void* workspace, size_t workspace_bytes, void* cuda_stream) {
    Opts o;
    const int rc = opts_from(opt, &o);
    if (rc != FRNN_OK) return rc;
    return build_batched(o, points, event_offsets, n_events, dim, r, k_max, out_src, out_dst, out_d2, edge_capacity,
                         out_edge_offsets, out_status, out_row_ptr, workspace, workspace_bytes, cuda_stream);
}

int frnn_build(const float* points, int64_t n, int dim, float r, int k_max,
               int32_t* out_src, int32_t* out_dst, float* out_d2, int64_t* out_count) {
    if (!out_count) return FRNN_ERR_INVALID_ARG;
    const int64_t cap = n > 0 ? n * static_cast<int64_t>(k_max > 0 ? k_max : 0) : 0;
    int rc = check_common(points, n, dim, r, k_max, out_src, out_dst, out_d2, cap);
    if (rc != FRNN_OK) return rc;
    const Opts o = default_opts();
    std::lock_guard<std::mutex> lock(g_cache_mutex);
    const size_t need = workspace_bytes_for(o, n, 1, dim, k_max);
    size_t misc_have = g_cache.misc ? 64 : 0;
    if ((rc = ensure(&g_cache.ws, &g_cache.ws_bytes, need)) != FRNN_OK) return rc;
    if ((rc = ensure(&g_cache.misc, &misc_have, 64)) != FRNN_OK) return rc;
    int64_t* d_count = static_cast<int64_t*>(g_cache.misc);
    int32_t* d_status = reinterpret_cast<int32_t*>(static_cast<char*>(g_cache.misc) + 8);
    rc = build_single(o, false, points, n, dim, r, k_max, out_src, out_dst, out_d2, cap, d_count, d_status, nullptr, g_cache.ws,
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
    int rc = check_common(points, n, dim, r, k_max, out_src, out_dst, out_d2, edge_capacity, true);
    if (rc != FRNN_OK) return rc;
    const Opts o = default_opts();
    std::lock_guard<std::mutex> lock(g_cache_mutex);
    const size_t need = workspace_bytes_for(o, n, 1, dim, k_max);
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
    rc = build_single(o, false, static_cast<const float*>(g_cache.pts), n, dim, r, k_max, d_src, d_dst, d_d2, edge_capacity, d_count, d_status,
                      nullptr, g_cache.ws, g_cache.ws_bytes, st);
    if (rc != FRNN_OK) return rc;
    CK(cudaMemcpyAsync(out_count, d_count, 8, cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    if (*out_count > edge_capacity) return FRNN_ERR_CAPACITY;
    const size_t e = static_cast<size_t>(*out_count);
    if (e) {
        static const void* refused = nullptr;                     // (under g_cache_mutex)
        if ((rc = copy_edges_to_host(out_src, out_dst, out_d2, d_src, g_cache.edge_cap, e, st, &refused)) != FRNN_OK) return rc;
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
        const void* refused_2d = nullptr;                         // see copy_edges_to_host
        State state = FREE;
    };
    std::vector<Slot> slots;
    int64_t n_max = 0, cap = 0;
    int k_max = 0, next = 0;
    size_t ws_bytes = 0;
    Opts opts;                                                    // fixed at creation: the workspaces are sized for it
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
    const int crc = copy_edges_to_host(s.h_src, s.h_dst, s.h_d2, s.src, static_cast<size_t>(p->cap), e, s.stream, &s.refused_2d);
    if (crc != FRNN_OK) return crc;
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

int frnn_host_pipeline_create_opt(const frnn_options* opt, int64_t n_max, int dim, int k_max, int64_t edge_capacity, int depth,
                                  frnn_host_pipeline** out) {
    if (!out || n_max < 1 || k_max < 1 || edge_capacity < 1 || depth < 1 || depth > 16) return FRNN_ERR_INVALID_ARG;
    if (dim != kDim) return FRNN_ERR_UNSUPPORTED;
    Opts o;
    const int orc = opts_from(opt, &o);
    if (orc != FRNN_OK) return orc;
    frnn_host_pipeline* p = new (std::nothrow) frnn_host_pipeline;
    if (!p) return FRNN_ERR_CUDA;
    p->n_max = n_max; p->k_max = k_max;
    p->cap = edge_capacity;
    p->opts = o;
    // events of any size up to n_max: the largest workspace over the grid classes an event of at most n_max rows can fall in
    p->ws_bytes = 0;
    for (int64_t n : {n_max, static_cast<int64_t>(399999), static_cast<int64_t>(16383)}) {
        if (n > n_max) continue;
        const size_t b = workspace_bytes_for(o, n, 1, dim, k_max);
        if (b > p->ws_bytes) p->ws_bytes = b;
    }
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
        if (!ok) { const int rc = cuda_fail(cudaGetLastError(), "frnn_host_pipeline_create"); pipeline_free(p); return rc; }
        s.dst = s.src + p->cap;
        s.d2 = reinterpret_cast<float*>(s.dst + p->cap);
    }
    *out = p;
    return FRNN_OK;
}

int frnn_host_pipeline_create(int64_t n_max, int dim, int k_max, int64_t edge_capacity, int depth, frnn_host_pipeline** out) {
    return frnn_host_pipeline_create_opt(nullptr, n_max, dim, k_max, edge_capacity, depth, out);
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
    rc = build_single(p->opts, false, s.pts, n, kDim, r, p->k_max, s.src, s.dst, s.d2, p->cap, s.count, d_status, nullptr, s.ws, p->ws_bytes, s.stream);
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

long long frnn_graph_builds(void) { return g_graph_builds.load(std::memory_order_relaxed); }

int frnn_set_profiling(int enabled) {
    {
        std::lock_guard<std::mutex> lock(g_defaults_mutex);
        g_defaults.timeline = enabled == 2;
    }
    if (enabled == 2) enabled = 0;
    if (enabled && !g_ev_valid) {
        for (int i = 0; i <= kPhases; ++i) CK(cudaEventCreate(&g_ev[i]));
        g_ev_valid = true;
    }
    g_profiling = enabled != 0;
    return FRNN_OK;
}

int frnn_get_profile(float* phase_ms, int max_phases) {
    if (!g_ev_valid || !phase_ms) return FRNN_ERR_INVALID_ARG;
    CK(cudaEventSynchronize(g_ev[kPhases]));
    const int n = max_phases < kPhases ? max_phases : kPhases;
    for (int i = 0; i < n; ++i) CK(cudaEventElapsedTime(&phase_ms[i], g_ev[i], g_ev[i + 1]));
    return n;
}

int frnn_get_timeline(const void* workspace, int64_t n_total, int n_events, int dim, double* begin_us, double* end_us, int max_phases) {
    if (!workspace || !begin_us || !end_us || n_total <= 0 || n_events < 1 || dim < 1 || dim > kDimMax) return FRNN_ERR_INVALID_ARG;
    static_assert(kStampsOffset + 2 * kTimelinePhases * 8 <= kCountersBytes, "the stamps fit the counters block");
    unsigned long long h[2 * kTimelinePhases];              // the stamps sit at a fixed offset from the workspace's base (make_layout)
    CK(cudaMemcpy(h, static_cast<const char*>(workspace) + kStampsOffset, sizeof(h), cudaMemcpyDeviceToHost));
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
        std::lock_guard<std::mutex> lock(g_exec_mutex);
        g_execs.clear();
    }
    std::lock_guard<std::mutex> lock(g_cache_mutex);
    if (g_cache.ws) cudaFree(g_cache.ws);
    if (g_cache.misc) cudaFree(g_cache.misc);
    if (g_cache.pts) cudaFree(g_cache.pts);
    if (g_cache.edges) cudaFree(g_cache.edges);
    if (g_cache.stream) cudaStreamDestroy(g_cache.stream);
    g_cache = Cache{};
}

}  // extern "C"
