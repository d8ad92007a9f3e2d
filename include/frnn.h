/*
 * frnn.h -- C ABI of the B200-native fixed-radius nearest-neighbour (FRNN) graph builder.
 *
 * Operation (what every entry point computes):
 *   PAPER.md:31 (section 2): "it is necessary to construct a fixed-radius nearest neighbor (FRNN)
 *     graph in this embedded space. The FRNN graph has only edges connecting neighboring
 *     spacepoints residing within a constant radius".
 *   PAPER.md:69 (section 3.4): "all the neighboring points residing within a certain distance from
 *     each query spacepoint"; solved by a grid ("cell technique") over a low-dimensional projection
 *     of the embedding, worst case O(n).
 *   BASELINE.json north_star: directed edge list, at most k_max nearest per query, (src,dst) sorted.
 *
 * Result, for each query row i of an event (readings R1..R10 in DESIGN.md section 2):
 *   S_i = { j != i : d2(i,j) <= r2 },  r2 = fl32(r*r);
 *   d2(i,j) = fp32 chain  acc = 0; for d = 0..dim-1: t = fl32(x[i][d]-x[j][d]); acc = fma(t,t,acc);
 *   if |S_i| > k_max keep the k_max smallest under (d2 ascending, then j ascending);
 *   emit (src=i, dst=j, d2) for the kept j in ascending j; rows i in ascending order.
 * The result is exact (not approximate): the grid only prunes candidates.
 *
 * Conventions
 *   - Every pointer is a DEVICE pointer owned by the caller unless marked HOST.  The library never
 *     allocates or frees caller-visible memory.  frnn_build_ex / frnn_build_batched only enqueue
 *     work on `cuda_stream` (a cudaStream_t; NULL = legacy default stream) and never synchronise.
 *   - points: row-major n x dim fp32, 1 <= dim <= 16 (FRNN_ERR_UNSUPPORTED otherwise).  dim == 8 is the fast path:
 *     base 32-byte aligned (a row moves as one 256-bit transaction; FRNN_ERR_INVALID_ARG otherwise).  Other dims
 *     (SURVEY.md 8(f) f3): rows are read float by float and padded with zeros internally -- to 8 floats, or to 16 in
 *     two internal rows when dim > 8 -- which leaves every d2 bit-identical to the dim-term chain; the grid bins at
 *     most dim coordinates and never a coordinate beyond the 8th.  Finite values (non-finite coordinates
 *     are a precondition violation; they can never cause an out-of-bounds access).
 *   - src/dst are int32 row indices (local to the event in the batched call); counts and offsets
 *     are int64.  Edges of one call are sorted by (src, dst) ascending and free of duplicates.
 *   - Return value: FRNN_OK or a negative frnn_status for faults the host can detect; in that case
 *     no output is touched and nothing is enqueued.  Faults only the device can detect are
 *     reported in *out_status (device int32): FRNN_OK, or FRNN_ERR_CAPACITY when the edge count
 *     exceeds edge_capacity; then *out_count holds the needed size and only edges at positions
 *     < edge_capacity are written.
 *   - Thread safety: frnn_build_ex/_opt/_dense_ex/_batched(_opt) calls that use DISTINCT workspaces may run
 *     concurrently from different host threads on different streams (tests/test_parity_gpu.py runs two threads
 *     against the oracle).  Per-call choices travel in a frnn_options argument; the process-wide setters below
 *     (frnn_set_grid, frnn_set_bin_order, frnn_set_graph_mode) only change the DEFAULTS used by calls without
 *     options: every call snapshots them once under a lock, and a workspace must be sized
 *     (frnn_workspace_bytes[_opt]) with the same defaults / options as the call that uses it.
 *     frnn_set_profiling(1) / frnn_get_profile are bench instrumentation and not thread safe.
 *     No C++ exception crosses this boundary.
 *   - There is no CPU fallback: without a CUDA device every compute entry point fails with
 *     FRNN_ERR_CUDA.
 */
#ifndef FRNN_B200_H
#define FRNN_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    FRNN_OK = 0,
    FRNN_ERR_INVALID_ARG = -1,  /* null or misaligned pointer, n < 0, r < 0 or not finite, k_max < 1, bad offsets */
    FRNN_ERR_UNSUPPORTED = -2,  /* dim outside 1..16 (host pipeline and edge-row calls: dim != 8), more than 2^31-1 rows */
    FRNN_ERR_CAPACITY = -3,     /* device-detected: more edges than edge_capacity */
    FRNN_ERR_WORKSPACE = -4,    /* workspace_bytes < frnn_workspace_bytes(...) */
    FRNN_ERR_CUDA = -5          /* a CUDA runtime call failed (or no device) */
} frnn_status;

/* Library/ABI version: major*10000 + minor*100 + patch. */
int frnn_version(void);

/* Static string for a frnn_status value (never NULL). */
const char* frnn_status_string(int status);

/* Text of the last CUDA failure behind a FRNN_ERR_CUDA returned on THIS host thread ("call: message (name)"; "" if
 * none yet).  The library clears the runtime's non-sticky error state before returning FRNN_ERR_CUDA.  frnn_build_static
 * leaves its own sentence here when it refuses an event beyond its size limit (FRNN_ERR_UNSUPPORTED). */
const char* frnn_last_error_string(void);

/*
 * Per-call options.  Fill with frnn_options_init, change what is needed, pass to the *_opt entry
 * points; NULL there means "the process defaults".  PAPER.md:69 (section 3.4): the paper's grid bins "three
 * dimensions" of the embedding and notes that the cost of the cells grows as O(3^k k n) with the number k of binned
 * coordinates; which and how many coordinates are binned, and how many cells the toroidal grid has per coordinate,
 * never change the RESULT (R8/R9), only the amount of pruning and the size of the cell table.
 *   grid_dims   number of binned coordinates, 1..6; 0 = from the event size alone (no look at the data, no synchronisation);
 *               FRNN_GRID_AUTO (-1) = chosen PER CALL from the call's own rows: the call first runs the estimate of
 *               frnn_suggest_grid (measure = 0: cell histograms of a sample, cost model, default coordinate order) on
 *               cuda_stream and SYNCHRONISES that stream once (about 60 us), then enqueues the build on the grid it picked;
 *               grid_bits is ignored; the workspace must hold frnn_workspace_bytes_opt() with the same options (room for any
 *               grid the call may pick).  For streams whose statistics really change from event to event; otherwise choose
 *               once with frnn_suggest_grid and reuse the options.  A stream that is being captured cannot be
 *               synchronised: the call then returns FRNN_ERR_UNSUPPORTED (so do frnn_suggest_grid / _bin_order).
 *   grid_bits   log2 of the toroidal grid extent per binned coordinate, 2..8; 0 = automatic (5).  With fewer cells
 *               than the data's extent / r, far-apart cells alias onto one table entry: exact, more candidates.
 *   order       order[0..order_count) = coordinates (0..15, distinct) binned first and keyed next, as in
 *               frnn_set_bin_order; order_count = 0: the first grid_dims coordinates are binned, the next four keyed
 *   launch_mode FRNN_LAUNCH_DEFAULT (process default, see frnn_set_graph_mode), FRNN_LAUNCH_GRAPH, FRNN_LAUNCH_PLAIN
 *   timeline    != 0: the kernels leave %globaltimer stamps in the workspace (frnn_get_timeline); 0 leaves the
 *               process-wide setting (frnn_set_profiling(2)) as it is
 * What a non-NULL options argument inherits from the process-wide setters: launch_mode 0 takes frnn_set_graph_mode's
 * default and timeline 0 takes frnn_set_profiling(2)'s; the GRID and the coordinate ORDER are never inherited -- grid_dims
 * 0 / grid_bits 0 / order_count 0 mean "from the event size" / 5 / "the default order" even after frnn_set_grid or
 * frnn_set_bin_order (those two only serve calls made without options).  frnn_get_grid_opt reports the grid a call
 * with given options runs on.
 * struct_bytes must be sizeof(frnn_options) of the caller's header (frnn_options_init sets it).
 */
enum { FRNN_LAUNCH_DEFAULT = 0, FRNN_LAUNCH_GRAPH = 1, FRNN_LAUNCH_PLAIN = 2 };
enum { FRNN_GRID_AUTO = -1 };
typedef struct frnn_options {
    uint32_t struct_bytes;
    int32_t grid_dims;
    int32_t grid_bits;
    int32_t order_count;
    int32_t order[8];
    int32_t launch_mode;
    int32_t timeline;
    int32_t reserved[4];
} frnn_options;
void frnn_options_init(frnn_options* opt);

/*
 * Bytes of scratch needed for a call over n_total rows in n_events events (n_events = 1 for
 * frnn_build_ex).  Depends on the grid chosen from (n_total / n_events); 0 on invalid arguments.
 * The workspace holds S2..S9 of SURVEY.md section 8(a): cell table, cell-ordered point copy,
 * permutation, per-row counts and the CSR row pointer.  256-byte aligned base required.
 */
size_t frnn_workspace_bytes(int64_t n_total, int n_events, int dim, int k_max);
/* The same for calls made with `opt` (NULL: the process defaults, i.e. frnn_workspace_bytes). */
size_t frnn_workspace_bytes_opt(const frnn_options* opt, int64_t n_total, int n_events, int dim, int k_max);

/*
 * Default grid (process-wide DEFAULT for calls without options; affects frnn_workspace_bytes as well, so set it
 * before sizing workspaces): grid_dims = number of leading coordinates that are binned (1..6), grid_bits = log2 of
 * the toroidal grid extent per binned coordinate (2..8).  0 restores the automatic choice.  The result never
 * depends on the grid (R8/R9).  Returns FRNN_OK or FRNN_ERR_INVALID_ARG.
 */
int frnn_set_grid(int grid_dims, int grid_bits);
/* The grid a call without options over (n_total, n_events, dim) would use. */
void frnn_get_grid(int64_t n_total, int n_events, int dim, int* grid_dims, int* grid_bits);
/* The same for a call made with `opt` (NULL: frnn_get_grid).  FRNN_GRID_AUTO or invalid options: both outputs are set to 0
 * (the grid is then only known per call). */
void frnn_get_grid_opt(const frnn_options* opt, int64_t n_total, int n_events, int dim, int* grid_dims, int* grid_bits);

/*
 * S1 from the data (section 3.4: the O(3^k k n) trade-off behind the paper's
 * "three dimensions").  Looks at a sample (<= 65,536 rows, evenly strided) of `points` (DEVICE, n x dim; the rows
 * of n_events events of about n / n_events rows each): per coordinate the histogram of the cell coordinate (cells of
 * side r (1 + 2^-7), modulo 256), its minimum and maximum.  From the histograms folded to 2^bits cells it gets, per
 * coordinate and per bits, the probability s that two random points fall within one cell of each other on that
 * torus; the expected candidates per query of a grid are n * product of s over its binned coordinates, the survivors
 * of the key filter that times the product of s(64 cells) over the keyed ones.  It then picks the (grid_dims,
 * grid_bits) -- and, only when that is predicted to gain more than 10 %, an order of the coordinates -- that minimise
 * a cost model of the path (fixed latency; table entries to zero and scan; per query: neighbour rows, keys, survivors;
 * constants in DESIGN.md section 7), over grids whose table stays within 64 cells per point of an event.
 *   measure == 0: the model's best is taken as it is (one small kernel, a stream synchronise).
 *   measure != 0: the model only makes a SHORTLIST (at most FRNN_GRID_REPORT_TRIES grids within 2.5x of its best); each
 *                 is then run for real on the first event of `points` (edge capacity 0: everything but the output
 *                 stores; plain launches; 1 warm-up + 3 timed calls, CUDA events on cuda_stream) and the fastest wins.
 *                 Allocates and frees its own scratch (cudaMalloc); a few milliseconds: a set-up call.
 * The choice is written into *opt (which must have been initialised; launch_mode and timeline are left alone); an
 * order of the coordinates other than the default is chosen only for a predicted gain of more than 10 %.  *report
 * (optional) receives what was seen, predicted and measured.  The statistics of an embedding belong to the trained
 * model more than to the event: choose once per model and radius, reuse the options -- the per-event path stays
 * reduction-free.  SYNCHRONOUS.  Never changes any result.
 */
#define FRNN_GRID_REPORT_TRIES 12
typedef struct frnn_grid_report {
    int32_t grid_dims, grid_bits, reordered, n_tried;
    int64_t sampled;                 /* rows looked at */
    float predicted_candidates;      /* per query, both directions */
    float predicted_survivors;       /* candidates that pass the key filter, per query */
    float predicted_us;              /* the cost model's figure for one call */
    float measured_us;               /* measure != 0: device time of one call on the chosen grid (capacity 0) */
    float extent_cells[16];          /* (max - min) / cell side per coordinate */
    float pair_probability[16];      /* s at the chosen grid_bits per coordinate */
    float key_probability[16];       /* s at the key filter's 64 cells per coordinate */
    int32_t tried_dims[FRNN_GRID_REPORT_TRIES], tried_bits[FRNN_GRID_REPORT_TRIES], tried_reordered[FRNN_GRID_REPORT_TRIES];
    float tried_predicted_us[FRNN_GRID_REPORT_TRIES], tried_measured_us[FRNN_GRID_REPORT_TRIES];   /* the shortlist */
} frnn_grid_report;
int frnn_suggest_grid(const float* points, int64_t n, int n_events, int dim, float r, int measure,
                      frnn_options* opt /* HOST, in/out */, frnn_grid_report* report /* HOST, optional */, void* cuda_stream);

/*
 * Which coordinates the grid bins and which the key filter tests (PAPER.md:69 says only that the
 * paper's grid uses "three dimensions" of the embedding, not which).  order[0..count) lists coordinate indices in
 * [0, 16), distinct; a call whose grid bins g coordinates bins order[0..g) and keys the next four; entries not given
 * are filled with the unused coordinates in ascending order.  count == 0 (or order == NULL) restores the default (the
 * first g coordinates binned, the next four keyed -- the fast path).  Process-wide DEFAULT for calls without options.  The RESULT never depends on the
 * order: every binned or keyed coordinate is a necessary condition by itself (R8); only the amount of pruning
 * does.  The statistics of an embedding belong to the trained model, not to the event: choose once, reuse.
 * frnn_suggest_bin_order ranks the coordinates of a sample of `points` (DEVICE, n x dim) by the probability that two
 * random points fall within one cell (side r) of each other along that coordinate -- the smaller, the more it prunes --
 * writes the best eight to order[0..8) (HOST) and, if score != NULL, the 16 probabilities to score (HOST; absent
 * coordinates: 2.0).  Synchronous (one small kernel, a stream synchronise).
 */
int frnn_set_bin_order(const int* order /* HOST */, int count);
int frnn_suggest_bin_order(const float* points, int64_t n, int dim, float r, int* order /* HOST, 8 */,
                           float* score /* HOST, 16, optional */, void* cuda_stream);

/*
 * Launch mode (process-wide DEFAULT for calls without options).  1 (default): a call on a non-default stream runs
 * as ONE launch of an instantiated CUDA graph that belongs to the call's workspace.  The graph depends only on the
 * SHAPE of the call (which kernels run: grid_dims, dim <= 8 or > 8, single event or batch, bin order on/off, brute
 * force or grid) -- never on n, the pointers, r, k_max or the capacity: those are written into the graph's nodes
 * before the launch (only the nodes whose values changed since the workspace's previous call), so events of
 * different sizes and rotating buffers replay the same graph (section 3: events differ in size).
 * First use of a (workspace, shape) pair builds the graph (about 0.1 ms, bench.py prints it); at most 64 are kept,
 * least recently used evicted; threads on distinct workspaces do not wait for each other.  About 1 us per kernel
 * boundary instead of about 3 us per stream launch.
 * 0: kernels are launched one by one.  Calls on the legacy default stream, calls made while the caller is itself
 * capturing the stream, and event-profiled calls always launch one by one.
 */
int frnn_set_graph_mode(int enabled);
/* Number of CUDA graphs this process has built and instantiated so far (monotonic).  A stream of calls of one shape on
 * one workspace must not move it after the first call, whatever n, the buffers and the parameters are. */
long long frnn_graph_builds(void);

/*
 * The north_star 9-argument form.  Current device, legacy default stream, internally cached
 * workspace, output capacity assumed n*k_max edges (caller guarantees that much room, or at
 * least as many edges as the result has -- nothing is written beyond n*k_max).  SYNCHRONOUS:
 * returns after completion.  out_count is a HOST pointer (here and only here).
 * Calls are serialised by an internal lock (shared cached workspace).
 */
int frnn_build(const float* points, int64_t n, int dim, float r, int k_max,
               int32_t* out_src, int32_t* out_dst, float* out_d2, int64_t* out_count /* HOST */);

/*
 * Full single-event form: asynchronous on cuda_stream.
 *   out_src/out_dst/out_d2 : room for edge_capacity edges each
 *   out_count              : device int64, number of edges of the result (even on overflow)
 *   out_status             : device int32, see above
 *   out_row_ptr            : optional (may be NULL) device int64[n+1], CSR offsets by src row
 *   workspace              : device scratch of >= frnn_workspace_bytes(n, 1, dim, k_max) bytes
 * n == 0 and n == 1 are legal (count 0).  r == 0 is legal (edges between exact duplicates).
 */
int frnn_build_ex(const float* points, int64_t n, int dim, float r, int k_max,
                  int32_t* out_src, int32_t* out_dst, float* out_d2, int64_t edge_capacity,
                  int64_t* out_count, int32_t* out_status, int64_t* out_row_ptr,
                  void* workspace, size_t workspace_bytes, void* cuda_stream);
/* frnn_build_ex with per-call options (opt == NULL: the process defaults); workspace >= frnn_workspace_bytes_opt(opt, ...). */
int frnn_build_opt(const frnn_options* opt, const float* points, int64_t n, int dim, float r, int k_max,
                   int32_t* out_src, int32_t* out_dst, float* out_d2, int64_t edge_capacity,
                   int64_t* out_count, int32_t* out_status, int64_t* out_row_ptr,
                   void* workspace, size_t workspace_bytes, void* cuda_stream);

/*
 * The brute-force variant.  PAPER.md:57 (section 3.1): the graph can be built by querying every
 * point against a flat index (no grid) and cutting the neighbours at the radius; "brute force ...
 * quadratic".  Same arguments, same result (bit for bit) and same error behaviour as frnn_build_ex: the K nearest
 * within r of a flat search ARE the K-capped radius neighbourhood.  Cost O(n^2): every unordered pair is evaluated
 * once; meant as the on-GPU second opinion and as the baseline the grid is measured against.  n <= 8,388,480.
 */
int frnn_build_dense_ex(const float* points, int64_t n, int dim, float r, int k_max,
                        int32_t* out_src, int32_t* out_dst, float* out_d2, int64_t edge_capacity,
                        int64_t* out_count, int32_t* out_status, int64_t* out_row_ptr,
                        void* workspace, size_t workspace_bytes, void* cuda_stream);

/*
 * frnn_build_static -- frnn_build_ex for callers that must not (or cannot) allocate device memory.
 *
 * Who this is for.  Track finding runs inside larger programs that often forbid allocation on the path where an
 * event is processed: an online / trigger process that hands all of the GPU's memory to its framework's arena when
 * it is configured, so that a later cudaMalloc fails or breaks the memory budget; a latency-bound event loop, where
 * cudaMalloc and cudaFree are ruled out because they stall the whole device for an unpredictable time; a plug-in
 * that runs under somebody else's allocator and has no way to ask it for scratch.  Such a caller can still hand
 * over its input and output arrays, but has nowhere to take a workspace from.
 *
 * What it does.  Same operation, same arguments, same result (bit for bit) and same error behaviour as
 * frnn_build_ex (section 2, section 3.4; S1..S10 of SURVEY.md section 8(a)), minus the two
 * workspace arguments: the scratch is a fixed array of frnn_static_scratch_bytes() = 3 MiB that is part of the
 * library's device image.  Every GPU on which the library's code is loaded holds those 3 MiB until the process ends,
 * used or not -- hence the small limit:
 *     n <= FRNN_STATIC_MAX_ROWS (8192 rows), any dim 1..16.
 * A larger n returns FRNN_ERR_UNSUPPORTED, enqueues nothing, touches no output, and leaves a sentence saying so in
 * frnn_last_error_string().  The entry point calls no cudaMalloc / cudaFree and nothing that allocates device memory:
 * it uses the automatic grid and the default coordinate order (frnn_set_grid / frnn_set_bin_order do not apply, the
 * array is sized for that layout) and enqueues its memset and kernels one by one on cuda_stream (no CUDA-graph
 * executable is built; frnn_set_graph_mode does not apply).  Asynchronous like frnn_build_ex.
 *
 * Rules that come with a shared array:
 *   - First call on a device: it looks up the array's device address (once per device, for the device that is
 *     current at the call) before enqueuing.  Make that first call at set-up time, outside any stream capture.
 *   - All calls on one device use the SAME array.  The call clears what it needs cleared itself, so leftovers of an
 *     earlier call are harmless; but two calls whose work overlaps on the GPU (different streams without an
 *     ordering between them, or two host threads) overwrite each other's scratch and produce garbage.  Keep the
 *     calls of a device on one stream, or order them with events.
 *   - Devices are independent: each has its own copy of the array.
 */
#define FRNN_STATIC_MAX_ROWS 8192
size_t frnn_static_scratch_bytes(void);
int frnn_build_static(const float* points, int64_t n, int dim, float r, int k_max,
                      int32_t* out_src, int32_t* out_dst, float* out_d2, int64_t edge_capacity,
                      int64_t* out_count, int32_t* out_status, int64_t* out_row_ptr, void* cuda_stream);

/*
 * Batched events (BASELINE.json config 3): n_events independent events concatenated in `points`;
 * event e owns rows [event_offsets[e], event_offsets[e+1]) (HOST int64[n_events+1], ascending,
 * event_offsets[0] == 0).  No cross-event edges.  src/dst are LOCAL to the event.  Edges of event
 * e occupy [out_edge_offsets[e], out_edge_offsets[e+1]) (device int64[n_events+1]); the total is
 * out_edge_offsets[n_events].  out_row_ptr (optional) has event_offsets[n_events]+1 entries over
 * the concatenated rows.  workspace >= frnn_workspace_bytes(total rows, n_events, dim, k_max).
 */
int frnn_build_batched(const float* points, const int64_t* event_offsets /* HOST */, int n_events,
                       int dim, float r, int k_max,
                       int32_t* out_src, int32_t* out_dst, float* out_d2, int64_t edge_capacity,
                       int64_t* out_edge_offsets, int32_t* out_status, int64_t* out_row_ptr,
                       void* workspace, size_t workspace_bytes, void* cuda_stream);
int frnn_build_batched_opt(const frnn_options* opt, const float* points, const int64_t* event_offsets /* HOST */, int n_events,
                           int dim, float r, int k_max,
                           int32_t* out_src, int32_t* out_dst, float* out_d2, int64_t edge_capacity,
                           int64_t* out_edge_offsets, int32_t* out_status, int64_t* out_row_ptr,
                           void* workspace, size_t workspace_bytes, void* cuda_stream);

/*
 * Host-buffer convenience: points and all outputs are HOST pointers (pinned memory makes the copies
 * asynchronous; `points` needs only the 4-byte alignment of a float array); device staging buffers are
 * cached inside the library.  Copies the points in, runs frnn_build_ex, copies count + edges
 * out, synchronises.  Returns FRNN_ERR_CAPACITY if the result has more than edge_capacity edges
 * (*out_count = needed size, nothing else copied).  Calls are serialised by an internal lock (one shared cache).
 */
int frnn_build_host(const float* points /* HOST */, int64_t n, int dim, float r, int k_max,
                    int32_t* out_src /* HOST */, int32_t* out_dst /* HOST */, float* out_d2 /* HOST */,
                    int64_t edge_capacity, int64_t* out_count /* HOST */);

/*
 * Host pipeline: the end-to-end path for a STREAM of events in host memory.  Each submit enqueues, on the next of
 * `depth` internal slots (one CUDA stream, one workspace, one set of device buffers each): the H2D copy of the
 * points, frnn_build_ex and the copy of the edge COUNT to the host.  As soon as the host sees (at a later submit or
 * in wait) that a build has completed, it hands the copy of exactly that many edges to the copy engine.  So the H2D
 * copy of event i+1, the build of event i and the D2H copy of event i-1 overlap; the only blocking point is the
 * retirement of the oldest event in flight.
 *   create : n_max = largest event, edge_capacity = room (in edges) of every output buffer passed later,
 *            depth = events in flight (1..16; 3 or 4 is enough).
 *   submit : points HOST n x 8 fp32; out_src/out_dst/out_d2/out_count HOST (page-locked memory makes the copies
 *            asynchronous and is what bench.py uses; pageable memory works, slower).  Returns immediately unless the
 *            slot it needs is still busy (then it retires that event first).  The outputs of an event are valid after
 *            frnn_host_pipeline_wait, or after `depth` further submits.  *out_count = number of edges, or -(needed) - 1
 *            when the result has more than edge_capacity edges (then only edge_capacity are written).
 *   wait   : blocks until every submitted event is complete (oldest first).
 * Events of any size 1..n_max may follow each other: every slot replays one graph whatever n is.
 * When out_src, out_dst and out_d2 are equally spaced in memory (one block holding src | dst | d2, each of at least `count`
 * entries) the edges of an event travel as ONE 2-D copy instead of three copies (about 15 % faster end to end on a PCIe
 * gen5 box); any other placement works the same way, with three copies.  The same holds for frnn_build_host.
 * Not thread safe per pipeline; distinct pipelines are independent.
 */
typedef struct frnn_host_pipeline frnn_host_pipeline;
int frnn_host_pipeline_create(int64_t n_max, int dim, int k_max, int64_t edge_capacity, int depth, frnn_host_pipeline** out);
/* The same with options fixed for the pipeline's lifetime (NULL: the process defaults at creation). */
int frnn_host_pipeline_create_opt(const frnn_options* opt, int64_t n_max, int dim, int k_max, int64_t edge_capacity, int depth,
                                  frnn_host_pipeline** out);
int frnn_host_pipeline_submit(frnn_host_pipeline* pipeline, const float* points /* HOST */, int64_t n, float r,
                              int32_t* out_src /* HOST */, int32_t* out_dst /* HOST */,
                              float* out_d2 /* HOST */, int64_t* out_count /* HOST */);
int frnn_host_pipeline_wait(frnn_host_pipeline* pipeline);
void frnn_host_pipeline_destroy(frnn_host_pipeline* pipeline);

/* Number of kernel launches (memset nodes included) the last frnn_build_ex/_batched call enqueued
 * on this thread; what bench.py reports as gpu_launches. */
int frnn_last_launch_count(void);

/*
 * Per-phase device timing for bench.py's roofline line.  frnn_set_profiling(1) makes every later
 * frnn_build_ex/_batched call record one CUDA event after each phase of the path (on the call's
 * stream); frnn_get_profile waits for the LAST profiled call and writes the duration in ms of
 * each phase (memset, bin, scan_cells, scatter, search, emit) into phase_ms[0..max_phases), returning the number of phases written or a negative
 * status.  Process-global, not thread safe; leave it off when timing whole calls.
 */
int frnn_set_profiling(int enabled);
int frnn_get_profile(float* phase_ms /* HOST */, int max_phases);
const char* frnn_phase_name(int phase);

/*
 * In-graph timeline.  frnn_set_profiling(2) (instead of 1) keeps the CUDA-graph replay and makes every
 * kernel of later calls leave the earliest start and the latest end of its warps (%globaltimer) in the
 * call's workspace; frnn_get_timeline synchronises nothing itself (the caller waits for the call first),
 * copies the stamps of the LAST call that used `workspace` (a device pointer: the base the call was given.  The stamps
 * sit at a fixed offset from it, so the call may have been made with any options -- per-call grid, coordinate order,
 * FRNN_GRID_AUTO; n_total / n_events / dim are only checked for plausibility) and writes, per kernel (bin, scan_cells, scatter, search, emit), begin and end in
 * microseconds relative to the start of the first kernel.  Returns the number of kernels written or a
 * negative status.  Unlike mode 1 this does not perturb the launch sequence.
 */
int frnn_get_timeline(const void* workspace, int64_t n_total, int n_events, int dim,
                      double* begin_us /* HOST */, double* end_us /* HOST */, int max_phases);
const char* frnn_timeline_name(int phase);

/*
 * ---- The two steps that consume the edge list ----
 *
 * frnn_gather_edge_rows -- input rows of the edge-filtering stage.  PAPER.md:31 (section 2): the filter is a
 * classifier on EDGES, i.e. on the features of both end points; PAPER.md:37 (section 3): it is fed "in batches of
 * 800,000 edges".  For every edge e in [e_begin, min(e_begin + e_max, *edge_count)):
 *     out[(e - e_begin) * 2*dim + 0 .. dim)      = points[(src[e] + row_base) * dim ..]
 *     out[(e - e_begin) * 2*dim + dim .. 2*dim)  = points[(dst[e] + row_base) * dim ..]
 * All pointers are DEVICE pointers.  points: n x dim fp32 (dim == 8), 32-byte aligned; out: room for e_max rows of
 * 2*dim floats, 32-byte aligned; edge_count: device int64 (the out_count of frnn_build_ex) or NULL (then exactly
 * e_max edges are gathered); row_base: added to src/dst (event_offsets[e] for the local indices of a batched
 * build, else 0).  src/dst + row_base must lie in [0, n) (precondition; indices are clamped, never read out of
 * bounds).  Asynchronous on cuda_stream.  Returns FRNN_OK or a negative status; nothing is enqueued on error.
 */
int frnn_gather_edge_rows(const float* points, int64_t n, int dim, const int32_t* src, const int32_t* dst,
                          const int64_t* edge_count, int64_t e_begin, int64_t e_max, int64_t row_base,
                          float* out, void* cuda_stream);

/*
 * frnn_label_components -- track labelling.  PAPER.md:33 (section 2): edges whose score passes a threshold are
 * kept and the connected components of what remains are the track candidates; PAPER.md:61 (section 3.2): weakly
 * connected components on the GPU.  Over the nodes 0..n-1 and the edges e < min(edge_max, *edge_count) with
 * score[e] >= threshold (score == NULL: every edge), direction ignored:
 *     labels[i] = the smallest node index in the component of node i   (canonical: one correct answer)
 *     *n_components = number of components (isolated nodes count)      (optional, may be NULL)
 * All pointers are DEVICE pointers (labels int32[n], n_components int32[1], edge_count int64[1] or NULL).
 * Edges with an end point outside [0, n) and self loops are ignored.  No workspace: labels doubles as the
 * union-find parent array.  Asynchronous on cuda_stream.  Returns FRNN_OK or a negative status.
 * On a non-default stream the three kernels replay one CUDA graph that belongs to the STREAM; labels, the edge arrays
 * and every other argument are rewritten in its nodes when they change (frnn_graph_builds does not move when a
 * consumer rotates its arrays).  Calls that share a stream must come from one host thread at a time.
 */
int frnn_label_components(int64_t n, const int32_t* src, const int32_t* dst, const float* score, float threshold,
                          const int64_t* edge_count, int64_t edge_max, int32_t* labels, int32_t* n_components,
                          void* cuda_stream);

/* Release the cached workspace / staging buffers of frnn_build and frnn_build_host. */
void frnn_release_cached(void);

#ifdef __cplusplus
}
#endif
#endif /* FRNN_B200_H */
