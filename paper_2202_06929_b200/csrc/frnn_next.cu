// frnn_next.cu -- the two steps that consume the edge list right after graph building:
//   frnn_gather_edge_rows    [x_src || x_dst] feature rows per edge, the input of the filter stage, which the paper
//                            feeds in batches of 800,000 edges
//   frnn_label_components    weakly connected components of the thresholded edge list = track labelling
//                            (PAPER.md:33 threshold on the edge score, PAPER.md:61 weakly connected components)
// Product code: shares nothing with oracle/.  No CPU fallback.
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>

#include "../../include/frnn.h"
#include "launch_plan.h"

namespace {

constexpr int kDim = 8;

__device__ __forceinline__ void load_row_nc(const float4* p, float4& a, float4& b) {
    asm("ld.global.nc.v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
        : "=f"(a.x), "=f"(a.y), "=f"(a.z), "=f"(a.w), "=f"(b.x), "=f"(b.y), "=f"(b.z), "=f"(b.w) : "l"(p));
}
// streaming store: the gathered rows are written once and read by another stage, they should not push the
// points out of L2
__device__ __forceinline__ void store_row_cs(float4* p, const float4& a, const float4& b) {
    asm volatile("st.global.cs.v8.f32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};"
                 :: "l"(p), "f"(a.x), "f"(a.y), "f"(a.z), "f"(a.w), "f"(b.x), "f"(b.y), "f"(b.z), "f"(b.w) : "memory");
}

// ---------------------------------------------------------------------------------------------------------
// f4: one thread per edge: both indices, then both 256-bit row loads in flight (random 32-byte sectors served by L2:
// one event = 3.84 MB), then 64 contiguous bytes stored; a warp writes 2 KB contiguous (streaming stores).
// ---------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) gather_edge_rows_kernel(const float4* __restrict__ pts, int64_t n,
                                                               const int32_t* __restrict__ src, const int32_t* __restrict__ dst,
                                                               const int64_t* __restrict__ edge_count, int64_t e_begin, int64_t e_max,
                                                               int64_t row_base, float4* __restrict__ out) {
    int64_t e_end = e_begin + e_max;
    if (edge_count) { const int64_t c = *edge_count; e_end = c < e_end ? c : e_end; }
    const int64_t t = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    const int64_t e = e_begin + t;
    if (e >= e_end) return;
    int64_t ra = static_cast<int64_t>(src[e]) + row_base, rb = static_cast<int64_t>(dst[e]) + row_base;
    ra = ra < 0 ? 0 : (ra >= n ? n - 1 : ra);                     // indices are a precondition; never read out of bounds
    rb = rb < 0 ? 0 : (rb >= n ? n - 1 : rb);
    float4 a0, a1, b0, b1;
    load_row_nc(pts + 2 * ra, a0, a1);
    load_row_nc(pts + 2 * rb, b0, b1);
    store_row_cs(out + 4 * t, a0, a1);
    store_row_cs(out + 4 * t + 2, b0, b1);
}

// ---------------------------------------------------------------------------------------------------------
// f2: lock-free union-find.  parent[] lives in `labels`.  A root is only ever linked to a SMALLER index, so the
// root of a tree is the smallest index of its component and the final label is canonical.
// ---------------------------------------------------------------------------------------------------------
// (one by-value argument struct per kernel: the three launches are the nodes of a cached CUDA graph, see launch_plan.h)
struct CcArgs {
    int32_t* parent;
    int64_t n;
    const int32_t* src;
    const int32_t* dst;
    const float* score;
    float threshold;
    const int64_t* edge_count;
    int64_t edge_max;
    int32_t* n_components;
};
__global__ void __launch_bounds__(256) cc_init_kernel(CcArgs a) {
    const int64_t i = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (i < a.n) a.parent[i] = static_cast<int32_t>(i);
    if (i == 0 && a.n_components) *a.n_components = 0;
}

// find with path halving, starting from x whose parent px has already been loaded (L2-coherent loads: other blocks
// update the array concurrently); the racing writes only ever replace a pointer by one of its ancestors
__device__ __forceinline__ int32_t cc_find(int32_t* parent, int32_t x, int32_t px) {
    while (px != x) {
        const int32_t gp = __ldcg(parent + px);
        if (gp != px) __stcg(parent + x, gp);
        x = px;
        px = gp;
    }
    return x;
}

__global__ void __launch_bounds__(256) cc_hook_kernel(CcArgs a) {
    int32_t* __restrict__ parent = a.parent;
    const int64_t n = a.n;
    const int32_t* __restrict__ src = a.src;
    const int32_t* __restrict__ dst = a.dst;
    const float* __restrict__ score = a.score;
    const float threshold = a.threshold;
    const int64_t* __restrict__ edge_count = a.edge_count;
    int64_t e_end = a.edge_max;
    if (edge_count) { const int64_t c = *edge_count; e_end = c < e_end ? c : e_end; }
    for (int64_t e = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x; e < e_end;
         e += static_cast<int64_t>(gridDim.x) * blockDim.x) {
        int32_t u = src[e], v = dst[e];
        const float sc = score ? score[e] : 0.0f;                   // the three loads of the edge travel together
        if (score && !(sc >= threshold)) continue;
        if (u < 0 || v < 0 || u >= n || v >= n || u == v) continue;
        int32_t pu = __ldcg(parent + u), pv = __ldcg(parent + v);   // both parents in flight
        if (pu == pv) continue;                                     // already in one tree (the usual case once a track is linked)
        while (true) {
            u = cc_find(parent, u, pu);
            v = cc_find(parent, v, pv);
            if (u == v) break;
            if (u < v) { const int32_t t = u; u = v; v = t; }      // u is the larger root
            const int32_t old = atomicCAS(&parent[u], u, v);       // link it under the smaller one
            if (old == u) break;
            pu = old;                                              // somebody linked u first: go on from there
            pv = v;                                                // v was a root a moment ago
        }

    }
}

__global__ void __launch_bounds__(256) cc_flatten_kernel(CcArgs a) {
    int32_t* __restrict__ parent = a.parent;
    const int64_t n = a.n;
    int32_t* __restrict__ n_components = a.n_components;
    const int64_t i = static_cast<int64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
    bool root = false;
    if (i < n) {
        volatile int32_t* p = parent;
        int32_t r = static_cast<int32_t>(i);
        int32_t pr = p[r];
        while (pr != r) { r = pr; pr = p[r]; }                     // roots do not change in this kernel
        p[i] = r;
        root = r == static_cast<int32_t>(i);
    }
    if (n_components) {                                            // one atomic per block
        __shared__ int s_roots;
        if (threadIdx.x == 0) s_roots = 0;
        __syncthreads();
        const unsigned m = __ballot_sync(0xffffffffu, root);
        if ((threadIdx.x & 31) == 0 && m) atomicAdd(&s_roots, __popc(m));
        __syncthreads();
        if (threadIdx.x == 0 && s_roots) atomicAdd(n_components, s_roots);
    }
}

unsigned blocks_for(int64_t items, int threads, int64_t cap) {
    int64_t b = (items + threads - 1) / threads;
    if (b < 1) b = 1;
    if (b > cap) b = cap;
    return static_cast<unsigned>(b);
}

}  // namespace

extern "C" {

int frnn_gather_edge_rows(const float* points, int64_t n, int dim, const int32_t* src, const int32_t* dst,
                          const int64_t* edge_count, int64_t e_begin, int64_t e_max, int64_t row_base,
                          float* out, void* cuda_stream) {
    if (n < 0 || e_begin < 0 || e_max < 0) return FRNN_ERR_INVALID_ARG;
    if (dim != kDim) return FRNN_ERR_UNSUPPORTED;
    if (e_max == 0) return FRNN_OK;
    if (n == 0 || !points || !src || !dst || !out) return FRNN_ERR_INVALID_ARG;
    if (reinterpret_cast<uintptr_t>(points) % 32 || reinterpret_cast<uintptr_t>(out) % 32) return FRNN_ERR_INVALID_ARG;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    gather_edge_rows_kernel<<<blocks_for(e_max, 256, 0x7fffffff), 256, 0, st>>>(
        reinterpret_cast<const float4*>(points), n, src, dst, edge_count, e_begin, e_max, row_base, reinterpret_cast<float4*>(out));
    return cudaGetLastError() == cudaSuccess ? FRNN_OK : FRNN_ERR_CUDA;
}

int frnn_label_components(int64_t n, const int32_t* src, const int32_t* dst, const float* score, float threshold,
                          const int64_t* edge_count, int64_t edge_max, int32_t* labels, int32_t* n_components,
                          void* cuda_stream) {
    if (n < 0 || edge_max < 0 || n > 0x7fffffffll) return FRNN_ERR_INVALID_ARG;
    if (score && isnan(threshold)) return FRNN_ERR_INVALID_ARG;
    if (n > 0 && !labels) return FRNN_ERR_INVALID_ARG;
    if (edge_max > 0 && (!src || !dst)) return FRNN_ERR_INVALID_ARG;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    if (n == 0) {
        if (n_components && cudaMemsetAsync(n_components, 0, 4, st) != cudaSuccess) return FRNN_ERR_CUDA;
        return FRNN_OK;
    }
    // the three kernels as a plan: on a non-default stream they replay the graph that belongs to that STREAM (every
    // argument, the labels array included, is a node parameter rewritten when it changed: a consumer that rotates its
    // label arrays keeps one graph instead of building one per array and pushing the build graphs out of the cache),
    // else they are launched one by one
    thread_local frnn::Plan plan;
    plan.clear();
    const CcArgs a{labels, n, src, dst, score, threshold, edge_count, edge_max, n_components};
    plan.add(frnn::fptr(cc_init_kernel), blocks_for(n, 256, 0x7fffffff), 1, 256, 0, a);
    if (edge_max > 0) plan.add(frnn::fptr(cc_hook_kernel), blocks_for(edge_max, 256, 148 * 64), 1, 256, 0, a);
    plan.add(frnn::fptr(cc_flatten_kernel), blocks_for(n, 256, 0x7fffffff), 1, 256, 0, a);
    return frnn::run_plan(plan, cuda_stream, st, frnn::default_use_graph());
}

}  // extern "C"
