// launch_plan.h -- private to csrc/: a call of the library as a PLAN (one optional memset + a list of kernel launches with
// by-value argument structs) and the entry point that runs it, either node by node or through the CUDA graph that belongs to
// (key, list of kernel functions).  Defined in frnn.cu; used by frnn.cu and frnn_next.cu.  Not part of the C ABI.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string.h>

#include <vector>

namespace frnn {

struct Node {
    const void* func;
    unsigned grid_x, grid_y, block;
    int phase;                    // frnn_phase_name index (per-phase event timing of the build path)
    uint32_t arg_off, arg_bytes;  // the by-value argument struct inside Plan::args
};
struct Plan {
    void* ms_dst = nullptr;       // memset at the head of the plan (ms_bytes == 0: none)
    size_t ms_bytes = 0;
    std::vector<Node> nodes;
    std::vector<unsigned char> args;
    void clear() { ms_dst = nullptr; ms_bytes = 0; nodes.clear(); args.clear(); }
    template <class A>
    void add(const void* func, unsigned grid_x, unsigned grid_y, unsigned block, int phase, const A& a) {
        static_assert(sizeof(A) <= 4096, "kernel arguments are limited to 4 KB");
        const size_t off = (args.size() + 15) & ~static_cast<size_t>(15);
        args.resize(off + sizeof(A));
        memcpy(args.data() + off, &a, sizeof(A));
        nodes.push_back(Node{func, grid_x, grid_y, block, phase, static_cast<uint32_t>(off), static_cast<uint32_t>(sizeof(A))});
    }
};

template <class K> const void* fptr(K k) { return reinterpret_cast<const void*>(k); }

// Runs the plan on `st`.  want_graph (and a stream that allows it: not the legacy default stream, not being captured, no
// per-phase profiling) -> one launch of the graph executable that belongs to (key, the plan's kernel functions), its node
// parameters rewritten where they changed; otherwise the memset and the kernels one by one.  Returns an frnn_status.
int run_plan(const Plan& P, void* key, cudaStream_t st, bool want_graph);
bool default_use_graph();         // the process default of frnn_set_graph_mode

}  // namespace frnn
