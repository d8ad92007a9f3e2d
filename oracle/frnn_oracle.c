/*
 * frnn_oracle.c -- CPU oracle for the fixed-radius nearest-neighbour (FRNN) graph.
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference leg may build, load or call this file.  It shares no code, header, table or
 * helper with the CUDA path under paper_2202_06929_b200/csrc/ and includes nothing from include/.
 *
 * What it computes (DESIGN.md section 2 lists every reading R1..R10 used below):
 *   PAPER.md:31 (section 2): "The FRNN graph has only edges connecting neighboring spacepoints
 *     residing within a constant radius" in the embedded space.
 *   PAPER.md:69 (section 3.4): "an unsorted list of all the neighboring points residing within a
 *     certain distance from each query spacepoint"; brute force is O(n^2); "cell techniques" /
 *     "grid-based techniques" are O(n); the custom library projects to three dimensions for the
 *     cell search.
 *   BASELINE.json north_star: directed edge list, capped at the K nearest per query, (src,dst)
 *     sorted, d2 in a fixed fp32 summation order, index tiebreak.
 *
 * Definition, per query i (mode A = brute force, "brute force ... quadratic"):
 *   1. S_i = { j != i : d2(i,j) <= r2 },  r2 = fl32(r*r)                          [R1, R2, R4]
 *      d2(i,j): acc = 0; for d = 0..D-1 in order: t = fl32(x[i][d]-x[j][d]);
 *               acc = fmaf(t, t, acc)   (one rounding per step)                    [R3]
 *   2. if |S_i| > K keep the K smallest under (d2 ascending, then j ascending)     [R6]
 *   3. emit (i, j, d2) for the kept j in ascending j; queries in ascending i       [R5, R7]
 *
 * Mode B (cell list, "cell techniques"): bin the first min(D,3) coordinates in
 * DOUBLE with cell side 1.001*r, sorted table of occupied cells, visit the 3^g adjacent cells,
 * then apply exactly steps 1-3.  It is exact because ||x-y|| <= r implies |x_d-y_d| <= r for
 * every d, so the two cells differ by at most 1 per binned coordinate (R8).  Mode B
 * must equal mode A bit for bit (tests/test_oracle_pins.py); mode B is the one bench.py times.
 *
 * Parity pins: tests/test_oracle_pins.py (closed-form lattice counts, hand-worked fixture under
 * tests/golden/, exact-rational d2, scipy cKDTree in float64, invariants, mode A == mode B).
 * Nothing here is "parity unpinned".
 *
 * Build: gcc -O2 -fopenmp -mfma -ffp-contract=off -fno-fast-math -shared -fPIC (oracle/build.py).
 * -ffp-contract=off: the only fused operation is the explicit fmaf().  No fast-math anywhere.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    float d2;
    int32_t j;
} hit_t;

typedef struct {
    int64_t n_queries;   /* number of query rows evaluated */
    int64_t count;       /* number of edges emitted = sum_i min(|S_i|, K) */
    int32_t* src;        /* [count] query index i (original row index) */
    int32_t* dst;        /* [count] neighbour index j */
    float* d2;           /* [count] pinned-order squared distance */
    int64_t* uncapped;   /* [n_queries] |S_i| before the K cap, in query order */
    int threads;         /* OpenMP threads actually used */
} frnn_oracle_result;

/* R3: sequential FMA chain over d = 0..D-1, one rounding per step. */
static float d2_pinned(const float* a, const float* b, int dim) {
    float acc = 0.0f;
    for (int d = 0; d < dim; ++d) {
        float t = a[d] - b[d];
        acc = fmaf(t, t, acc);
    }
    return acc;
}

static int cmp_d2_then_j(const void* pa, const void* pb) {
    const hit_t* a = (const hit_t*)pa;
    const hit_t* b = (const hit_t*)pb;
    if (a->d2 < b->d2) return -1;
    if (a->d2 > b->d2) return 1;
    return (a->j > b->j) - (a->j < b->j);
}

static int cmp_j(const void* pa, const void* pb) {
    const hit_t* a = (const hit_t*)pa;
    const hit_t* b = (const hit_t*)pb;
    return (a->j > b->j) - (a->j < b->j);
}

typedef struct {
    hit_t* v;
    int64_t len, cap;
} hitvec;

static void hv_push(hitvec* h, float d2, int32_t j) {
    if (h->len == h->cap) {
        h->cap = h->cap ? 2 * h->cap : 64;
        h->v = (hit_t*)realloc(h->v, (size_t)h->cap * sizeof(hit_t));
    }
    h->v[h->len].d2 = d2;
    h->v[h->len].j = j;
    h->len++;
}

/* Steps 2 and 3 of the definition on the collected S_i.  Returns the kept length. */
static int64_t cap_and_order(hitvec* h, int k_max) {
    if (h->len == 0) return 0;                 /* S_i empty: nothing to order (and h->v may still be NULL: not for qsort) */
    if (h->len > k_max) {
        qsort(h->v, (size_t)h->len, sizeof(hit_t), cmp_d2_then_j);
        h->len = k_max;
    }
    qsort(h->v, (size_t)h->len, sizeof(hit_t), cmp_j);
    return h->len;
}

/* ---- mode B helpers: occupied-cell table over the first g coordinates, in double ---- */
#define ORACLE_GMAX 3
typedef struct {
    int64_t c[ORACLE_GMAX];
    int32_t idx;
} cellkey;

/* unused coordinates (d >= g) are stored as 0, so comparing all three is comparing the first g */
static int cmp_cell(const void* pa, const void* pb) {
    const cellkey* a = (const cellkey*)pa;
    const cellkey* b = (const cellkey*)pb;
    for (int d = 0; d < ORACLE_GMAX; ++d) {
        if (a->c[d] < b->c[d]) return -1;
        if (a->c[d] > b->c[d]) return 1;
    }
    return 0;
}

/* first position in keys[0..n) whose cell is not less than c (binary search) */
static int64_t lower_bound_cell(const cellkey* keys, int64_t n, const cellkey* c) {
    int64_t lo = 0, hi = n;
    while (lo < hi) {
        int64_t mid = lo + (hi - lo) / 2;
        if (cmp_cell(&keys[mid], c) < 0) lo = mid + 1; else hi = mid;
    }
    return lo;
}

/*
 * mode: 0 = brute force (A), 1 = cell list (B).
 * x: n x dim fp32 row-major.  queries: optional list of n_q query row indices (NULL = all rows,
 * n_q ignored); candidates are always all n rows.  Returns NULL on bad arguments.
 */
frnn_oracle_result* frnn_oracle_run(int mode, const float* x, int64_t n, int dim, float r, int k_max,
                                    const int64_t* queries, int64_t n_q, int n_threads) {
    if (n < 0 || dim < 1 || !(r >= 0.0f) || k_max < 1 || (n > 0 && !x) || n > INT32_MAX) return NULL;
    if (!queries) n_q = n;
    const float r2 = r * r;                                   /* R2: fl32(r*r), formed once */
    frnn_oracle_result* res = (frnn_oracle_result*)calloc(1, sizeof(*res));
    hit_t** per_q = (hit_t**)calloc((size_t)(n_q > 0 ? n_q : 1), sizeof(hit_t*));
    int64_t* kept = (int64_t*)calloc((size_t)(n_q > 0 ? n_q : 1), sizeof(int64_t));
    res->uncapped = (int64_t*)calloc((size_t)(n_q > 0 ? n_q : 1), sizeof(int64_t));
    res->n_queries = n_q;

    /* mode B: cells on the first g coordinates, double arithmetic, side 1.001*r (R8, R9).
       r == 0: any positive side is valid (side >= r is all the argument needs); use 1.0. */
    const int g = dim < ORACLE_GMAX ? dim : ORACLE_GMAX;
    cellkey* keys = NULL;
    if (mode == 1 && n > 0) {
        const double side = r > 0.0f ? 1.001 * (double)r : 1.0;
        keys = (cellkey*)malloc((size_t)n * sizeof(cellkey));
        for (int64_t p = 0; p < n; ++p) {
            for (int d = 0; d < ORACLE_GMAX; ++d)
                keys[p].c[d] = d < g ? (int64_t)floor((double)x[p * dim + d] / side) : 0;
            keys[p].idx = (int32_t)p;
        }
        qsort(keys, (size_t)n, sizeof(cellkey), cmp_cell);
    }
    int threads_used = 1;
    int nt = 1;
#ifdef _OPENMP
    nt = n_threads > 0 ? n_threads : omp_get_num_procs();
#endif
#pragma omp parallel num_threads(nt)
    {
#ifdef _OPENMP
#pragma omp single
        threads_used = omp_get_num_threads();
#endif
        hitvec h = {0, 0, 0};
#pragma omp for schedule(dynamic, 64)
        for (int64_t q = 0; q < n_q; ++q) {
            const int64_t i = queries ? queries[q] : q;
            const float* xi = x + i * dim;
            h.len = 0;
            if (mode == 0) {
                for (int64_t j = 0; j < n; ++j) {
                    if (j == i) continue;                                  /* R4: by index */
                    float d2 = d2_pinned(xi, x + j * dim, dim);
                    if (d2 <= r2) hv_push(&h, d2, (int32_t)j);             /* R1: inclusive */
                }
            } else {
                const double side = r > 0.0f ? 1.001 * (double)r : 1.0;
                int64_t ci[ORACLE_GMAX] = {0, 0, 0};
                for (int d = 0; d < g; ++d) ci[d] = (int64_t)floor((double)xi[d] / side);
                int64_t off[ORACLE_GMAX];
                for (off[0] = -1; off[0] <= 1; ++off[0])
                for (off[1] = (g > 1 ? -1 : 0); off[1] <= (g > 1 ? 1 : 0); ++off[1])
                for (off[2] = (g > 2 ? -1 : 0); off[2] <= (g > 2 ? 1 : 0); ++off[2]) {
                    cellkey c;
                    for (int d = 0; d < ORACLE_GMAX; ++d) c.c[d] = d < g ? ci[d] + off[d] : 0;
                    for (int64_t p = lower_bound_cell(keys, n, &c); p < n && cmp_cell(&keys[p], &c) == 0; ++p) {
                        const int64_t j = keys[p].idx;
                        if (j == i) continue;
                        float d2 = d2_pinned(xi, x + j * dim, dim);
                        if (d2 <= r2) hv_push(&h, d2, (int32_t)j);
                    }
                }
            }
            res->uncapped[q] = h.len;
            kept[q] = cap_and_order(&h, k_max);
            if (kept[q] > 0) {
                per_q[q] = (hit_t*)malloc((size_t)kept[q] * sizeof(hit_t));
                memcpy(per_q[q], h.v, (size_t)kept[q] * sizeof(hit_t));
            }
        }
        free(h.v);
    }
    res->threads = threads_used;
    int64_t total = 0;
    for (int64_t q = 0; q < n_q; ++q) total += kept[q];
    res->count = total;
    res->src = (int32_t*)malloc((size_t)(total > 0 ? total : 1) * sizeof(int32_t));
    res->dst = (int32_t*)malloc((size_t)(total > 0 ? total : 1) * sizeof(int32_t));
    res->d2 = (float*)malloc((size_t)(total > 0 ? total : 1) * sizeof(float));
    int64_t e = 0;
    for (int64_t q = 0; q < n_q; ++q) {
        const int64_t i = queries ? queries[q] : q;
        for (int64_t t = 0; t < kept[q]; ++t, ++e) {
            res->src[e] = (int32_t)i;
            res->dst[e] = per_q[q][t].j;
            res->d2[e] = per_q[q][t].d2;
        }
        free(per_q[q]);
    }
    free(per_q);
    free(kept);
    free(keys);
    return res;
}

void frnn_oracle_free(frnn_oracle_result* res) {
    if (!res) return;
    free(res->src);
    free(res->dst);
    free(res->d2);
    free(res->uncapped);
    free(res);
}

/* The pinned d2 alone, for tests that check the summation order against exact rational arithmetic. */
float frnn_oracle_d2(const float* a, const float* b, int dim) { return d2_pinned(a, b, dim); }
