/* Test-side driver: runs oracle/frnn_oracle.c -- the file itself, included below -- under AddressSanitizer and
 * UndefinedBehaviorSanitizer ("ASan/UBSan on the CPU oracle").  Built and run by
 * tests/test_oracle_sanitizers.py; never part of the product, never linked into libfrnn_oracle.so.
 *
 * usage: driver <case file>
 * case file (binary, little endian): int64 n, int32 dim, int32 k_max, int32 mode, float r, int64 n_q,
 *                                    n*dim floats, n_q int64 query indices (n_q = -1: all rows, no list)
 * prints: "<count> <sum src> <sum dst> <xor of the d2 bit patterns> <sum uncapped>"
 */
#include "../oracle/frnn_oracle.c"

#include <stdio.h>

int main(int argc, char** argv) {
    if (argc != 2) return 2;
    FILE* f = fopen(argv[1], "rb");
    if (!f) return 2;
    int64_t n = 0, n_q = 0;
    int32_t dim = 0, k_max = 0, mode = 0;
    float r = 0.0f;
    if (fread(&n, 8, 1, f) != 1 || fread(&dim, 4, 1, f) != 1 || fread(&k_max, 4, 1, f) != 1 || fread(&mode, 4, 1, f) != 1 ||
        fread(&r, 4, 1, f) != 1 || fread(&n_q, 8, 1, f) != 1) return 2;
    float* x = (float*)malloc((size_t)(n * dim > 0 ? n * dim : 1) * sizeof(float));
    if (n * dim > 0 && fread(x, sizeof(float), (size_t)(n * dim), f) != (size_t)(n * dim)) return 2;
    int64_t* q = NULL;
    if (n_q >= 0) {
        q = (int64_t*)malloc((size_t)(n_q > 0 ? n_q : 1) * sizeof(int64_t));
        if (n_q > 0 && fread(q, 8, (size_t)n_q, f) != (size_t)n_q) return 2;
    }
    fclose(f);
    frnn_oracle_result* res = frnn_oracle_run(mode, x, n, dim, r, k_max, q, n_q >= 0 ? n_q : 0, 0);
    if (!res) { printf("null\n"); free(x); free(q); return 0; }
    int64_t s_src = 0, s_dst = 0, s_unc = 0;
    uint32_t x_d2 = 0;
    for (int64_t e = 0; e < res->count; ++e) {
        uint32_t bits;
        memcpy(&bits, &res->d2[e], 4);
        s_src += res->src[e];
        s_dst += res->dst[e];
        x_d2 ^= bits;
    }
    for (int64_t i = 0; i < res->n_queries; ++i) s_unc += res->uncapped[i];
    printf("%lld %lld %lld %u %lld\n", (long long)res->count, (long long)s_src, (long long)s_dst, x_d2, (long long)s_unc);
    frnn_oracle_free(res);
    free(x);
    free(q);
    return 0;
}
