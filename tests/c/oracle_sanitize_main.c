/*
 * oracle_sanitize_main.c -- drives the C oracle (oracle/lcs_oracle.c) and the CPU context baseline
 * (oracle/bitpar_cpu.c) under AddressSanitizer + UndefinedBehaviorSanitizer (SURVEY.md section 5:
 * "ASan/UBSan on the oracle").  Built and run by tests/test_oracle_sanitizers.py:
 *   gcc -O1 -g -fsanitize=address,undefined -fno-sanitize-recover=all -pthread \
 *       tests/c/oracle_sanitize_main.c oracle/lcs_oracle.c oracle/bitpar_cpu.c -lm
 * Random ragged sets (lengths 1..700, word-boundary lengths included) go through every entry point; the
 * threaded pair driver and every lane count of the multi-pair baseline must agree with the single-pair DP.
 * Exit code 0 = no sanitizer report and no disagreement.
 */
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>

int64_t oracle_encode(const uint8_t *in, int64_t n, uint8_t *out);
int32_t oracle_lcs_len(const uint8_t *a, int32_t la, const uint8_t *b, int32_t lb);
int64_t oracle_indel(int64_t la, int64_t lb, int64_t lcs);
double oracle_similarity(int64_t la, int64_t lb, int64_t lcs);
int oracle_pairs(const uint8_t *codes, const int64_t *offsets, const int64_t *pi, const int64_t *pj, int64_t n,
                 int32_t *lcs_out, double *sim_out, int32_t n_threads);
int bitpar_rowsets(const uint8_t *codes, const int64_t *offsets, const int64_t *row_i, const int64_t *col_ptr,
                   const int64_t *col_j, int64_t n_rows, int32_t max_len, int32_t *lcs_out, int32_t n_threads, int isa);
int bitpar_best_isa(void);

static uint64_t rng_state = 0x9E3779B97F4A7C15ull;
static uint32_t rnd(void) { rng_state ^= rng_state << 13; rng_state ^= rng_state >> 7; rng_state ^= rng_state << 17; return (uint32_t)(rng_state >> 32); }

int main(void)
{
    enum { K = 48 };
    static const int fixed[] = { 1, 2, 63, 64, 65, 127, 128, 129, 255, 256, 257, 700 };
    static const char letters[] = "ACDEFGHIKLMNPQRSTVWYBZXUOJacdxyz";
    int64_t offsets[K + 1], total = 0;
    int32_t lens[K], max_len = 0;
    int s, t, isa_list[] = { 0, 2, 4, 8, -1 };
    for (s = 0; s < K; ++s) {
        lens[s] = s < (int)(sizeof fixed / sizeof fixed[0]) ? fixed[s] : 1 + (int32_t)(rnd() % 400);
        if (lens[s] > max_len) max_len = lens[s];
        offsets[s] = total; total += lens[s];
    }
    offsets[K] = total;
    uint8_t *raw = malloc((size_t)total), *codes = malloc((size_t)total);
    for (t = 0; t < total; ++t) raw[t] = (uint8_t)letters[rnd() % (sizeof letters - 1)];
    if (oracle_encode(raw, total, codes) != -1) { fprintf(stderr, "encode rejected a letter\n"); return 2; }
    raw[5] = '*';
    if (oracle_encode(raw, total, codes) != 5) { fprintf(stderr, "encode missed a bad byte\n"); return 2; }
    raw[5] = 'A';
    oracle_encode(raw, total, codes);

    const int64_t n = (int64_t)K * K;
    int64_t *pi = malloc(sizeof(int64_t) * n), *pj = malloc(sizeof(int64_t) * n), col_ptr[K + 1], row_i[K];
    int32_t *ref = malloc(sizeof(int32_t) * n), *thr = malloc(sizeof(int32_t) * n), *bp = malloc(sizeof(int32_t) * n);
    double *sim = malloc(sizeof(double) * n);
    for (s = 0; s < K; ++s) {
        row_i[s] = s; col_ptr[s] = (int64_t)s * K;
        for (t = 0; t < K; ++t) {
            pi[s * K + t] = s; pj[s * K + t] = t;
            ref[s * K + t] = oracle_lcs_len(codes + offsets[s], lens[s], codes + offsets[t], lens[t]);
        }
    }
    col_ptr[K] = n;
    oracle_pairs(codes, offsets, pi, pj, n, thr, sim, 4);
    for (t = 0; t < n; ++t) {
        int64_t la = lens[pi[t]], lb = lens[pj[t]];
        if (thr[t] != ref[t]) { fprintf(stderr, "oracle_pairs disagrees at %d\n", t); return 3; }
        if (oracle_indel(la, lb, ref[t]) != la + lb - 2 * ref[t]) { fprintf(stderr, "indel\n"); return 3; }
        if (sim[t] != oracle_similarity(la, lb, ref[t])) { fprintf(stderr, "similarity\n"); return 3; }
    }
    for (s = 0; s < (int)(sizeof isa_list / sizeof isa_list[0]); ++s) {
        if (bitpar_rowsets(codes, offsets, row_i, col_ptr, pj, K, max_len, bp, 3, isa_list[s]) != 0) { fprintf(stderr, "isa %d refused\n", isa_list[s]); return 4; }
        for (t = 0; t < n; ++t)
            if (bp[t] != ref[t]) { fprintf(stderr, "bitpar isa %d disagrees at %d: %d vs %d\n", isa_list[s], t, bp[t], ref[t]); return 4; }
    }
    free(raw); free(codes); free(pi); free(pj); free(ref); free(thr); free(bp); free(sim);
    printf("sanitized ok: %lld pairs, best isa %d\n", (long long)n, bitpar_best_isa());
    return 0;
}
