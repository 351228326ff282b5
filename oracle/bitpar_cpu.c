/*
 * bitpar_cpu.c -- CONTEXT BASELINE for bench.py, NOT a parity oracle and NOT product code.
 *
 * The paper's own stage-I design on a CPU: the bit-parallel LCS length with
 * w = 64-bit words, one pair per task, spread over threads (the paper additionally packs several
 * pairs into AVX registers; this scalar version does not).  It exists so that the benchmark can put
 * "the paper's method on this box's host cores" beside the GPU number, because the paper prints no
 * stage-I throughput.  It shares the recurrence with the CUDA path, so it proves nothing about
 * parity; it is itself checked against the plain-DP oracle in tests/test_oracle_pins.py.
 * Shares no code with paper_1603_06958_b200/csrc.  Build: gcc -O2 (oracle/build.py).
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <pthread.h>

#define SYMS 32

/* LCS length of a (length la, the side that carries the bit-vector) and b; codes < 32. */
static int32_t bitpar_lcs(const uint8_t *a, int32_t la, const uint8_t *b, int32_t lb, uint64_t *M, uint64_t *V)
{
    int32_t W = (la + 63) / 64, i, j, w, lcs = 0;
    memset(M, 0, sizeof(uint64_t) * SYMS * (size_t)W);
    for (i = 0; i < la; ++i) M[(size_t)a[i] * W + (i >> 6)] |= 1ull << (i & 63);
    for (w = 0; w < W; ++w) V[w] = ~0ull;
    for (j = 0; j < lb; ++j) {
        const uint64_t *m = M + (size_t)b[j] * W;
        unsigned long long carry = 0;
        for (w = 0; w < W; ++w) {
            uint64_t u = V[w] & m[w];
            uint64_t t = V[w] + u;                      /* add with carry in and out, across words */
            uint64_t s = t + carry;
            carry = (unsigned long long)((t < u) | (s < t));
            V[w] = s | (V[w] & ~m[w]);
        }
    }
    for (w = 0; w < W; ++w) lcs += __builtin_popcountll(~V[w]);
    return lcs;
}

typedef struct {
    const uint8_t *codes; const int64_t *offsets; const int64_t *pi, *pj; int64_t n;
    int32_t *out; int64_t *next; pthread_mutex_t *mu; int32_t max_len;
} bp_job;

static void *bp_worker(void *arg)
{
    bp_job *jb = (bp_job *)arg;
    int32_t W = (jb->max_len + 63) / 64;
    uint64_t *M = (uint64_t *)malloc(sizeof(uint64_t) * SYMS * (size_t)(W + 1));
    uint64_t *V = (uint64_t *)malloc(sizeof(uint64_t) * (size_t)(W + 1));
    for (;;) {
        int64_t p0, p1, p;
        pthread_mutex_lock(jb->mu);
        p0 = *jb->next; *jb->next = p0 + 256;
        pthread_mutex_unlock(jb->mu);
        if (p0 >= jb->n) break;
        p1 = p0 + 256 < jb->n ? p0 + 256 : jb->n;
        for (p = p0; p < p1; ++p) {
            int64_t i = jb->pi[p], j = jb->pj[p];
            int32_t li = (int32_t)(jb->offsets[i + 1] - jb->offsets[i]);
            int32_t lj = (int32_t)(jb->offsets[j + 1] - jb->offsets[j]);
            const uint8_t *si = jb->codes + jb->offsets[i], *sj = jb->codes + jb->offsets[j];
            jb->out[p] = li <= lj ? bitpar_lcs(si, li, sj, lj, M, V) : bitpar_lcs(sj, lj, si, li, M, V);
        }
    }
    free(M); free(V);
    return NULL;
}

/* codes must already be encoded (< 32).  max_len = the longest sequence among the pairs. */
int bitpar_pairs(const uint8_t *codes, const int64_t *offsets, const int64_t *pi, const int64_t *pj,
                 int64_t n, int32_t max_len, int32_t *lcs_out, int32_t n_threads)
{
    pthread_t th[256];
    pthread_mutex_t mu = PTHREAD_MUTEX_INITIALIZER;
    int64_t next = 0;
    bp_job jb;
    int t;
    if (n_threads < 1) n_threads = 1;
    if (n_threads > 256) n_threads = 256;
    jb.codes = codes; jb.offsets = offsets; jb.pi = pi; jb.pj = pj; jb.n = n; jb.out = lcs_out;
    jb.next = &next; jb.mu = &mu; jb.max_len = max_len;
    for (t = 0; t < n_threads; ++t)
        if (pthread_create(&th[t], NULL, bp_worker, &jb) != 0) { n_threads = t; break; }
    if (n_threads == 0) bp_worker(&jb);
    for (t = 0; t < n_threads; ++t) pthread_join(th[t], NULL);
    return 0;
}
