/*
 * bitpar_cpu.c -- CONTEXT BASELINE for bench.py, NOT a parity oracle and NOT product code.
 *
 * The paper's own stage-I design on a CPU: the bit-parallel LCS length with
 * w = 64-bit words, the pairs spread over threads, and "multiple pairs of sequences ... processed
 * simultaneously by the same thread" in SIMD registers -- a = 2 (128-bit), 4 (AVX2) or 8 (AVX-512)
 * 64-bit words per vector.  One task = one ROW sequence A (its match bit-vectors are built once) against
 * a list of column sequences B, `a` of them at a time: lane l of every vector belongs to pair (A, B_l);
 * the add carry between words is a per-lane mask obtained by unsigned compares.
 * It exists so that the benchmark can put "the paper's method on this box's host cores" beside the GPU
 * number, because the paper prints no stage-I throughput.  It shares the recurrence with the CUDA path,
 * so it proves nothing about parity; it is itself checked against the plain-DP oracle in
 * tests/test_oracle_pins.py (every lane count, through the generic code path where the host lacks the ISA).
 * Shares no code with paper_1603_06958_b200/csrc.  Build: gcc -O2 (oracle/build.py).
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <pthread.h>
#if defined(__x86_64__)
#include <immintrin.h>
#endif

#define SYMS 32
#define PAD_SYM 31           /* never a residue code (codes are < 25): its match words are all zero */

/* Match bit-vectors of a, layout M[word][symbol] (one row of 32 words per 64 residues). */
static void build_table(const uint8_t *a, int32_t la, int32_t W, uint64_t *M)
{
    int32_t i;
    memset(M, 0, sizeof(uint64_t) * SYMS * (size_t)W);
    for (i = 0; i < la; ++i) M[(size_t)(i >> 6) * SYMS + a[i]] |= 1ull << (i & 63);
}

/* scalar: one pair.  LCS length of the table's sequence (W words) and b. */
static int32_t lcs_scalar(const uint64_t *M, int32_t W, const uint8_t *b, int32_t lb, uint64_t *V)
{
    int32_t j, w, lcs = 0;
    for (w = 0; w < W; ++w) V[w] = ~0ull;
    for (j = 0; j < lb; ++j) {
        const uint64_t *m = M + b[j];
        unsigned long long carry = 0;
        for (w = 0; w < W; ++w) {
            uint64_t mw = m[(size_t)w * SYMS];
            uint64_t u = V[w] & mw;
            uint64_t t = V[w] + u;                      /* add with carry in and out, across words */
            uint64_t s = t + carry;
            carry = (unsigned long long)((t < u) | (s < t));
            V[w] = s | (V[w] & ~mw);
        }
    }
    for (w = 0; w < W; ++w) lcs += __builtin_popcountll(~V[w]);
    return lcs;
}

/* SIMD: N pairs (one table, N column sequences) per vector of N 64-bit lanes.  V: N*W words of scratch
 * (vector-aligned).  Columns shorter than the group's longest are padded with PAD_SYM (a no-op step).
 * The body is written once with GCC vector extensions and instantiated per lane count and target ISA. */
/* GATHER(mw, row, sym): lane l of mw = row[sym[l]] -- element-wise for the generic vectors, the hardware    */
/* gather instruction where the ISA has one.                                                               */
#define GATHER_GENERIC(N, mw, row, sym) do { int l_; for (l_ = 0; l_ < N; ++l_) (mw)[l_] = (row)[(sym)[l_]]; } while (0)
#define DEFINE_LCS_VEC(NAME, N, TARGET, GATHER)                                                           \
    typedef uint64_t NAME##_vec __attribute__((vector_size(8 * N)));                                      \
    TARGET static void NAME(const uint64_t *M, int32_t W, const uint8_t *const *b, const int32_t *lb,     \
                            int32_t n, NAME##_vec *V, int32_t *out)                                       \
    {                                                                                                     \
        int32_t j, w, l, maxlen = 0;                                                                      \
        const NAME##_vec ones = ~(NAME##_vec){0};                                                         \
        for (l = 0; l < n; ++l) if (lb[l] > maxlen) maxlen = lb[l];                                       \
        for (w = 0; w < W; ++w) V[w] = ones;                                                              \
        for (j = 0; j < maxlen; ++j) {                                                                    \
            long long sym[N] __attribute__((aligned(64)));                                                \
            NAME##_vec carry = (NAME##_vec){0};                                                           \
            for (l = 0; l < N; ++l) sym[l] = (l < n && j < lb[l]) ? b[l][j] : PAD_SYM;                    \
            for (w = 0; w < W; ++w) {                                                                     \
                const uint64_t *row = M + (size_t)w * SYMS;                                               \
                NAME##_vec mw, u, t, s;                                                                   \
                GATHER(mw, row, sym);                                   /* lane l's symbol */              \
                u = V[w] & mw;                                                                            \
                t = V[w] + u;                                                                             \
                s = t - carry;                                          /* carry is a 0 / -1 lane mask */  \
                carry = (NAME##_vec)(t < u) | (NAME##_vec)(s < t);                                        \
                V[w] = s | (V[w] & ~mw);                                                                  \
            }                                                                                             \
        }                                                                                                 \
        for (l = 0; l < n; ++l) {                                                                         \
            int32_t lcs = 0;                                                                              \
            for (w = 0; w < W; ++w) lcs += __builtin_popcountll(~V[w][l]);                                \
            out[l] = lcs;                                                                                 \
        }                                                                                                 \
    }

#define GATHER_2(mw, row, sym) GATHER_GENERIC(2, mw, row, sym)
#define GATHER_4(mw, row, sym) GATHER_GENERIC(4, mw, row, sym)
#define GATHER_8(mw, row, sym) GATHER_GENERIC(8, mw, row, sym)
DEFINE_LCS_VEC(lcs_v2, 2, , GATHER_2)
DEFINE_LCS_VEC(lcs_v4, 4, , GATHER_4)
DEFINE_LCS_VEC(lcs_v8, 8, , GATHER_8)
#if defined(__x86_64__)
#define GATHER_AVX2(mw, row, sym) \
    (mw) = (__typeof__(mw))_mm256_i64gather_epi64((const long long *)(row), _mm256_load_si256((const __m256i *)(sym)), 8)
#define GATHER_AVX512(mw, row, sym) \
    (mw) = (__typeof__(mw))_mm512_i64gather_epi64(_mm512_load_si512((const void *)(sym)), (const void *)(row), 8)
DEFINE_LCS_VEC(lcs_v4_avx2, 4, __attribute__((target("avx2"))), GATHER_AVX2)
DEFINE_LCS_VEC(lcs_v8_avx512, 8, __attribute__((target("avx512f,avx512bw,avx512dq,avx512vl"))), GATHER_AVX512)
#endif

/* ISA codes of bitpar_rowsets: 0 scalar; 2 / 4 / 8 generic vectors of that many lanes (compiled for the
 * baseline ISA: the code path of the wide variants on any host); 14 = AVX2 (a = 4); 18 = AVX-512 (a = 8);
 * -1 = the widest the host supports natively. */
int bitpar_best_isa(void)
{
#if defined(__x86_64__)
    __builtin_cpu_init();
    if (__builtin_cpu_supports("avx512f") && __builtin_cpu_supports("avx512bw") &&
        __builtin_cpu_supports("avx512dq") && __builtin_cpu_supports("avx512vl")) return 18;
    if (__builtin_cpu_supports("avx2")) return 14;
#endif
    return 2;
}

static int isa_lanes(int isa) { return isa == 0 ? 1 : (isa == 14 ? 4 : (isa == 18 ? 8 : isa)); }

typedef struct {
    const uint8_t *codes; const int64_t *offsets;
    const int64_t *row_i, *col_ptr, *col_j; int64_t n_rows;
    int32_t *out; int64_t *next; pthread_mutex_t *mu; int32_t max_len; int isa;
} bp_job;

static void *bp_worker(void *arg)
{
    bp_job *jb = (bp_job *)arg;
    const int32_t Wmax = (jb->max_len + 63) / 64;
    const int lanes = isa_lanes(jb->isa);
    uint64_t *M = NULL, *V = NULL;
    if (posix_memalign((void **)&M, 64, sizeof(uint64_t) * SYMS * (size_t)(Wmax + 1)) != 0) return NULL;
    if (posix_memalign((void **)&V, 64, sizeof(uint64_t) * 8 * (size_t)(Wmax + 1)) != 0) { free(M); return NULL; }
    for (;;) {
        int64_t r, c;
        pthread_mutex_lock(jb->mu);
        r = *jb->next; *jb->next = r + 1;
        pthread_mutex_unlock(jb->mu);
        if (r >= jb->n_rows) break;
        {
            const int64_t i = jb->row_i[r];
            const uint8_t *a = jb->codes + jb->offsets[i];
            const int32_t la = (int32_t)(jb->offsets[i + 1] - jb->offsets[i]);
            const int32_t W = (la + 63) / 64;
            build_table(a, la, W, M);                    /* once per row: shared by all its columns */
            for (c = jb->col_ptr[r]; c < jb->col_ptr[r + 1]; c += lanes) {
                const uint8_t *b[8]; int32_t lb[8]; int32_t n = 0, l;
                for (l = 0; l < lanes && c + l < jb->col_ptr[r + 1]; ++l, ++n) {
                    const int64_t j = jb->col_j[c + l];
                    b[l] = jb->codes + jb->offsets[j];
                    lb[l] = (int32_t)(jb->offsets[j + 1] - jb->offsets[j]);
                }
                switch (jb->isa) {
                case 0:  jb->out[c] = lcs_scalar(M, W, b[0], lb[0], V); break;
                case 2:  lcs_v2(M, W, b, lb, n, (lcs_v2_vec *)V, jb->out + c); break;
                case 4:  lcs_v4(M, W, b, lb, n, (lcs_v4_vec *)V, jb->out + c); break;
                case 8:  lcs_v8(M, W, b, lb, n, (lcs_v8_vec *)V, jb->out + c); break;
#if defined(__x86_64__)
                case 14: lcs_v4_avx2(M, W, b, lb, n, (lcs_v4_avx2_vec *)V, jb->out + c); break;
                case 18: lcs_v8_avx512(M, W, b, lb, n, (lcs_v8_avx512_vec *)V, jb->out + c); break;
#endif
                default: break;
                }
            }
        }
    }
    free(M); free(V);
    return NULL;
}

/*
 * LCS of row sequence row_i[r] against each of col_j[col_ptr[r] .. col_ptr[r+1]) (ORIGINAL indices, codes
 * already encoded, < 25), r = 0..n_rows-1; lcs_out is parallel to col_j.  The row carries the bit-vectors
 * whatever the lengths (LCS is symmetric).  Returns 0, or -1 for an ISA the host cannot run.
 */
int bitpar_rowsets(const uint8_t *codes, const int64_t *offsets, const int64_t *row_i, const int64_t *col_ptr,
                   const int64_t *col_j, int64_t n_rows, int32_t max_len, int32_t *lcs_out, int32_t n_threads, int isa)
{
    pthread_t th[256];
    pthread_mutex_t mu = PTHREAD_MUTEX_INITIALIZER;
    int64_t next = 0;
    bp_job jb;
    int t, best = bitpar_best_isa();
    if (isa < 0) isa = best;
    if (isa != 0 && isa != 2 && isa != 4 && isa != 8 && isa != 14 && isa != 18) return -1;
    if ((isa == 14 && best != 14 && best != 18) || (isa == 18 && best != 18)) return -1;
    if (n_threads < 1) n_threads = 1;
    if (n_threads > 256) n_threads = 256;
    jb.codes = codes; jb.offsets = offsets; jb.row_i = row_i; jb.col_ptr = col_ptr; jb.col_j = col_j;
    jb.n_rows = n_rows; jb.out = lcs_out; jb.next = &next; jb.mu = &mu; jb.max_len = max_len; jb.isa = isa;
    for (t = 0; t < n_threads; ++t)
        if (pthread_create(&th[t], NULL, bp_worker, &jb) != 0) { n_threads = t; break; }
    if (n_threads == 0) bp_worker(&jb);
    for (t = 0; t < n_threads; ++t) pthread_join(th[t], NULL);
    return 0;
}
