/*
 * lcs_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, obviously-correct CPU oracle for FAMSA stage I (arxiv 1603.06958,
 * "Pairwise similarities calculation").  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * call it.  It shares no code, header, table or constant with the CUDA path under
 * paper_1603_06958_b200/csrc/ and never uses the bit-parallel recurrence: the
 * method is exact ("the calculation can be made using the bit-parallel
 * approach"), so the oracle is the plain definition written out.
 *
 * Pins (tests/test_oracle_pins.py): brute-force subsequence enumeration, closed
 * forms, invariants, an independent insertion/deletion edit-distance DP, planted
 * structure.  Conventions the paper cannot pin ("parity unpinned", R9-R12,
 * R15): the 25-letter code table, similarity at indel = 0, the sort tie-break.
 *
 * Build: gcc -O2 -shared -fPIC -pthread (oracle/build.py).  Never tuned.
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <math.h>
#include <pthread.h>

/* ---- alphabet (reading R9/R10; PAPER.md:85 names "twenty amino acids and
 * several special symbols" but prints no table).  Codes 0..19 = ACDEFGHIKLMNPQRSTVWY,
 * 20=B 21=Z 22=X 23=U 24=O, J->X, lower case folded.  A byte < 25 is already a code. */
static int encode_byte(uint8_t c)
{
    static const char letters[] = "ACDEFGHIKLMNPQRSTVWYBZXUO";
    int i;
    if (c < 25) return (int)c;
    if (c >= 'a' && c <= 'z') c = (uint8_t)(c - 'a' + 'A');
    if (c == 'J') return 22;
    for (i = 0; i < 25; ++i)
        if ((uint8_t)letters[i] == c) return i;
    return -1;
}

/* Encode n bytes.  Returns -1 on success, else the position of the first byte that is
 * neither a code nor a letter. */
int64_t oracle_encode(const uint8_t *in, int64_t n, uint8_t *out)
{
    int64_t p;
    for (p = 0; p < n; ++p) {
        int c = encode_byte(in[p]);
        if (c < 0) return p;
        out[p] = (uint8_t)c;
    }
    return -1;
}

/* ---- LCS length: the "straightforward dynamic programming (DP) rule",
 * i.e. the textbook recurrence (the paper does not print it; R1):
 *   D[0][.] = D[.][0] = 0
 *   D[i][j] = D[i-1][j-1] + 1            if A[i] == B[j]
 *           = max(D[i-1][j], D[i][j-1])  otherwise
 * result D[|A|][|B|] = "the maximal number of perfectly matching columns".
 * Two rolling rows of int32. */
int32_t oracle_lcs_len(const uint8_t *a, int32_t la, const uint8_t *b, int32_t lb)
{
    int32_t *prev, *cur, *tmp, res;
    int32_t i, j;
    if (la <= 0 || lb <= 0) return 0;
    prev = (int32_t *)calloc((size_t)lb + 1, sizeof(int32_t));
    cur = (int32_t *)calloc((size_t)lb + 1, sizeof(int32_t));
    if (!prev || !cur) { free(prev); free(cur); return -1; }
    for (i = 1; i <= la; ++i) {
        cur[0] = 0;
        for (j = 1; j <= lb; ++j) {
            if (a[i - 1] == b[j - 1]) {
                cur[j] = prev[j - 1] + 1;
            } else {
                cur[j] = prev[j] > cur[j - 1] ? prev[j] : cur[j - 1];
            }
        }
        tmp = prev; prev = cur; cur = tmp;
    }
    res = prev[lb];
    free(prev); free(cur);
    return res;
}

/* indel(A,B) = |A| + |B| - 2 * LCS_len(A,B) */
int64_t oracle_indel(int64_t la, int64_t lb, int64_t lcs)
{
    return la + lb - 2 * lcs;
}

/* similarity(A,B) = LCS_len(A,B) / indel(A,B)^2, in double.
 * indel = 0 (identical sequences): IEEE division, LCS > 0 gives +inf (R12). */
double oracle_similarity(int64_t la, int64_t lb, int64_t lcs)
{
    double d = (double)oracle_indel(la, lb, lcs);
    return (double)lcs / (d * d);
}

/* ---- batch driver: one pair per task over pthread workers (the timed cpu_baseline).
 * codes/offsets describe n_seq encoded sequences; pair p is (pi[p], pj[p]). */
typedef struct {
    const uint8_t *codes; const int64_t *offsets;
    const int64_t *pi, *pj; int64_t n_pairs;
    int32_t *lcs_out; double *sim_out;
    int64_t *next; pthread_mutex_t *mu;
} job_t;

static void *worker(void *arg)
{
    job_t *jb = (job_t *)arg;
    for (;;) {
        int64_t p0, p1, p;
        pthread_mutex_lock(jb->mu);
        p0 = *jb->next; *jb->next = p0 + 64;
        pthread_mutex_unlock(jb->mu);
        if (p0 >= jb->n_pairs) break;
        p1 = p0 + 64 < jb->n_pairs ? p0 + 64 : jb->n_pairs;
        for (p = p0; p < p1; ++p) {
            int64_t i = jb->pi[p], j = jb->pj[p];
            int64_t la = jb->offsets[i + 1] - jb->offsets[i];
            int64_t lb = jb->offsets[j + 1] - jb->offsets[j];
            int32_t l = oracle_lcs_len(jb->codes + jb->offsets[i], (int32_t)la,
                                       jb->codes + jb->offsets[j], (int32_t)lb);
            jb->lcs_out[p] = l;
            if (jb->sim_out) jb->sim_out[p] = oracle_similarity(la, lb, l);
        }
    }
    return NULL;
}

int oracle_pairs(const uint8_t *codes, const int64_t *offsets,
                 const int64_t *pi, const int64_t *pj, int64_t n_pairs,
                 int32_t *lcs_out, double *sim_out, int32_t n_threads)
{
    pthread_t th[256];
    pthread_mutex_t mu = PTHREAD_MUTEX_INITIALIZER;
    int64_t next = 0;
    job_t jb;
    int t;
    if (n_threads < 1) n_threads = 1;
    if (n_threads > 256) n_threads = 256;
    jb.codes = codes; jb.offsets = offsets; jb.pi = pi; jb.pj = pj; jb.n_pairs = n_pairs;
    jb.lcs_out = lcs_out; jb.sim_out = sim_out; jb.next = &next; jb.mu = &mu;
    for (t = 0; t < n_threads; ++t)
        if (pthread_create(&th[t], NULL, worker, &jb) != 0) { n_threads = t; break; }
    if (n_threads == 0) worker(&jb);
    for (t = 0; t < n_threads; ++t) pthread_join(th[t], NULL);
    return 0;
}
