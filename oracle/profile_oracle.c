/*
 * profile_oracle.c -- TEST INFRASTRUCTURE (oracle for SURVEY.md 8(f) NEXT-4): the sequence-versus-profile
 * dynamic programming of FAMSA's stage III ("specialised variants of the general DP procedure
 * ... profile alignments are made against a single sequence"; profile arrays PAPER.md:75-79; gap types
 * PAPER.md:111-116; gap scaling PAPER.md:133-137; consecutive gap columns in both inputs PAPER.md:139).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may use it; it
 * shares no code with paper_1603_06958_b200/csrc.  Plain, slow, obviously correct: three full
 * (n1+1) x (n2+1) tables, one cell at a time, in the order of the recurrence below.  The paper calls the
 * recurrence "classical" and does not print it; every choice is a reading recorded in DESIGN.md (P1-P9).
 *
 * Inputs of one alignment
 *   cost[i][c]  i < n1, c < 32: score of aligning symbol c to profile column i (the paper's second profile
 *               array, "costs of alignment of consecutive columns to each possible alphabet symbol")
 *   y[j]        j < n2: the sequence, codes < 32
 *   g[4]        gap_terminal_open T_o, gap_terminal_extension T_e, gap_open G_o, gap_extension G_e, already
 *               multiplied by g_scale; a run of L gaps costs open + (L-1) * extension
 *   nseq        sequences in the profile: a gap COLUMN inserted into the profile puts one gap into each of them
 * States at cell (i, j) = prefixes of i profile columns and j residues:
 *   M  column i aligned to residue j
 *   X  column i aligned to a gap in the sequence   (cost per gap: 1 x)
 *   Y  residue j aligned to a gap column inserted into the profile   (cost per gap: nseq x)
 * A gap in the sequence is TERMINAL when it lies before the first or after the last residue (j = 0 or
 * j = n2); a gap column in the profile is terminal when i = 0 or i = n1.  Score = max over the three states
 * at (n1, n2).  Ties: M before X before Y (first maximum).
 *
 * REAL selects the arithmetic: double (the oracle proper) or float (the kernel's precision, used only where a
 * floating-point comparison decides the traceback: both sides then decide in the same precision).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>

#define SYMS 32

#define DEFINE_ALIGN(NAME, REAL, NEG)                                                                          \
    /* returns the score; if path != NULL writes the optimal path's operations (0 = M, 1 = X, 2 = Y) from   */ \
    /* the first alignment column to the last and its length to *path_len (<= n1 + n2)                      */ \
    int NAME(const float *cost, int32_t n1, const uint8_t *y, int32_t n2, const float *g, int32_t nseq,        \
             double *score_out, uint8_t *path, int32_t *path_len)                                              \
    {                                                                                                          \
        const size_t W = (size_t)n2 + 1, N = ((size_t)n1 + 1) * W;                                             \
        REAL *M = (REAL *)malloc(sizeof(REAL) * N), *X = (REAL *)malloc(sizeof(REAL) * N);                     \
        REAL *Y = (REAL *)malloc(sizeof(REAL) * N);                                                            \
        uint8_t *D = (uint8_t *)malloc(N);   /* bits 0-1 / 2-3 / 4-5: where M / X / Y came from */             \
        const REAL To = (REAL)g[0], Te = (REAL)g[1], Go = (REAL)g[2], Ge = (REAL)g[3], ns = (REAL)nseq;        \
        int32_t i, j;                                                                                          \
        if (!M || !X || !Y || !D) { free(M); free(X); free(Y); free(D); return -1; }                           \
        M[0] = 0; X[0] = NEG; Y[0] = NEG; D[0] = 0;                                                            \
        for (j = 1; j <= n2; ++j) {          /* row 0: residues before the first column: terminal gap columns */ \
            M[j] = NEG; X[j] = NEG;                                                                            \
            Y[j] = j == 1 ? M[0] - ns * To : Y[j - 1] - ns * Te;                                               \
            D[j] = (uint8_t)((j == 1 ? 0 : 2) << 4);                                                           \
        }                                                                                                      \
        for (i = 1; i <= n1; ++i) {                                                                            \
            const float *ci = cost + (size_t)(i - 1) * SYMS;                                                   \
            const size_t r = (size_t)i * W, u = r - W;                                                         \
            M[r] = NEG; Y[r] = NEG;          /* column 0: columns before the first residue: terminal gaps */   \
            X[r] = i == 1 ? M[0] - To : X[u] - Te;                                                             \
            D[r] = (uint8_t)((i == 1 ? 0 : 1) << 2);                                                           \
            for (j = 1; j <= n2; ++j) {                                                                        \
                const REAL gox = j == n2 ? To : Go, gex = j == n2 ? Te : Ge;      /* gaps in the sequence */   \
                const REAL goy = ns * (i == n1 ? To : Go), gey = ns * (i == n1 ? Te : Ge);                     \
                REAL b, v; uint8_t d, from;                                                                    \
                /* M: from the diagonal */                                                                     \
                b = M[u + j - 1]; from = 0;                                                                    \
                if (X[u + j - 1] > b) { b = X[u + j - 1]; from = 1; }                                          \
                if (Y[u + j - 1] > b) { b = Y[u + j - 1]; from = 2; }                                          \
                M[r + j] = b + (REAL)ci[y[j - 1]]; d = from;                                                   \
                /* X: from above */                                                                            \
                b = M[u + j] - gox; from = 0;                                                                  \
                v = X[u + j] - gex; if (v > b) { b = v; from = 1; }                                            \
                v = Y[u + j] - gox; if (v > b) { b = v; from = 2; }                                            \
                X[r + j] = b; d |= (uint8_t)(from << 2);                                                       \
                /* Y: from the left */                                                                         \
                b = M[r + j - 1] - goy; from = 0;                                                              \
                v = X[r + j - 1] - goy; if (v > b) { b = v; from = 1; }                                        \
                v = Y[r + j - 1] - gey; if (v > b) { b = v; from = 2; }                                        \
                Y[r + j] = b; d |= (uint8_t)(from << 4);                                                       \
                D[r + j] = d;                                                                                  \
            }                                                                                                  \
        }                                                                                                      \
        {                                                                                                      \
            const size_t e = (size_t)n1 * W + n2;                                                              \
            REAL b = M[e]; int st = 0;                                                                         \
            if (X[e] > b) { b = X[e]; st = 1; }                                                                \
            if (Y[e] > b) { b = Y[e]; st = 2; }                                                                \
            *score_out = (double)b;                                                                            \
            if (path) {                                                                                        \
                int32_t n = 0, a, z;                                                                           \
                i = n1; j = n2;                                                                                \
                while (i > 0 || j > 0) {                                                                       \
                    const uint8_t d = D[(size_t)i * W + j];                                                    \
                    path[n++] = (uint8_t)st;                                                                   \
                    if (st == 0) { st = d & 3; --i; --j; }                                                     \
                    else if (st == 1) { st = (d >> 2) & 3; --i; }                                              \
                    else { st = (d >> 4) & 3; --j; }                                                           \
                }                                                                                              \
                for (a = 0, z = n - 1; a < z; ++a, --z) { uint8_t t = path[a]; path[a] = path[z]; path[z] = t; } \
                *path_len = n;                                                                                 \
            }                                                                                                  \
        }                                                                                                      \
        free(M); free(X); free(Y); free(D);                                                                    \
        return 0;                                                                                              \
    }

DEFINE_ALIGN(oracle_seqprof_align_f64, double, (-1.0e300))
DEFINE_ALIGN(oracle_seqprof_align_f32, float, (-3.0e38f))

/* cost[i][c] = sum_d counts[i][d] * subst[d][c]  (the counters array and the costs array;
 * sum-of-pairs of column i against symbol c).  Double accumulation, rounded once to float. */
void oracle_profile_costs(const uint32_t *counts, const float *subst, int32_t n1, float *cost)
{
    int32_t i, c, d;
    for (i = 0; i < n1; ++i)
        for (c = 0; c < SYMS; ++c) {
            double s = 0.0;
            for (d = 0; d < SYMS; ++d) s += (double)counts[(size_t)i * SYMS + d] * (double)subst[d * SYMS + c];
            cost[(size_t)i * SYMS + c] = (float)s;
        }
}

/* g_scale = 1 + log(k / g_l) / g_d  (g_l printed "g_1"; natural logarithm: reading P3). */
double oracle_gap_scale(double k, double g_l, double g_d) { return 1.0 + log(k / g_l) / g_d; }
