/*
 * famsa_profile.h -- C-ABI boundary of SURVEY.md 8(f) NEXT-4: the sequence-versus-profile dynamic programming
 * of FAMSA's stage III (arxiv 1603.06958, "Progressive construction of the alignment": "the
 * majority of profile alignments are made against a single sequence ... specialised variants of the general DP
 * procedure").  Part of libfamsa_lcs.so; error codes and famsa_last_error() as in famsa_lcs.h.
 *
 * The paper calls the recurrence "classical" and prints neither it, nor the MIQS matrix, nor the gap constants,
 * so the substitution matrix and the four gap costs are INPUTS here and every other choice is a reading
 * (P1-P9).  One alignment = a profile of n1 columns against a sequence of n2 residues:
 *   cost[i][c]   fp32, i < n1, c < 32: score of symbol c against column i -- the paper's second profile array
 *                ("costs of alignment of consecutive columns to each possible alphabet symbol", 32 words per
 *                column); famsa_profile_costs builds it from the first one (symbol counters)
 *   y[j]         residue codes < 32
 *   gaps[4]      gap_terminal_open, gap_terminal_extension, gap_open, gap_extension, already
 *                multiplied by famsa_gap_scale; a run of L gaps costs open + (L-1) * extension; terminal = before
 *                the first / after the last residue (gaps in the sequence) or column (gap columns in the profile)
 *   nseq         sequences in the profile: a gap column inserted into the profile costs nseq gaps
 * States M (column ~ residue), X (column ~ gap in the sequence), Y (residue ~ gap column in the profile), every
 * transition allowed -- including X <-> Y, "consecutive insertions of gap columns to both profiles",
 * PAPER.md:139.  score = max over the states at (n1, n2); ties M before X before Y.
 */
#ifndef FAMSA_PROFILE_H
#define FAMSA_PROFILE_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define FAMSA_SEQPROF_MAX_SEQ 1024   /* residues per sequence (the sequence side lives in registers across a warp) */

/*
 * cost[i][c] = sum_d counts[i][d] * subst[d][c] for n_cols profile columns.
 *   counts_dev  DEVICE uint32 [n_cols][32]   subst_dev  DEVICE float [32][32]   cost_dev  DEVICE float [n_cols][32]
 * Accumulated in double, rounded once.  Enqueued on cuda_stream.
 */
int famsa_profile_costs(const uint32_t* counts_dev, const float* subst_dev, int64_t n_cols, float* cost_dev,
                        void* cuda_stream);

/* g_scale = 1 + ln(k / g_l) / g_d, the factor every gap cost is multiplied by (defaults 45, 7). */
double famsa_gap_scale(double k, double g_l, double g_d);

/* Bytes of DEVICE workspace (traceback directions) that famsa_seqprof_align needs for this batch; -1 on bad input. */
int64_t famsa_seqprof_workspace(const int64_t* col_off_host, const int64_t* seq_off_host, int64_t n_align);

/*
 * famsa_seqprof_align -- a batch of n_align INDEPENDENT alignments ("profile alignments in the bottom part of the
 * guide tree are independent, they can be performed in parallel").  One warp per alignment (16 lanes per
 * alignment, two alignments per warp, when n2 <= 256): lane l
 * owns J = 4 ceil(n2/128) (4 ceil(n2/64) with 16 lanes) consecutive residues with its three previous-row values per residue in registers and
 * sweeps the profile columns in a skewed wavefront (lane l works on column t - l at step t; the boundary values
 * move right by one shuffle per step); one direction byte per cell goes to the workspace and a second kernel
 * walks it back.
 *   cost_dev      DEVICE float: the concatenated cost rows of all profiles; profile b = rows [col_off[b], col_off[b+1])
 *   col_off_host  HOST  int64 [n_align+1]
 *   seq_dev       DEVICE uint8: concatenated residue codes (< 32); sequence b = [seq_off[b], seq_off[b+1])
 *   seq_off_host  HOST  int64 [n_align+1]; every sequence has 1..FAMSA_SEQPROF_MAX_SEQ residues, every profile >= 1 column
 *   gaps_dev      DEVICE float [n_align][4]      nseq_dev  DEVICE int32 [n_align]
 *   score_dev     DEVICE float [n_align]
 *   path_dev      DEVICE uint8 or NULL: operations 0 = M, 1 = X, 2 = Y of alignment b, first alignment column
 *                 first, RIGHT-ALIGNED in the segment [col_off[b] + seq_off[b], col_off[b+1] + seq_off[b+1]) (its
 *                 capacity n1 + n2): they start at segment_end - path_len[b]
 *   path_len_dev  DEVICE int32 [n_align] (required with path_dev)
 *   workspace_dev DEVICE, famsa_seqprof_workspace bytes, 16-byte aligned (may be NULL when path_dev is NULL)
 * Enqueued on cuda_stream; the offset arrays are copied before the call returns.
 * Errors: FAMSA_EINVAL (null pointers, offsets), FAMSA_ELENGTH (an empty or too long sequence, an empty profile),
 * FAMSA_ENOMEM, FAMSA_ECUDA.
 */
int famsa_seqprof_align(const float* cost_dev, const int64_t* col_off_host, const uint8_t* seq_dev,
                        const int64_t* seq_off_host, const float* gaps_dev, const int32_t* nseq_dev, int64_t n_align,
                        float* score_dev, uint8_t* path_dev, int32_t* path_len_dev, void* workspace_dev,
                        void* cuda_stream);

#define FAMSA_SEQPROF_STATIC_MAX 16384   /* alignments per famsa_seqprof_scores_static call */

/*
 * famsa_seqprof_scores_static -- famsa_seqprof_align in score-only mode for callers that cannot allocate (code under
 * CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc): the call makes NO cudaMalloc / cudaFree /
 * cudaMallocAsync / cudaMallocHost call and no heap allocation.  Its scratch (the device copy of the alignment
 * descriptors + one final-state byte per alignment) is a file-scope `static __device__` array of
 * FAMSA_SEQPROF_STATIC_MAX x 49 bytes = 0.8 MB that every GPU which loads the library holds until the process exits.
 * Arguments as famsa_seqprof_align (scores only: no path, no workspace); the CURRENT device is used; enqueued on
 * cuda_stream.  Scores are bit-identical to famsa_seqprof_align's.
 *   - n_align > FAMSA_SEQPROF_STATIC_MAX: FAMSA_ERANGE (split the batch or use famsa_seqprof_align).
 *   - Every call on a device shares the one array, which keeps the previous call's contents; a call overwrites all it
 *     reads, so calls ORDERED on the device (same stream, or ordered by events) are independent of one another, but
 *     calls that OVERLAP on the GPU (different streams without ordering, several host threads on different streams)
 *     RACE on it and give undefined scores.
 */
int famsa_seqprof_scores_static(const float* cost_dev, const int64_t* col_off_host, const uint8_t* seq_dev,
                                const int64_t* seq_off_host, const float* gaps_dev, const int32_t* nseq_dev,
                                int64_t n_align, float* score_dev, void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* FAMSA_PROFILE_H */
