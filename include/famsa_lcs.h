/*
 * famsa_lcs.h -- C-ABI boundary of the B200-native FAMSA stage I hot path
 * (arxiv 1603.06958, "Pairwise similarities calculation"):
 * all-pairs LCS length (bit-parallel), indel distance
 * and similarity = LCS / indel^2, streamed in row blocks so that the
 * single-linkage consumer needs O(k) memory.
 *
 * Plain pointers and sizes only; each pointer is marked HOST or DEVICE.  No exception
 * crosses the ABI.  Every int-returning call returns 0 (FAMSA_OK) or a negative
 * FAMSA_E* code; famsa_last_error() gives the text for the calling thread.
 * There is NO CPU fallback: without an sm_100 CUDA device famsa_pack fails with
 * FAMSA_ECUDA.
 *
 * Index space.  famsa_pack sorts sequences by DESCENDING length, ties by ascending
 * original index (stable).  All row/column indices below are SORTED indices;
 * famsa_perm maps sorted -> original.  Row i holds pairs (i, j) for 0 <= j < i; in each
 * such pair sequence i is the shorter one and carries the bit-vectors (LCS is symmetric).
 *
 * Output layout.  For a call over rows [i0, i1): entry (i, j) is at
 *     i*(i-1)/2 - i0*(i0-1)/2 + j
 * in both lcs_out and sim_out (two arrays, packed triangular by rows; row i contiguous).
 */
#ifndef FAMSA_LCS_H
#define FAMSA_LCS_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct famsa_ctx famsa_ctx;   /* opaque; owns every device allocation it makes */

enum {
    FAMSA_OK      = 0,
    FAMSA_EINVAL  = -1,  /* null pointer, k < 0, offsets[0] != 0 or offsets decreasing     */
    FAMSA_ESYMBOL = -2,  /* a byte that is neither a code (< 25) nor an amino-acid letter  */
    FAMSA_ELENGTH = -3,  /* an empty sequence, or one longer than FAMSA_MAX_LEN            */
    FAMSA_ERANGE  = -4,  /* i0 > i1, i0 < 0 or i1 > k                                      */
    FAMSA_ENOMEM  = -5,  /* host or device allocation failed                               */
    FAMSA_ECUDA   = -6   /* any CUDA runtime error, or no sm_100 device                    */
};

#define FAMSA_MAX_LEN 65535   /* so that every LCS length fits uint16 */

/*
 * famsa_pack -- steps a1-a3 of the path (encode, length sort, match-table build); one-off,
 * O(sum |S|), runs on the device.
 *   seqs     HOST  concatenated residues, no terminators.  A byte < 25 is already a code;
 *                  ASCII letters (either case) map to the 25-letter code
 *                  ACDEFGHIKLMNPQRSTVWY + B Z X U O (J -> X).  Anything else: FAMSA_ESYMBOL.
 *   offsets  HOST  k+1 entries, offsets[0] = 0, sequence s = seqs[offsets[s], offsets[s+1]).
 *   k        number of sequences (0 and 1 are legal: zero pairs).
 *   device   CUDA device ordinal to pack onto (the ctx stays bound to it).
 *   out      receives the handle.  Inputs are copied; the caller may free them on return.
 * Builds, per sequence S and symbol c, the match bit-vectors M_S[c] (bit i set iff
 * S[i] == c; "bit-parallel approach") and the pre-scaled, lane-interleaved
 * residue streams the sweep reads.  Synchronises the device before returning.
 */
int famsa_pack(const uint8_t* seqs, const int64_t* offsets, int64_t k, int device,
               famsa_ctx** out);

/*
 * famsa_lcs_rows -- steps a4-a7: the pair sweep for rows [i0, i1), all columns j < i.
 * For each pair, with A = sequence i (shorter) and B = sequence j: V <- all ones; for each
 * residue b of B: U = V & M_A[b]; V = (V + U) | (V - U) with the add carry propagated across
 * words; LCS = number of zero bits of V (recurrence as stated in BASELINE.json
 * north_star).  Then indel = |A| + |B| - 2 LCS and
 * similarity = LCS / indel^2 in fp32 (+inf when indel = 0).
 *   lcs_out  DEVICE  famsa_rows_pairs(i0, i1) uint16 entries, layout above.  May be NULL
 *                    only if sim_out is not.
 *   sim_out  DEVICE  same count of float entries, or NULL (LCS only).
 *   cuda_stream      a cudaStream_t (NULL = default stream).  Work is ENQUEUED, not
 *                    synchronised; the buffers belong to the caller and must stay valid
 *                    until the stream has run.  One ctx may serve concurrent calls on
 *                    different streams (it is read-only after pack).
 * Errors: FAMSA_EINVAL (null ctx, both outputs NULL), FAMSA_ERANGE, FAMSA_ECUDA.
 */
int famsa_lcs_rows(famsa_ctx* ctx, int64_t i0, int64_t i1,
                   uint16_t* lcs_out, float* sim_out, void* cuda_stream);

/*
 * famsa_lcs_rows_host -- the same call for HOST output buffers (the end-to-end path).  Synchronous.
 * Pinned buffers are written by the sweep kernels directly (see famsa_host_mode); for pageable ones the
 * rows are swept in chunks on the device and each chunk is copied back, device compute overlapped with
 * the device->host copy of the previous chunk.
 *   lcs_host, sim_host  HOST  as above (either may be NULL, not both); pageable or pinned.
 */
int famsa_lcs_rows_host(famsa_ctx* ctx, int64_t i0, int64_t i1,
                        uint16_t* lcs_host, float* sim_host);

/*
 * famsa_lcs_rows_host_async -- as above but returns once the work is ENQUEUED on the ctx's own streams, so
 * the sweep of the next row block overlaps the device->host copy of this one (a streaming consumer calls it
 * block after block with two host buffers).  The host buffers must be pinned for the copies to be
 * asynchronous, must stay valid, and hold the results only after famsa_sync(ctx).  Calls of one ctx are
 * ordered; do not mix concurrent host-path calls of one ctx from several threads.
 */
int famsa_lcs_rows_host_async(famsa_ctx* ctx, int64_t i0, int64_t i1,
                              uint16_t* lcs_host, float* sim_host);

/* Wait for everything the host path of this ctx has enqueued. */
int famsa_sync(famsa_ctx* ctx);

/*
 * famsa_host_mode -- how famsa_lcs_rows_host* moves the rows to the host (results never depend on it):
 *   -1  auto (default): if every non-NULL output buffer is PINNED (page-locked and mapped: cudaHostAlloc /
 *       cudaHostRegister / torch pin_memory), the sweep kernels store each row straight into the caller's
 *       buffer through its device alias -- the row store of step a7 is then itself the device->host transfer
 *       (coalesced streaming stores become posted PCIe writes), with no staging buffer, copy engine or chunk
 *       boundary; pageable buffers take the staged path (device row chunks + cudaMemcpyAsync).
 *    0  always staged.      1  direct, FAMSA_EINVAL if a buffer is not pinned.
 */
int famsa_host_mode(famsa_ctx* ctx, int mode);

/*
 * famsa_lcs_rows_checksum -- famsa_lcs_rows plus a 64-bit checksum of what the call stored (SURVEY.md 8(d):
 * "a 64-bit checksum per block is kept to prove the work was done"), accumulated by the sweep kernels' own
 * epilogue (warp reductions + one atomic per warp and row; nothing is re-read):
 *   checksum_dev  DEVICE  uint64[2], ADDED to (the caller zeroes it):
 *                         [0] += sum of the LCS lengths of the call's pairs,
 *                         [1] += sum of the fp32 similarities' bit patterns (untouched if sim_out is NULL).
 * Both are order-independent integer sums mod 2^64, so any reduction over the output arrays reproduces them.
 */
int famsa_lcs_rows_checksum(famsa_ctx* ctx, int64_t i0, int64_t i1, uint16_t* lcs_out, float* sim_out,
                            uint64_t* checksum_dev, void* cuda_stream);

/*
 * Per-phase timing of the HOST-output path (diagnostics for the end-to-end number).
 *   famsa_host_profile(ctx, 1)   from now on every row chunk of famsa_lcs_rows_host* is bracketed by CUDA
 *                                events on the ctx's compute and copy streams.
 *   famsa_host_profile_read      waits for the ctx's host path, then fills HOST out[5] and resets:
 *                                [0] sum of the chunks' sweep times (ms), [1] sum of their device->host copy
 *                                times (ms), [2] bytes copied, [3] first sweep start -> last copy end (ms),
 *                                [4] number of chunks.
 *   famsa_pack_profile           HOST ms4[4]: wall time of famsa_pack's phases for this ctx: host->device copy +
 *                                encode, length sort, host-side plan, device allocation + stream/table build.
 */
int famsa_host_profile(famsa_ctx* ctx, int enable);
int famsa_host_profile_read(famsa_ctx* ctx, double* out5);
int famsa_pack_profile(const famsa_ctx* ctx, double* ms4);

/*
 * The HOST-output path keeps its device staging (two row-chunk buffers, two streams) in a process-wide pool:
 * famsa_free returns a ctx's set to the pool and the next ctx on that device reuses it.  famsa_free likewise keeps
 * the ctx's device blocks (the packed set, up to 6 GB per process) for the next famsa_pack of about the same size,
 * so that pack / sweep / free in a loop does not go through cudaMalloc and cudaFree.  famsa_trim() releases every
 * idle set and block (call it before a large allocation of your own).
 */
int famsa_trim(void);

/* Number of (i, j < i) entries of rows [i0, i1): i1(i1-1)/2 - i0(i0-1)/2.  -1 if i0 > i1 or i0 < 0. */
int64_t famsa_rows_pairs(int64_t i0, int64_t i1);

/* True DP cells of rows [i0, i1): sum over pairs of |A|*|B| (what GCUPS counts; padding excluded). */
int famsa_rows_cells(const famsa_ctx* ctx, int64_t i0, int64_t i1, double* cells);

int famsa_k(const famsa_ctx* ctx, int64_t* k);
int famsa_perm(const famsa_ctx* ctx, int64_t* perm_host);      /* HOST, k entries: perm[sorted] = original */
int famsa_lengths(const famsa_ctx* ctx, uint32_t* len_host);   /* HOST, k entries, sorted order            */

/*
 * Introspection of what pack built (tests): decoded residues and match-table words.
 *   famsa_codes   HOST out, len entries: codes 0..24 of sorted sequence s, read back from the
 *                 device-resident interleaved stream.
 *   famsa_match   HOST out, ceil(len/32) words: M_s[c] read back from the device table.
 */
int famsa_codes(const famsa_ctx* ctx, int64_t s, uint8_t* codes_host);
int famsa_match(const famsa_ctx* ctx, int64_t s, int c, uint32_t* words_host);

/* Kernel launches enqueued by this ctx so far (pack + sweep), for bench.py's gpu_launches. */
int64_t famsa_launch_count(const famsa_ctx* ctx);

/*
 * famsa_alu_peak -- micro-benchmark that measures the chip's INT32 ALU-pipe issue rate
 * (independent LOP3/IADD3 chains, all SMs, full occupancy): the roofline denominator.
 *   device            CUDA device ordinal
 *   instr_per_s       HOST out: warp-lane INT32 instructions per second (thread-instr/s)
 *   instr_per_clk_sm  HOST out: the same per SM per clock, using sm_mhz below
 *   sm_mhz            HOST out: SM clock achieved during the run (clock64 / elapsed time)
 */
int famsa_alu_peak(int device, double* instr_per_s, double* instr_per_clk_sm, double* sm_mhz);

/*
 * famsa_mix_peak -- the same micro-benchmark with the sweep's instruction mix: per word-step 3 ALU-pipe
 * instructions (LOP3, IADD3.X, LOP3) plus ONE conflict-free 32-bit shared-memory load, V in registers,
 * no global traffic, 40 warps per SM.  What it reaches is the ceiling of this mix on the SM's issue
 * logic; bench.py prints it beside the ALU peak (roofline.mix_ceiling_instr_per_clk_sm).
 *   alu_instr_per_clk_sm  HOST out: ALU-pipe thread-instructions per clock per SM achieved (the 3 per word-step)
 *   sm_mhz                HOST out: SM clock during the run
 */
int famsa_mix_peak(int device, double* alu_instr_per_clk_sm, double* sm_mhz);


/* ---------------------------------------------------------------------------------------------
 * Stage II consumer: the single-linkage guide tree over the similarities,
 * built incrementally from the streamed row blocks in O(k) memory ("it can be
 * computed incrementally, i.e., without storing the complete similarity matrix ... first two stages
 * of FAMSA are performed simultaneously").  The paper uses SLINK, whose row update is a serial
 * pointer chase; here the state is the maximum spanning forest of the rows consumed so far (the
 * single-linkage dendrogram is its edges taken by decreasing similarity).  A row block is merged in
 * with ONE read of the block and no host round trip: round 0 of Boruvka on the block's own graph
 * (best entry per row and per column -- the sweep's epilogue delivers these when the block comes from
 * famsa_guide_forest), one pass that keeps the best edge from every block row into every other
 * component (at most 1024 components remain after round 0), and a persistent cooperative kernel that
 * merges the resulting sparse edge set into the forest by Boruvka rounds with grid-wide barriers.
 * Under ties in the similarities the tree is not unique; the sorted merge similarities are.
 */
typedef struct famsa_tree famsa_tree;

/* O(k) device state for k leaves on CUDA device `device`. */
int famsa_tree_create(int64_t k, int device, famsa_tree** out);

/*
 * Consume rows [i0, i1) of the similarity matrix.  Row blocks may arrive in ANY order and each row
 * once (the state is the maximum spanning forest of the entries seen so far), so a rank of a
 * multi-GPU job can feed only the blocks it swept.
 *   sim_block  DEVICE  famsa_rows_pairs(i0, i1) floats in the famsa_lcs_rows layout, similarities >= 0
 *                      (+inf allowed; entries with the sign bit set are ignored).
 * The work is ENQUEUED on `cuda_stream` (NULL = default stream) and not synchronised: sim_block must stay
 * valid and unchanged until the stream has run; calls for one tree must be stream-ordered with one
 * another.  famsa_tree_edge_count / _edges / _finish wait for the device.  Errors found on the device
 * (no convergence, internal overflow) are reported by those calls as FAMSA_EINVAL.
 */
int famsa_tree_update(famsa_tree* t, int64_t i0, int64_t i1, const float* sim_block, void* cuda_stream);

/*
 * Merge m weighted edges (a[e], b[e], sim[e]) into the forest: MSF(E1 u E2) = MSF(MSF(E1) u MSF(E2)),
 * so the forests of several ranks (famsa_tree_edges of each, gathered) merged into one tree give the
 * tree of the whole matrix.  HOST inputs; leaves in [0, k), similarities >= 0.
 */
int famsa_tree_merge_edges(famsa_tree* t, const int64_t* a_host, const int64_t* b_host, const float* sim_host, int64_t m);

/* Edges in the current forest (k-1 once every row has been consumed or merged in); waits for the device;
 * -1 if the device reported an error. */
int64_t famsa_tree_edge_count(const famsa_tree* t);

/* HOST outputs, famsa_tree_edge_count entries each: the current forest's edges (a > b, leaf indices). */
int famsa_tree_edges(famsa_tree* t, int64_t* a_host, int64_t* b_host, float* sim_host);

/*
 * The dendrogram, k-1 merges by decreasing similarity (ties: by ascending (a, b) of the tree edge):
 * merge t joins clusters id_a[t] < id_b[t] into cluster k + t (leaves are 0..k-1, scipy convention);
 * sim[t] is the merge similarity, size[t] the leaves in the new cluster.  HOST outputs, k-1 entries.
 * Every row must have been consumed (or the missing ones merged in as edges): else FAMSA_ERANGE.
 */
int famsa_tree_finish(famsa_tree* t, int64_t* id_a_host, int64_t* id_b_host, float* sim_host, int64_t* size_host);

void famsa_tree_free(famsa_tree* t);

/*
 * famsa_guide_tree -- stages I and II together, as the paper runs them: sweeps the
 * packed set in row blocks of `block_rows` rows (0 = default 1024 = the maximum) and feeds each block to
 * the tree while the next block is being swept on a second stream; row blocks never leave the device and
 * the host only enqueues (the sweep of block n+2 waits on an event for the merge of block n).
 * Outputs as famsa_tree_finish, in SORTED leaf indices (map through famsa_perm).
 */
int famsa_guide_tree(famsa_ctx* ctx, int64_t block_rows, int64_t* id_a_host, int64_t* id_b_host,
                     float* sim_host, int64_t* size_host);

/*
 * famsa_guide_forest -- the same pipeline over one part of the row blocks: blocks part, part + parts,
 * part + 2*parts, ... (0 <= part < parts), the cyclic deal that balances the triangle over `parts`
 * GPUs.  Returns the tree handle (its forest spans only what this part saw); gather every part's
 * famsa_tree_edges, famsa_tree_merge_edges them into one tree and famsa_tree_finish it.
 * The caller frees *out with famsa_tree_free.
 */
int famsa_guide_forest(famsa_ctx* ctx, int64_t block_rows, int64_t part, int64_t parts, famsa_tree** out);

/*
 * Tuning knobs of ONE ctx (tests sweep them; concurrent calls on other ctxs are unaffected).  Results never
 * depend on them.  0 (or -1 for small_job_mode) restores the default.
 *   rows_per_cta    rows of A per CTA on the register path, 1..12 (default 2)
 *   small_job_mode  -1 auto: calls with fewer than 2048 x SM-count pairs run one pair per thread in one-warp
 *                   CTAs (the hardware then balances the job at warp granularity); 0 never; 1 always
 *   l2_group_mb     size of the residue-stream slice that one column group of a launch re-reads from L2
 *                   (default 24)
 */
int famsa_ctx_set_tuning(famsa_ctx* ctx, int rows_per_cta, int small_job_mode, int l2_group_mb);

void famsa_free(famsa_ctx* ctx);            /* famsa_free(NULL) is a no-op */
const char* famsa_strerror(int code);       /* static text for a FAMSA_E* code */
const char* famsa_last_error(void);         /* detail of the calling thread's last failure */

#ifdef __cplusplus
}
#endif
#endif /* FAMSA_LCS_H */
