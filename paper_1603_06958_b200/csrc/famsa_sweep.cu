// famsa_sweep.cu -- steps a4-a7 of the path: the all-pairs bit-parallel LCS sweep, zero count,
// similarity epilogue and packed-triangular row store (recurrence as
// stated in BASELINE.json north_star, cited by the paper as Hyyro [15]).
//
// Mapping: one thread sweeps NR = 1-3 rows (A side) against one column (B side).
// A CTA owns TA rows (their match tables arrive in shared memory by one TMA bulk copy; layout
// [word][symbol], so one warp load = one 128-byte row and no residue mix can bank-conflict) x TB = 128
// columns (thread t walks sequence j0 + t; a warp = one 32-lane interleave group, so each uint4 load
// is 512 contiguous bytes).  V lives in NR x W registers; the add carry runs through the hardware
// carry flag (add.cc / addc.cc -> IADD3 / IADD3.X).  Per 32-bit word-step: LOP3, IADD3.X, LOP3 + one
// LDS.  Rows longer than 32 words are cut into blocks of Wb <= 32 words; the carry out of block t at
// residue p is kept in a per-thread bit-vector and fed to block t+1 at residue p.
#include <algorithm>

#include "famsa_internal.h"

namespace famsa {

#ifndef FAMSA_TB
#define FAMSA_TB 128
#endif
constexpr int TB = FAMSA_TB;     // threads (= columns) per CTA
constexpr int MAX_ROWS_PER_LAUNCH = 1024;

struct SweepArgs {
    const uint4*    stream;      // interleaved residue stream
    const uint32_t* goff;        // group offsets (512-byte units)
    const uint4*    tables;      // match tables, 128-byte rows
    const uint32_t* toff;        // table row offset per sequence
    const uint32_t* len;         // lengths, sorted order
    uint16_t*       lcs_out;
    float*          sim_out;
    int64_t         out_base;    // i0*(i0-1)/2 of the call
    uint32_t        r0, r1;      // rows of this launch
    uint32_t        ta;          // rows per CTA
    uint32_t        n_col_tiles;
    uint32_t        nblk;        // table blocks per row (1 on the register path)
    uint32_t        row_tiles;   // row tiles of this launch
    uint32_t        cg_tiles;    // column tiles per column group (L2 blocking of the residue stream, see tile_coords)
    unsigned long long* checksum;   // DEVICE u64[2] or nullptr: += sum of LCS, += sum of similarity bit patterns
    unsigned long long* cand_row;   // DEVICE or nullptr: round-0 candidates of the guide tree (TreeCand, famsa_internal.h)
    unsigned long long* cand_col;
};

// CTA -> (row tile, column tile).  The grid is walked column GROUP by column group: inside a group of
// cg_tiles column tiles every row tile of the launch is swept before the next group starts, so the slice
// of the residue stream in use (cg_tiles x 128 sequences, sized to ~24 MB by the host) is re-read from L2
// by each of the launch's row tiles instead of the whole 129 MB stream cycling through the 126 MB L2 once
// per row tile (r01: 22 GB of DRAM reads for a launch whose algorithmic traffic is 1.6 GB).
// Columns ascend inside and across groups, so the longest sequences are still scheduled first.
__device__ __forceinline__ void tile_coords(const SweepArgs& a, uint32_t& row_tile, uint32_t& col_tile) {
    const uint32_t per_group = a.row_tiles * a.cg_tiles;
    const uint32_t cg = blockIdx.x / per_group;
    const uint32_t rem = blockIdx.x - cg * per_group;
    const uint32_t c0 = cg * a.cg_tiles;
    const uint32_t gc = min(a.cg_tiles, a.n_col_tiles - c0);        // the last group may be narrower
    row_tile = rem / gc;
    col_tile = c0 + rem % gc;
}

// ---- table staging: one TMA bulk copy (cp.async.bulk, global -> shared) per tile, completion on an
// mbarrier; no registers or LSU instructions are spent on it and the waiting warps sleep on the barrier.
__device__ __forceinline__ void mbar_init(uint32_t bar) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" :: "r"(bar));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void bulk_load(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");        // earlier generic reads of dst vs. this async write
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(bar), "r"(bytes) : "memory");
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 :: "r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile("{\n\t.reg .pred p;\n\tWAIT_%=:\n\t"
                 "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
                 "@p bra DONE_%=;\n\tbra WAIT_%=;\n\tDONE_%=:\n\t}" :: "r"(bar), "r"(parity) : "memory");
}

template <int IMM>
__device__ __forceinline__ uint32_t lds32(uint32_t addr) {
    uint32_t v;
    asm("ld.shared.u32 %0, [%1+%2];" : "=r"(v) : "r"(addr), "n"(IMM));
    return v;
}
// m[w] = table word w of the symbol column at `addr` (static unroll so the offset is an immediate)
template <int W, int I = 0>
struct LoadWords {
    static __device__ __forceinline__ void run(uint32_t (&m)[W], uint32_t addr) {
        m[I] = lds32<I * ROW_BYTES>(addr);
        LoadWords<W, I + 1>::run(m, addr);
    }
};
template <int W>
struct LoadWords<W, W> {
    static __device__ __forceinline__ void run(uint32_t (&)[W], uint32_t) {}
};

// One residue against W words of V.  `addr` = shared-memory address of the symbol's column in
// word-row 0 (table base | code*4).  CARRY: the chain starts from / ends in the hardware carry.
template <int W, bool CARRY>
__device__ __forceinline__ void residue_step(uint32_t (&V)[W], uint32_t addr, uint32_t& cin, uint32_t& cout) {
    uint32_t m[W], s[W];
    LoadWords<W>::run(m, addr);
    if (CARRY) asm volatile("add.cc.u32 %0, %0, %0;" : "+r"(cin));            // carry flag <- top bit of cin
#pragma unroll
    for (int w = 0; w < W; ++w) {
        uint32_t u = V[w] & m[w];
        if (w == 0 && !CARRY) asm volatile("add.cc.u32 %0, %1, %2;" : "=r"(s[w]) : "r"(V[w]), "r"(u));
        else                  asm volatile("addc.cc.u32 %0, %1, %2;" : "=r"(s[w]) : "r"(V[w]), "r"(u));
    }
    if (CARRY) asm volatile("addc.u32 %0, %0, %0;" : "+r"(cout));             // shift the carry out in
#pragma unroll
    for (int w = 0; w < W; ++w) V[w] = s[w] | (V[w] & ~m[w]);
}

// Shared-memory address of residue R's symbol column: the table base with byte R of bword (= code*4
// < 128) spliced into its low byte -- tbase is 256-byte aligned, so one PRMT does extract + add.
// (Tried and rejected, r01: doing this on the FMA pipe with IMAD + IMAD.HI against __constant__
// multipliers -- 7 FMA-pipe instructions per 4 residues instead of 4 ALU ones -- ran 3 % slower.)
template <int R>
__device__ __forceinline__ uint32_t residue_addr(uint32_t bword, uint32_t tbase) {
    return __byte_perm(bword, tbase, 0x7650 + R);
}

template <int W, bool CARRY>
__device__ __forceinline__ void word_step(uint32_t (&V)[W], uint32_t bword, uint32_t tbase, uint32_t& cin, uint32_t& cout) {
    residue_step<W, CARRY>(V, residue_addr<0>(bword, tbase), cin, cout);
    residue_step<W, CARRY>(V, residue_addr<1>(bword, tbase), cin, cout);
    residue_step<W, CARRY>(V, residue_addr<2>(bword, tbase), cin, cout);
    residue_step<W, CARRY>(V, residue_addr<3>(bword, tbase), cin, cout);
}

// Sweep this warp's group (nwords 4-residue words, i.e. up to the group's longest sequence) against
// one table block.  cv: carry bit-vector, 16 bits per 16-residue chunk (blocked path only).
template <int W, bool CARRY>
__device__ __forceinline__ void sweep_block(uint32_t (&V)[W], const uint4* __restrict__ bp, uint32_t nwords, uint32_t tbase,
                                            unsigned short* cv, bool read_cv, bool write_cv) {
    const uint32_t nfull = nwords >> 2, tail = nwords & 3;
    uint4 cur = nwords ? __ldg(bp) : make_uint4(0, 0, 0, 0);
    for (uint32_t c = 0; c < nfull; ++c) {
        uint4 nxt = cur;
        if ((c + 1) * 4 < nwords) nxt = __ldg(bp + (size_t)(c + 1) * GROUP);
        uint32_t cin = 0, cout = 0;
        if (CARRY && read_cv) cin = (uint32_t)cv[c] << 16;
        word_step<W, CARRY>(V, cur.x, tbase, cin, cout);
        word_step<W, CARRY>(V, cur.y, tbase, cin, cout);
        word_step<W, CARRY>(V, cur.z, tbase, cin, cout);
        word_step<W, CARRY>(V, cur.w, tbase, cin, cout);
        if (CARRY && write_cv) cv[c] = (unsigned short)cout;
        cur = nxt;
    }
    if (tail) {                                           // last, partial chunk: 1-3 words
        uint32_t cin = 0, cout = 0;
        if (CARRY && read_cv) cin = (uint32_t)cv[nfull] << 16;
#pragma unroll 1
        for (uint32_t q = 0; q < tail; ++q) {
            const uint32_t w = q == 0 ? cur.x : (q == 1 ? cur.y : cur.z);
            word_step<W, CARRY>(V, w, tbase, cin, cout);
        }
        if (CARRY && write_cv) cv[nfull] = (unsigned short)(cout << (16 - 4 * tail));   // first residue's carry at bit 15
    }
}

// Epilogue (a6, a7) for one row of a warp: indel = |A| + |B| - 2 LCS, similarity = LCS / indel^2
// (PAPER.md:42).  Plain stores: with the column-group rasterisation the residue-stream slice in use stays in L2
// whatever the output does (measured r02: st.global.cs was 0.3 % slower and saved 0.3 GB of 35 GB DRAM traffic
// per step).  Called by ALL lanes of the warp (`valid` says which lanes own an entry) so that the optional
// checksum and the guide tree's candidates can use warp reductions.  Returns the entry as a candidate of
// column j (0 when candidates are off).
template <bool CAND>
__device__ __forceinline__ unsigned long long store_pair(const SweepArgs& a, bool valid, uint32_t i, uint32_t j, uint32_t la, uint32_t lb, uint32_t lcs) {
    const int64_t pos = (int64_t)i * (i - 1) / 2 - a.out_base + j;
    uint32_t sim_bits = 0;
    if (valid) {
        if (a.lcs_out) a.lcs_out[pos] = (unsigned short)lcs;
        if (a.sim_out || CAND) {
            const unsigned long long indel = (unsigned long long)la + lb - 2ull * lcs;
            const float sim = __fdiv_rn(__uint2float_rn(lcs), __ull2float_rn(indel * indel));
            if (a.sim_out) a.sim_out[pos] = sim;
            sim_bits = __float_as_uint(sim);
        }
    }
    if (a.checksum) {                                       // kernel-uniform
        const uint32_t sl = __reduce_add_sync(0xffffffffu, valid ? lcs : 0u);          // <= 32 x 65535
        const uint32_t s_lo = __reduce_add_sync(0xffffffffu, sim_bits & 0xFFFFu);
        const uint32_t s_hi = __reduce_add_sync(0xffffffffu, sim_bits >> 16);
        if ((threadIdx.x & 31) == 0) {
            if (sl) atomicAdd(a.checksum, (unsigned long long)sl);
            if (a.sim_out && (s_lo | s_hi)) atomicAdd(a.checksum + 1, ((unsigned long long)s_hi << 16) + s_lo);
        }
    }
    if (CAND) {                                             // compile-time: the guide tree's round-0 candidates
        const uint32_t hi = valid ? sim_bits + 1u : 0u;     // similarities are >= +0: bit order == value order
        const uint32_t hmax = __reduce_max_sync(0xffffffffu, hi);
        const uint32_t lmax = __reduce_max_sync(0xffffffffu, hi == hmax ? ~j : 0u);    // ties: the smallest column
        if ((threadIdx.x & 31) == 0 && hmax) {
            const unsigned long long key = ((unsigned long long)hmax << 32) | lmax;
            if (key > a.cand_row[i]) atomicMax(a.cand_row + i, key);                   // monotone filter: a stale read only costs an atomic
        }
        return valid ? ((unsigned long long)hi << 32) | (uint32_t)~i : 0ull;           // this entry as a candidate of column j
    }
    return 0ull;
}

// Column candidates of one row step of a thread (<= 3 rows): one filtered atomicMax.
__device__ __forceinline__ void store_col_cand(const SweepArgs& a, uint32_t j, unsigned long long key) {
    if (key && key > a.cand_col[j]) atomicMax(a.cand_col + j, key);
}

// ---- register path: every row of the launch fits one block of W words --------------------------
// NR rows per thread at once (3 for W <= 8, 2 for W <= 16, else 1) while NR x W words of V fit
// comfortably in registers: the rows see the same residue, so the address PRMT and the residue-stream
// loads are shared and the NR carry chains are independent (more ILP per warp).  Small jobs (too few
// pairs to fill the SMs' warp slots) use NR = 1 and one-warp CTAs instead: see sweep_rows().
__host__ __device__ constexpr int rows_per_thread(int w) { return w <= 8 ? 3 : (w <= 16 ? 2 : 1); }

template <int W, int NR, int TS>
__device__ __forceinline__ void residue_step_rows(uint32_t (&V)[NR][W], uint32_t addr) {
    uint32_t m[NR][W], s[NR][W];
#pragma unroll
    for (int p = 0; p < NR; ++p) LoadWords<W>::run(m[p], addr + p * TS);
#pragma unroll
    for (int p = 0; p < NR; ++p) {
#pragma unroll
        for (int w = 0; w < W; ++w) {
            uint32_t u = V[p][w] & m[p][w];
            if (w == 0) asm volatile("add.cc.u32 %0, %1, %2;" : "=r"(s[p][w]) : "r"(V[p][w]), "r"(u));
            else        asm volatile("addc.cc.u32 %0, %1, %2;" : "=r"(s[p][w]) : "r"(V[p][w]), "r"(u));
        }
    }
#pragma unroll
    for (int p = 0; p < NR; ++p)
#pragma unroll
        for (int w = 0; w < W; ++w) V[p][w] = s[p][w] | (V[p][w] & ~m[p][w]);
}

template <int W, int NR, int TS>
__device__ __forceinline__ void word_step_rows(uint32_t (&V)[NR][W], uint32_t bword, uint32_t tbase) {
    residue_step_rows<W, NR, TS>(V, residue_addr<0>(bword, tbase));
    residue_step_rows<W, NR, TS>(V, residue_addr<1>(bword, tbase));
    residue_step_rows<W, NR, TS>(V, residue_addr<2>(bword, tbase));
    residue_step_rows<W, NR, TS>(V, residue_addr<3>(bword, tbase));
}

template <int W, int NR, int TS>
__device__ __forceinline__ void sweep_rows_block(uint32_t (&V)[NR][W], const uint4* __restrict__ bp, uint32_t nwords, uint32_t tbase) {
    const uint32_t nfull = nwords >> 2, tail = nwords & 3;
    uint4 cur = nwords ? __ldg(bp) : make_uint4(0, 0, 0, 0);
    for (uint32_t c = 0; c < nfull; ++c) {
        uint4 nxt = cur;
        if ((c + 1) * 4 < nwords) nxt = __ldg(bp + (size_t)(c + 1) * GROUP);
        word_step_rows<W, NR, TS>(V, cur.x, tbase);
        word_step_rows<W, NR, TS>(V, cur.y, tbase);
        word_step_rows<W, NR, TS>(V, cur.z, tbase);
        word_step_rows<W, NR, TS>(V, cur.w, tbase);
        cur = nxt;
    }
#pragma unroll 1
    for (uint32_t q = 0; q < tail; ++q)                    // last, partial chunk: 1-3 words
        word_step_rows<W, NR, TS>(V, q == 0 ? cur.x : (q == 1 ? cur.y : cur.z), tbase);
}

// Every launch is a PROGRAMMATIC dependent of the kernel before it in the stream (launch_sweep): it may start
// while its predecessor drains, and every warp executes griddepcontrol.wait BEFORE ITS FIRST STORE (the sweep
// itself only reads the packed set, which nothing writes after famsa_pack).  The wait returns once the
// predecessor grid has completed and its memory operations are visible, so (1) stores of consecutive
// launches -- of one call or of consecutive calls on the stream -- land in stream order even when they hit
// the same addresses, (2) a grid cannot complete before its predecessor (every launch has at least one
// storing warp), so "the last launch is done" implies "every launch is done", which is what an event
// recorded after a call relies on, and (3) a predecessor that is NOT one of these kernels (a consumer of the
// previous row block, a memcpy) never triggers early, so the launch is then an ordinary stream-ordered one.
// (Without the launch attribute the instruction is a no-op.)
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

template <int W, int NR, bool CAND>
__global__ void __launch_bounds__(TB) sweep_short_kernel(const SweepArgs a) {
    extern __shared__ __align__(256) uint8_t smem[];
    asm volatile("griddepcontrol.launch_dependents;");
    constexpr int WST = (W + 1) & ~1;
    constexpr int TS = WST * ROW_BYTES;                  // bytes between the tables of consecutive rows
    uint32_t row_tile, col_tile;
    tile_coords(a, row_tile, col_tile);
    const uint32_t r_lo = a.r0 + row_tile * a.ta;
    const uint32_t r_hi = min(r_lo + a.ta, a.r1);
    const uint32_t j0 = col_tile * blockDim.x;           // blockDim.x = 128 columns, or 32 for small jobs
    if (j0 + 1 >= r_hi) return;                          // whole tile on or above the diagonal
    // stage the tile's tables: rows r_lo..r_hi-1 are contiguous (same stride each).  With NR > 1 the
    // last step of a warp may run past row r_hi-1: the launch allocates NR-1 extra table slots, whose
    // (uninitialised) content feeds V's that are never stored.
    const uint32_t smem_base = (uint32_t)__cvta_generic_to_shared(smem);   // 256-byte aligned: no static shared memory
    const uint32_t mbar = smem_base + (a.ta + NR - 1) * TS;                  // the mbarrier sits after the table slots
    if (threadIdx.x == 0) mbar_init(mbar);
    __syncthreads();
    if (threadIdx.x == 0)
        bulk_load(smem_base, a.tables + (size_t)a.toff[r_lo] * (ROW_BYTES / 16), (r_hi - r_lo) * TS, mbar);
    const uint32_t lane = threadIdx.x & 31;
    const uint32_t jw = j0 + (threadIdx.x & ~31u);       // first column of this warp
    if (jw + 1 >= r_hi) return;                          // this warp's columns are all >= every row (no barrier follows)
    const uint32_t j = jw + lane;
    const uint32_t gb = a.goff[jw / GROUP];              // jw < k, so this is a real group
    const uint4* bp = a.stream + (size_t)gb * GROUP + lane;
    const uint32_t lb = j < r_hi ? a.len[j] : 0;         // columns >= r_hi are never stored
    const uint32_t nwords = (a.len[jw] + 3) >> 2;        // 4-residue words to sweep: jw is the group's longest sequence
    mbar_wait(mbar, 0);                                  // the tables have landed
    for (uint32_t i = max(r_lo, jw + 1); i < r_hi; i += NR) {   // rows NR at a time, from the first one below column jw
        uint32_t V[NR][W];
#pragma unroll
        for (int p = 0; p < NR; ++p)
#pragma unroll
            for (int w = 0; w < W; ++w) V[p][w] = 0xFFFFFFFFu;
        sweep_rows_block<W, NR, TS>(V, bp, nwords, smem_base + (i - r_lo) * TS);
        unsigned long long ckey = 0;
#pragma unroll
        for (int p = 0; p < NR; ++p) {
            uint32_t lcs = 0;
#pragma unroll
            for (int w = 0; w < W; ++w) lcs += __popc(~V[p][w]);
            const uint32_t row = i + p;                  // warp-uniform
            if (p == 0) pdl_wait();                      // stores only after the previous launch is complete
            if (row < r_hi) ckey = max(ckey, store_pair<CAND>(a, j < row, row, j, a.len[row], lb, lcs));
        }
        if (CAND) store_col_cand(a, j, ckey);
    }
}

// ---- blocked path: rows of nblk blocks x W words; one row per CTA; carry bit-vector per thread --
template <int W, int CW, bool CAND>
__global__ void __launch_bounds__(TB) sweep_long_kernel(const SweepArgs a) {
    extern __shared__ __align__(256) uint8_t smem[];
    asm volatile("griddepcontrol.launch_dependents;");
    constexpr int WST = (W + 1) & ~1;
    uint32_t row_tile, col_tile;
    tile_coords(a, row_tile, col_tile);
    const uint32_t i = a.r0 + row_tile;
    const uint32_t j0 = col_tile * TB;
    if (j0 >= i) return;
    const uint32_t lane = threadIdx.x & 31;
    const uint32_t jw = j0 + (threadIdx.x & ~31u);
    const uint32_t j = jw + lane;
    const bool active = jw < i;                          // warp-uniform
    const uint32_t gb = active ? a.goff[jw / GROUP] : 0;
    const uint32_t nwords = active ? (a.len[jw] + 3) >> 2 : 0;
    const uint4* bp = a.stream + (size_t)gb * GROUP + lane;
    const uint32_t smem_base = (uint32_t)__cvta_generic_to_shared(smem);
    unsigned short cv[CW * 2];                           // 16 carry bits per 16-residue chunk
    uint32_t lcs = 0;
    const uint4* src = a.tables + (size_t)a.toff[i] * (ROW_BYTES / 16);
    const uint32_t mbar = smem_base + WST * ROW_BYTES;   // the mbarrier sits after the table block
    if (threadIdx.x == 0) mbar_init(mbar);
    for (uint32_t blk = 0; blk < a.nblk; ++blk) {
        __syncthreads();                                 // barrier initialised / everyone done with the previous block
        if (threadIdx.x == 0) bulk_load(smem_base, src + (size_t)blk * WST * (ROW_BYTES / 16), WST * ROW_BYTES, mbar);
        mbar_wait(mbar, blk & 1);                        // phase flips once per block
        if (active) {
            uint32_t V[W];
#pragma unroll
            for (int w = 0; w < W; ++w) V[w] = 0xFFFFFFFFu;
            sweep_block<W, true>(V, bp, nwords, smem_base, cv, blk > 0, blk + 1 < a.nblk);
#pragma unroll
            for (int w = 0; w < W; ++w) lcs += __popc(~V[w]);
        }
    }
    if (active) {
        pdl_wait();
        const unsigned long long ckey = store_pair<CAND>(a, j < i, i, j, a.len[i], j < i ? a.len[j] : 0, lcs);
        if (CAND) store_col_cand(a, j, ckey);
    }
}

}  // namespace famsa

// ---- host side: buckets -> launches ------------------------------------------------------------
namespace famsa {

// Every launch carries the programmatic-stream-serialization attribute (see pdl_wait above): the next
// bucket's -- or the next call's -- CTAs fill the SMs while the previous launch drains its last wave.
template <typename K>
static cudaError_t launch_sweep(K kernel, const SweepArgs& a, unsigned grid, unsigned block, size_t smem, cudaStream_t st) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid); cfg.blockDim = dim3(block); cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, a);
}

// Variants: small jobs use NR = 1 (one-warp CTAs); the guide tree's sweeps (cand) carry the candidate epilogue
// as a compile-time variant, so the plain sweep pays nothing for it (measured r02: as a run-time branch it
// cost the plain sweep 0.8 %).
#define SHORT_CASE(W) case W: return cand ? launch_sweep(sweep_short_kernel<W, rows_per_thread(W), true>, a, grid, block, smem, st) \
                                   : small ? launch_sweep(sweep_short_kernel<W, 1, false>, a, grid, block, smem, st) \
                                           : launch_sweep(sweep_short_kernel<W, rows_per_thread(W), false>, a, grid, block, smem, st);
static cudaError_t dispatch_short(int w, bool small, bool cand, const SweepArgs& a, unsigned grid, unsigned block, size_t smem, cudaStream_t st) {
    switch (w) {
        SHORT_CASE(1) SHORT_CASE(2) SHORT_CASE(3) SHORT_CASE(4) SHORT_CASE(5) SHORT_CASE(6) SHORT_CASE(7) SHORT_CASE(8)
        SHORT_CASE(9) SHORT_CASE(10) SHORT_CASE(11) SHORT_CASE(12) SHORT_CASE(13) SHORT_CASE(14) SHORT_CASE(15) SHORT_CASE(16)
        SHORT_CASE(17) SHORT_CASE(18) SHORT_CASE(19) SHORT_CASE(20) SHORT_CASE(21) SHORT_CASE(22) SHORT_CASE(23) SHORT_CASE(24)
        SHORT_CASE(25) SHORT_CASE(26) SHORT_CASE(27) SHORT_CASE(28) SHORT_CASE(29) SHORT_CASE(30) SHORT_CASE(31) SHORT_CASE(32)
        default: return cudaErrorInvalidValue;
    }
}
#define LONG_CASE(W) case W: return cand ? launch_sweep(sweep_long_kernel<W, CW_SMALL, true>, a, grid, TB, smem, st) \
                                         : launch_sweep(sweep_long_kernel<W, CW_SMALL, false>, a, grid, TB, smem, st);
static cudaError_t dispatch_long(int w, bool large, bool cand, const SweepArgs& a, unsigned grid, size_t smem, cudaStream_t st) {
    if (large) {
        if (w != 32) return cudaErrorInvalidValue;
        return cand ? launch_sweep(sweep_long_kernel<32, CW_LARGE, true>, a, grid, TB, smem, st)
                    : launch_sweep(sweep_long_kernel<32, CW_LARGE, false>, a, grid, TB, smem, st);
    }
    switch (w) {
        LONG_CASE(17) LONG_CASE(18) LONG_CASE(19) LONG_CASE(20) LONG_CASE(21) LONG_CASE(22) LONG_CASE(23) LONG_CASE(24)
        LONG_CASE(25) LONG_CASE(26) LONG_CASE(27) LONG_CASE(28) LONG_CASE(29) LONG_CASE(30) LONG_CASE(31) LONG_CASE(32)
        default: return cudaErrorInvalidValue;
    }
}

// Column tiles per column group, so that one group's slice of the residue stream is ~l2_group_bytes.
static uint32_t column_group_tiles(const famsa_ctx* ctx, uint32_t r1, uint32_t n_col_tiles, double l2_group_bytes) {
    const int64_t g_end = std::min<int64_t>(((int64_t)r1 - 1 + GROUP - 1) / GROUP, ctx->n_groups);
    const double bytes = (double)ctx->goff[g_end] * (GROUP * CHUNK);          // stream bytes of columns [0, r1-1)
    const double per_tile = std::max(bytes / std::max<uint32_t>(n_col_tiles, 1), 1.0);
    const double t = l2_group_bytes / per_tile;
    return (uint32_t)std::min<double>(std::max(t, 1.0), (double)std::max<uint32_t>(n_col_tiles, 1));
}

int sweep_rows(famsa_ctx* ctx, int64_t i0, int64_t i1, uint16_t* lcs, float* sim, unsigned long long* checksum, const TreeCand* cand, cudaStream_t st) {
    SweepArgs a;
    a.stream = reinterpret_cast<const uint4*>(ctx->d_stream);
    a.goff = ctx->d_goff;
    a.tables = reinterpret_cast<const uint4*>(ctx->d_tables);
    a.toff = ctx->d_toff;
    a.len = ctx->d_len;
    a.lcs_out = lcs; a.sim_out = sim;
    a.checksum = checksum;
    a.cand_row = cand ? cand->row : nullptr; a.cand_col = cand ? cand->col : nullptr;
    a.out_base = i0 * (i0 - 1) / 2;
    const uint32_t rows_per_cta = ctx->rows_per_cta.load();
    const int small_mode = ctx->small_mode.load();
    const double l2_group_bytes = (double)ctx->l2_group_mb.load() * 1048576.0;
    // Small job: too few pairs to give every SM sub-partition a handful of warps at 2-3 rows per thread.
    // Then every pair gets its own thread (NR = 1, one row per CTA) in one-warp CTAs, so the hardware
    // scheduler balances the job over the SMs at warp granularity (configs[0]: 124 750 pairs = 3 898 warps
    // over 592 sub-partitions) instead of a few fat 128-thread CTAs per SM.
    const bool use_cand = cand != nullptr;
    const bool small = !use_cand && (small_mode == 1 || (small_mode < 0 && famsa_rows_pairs(i0, i1) < (int64_t)2048 * ctx->sm_count));
    const unsigned block = small ? 32 : TB;
    for (const Bucket& b : ctx->buckets) {
        int64_t lo = std::max(b.r0, std::max<int64_t>(i0, 1)), hi = std::min(b.r1, i1);   // row 0 is empty
        for (int64_t r = lo; r < hi; r += MAX_ROWS_PER_LAUNCH) {
            a.r0 = (uint32_t)r; a.r1 = (uint32_t)std::min<int64_t>(r + MAX_ROWS_PER_LAUNCH, hi);
            a.nblk = (uint32_t)b.nblk;
            const int wst = (b.wb + 1) & ~1;
            cudaError_t e;
            if (b.nblk == 1) {
                a.n_col_tiles = (a.r1 - 1 + block - 1) / block;          // columns 0 .. r1-2
                const uint32_t nr = small ? 1u : (uint32_t)rows_per_thread(b.wb);
                a.ta = small ? 1u : ((rows_per_cta + nr - 1) / nr) * nr;   // a whole number of NR-row steps per CTA
                while (a.ta > nr && (size_t)(a.ta + nr - 1) * wst * ROW_BYTES + 16 > 48 * 1024) a.ta -= nr;   // default dynamic smem limit
                a.row_tiles = (a.r1 - a.r0 + a.ta - 1) / a.ta;
                a.cg_tiles = column_group_tiles(ctx, a.r1, a.n_col_tiles, l2_group_bytes);
                e = dispatch_short(b.wb, small, use_cand, a, a.row_tiles * a.n_col_tiles, block, (size_t)(a.ta + nr - 1) * wst * ROW_BYTES + 16, st);
            } else {
                a.n_col_tiles = (a.r1 - 1 + TB - 1) / TB;
                a.ta = 1;
                a.row_tiles = a.r1 - a.r0;
                a.cg_tiles = column_group_tiles(ctx, a.r1, a.n_col_tiles, l2_group_bytes);
                e = dispatch_long(b.wb, ctx->large_cw, use_cand, a, a.row_tiles * a.n_col_tiles, (size_t)wst * ROW_BYTES + 16, st);
            }
            if (e != cudaSuccess) return cuda_fail(e, "sweep kernel launch");
            ctx->launches++;
        }
    }
    return FAMSA_OK;
}

// ---- staging sets of the HOST-output path: two device row-chunk buffers, two streams, four events.
// Pooled per process (idle sets are kept on famsa_free and reused by the next ctx on the same device), so
// that a caller that packs, sweeps and frees in a loop does not pay cudaMalloc/cudaFree of ~1.6 GB and
// stream/event creation every time.  famsa_trim() releases the idle sets.
static std::mutex g_pool_mu;
static std::vector<Staging*> g_pool;

static void staging_destroy(Staging* s) {
    if (!s) return;
    cudaSetDevice(s->device);
    for (int b = 0; b < 2; ++b) {
        cudaFree(s->lcs[b]); cudaFree(s->sim[b]);
        if (s->ev_done[b]) cudaEventDestroy(s->ev_done[b]);
        if (s->ev_copied[b]) cudaEventDestroy(s->ev_copied[b]);
    }
    if (s->s_compute) cudaStreamDestroy(s->s_compute);
    if (s->s_copy) cudaStreamDestroy(s->s_copy);
    delete s;
}

// An idle set of this device with room for `pairs` pairs per buffer, or a new one (idle sets of the device
// that are too small are released first, so the pool never holds more than it last needed).
static int staging_acquire(int device, size_t pairs, Staging** out) {
    *out = nullptr;
    std::vector<Staging*> drop;
    Staging* got = nullptr;
    {
        std::lock_guard<std::mutex> lk(g_pool_mu);
        for (size_t n = 0; n < g_pool.size();) {
            Staging* s = g_pool[n];
            if (s->device == device && !got && s->pairs >= pairs) { got = s; g_pool.erase(g_pool.begin() + n); }
            else if (s->device == device && s->pairs < pairs) { drop.push_back(s); g_pool.erase(g_pool.begin() + n); }
            else ++n;
        }
    }
    for (Staging* s : drop) staging_destroy(s);
    if (got) { *out = got; return FAMSA_OK; }
    Staging* s = new (std::nothrow) Staging();
    if (!s) { set_error("famsa_lcs_rows_host: host allocation failed"); return FAMSA_ENOMEM; }
    s->device = device;
    cudaError_t e = cudaStreamCreateWithFlags(&s->s_compute, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&s->s_copy, cudaStreamNonBlocking);
    for (int b = 0; b < 2 && e == cudaSuccess; ++b) {
        e = cudaEventCreateWithFlags(&s->ev_done[b], cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&s->ev_copied[b], cudaEventDisableTiming);
    }
    if (e != cudaSuccess) { staging_destroy(s); return cuda_fail(e, "famsa_lcs_rows_host: stream/event creation"); }
    for (int b = 0; b < 2; ++b) {
        cudaError_t e1 = cudaMalloc((void**)&s->lcs[b], pairs * sizeof(uint16_t));
        cudaError_t e2 = cudaMalloc((void**)&s->sim[b], pairs * sizeof(float));
        if (e1 != cudaSuccess || e2 != cudaSuccess) {
            cudaGetLastError(); staging_destroy(s);
            set_error("famsa_lcs_rows_host: device allocation failed"); return FAMSA_ENOMEM;
        }
    }
    s->pairs = pairs;
    *out = s;
    return FAMSA_OK;
}

void staging_release(Staging* s) {                         // called by famsa_free
    if (!s) return;
    cudaSetDevice(s->device);
    cudaStreamSynchronize(s->s_copy); cudaStreamSynchronize(s->s_compute);
    for (HostChunkTimers& t : s->timers) for (cudaEvent_t e : t.ev) if (e) cudaEventDestroy(e);
    s->timers.clear(); s->profile = false;
    std::lock_guard<std::mutex> lk(g_pool_mu);
    g_pool.push_back(s);
}

}  // namespace famsa

using namespace famsa;

extern "C" int famsa_trim(void) {
    std::vector<Staging*> all;
    { std::lock_guard<std::mutex> lk(g_pool_mu); all.swap(g_pool); }
    for (Staging* s : all) staging_destroy(s);
    cache_trim();
    return FAMSA_OK;
}

extern "C" int famsa_ctx_set_tuning(famsa_ctx* ctx, int rows_per_cta, int small_job_mode, int l2_group_mb) {
    if (!ctx) { set_error("famsa_ctx_set_tuning: ctx is NULL"); return FAMSA_EINVAL; }
    if (rows_per_cta < 0 || rows_per_cta > 12) { set_error("famsa_ctx_set_tuning: rows_per_cta must be 0 (default) or 1..12"); return FAMSA_EINVAL; }
    if (small_job_mode < -1 || small_job_mode > 1) { set_error("famsa_ctx_set_tuning: small_job_mode must be -1 (auto), 0 or 1"); return FAMSA_EINVAL; }
    if (l2_group_mb < 0 || l2_group_mb > 4096) { set_error("famsa_ctx_set_tuning: l2_group_mb must be 0 (default) or 1..4096"); return FAMSA_EINVAL; }
    ctx->rows_per_cta.store(rows_per_cta ? (uint32_t)rows_per_cta : DEFAULT_ROWS_PER_CTA);
    ctx->small_mode.store(small_job_mode);
    ctx->l2_group_mb.store(l2_group_mb ? (uint32_t)l2_group_mb : DEFAULT_L2_GROUP_MB);
    return FAMSA_OK;
}

static int rows_check(famsa_ctx* ctx, int64_t i0, int64_t i1, const void* lcs, const void* sim, const char* who) {
    if (!ctx) { set_error(std::string(who) + ": ctx is NULL"); return FAMSA_EINVAL; }
    if (i0 < 0 || i0 > i1 || i1 > ctx->k) { set_error(std::string(who) + ": bad row range"); return FAMSA_ERANGE; }
    if (!lcs && !sim) { set_error(std::string(who) + ": both outputs are NULL"); return FAMSA_EINVAL; }
    return FAMSA_OK;
}

extern "C" int famsa_lcs_rows(famsa_ctx* ctx, int64_t i0, int64_t i1, uint16_t* lcs_out, float* sim_out,
                              void* cuda_stream) {
    int rc = rows_check(ctx, i0, i1, lcs_out, sim_out, "famsa_lcs_rows");
    if (rc != FAMSA_OK) return rc;
    if (famsa_rows_pairs(i0, i1) == 0) return FAMSA_OK;
    FAMSA_CUDA(cudaSetDevice(ctx->device));
    return sweep_rows(ctx, i0, i1, lcs_out, sim_out, nullptr, nullptr, (cudaStream_t)cuda_stream);
}

extern "C" int famsa_lcs_rows_checksum(famsa_ctx* ctx, int64_t i0, int64_t i1, uint16_t* lcs_out, float* sim_out,
                                       uint64_t* checksum_dev, void* cuda_stream) {
    int rc = rows_check(ctx, i0, i1, lcs_out, sim_out, "famsa_lcs_rows_checksum");
    if (rc != FAMSA_OK) return rc;
    if (!checksum_dev) { set_error("famsa_lcs_rows_checksum: checksum_dev is NULL"); return FAMSA_EINVAL; }
    if (famsa_rows_pairs(i0, i1) == 0) return FAMSA_OK;
    FAMSA_CUDA(cudaSetDevice(ctx->device));
    static_assert(sizeof(unsigned long long) == sizeof(uint64_t), "uint64_t");
    return sweep_rows(ctx, i0, i1, lcs_out, sim_out, reinterpret_cast<unsigned long long*>(checksum_dev), nullptr, (cudaStream_t)cuda_stream);
}

// The device alias of a PINNED (page-locked, mapped) host address, or false for pageable memory.
static bool pinned_alias(const void* host, void** dev) {
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, host) != cudaSuccess) { cudaGetLastError(); return false; }
    if (at.type != cudaMemoryTypeHost || !at.devicePointer) return false;
    *dev = at.devicePointer;
    return true;
}

// Direct host path: the outputs are pinned, so the sweep kernels store each row straight into the caller's
// buffer through its device alias (coalesced 64 / 128-byte streaming stores become posted PCIe writes; the
// path produces ~11 GB/s of output against a ~55 GB/s link).  No staging buffers, no copy engine, no chunk
// boundaries (every chunk boundary of the staged path is a launch that cannot overlap its predecessor's tail).
static int rows_host_direct(famsa_ctx* ctx, int64_t i0, int64_t i1, uint16_t* lcs_dev, float* sim_dev, bool wait) {
    if (!ctx->s_direct) FAMSA_CUDA(cudaStreamCreateWithFlags(&ctx->s_direct, cudaStreamNonBlocking));
    HostChunkTimers* tm = nullptr;
    if (ctx->host_profile) {
        ctx->direct_timers.emplace_back();
        tm = &ctx->direct_timers.back();
        for (int q = 0; q < 2; ++q) FAMSA_CUDA(cudaEventCreate(&tm->ev[q]));
        tm->bytes = (double)famsa_rows_pairs(i0, i1) * ((lcs_dev ? 2 : 0) + (sim_dev ? 4 : 0));
        FAMSA_CUDA(cudaEventRecord(tm->ev[0], ctx->s_direct));
    }
    int rc = sweep_rows(ctx, i0, i1, lcs_dev, sim_dev, nullptr, nullptr, ctx->s_direct);
    if (rc != FAMSA_OK) { cudaStreamSynchronize(ctx->s_direct); return rc; }
    if (tm) FAMSA_CUDA(cudaEventRecord(tm->ev[1], ctx->s_direct));
    if (wait) FAMSA_CUDA(cudaStreamSynchronize(ctx->s_direct));
    return FAMSA_OK;
}

static int rows_host_impl(famsa_ctx* ctx, int64_t i0, int64_t i1, uint16_t* lcs_host, float* sim_host, bool wait) {
    int rc = rows_check(ctx, i0, i1, lcs_host, sim_host, "famsa_lcs_rows_host");
    if (rc != FAMSA_OK) return rc;
    if (famsa_rows_pairs(i0, i1) == 0) return FAMSA_OK;
    FAMSA_CUDA(cudaSetDevice(ctx->device));
    const int mode = ctx->host_mode.load();
    if (mode != 0) {
        void *ld = nullptr, *sd = nullptr;
        const bool pinned = (!lcs_host || pinned_alias(lcs_host, &ld)) && (!sim_host || pinned_alias(sim_host, &sd));
        if (pinned) return rows_host_direct(ctx, i0, i1, (uint16_t*)ld, (float*)sd, wait);
        if (mode == 1) { set_error("famsa_lcs_rows_host: host_mode 1 (direct) needs pinned output buffers"); return FAMSA_EINVAL; }
    }
    // chunk size: about 1/8 of the call (so the copy of chunk n overlaps the sweep of chunk n+1),
    // between 1 Mi and 128 Mi pairs, and never smaller than the longest row
    const int64_t total_pairs = famsa_rows_pairs(i0, i1);
    const int64_t chunk_pairs = std::max<int64_t>(std::min<int64_t>(std::max<int64_t>(total_pairs / 8, (int64_t)1 << 20), (int64_t)128 << 20), i1);
    const size_t want = (size_t)std::min<int64_t>(total_pairs, chunk_pairs);
    if (!ctx->stg || ctx->stg->pairs < want) {
        // size the staging once per ctx (1/8 of the whole triangle, 1 Mi .. 128 Mi pairs, at least one row),
        // so that a stream of growing row-block calls does not reallocate it
        const int64_t tri = ctx->k * (ctx->k - 1) / 2;
        const size_t cap = (size_t)std::max<int64_t>(std::max<int64_t>(std::min<int64_t>(std::max<int64_t>(tri / 8, (int64_t)1 << 20), (int64_t)128 << 20), ctx->k), (int64_t)want);
        if (ctx->stg) { staging_release(ctx->stg); ctx->stg = nullptr; }       // drains it first
        rc = staging_acquire(ctx->device, cap, &ctx->stg);
        if (rc != FAMSA_OK) return rc;
        ctx->stg->profile = ctx->host_profile;
        ctx->host_chunks = 0;
    }
    Staging* g = ctx->stg;
    // on any failure below: drain what is already in flight on the two streams, then report
    auto fail = [&](int code) { cudaStreamSynchronize(g->s_compute); cudaStreamSynchronize(g->s_copy); return code; };
#define HOST_CUDA(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) return fail(famsa::cuda_fail(e__, #call)); } while (0)
    // chunk the row range so that each chunk fits a buffer (a single row always fits: cap >= k)
    int64_t r = i0; int64_t done_pairs = 0;
    int64_t& n = ctx->host_chunks;                         // chunks enqueued so far by this ctx: the ping-pong continues across calls
    while (r < i1) {
        int64_t e = r + 1;
        while (e < i1 && famsa_rows_pairs(r, e + 1) <= (int64_t)want) ++e;
        const int64_t np = famsa_rows_pairs(r, e);
        if (np > (int64_t)g->pairs) { set_error("famsa_lcs_rows_host: a single row exceeds the staging buffer"); return fail(FAMSA_ENOMEM); }
        const int b = (int)(n & 1);
        HostChunkTimers* tm = nullptr;
        if (g->profile) {
            g->timers.emplace_back();
            tm = &g->timers.back();
            for (cudaEvent_t& ev : tm->ev) HOST_CUDA(cudaEventCreate(&ev));
            tm->bytes = (double)np * ((lcs_host ? 2 : 0) + (sim_host ? 4 : 0));
        }
        if (n >= 2) HOST_CUDA(cudaStreamWaitEvent(g->s_compute, g->ev_copied[b], 0));
        if (tm) HOST_CUDA(cudaEventRecord(tm->ev[0], g->s_compute));
        rc = sweep_rows(ctx, r, e, lcs_host ? g->lcs[b] : nullptr, sim_host ? g->sim[b] : nullptr, nullptr, nullptr, g->s_compute);
        if (rc != FAMSA_OK) return fail(rc);
        if (tm) HOST_CUDA(cudaEventRecord(tm->ev[1], g->s_compute));
        HOST_CUDA(cudaEventRecord(g->ev_done[b], g->s_compute));
        HOST_CUDA(cudaStreamWaitEvent(g->s_copy, g->ev_done[b], 0));
        if (tm) HOST_CUDA(cudaEventRecord(tm->ev[2], g->s_copy));
        if (lcs_host) HOST_CUDA(cudaMemcpyAsync(lcs_host + done_pairs, g->lcs[b], np * sizeof(uint16_t), cudaMemcpyDeviceToHost, g->s_copy));
        if (sim_host) HOST_CUDA(cudaMemcpyAsync(sim_host + done_pairs, g->sim[b], np * sizeof(float), cudaMemcpyDeviceToHost, g->s_copy));
        if (tm) HOST_CUDA(cudaEventRecord(tm->ev[3], g->s_copy));
        HOST_CUDA(cudaEventRecord(g->ev_copied[b], g->s_copy));
        done_pairs += np; r = e; ++n;
    }
    if (wait) {
        HOST_CUDA(cudaStreamSynchronize(g->s_copy));
        HOST_CUDA(cudaStreamSynchronize(g->s_compute));
    }
#undef HOST_CUDA
    return FAMSA_OK;
}

extern "C" int famsa_lcs_rows_host(famsa_ctx* ctx, int64_t i0, int64_t i1, uint16_t* lcs_host, float* sim_host) {
    return rows_host_impl(ctx, i0, i1, lcs_host, sim_host, true);
}

extern "C" int famsa_lcs_rows_host_async(famsa_ctx* ctx, int64_t i0, int64_t i1, uint16_t* lcs_host, float* sim_host) {
    return rows_host_impl(ctx, i0, i1, lcs_host, sim_host, false);
}

extern "C" int famsa_sync(famsa_ctx* ctx) {
    if (!ctx) { set_error("famsa_sync: ctx is NULL"); return FAMSA_EINVAL; }
    FAMSA_CUDA(cudaSetDevice(ctx->device));
    if (ctx->stg) {
        FAMSA_CUDA(cudaStreamSynchronize(ctx->stg->s_copy));
        FAMSA_CUDA(cudaStreamSynchronize(ctx->stg->s_compute));
    }
    if (ctx->s_direct) FAMSA_CUDA(cudaStreamSynchronize(ctx->s_direct));
    return FAMSA_OK;
}

extern "C" int famsa_host_mode(famsa_ctx* ctx, int mode) {
    if (!ctx) { set_error("famsa_host_mode: ctx is NULL"); return FAMSA_EINVAL; }
    if (mode < -1 || mode > 1) { set_error("famsa_host_mode: mode must be -1 (auto), 0 (staged) or 1 (direct)"); return FAMSA_EINVAL; }
    ctx->host_mode.store(mode);
    return FAMSA_OK;
}

extern "C" int famsa_host_profile(famsa_ctx* ctx, int enable) {
    if (!ctx) { set_error("famsa_host_profile: ctx is NULL"); return FAMSA_EINVAL; }
    ctx->host_profile = enable != 0;
    if (ctx->stg) ctx->stg->profile = ctx->host_profile;
    return FAMSA_OK;
}

extern "C" int famsa_host_profile_read(famsa_ctx* ctx, double* out) {
    if (!ctx || !out) { set_error("famsa_host_profile_read: null argument"); return FAMSA_EINVAL; }
    for (int q = 0; q < 5; ++q) out[q] = 0.0;
    int rc = famsa_sync(ctx);
    if (rc != FAMSA_OK) return rc;
    float ms = 0.0f;
    if (!ctx->direct_timers.empty()) {                     // direct path: the stores ARE the transfer, so [1] stays 0
        for (HostChunkTimers& t : ctx->direct_timers) {
            FAMSA_CUDA(cudaEventElapsedTime(&ms, t.ev[0], t.ev[1])); out[0] += ms;
            out[2] += t.bytes;
        }
        FAMSA_CUDA(cudaEventElapsedTime(&ms, ctx->direct_timers.front().ev[0], ctx->direct_timers.back().ev[1]));
        out[3] = ms; out[4] = (double)ctx->direct_timers.size();
        for (HostChunkTimers& t : ctx->direct_timers) for (cudaEvent_t e : t.ev) if (e) cudaEventDestroy(e);
        ctx->direct_timers.clear();
        return FAMSA_OK;
    }
    if (!ctx->stg || ctx->stg->timers.empty()) return FAMSA_OK;
    Staging* g = ctx->stg;
    for (HostChunkTimers& t : g->timers) {
        FAMSA_CUDA(cudaEventElapsedTime(&ms, t.ev[0], t.ev[1])); out[0] += ms;
        FAMSA_CUDA(cudaEventElapsedTime(&ms, t.ev[2], t.ev[3])); out[1] += ms;
        out[2] += t.bytes;
    }
    FAMSA_CUDA(cudaEventElapsedTime(&ms, g->timers.front().ev[0], g->timers.back().ev[3]));
    out[3] = ms; out[4] = (double)g->timers.size();
    for (HostChunkTimers& t : g->timers) for (cudaEvent_t e : t.ev) cudaEventDestroy(e);
    g->timers.clear();
    return FAMSA_OK;
}
