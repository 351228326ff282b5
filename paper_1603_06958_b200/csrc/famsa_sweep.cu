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
};

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

__device__ __forceinline__ void store_pair(const SweepArgs& a, uint32_t i, uint32_t j, uint32_t la, uint32_t lb, uint32_t lcs) {
    int64_t pos = (int64_t)i * (i - 1) / 2 - a.out_base + j;
    if (a.lcs_out) a.lcs_out[pos] = (unsigned short)lcs;
    if (a.sim_out) {
        // indel = |A| + |B| - 2 LCS; similarity = LCS / indel^2
        unsigned long long indel = (unsigned long long)la + lb - 2ull * lcs;
        a.sim_out[pos] = __fdiv_rn(__uint2float_rn(lcs), __ull2float_rn(indel * indel));
    }
}

// ---- register path: every row of the launch fits one block of W words --------------------------
// Two rows per thread at once (NR = 2) while 2W words of V fit comfortably in registers: both rows
// see the same residue, so the address PRMT and the residue-stream loads are shared and the two
// carry chains are independent (more ILP per warp).
#ifndef FAMSA_NR_POLICY
#define FAMSA_NR_POLICY 2
#endif
__host__ __device__ constexpr int rows_per_thread(int w) {
#if FAMSA_NR_POLICY == 0
    return w <= 16 ? 2 : 1;
#elif FAMSA_NR_POLICY == 1
    return w <= 6 ? 4 : (w <= 10 ? 3 : (w <= 16 ? 2 : 1));
#elif FAMSA_NR_POLICY == 2
    return w <= 8 ? 3 : (w <= 16 ? 2 : 1);
#elif FAMSA_NR_POLICY == 3
    return w <= 4 ? 4 : (w <= 7 ? 3 : (w <= 20 ? 2 : 1));
#else
    return 1;
#endif
}

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

template <int W>
__global__ void __launch_bounds__(TB) sweep_short_kernel(const SweepArgs a) {
    extern __shared__ __align__(256) uint8_t smem[];
    asm volatile("griddepcontrol.launch_dependents;");
    constexpr int WST = (W + 1) & ~1;
    constexpr int TS = WST * ROW_BYTES;                  // bytes between the tables of consecutive rows
    constexpr int NR = rows_per_thread(W);
    const uint32_t col_tile = blockIdx.x % a.n_col_tiles, row_tile = blockIdx.x / a.n_col_tiles;
    const uint32_t r_lo = a.r0 + row_tile * a.ta;
    const uint32_t r_hi = min(r_lo + a.ta, a.r1);
    const uint32_t j0 = col_tile * TB;
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
#pragma unroll
        for (int p = 0; p < NR; ++p) {
            uint32_t lcs = 0;
#pragma unroll
            for (int w = 0; w < W; ++w) lcs += __popc(~V[p][w]);
            const uint32_t row = i + p;
            if (row < r_hi && j < row) store_pair(a, row, j, a.len[row], lb, lcs);
        }
    }
}

// ---- blocked path: rows of nblk blocks x W words; one row per CTA; carry bit-vector per thread --
template <int W, int CW>
__global__ void __launch_bounds__(TB) sweep_long_kernel(const SweepArgs a) {
    extern __shared__ __align__(256) uint8_t smem[];
    asm volatile("griddepcontrol.launch_dependents;");
    constexpr int WST = (W + 1) & ~1;
    const uint32_t col_tile = blockIdx.x % a.n_col_tiles, row_tile = blockIdx.x / a.n_col_tiles;
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
    if (active && j < i) store_pair(a, i, j, a.len[i], a.len[j], lcs);
}

}  // namespace famsa

// ---- host side: buckets -> launches ------------------------------------------------------------
namespace famsa {

// Launches after the first one of a famsa_lcs_rows call carry the programmatic-stream-serialization
// attribute: the launches of one call read the same read-only set and write disjoint output ranges,
// so the next bucket's CTAs may fill the SMs while the previous launch drains its last wave
// (every sweep kernel executes griddepcontrol.launch_dependents on entry; none needs .wait).
template <typename K>
static cudaError_t launch_sweep(K kernel, const SweepArgs& a, unsigned grid, size_t smem, cudaStream_t st, bool overlap) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid); cfg.blockDim = dim3(TB); cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = overlap ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kernel, a);
}
template <int W>
static cudaError_t launch_short(const SweepArgs& a, unsigned grid, size_t smem, cudaStream_t st, bool overlap) {
    return launch_sweep(sweep_short_kernel<W>, a, grid, smem, st, overlap);
}
template <int W, int CW>
static cudaError_t launch_long(const SweepArgs& a, unsigned grid, size_t smem, cudaStream_t st, bool overlap) {
    return launch_sweep(sweep_long_kernel<W, CW>, a, grid, smem, st, overlap);
}

#define SHORT_CASE(W) case W: return launch_short<W>(a, grid, smem, st, overlap);
static cudaError_t dispatch_short(int w, const SweepArgs& a, unsigned grid, size_t smem, cudaStream_t st, bool overlap) {
    switch (w) {
        SHORT_CASE(1) SHORT_CASE(2) SHORT_CASE(3) SHORT_CASE(4) SHORT_CASE(5) SHORT_CASE(6) SHORT_CASE(7) SHORT_CASE(8)
        SHORT_CASE(9) SHORT_CASE(10) SHORT_CASE(11) SHORT_CASE(12) SHORT_CASE(13) SHORT_CASE(14) SHORT_CASE(15) SHORT_CASE(16)
        SHORT_CASE(17) SHORT_CASE(18) SHORT_CASE(19) SHORT_CASE(20) SHORT_CASE(21) SHORT_CASE(22) SHORT_CASE(23) SHORT_CASE(24)
        SHORT_CASE(25) SHORT_CASE(26) SHORT_CASE(27) SHORT_CASE(28) SHORT_CASE(29) SHORT_CASE(30) SHORT_CASE(31) SHORT_CASE(32)
        default: return cudaErrorInvalidValue;
    }
}
#define LONG_CASE(W) case W: return launch_long<W, CW_SMALL>(a, grid, smem, st, overlap);
static cudaError_t dispatch_long(int w, bool large, const SweepArgs& a, unsigned grid, size_t smem, cudaStream_t st, bool overlap) {
    if (large) return w == 32 ? launch_long<32, CW_LARGE>(a, grid, smem, st, overlap) : cudaErrorInvalidValue;
    switch (w) {
        LONG_CASE(17) LONG_CASE(18) LONG_CASE(19) LONG_CASE(20) LONG_CASE(21) LONG_CASE(22) LONG_CASE(23) LONG_CASE(24)
        LONG_CASE(25) LONG_CASE(26) LONG_CASE(27) LONG_CASE(28) LONG_CASE(29) LONG_CASE(30) LONG_CASE(31) LONG_CASE(32)
        default: return cudaErrorInvalidValue;
    }
}

static uint32_t g_rows_per_cta = 2;     // TA; tunable through famsa_set_tuning (tests sweep it)

int sweep_rows(famsa_ctx* ctx, int64_t i0, int64_t i1, uint16_t* lcs, float* sim, cudaStream_t st) {
    SweepArgs a;
    a.stream = reinterpret_cast<const uint4*>(ctx->d_stream);
    a.goff = ctx->d_goff;
    a.tables = reinterpret_cast<const uint4*>(ctx->d_tables);
    a.toff = ctx->d_toff;
    a.len = ctx->d_len;
    a.lcs_out = lcs; a.sim_out = sim;
    a.out_base = i0 * (i0 - 1) / 2;
    int n_launched = 0;
    for (const Bucket& b : ctx->buckets) {
        int64_t lo = std::max(b.r0, std::max<int64_t>(i0, 1)), hi = std::min(b.r1, i1);   // row 0 is empty
        for (int64_t r = lo; r < hi; r += MAX_ROWS_PER_LAUNCH) {
            a.r0 = (uint32_t)r; a.r1 = (uint32_t)std::min<int64_t>(r + MAX_ROWS_PER_LAUNCH, hi);
            a.nblk = (uint32_t)b.nblk;
            a.n_col_tiles = (a.r1 - 1 + TB - 1) / TB;                // columns 0 .. r1-2
            const int wst = (b.wb + 1) & ~1;
            cudaError_t e;
            if (b.nblk == 1) {
                const uint32_t nr = (uint32_t)rows_per_thread(b.wb);
                a.ta = ((g_rows_per_cta + nr - 1) / nr) * nr;       // a whole number of NR-row steps per CTA
                while (a.ta > nr && (size_t)(a.ta + nr - 1) * wst * ROW_BYTES + 16 > 48 * 1024) a.ta -= nr;   // default dynamic smem limit
                unsigned row_tiles = (a.r1 - a.r0 + a.ta - 1) / a.ta;
                e = dispatch_short(b.wb, a, row_tiles * a.n_col_tiles, (size_t)(a.ta + nr - 1) * wst * ROW_BYTES + 16, st, n_launched > 0);
            } else {
                a.ta = 1;
                e = dispatch_long(b.wb, ctx->large_cw, a, (a.r1 - a.r0) * a.n_col_tiles, (size_t)wst * ROW_BYTES + 16, st, n_launched > 0);
            }
            if (e != cudaSuccess) return cuda_fail(e, "sweep kernel launch");
            ctx->launches++; ++n_launched;
        }
    }
    return FAMSA_OK;
}

}  // namespace famsa

using namespace famsa;

extern "C" int famsa_set_tuning(int rows_per_cta) {
    if (rows_per_cta < 1 || rows_per_cta > 12) { set_error("famsa_set_tuning: rows_per_cta must be 1..12"); return FAMSA_EINVAL; }
    g_rows_per_cta = (uint32_t)rows_per_cta;
    return FAMSA_OK;
}

extern "C" int famsa_lcs_rows(famsa_ctx* ctx, int64_t i0, int64_t i1, uint16_t* lcs_out, float* sim_out,
                              void* cuda_stream) {
    if (!ctx) { set_error("famsa_lcs_rows: ctx is NULL"); return FAMSA_EINVAL; }
    if (i0 < 0 || i0 > i1 || i1 > ctx->k) { set_error("famsa_lcs_rows: bad row range"); return FAMSA_ERANGE; }
    if (!lcs_out && !sim_out) { set_error("famsa_lcs_rows: both outputs are NULL"); return FAMSA_EINVAL; }
    if (famsa_rows_pairs(i0, i1) == 0) return FAMSA_OK;
    FAMSA_CUDA(cudaSetDevice(ctx->device));
    return sweep_rows(ctx, i0, i1, lcs_out, sim_out, (cudaStream_t)cuda_stream);
}

static int rows_host_impl(famsa_ctx* ctx, int64_t i0, int64_t i1, uint16_t* lcs_host, float* sim_host, bool wait) {
    if (!ctx) { set_error("famsa_lcs_rows_host: ctx is NULL"); return FAMSA_EINVAL; }
    if (i0 < 0 || i0 > i1 || i1 > ctx->k) { set_error("famsa_lcs_rows_host: bad row range"); return FAMSA_ERANGE; }
    if (!lcs_host && !sim_host) { set_error("famsa_lcs_rows_host: both outputs are NULL"); return FAMSA_EINVAL; }
    if (famsa_rows_pairs(i0, i1) == 0) return FAMSA_OK;
    FAMSA_CUDA(cudaSetDevice(ctx->device));
    // lazily create the ping-pong staging (two staging buffers of 1 Mi .. 128 Mi pairs each)
    // chunk size: about 1/8 of the call (so the copy of chunk n overlaps the sweep of chunk n+1),
    // between 1 Mi and 128 Mi pairs, and never smaller than the longest row
    const int64_t total_pairs = famsa_rows_pairs(i0, i1);
    const int64_t chunk_pairs = std::max<int64_t>(std::min<int64_t>(std::max<int64_t>(total_pairs / 8, (int64_t)1 << 20), (int64_t)128 << 20), i1);
    const size_t want = (size_t)std::min<int64_t>(total_pairs, chunk_pairs);
    if (!ctx->s_compute) {
        FAMSA_CUDA(cudaStreamCreateWithFlags(&ctx->s_compute, cudaStreamNonBlocking));
        FAMSA_CUDA(cudaStreamCreateWithFlags(&ctx->s_copy, cudaStreamNonBlocking));
        for (int b = 0; b < 2; ++b) {
            FAMSA_CUDA(cudaEventCreateWithFlags(&ctx->ev_done[b], cudaEventDisableTiming));
            FAMSA_CUDA(cudaEventCreateWithFlags(&ctx->ev_copied[b], cudaEventDisableTiming));
        }
    }
    if (ctx->buf_pairs < want) {
        // size the staging once per ctx (1/8 of the whole triangle, 1 Mi .. 128 Mi pairs, at least one row),
        // so that a stream of growing row-block calls does not reallocate it
        const int64_t tri = ctx->k * (ctx->k - 1) / 2;
        const size_t cap = (size_t)std::max<int64_t>(std::max<int64_t>(std::min<int64_t>(std::max<int64_t>(tri / 8, (int64_t)1 << 20), (int64_t)128 << 20), ctx->k), (int64_t)want);
        FAMSA_CUDA(cudaDeviceSynchronize());
        for (int b = 0; b < 2; ++b) {
            cudaFree(ctx->d_lcs_buf[b]); cudaFree(ctx->d_sim_buf[b]);
            ctx->d_lcs_buf[b] = nullptr; ctx->d_sim_buf[b] = nullptr;
        }
        ctx->buf_pairs = 0;
        for (int b = 0; b < 2; ++b) {
            cudaError_t e1 = cudaMalloc((void**)&ctx->d_lcs_buf[b], cap * sizeof(uint16_t));
            cudaError_t e2 = cudaMalloc((void**)&ctx->d_sim_buf[b], cap * sizeof(float));
            if (e1 != cudaSuccess || e2 != cudaSuccess) {
                cudaGetLastError(); set_error("famsa_lcs_rows_host: device allocation failed"); return FAMSA_ENOMEM;
            }
        }
        ctx->buf_pairs = cap;
    }
    // chunk the row range so that each chunk fits a buffer (a single row always fits: i < 2^32 / ... k <= buf)
    int64_t r = i0; int64_t done_pairs = 0;
    int64_t& n = ctx->host_chunks;                         // chunks enqueued so far by this ctx: the ping-pong continues across calls
    while (r < i1) {
        int64_t e = r + 1;
        while (e < i1 && famsa_rows_pairs(r, e + 1) <= (int64_t)want) ++e;
        const int64_t np = famsa_rows_pairs(r, e);
        if (np > (int64_t)ctx->buf_pairs) { set_error("famsa_lcs_rows_host: a single row exceeds the staging buffer"); return FAMSA_ENOMEM; }
        const int b = (int)(n & 1);
        if (n >= 2) FAMSA_CUDA(cudaStreamWaitEvent(ctx->s_compute, ctx->ev_copied[b], 0));
        int rc = sweep_rows(ctx, r, e, lcs_host ? ctx->d_lcs_buf[b] : nullptr, sim_host ? ctx->d_sim_buf[b] : nullptr, ctx->s_compute);
        if (rc != FAMSA_OK) return rc;
        FAMSA_CUDA(cudaEventRecord(ctx->ev_done[b], ctx->s_compute));
        FAMSA_CUDA(cudaStreamWaitEvent(ctx->s_copy, ctx->ev_done[b], 0));
        if (lcs_host) FAMSA_CUDA(cudaMemcpyAsync(lcs_host + done_pairs, ctx->d_lcs_buf[b], np * sizeof(uint16_t), cudaMemcpyDeviceToHost, ctx->s_copy));
        if (sim_host) FAMSA_CUDA(cudaMemcpyAsync(sim_host + done_pairs, ctx->d_sim_buf[b], np * sizeof(float), cudaMemcpyDeviceToHost, ctx->s_copy));
        FAMSA_CUDA(cudaEventRecord(ctx->ev_copied[b], ctx->s_copy));
        done_pairs += np; r = e; ++n;
    }
    if (wait) {
        FAMSA_CUDA(cudaStreamSynchronize(ctx->s_copy));
        FAMSA_CUDA(cudaStreamSynchronize(ctx->s_compute));
    }
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
    if (ctx->s_copy) FAMSA_CUDA(cudaStreamSynchronize(ctx->s_copy));
    if (ctx->s_compute) FAMSA_CUDA(cudaStreamSynchronize(ctx->s_compute));
    return FAMSA_OK;
}
