// famsa_internal.h -- shared between the translation units of libfamsa_lcs.so (CUDA path only;
// nothing under oracle/ includes this).  Device data layout of a packed sequence set.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <atomic>
#include <deque>
#include <mutex>
#include <string>
#include <vector>

#include "famsa_lcs.h"

namespace famsa {

// ---- layout constants ---------------------------------------------------------------------
// Residue stream ("B side"): sorted sequences in groups of 32 (one group = the 32 lanes of a
// warp), 16-byte chunks interleaved by lane: byte p of lane l of group g sits at
//     stream[(goff[g] + p/16) * 512 + l*16 + p%16].
// Each byte is code*4 (the byte offset of the symbol inside a 128-byte table row); positions
// past the end of a sequence hold PAD_BYTE, whose table row (symbol 31) is all-zero, so a pad
// residue leaves V unchanged.
constexpr int      GROUP      = 32;
constexpr int      CHUNK      = 16;
constexpr uint8_t  PAD_BYTE   = 31 * 4;
// Match tables ("A side"): per sequence, words x 32 symbols, layout [word][symbol] uint32, so a
// warp reading one word for 32 different residues touches one 128-byte row (bank = symbol).
// A sequence of Ws = ceil(len/32) words is cut into nblk blocks of Wb <= 32 words; each block is
// stored with an even word stride Wst so every block base is 256-byte aligned.
constexpr int      SYMS       = 32;
constexpr int      ROW_BYTES  = SYMS * 4;       // 128
constexpr int      MAX_WB     = 32;             // V words held in registers per thread
constexpr int      CW_SMALL   = 128;            // carry-vector words (long path), |B| <= 4096
constexpr int      CW_LARGE   = 2048;           // |B| <= 65535

struct BlockPlan { int nblk; int wb; int wst; };   // wst = wb rounded up to even

inline BlockPlan plan_blocks(uint32_t len, bool force32) {
    int ws = (int)((len + 31) / 32);
    BlockPlan p;
    p.nblk = (ws + MAX_WB - 1) / MAX_WB;
    p.wb = (p.nblk > 1 && force32) ? MAX_WB : (ws + p.nblk - 1) / p.nblk;
    p.wst = (p.wb + 1) & ~1;
    return p;
}

struct Bucket { int64_t r0, r1; int nblk, wb; };   // rows [r0, r1) share one kernel variant

constexpr uint32_t DEFAULT_ROWS_PER_CTA = 2;       // TA on the register path (famsa_ctx_set_tuning)
constexpr uint32_t DEFAULT_L2_GROUP_MB  = 24;      // residue-stream slice one column group of a launch re-reads from L2

// Staging of the HOST-output path (famsa_lcs_rows_host*): two device row-chunk buffers, two streams and the
// events that order them; pooled per process (famsa_sweep.cu).
struct HostChunkTimers { cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr}; double bytes = 0.0; };   // sweep start/end, copy start/end
struct Staging {
    int       device = 0;
    size_t    pairs = 0;                            // capacity of each buffer, in pairs
    uint16_t* lcs[2] = {nullptr, nullptr};
    float*    sim[2] = {nullptr, nullptr};
    cudaStream_t s_compute = nullptr, s_copy = nullptr;
    cudaEvent_t  ev_done[2] = {nullptr, nullptr}, ev_copied[2] = {nullptr, nullptr};
    bool      profile = false;                      // famsa_host_profile: time every chunk's sweep and copy
    std::deque<HostChunkTimers> timers;
};

}  // namespace famsa

struct famsa_ctx {
    int      device = 0;
    int      sm_count = 0;
    int64_t  k = 0;
    int64_t  n_groups = 0;
    uint32_t max_len = 0;
    bool     large_cw = false;                  // some sequence longer than 4096
    // host copies
    std::vector<int64_t>  perm;                 // perm[sorted] = original
    std::vector<uint32_t> len;                  // sorted order
    std::vector<uint32_t> toff;                 // table offset of sorted sequence s, in 128-byte rows
    std::vector<uint32_t> goff;                 // n_groups+1: stream offset of group g, in 512-byte units
    std::vector<double>   len_prefix;           // k+1: sum of len[0..s)
    std::vector<famsa::Bucket> buckets;
    // device
    uint8_t*  d_stream = nullptr;  size_t stream_bytes = 0;
    uint32_t* d_tables = nullptr;  size_t table_bytes = 0;
    uint32_t* d_len = nullptr;
    uint32_t* d_toff = nullptr;
    uint32_t* d_goff = nullptr;
    // row-block staging of famsa_lcs_rows_host* (acquired lazily from the process-wide pool)
    famsa::Staging* stg = nullptr;
    int64_t   host_chunks = 0;                  // chunks enqueued by the host path so far
    bool      host_profile = false;
    // direct host path: PINNED host outputs are written by the sweep kernels themselves (their device alias,
    // posted PCIe writes), on this stream; no staging, no copy engine, no chunking
    cudaStream_t s_direct = nullptr;
    std::atomic<int> host_mode{-1};             // famsa_host_mode: -1 auto (direct if every output is pinned), 0 staged, 1 direct or fail
    std::deque<famsa::HostChunkTimers> direct_timers;
    // tuning (famsa_ctx_set_tuning): per ctx, so concurrent calls on other ctxs / streams are unaffected
    std::atomic<uint32_t> rows_per_cta{famsa::DEFAULT_ROWS_PER_CTA};
    std::atomic<int>      small_mode{-1};       // -1 auto, 0 never, 1 always: one-warp CTAs, one pair per thread
    std::atomic<uint32_t> l2_group_mb{famsa::DEFAULT_L2_GROUP_MB};
    double    pack_ms[4] = {0, 0, 0, 0};        // famsa_pack_profile: H2D + encode, sort, host plan, stream + table build
    std::atomic<int64_t> launches{0};
};

namespace famsa {
// Round-0 candidates of the guide tree (famsa_tree.cu), accumulated by the sweep's epilogue when given:
// row[i] = max over the row's entries of key(similarity, column), col[j] = max over the call's rows of
// key(similarity, row); key = (fp32 bits + 1) << 32 | ~other, so a 64-bit atomicMax picks the higher
// similarity and then the smaller `other`.  The caller zeroes both before the call.
struct TreeCand { unsigned long long* row; unsigned long long* col; };
void set_error(const std::string& msg);
int  cuda_fail(cudaError_t e, const char* what);          // records text, returns FAMSA_ECUDA
int  sweep_rows(famsa_ctx* ctx, int64_t i0, int64_t i1, uint16_t* lcs, float* sim, unsigned long long* checksum, const TreeCand* cand, cudaStream_t st);
void staging_release(Staging* s);                          // back to the pool (drains its streams first)
cudaError_t cache_alloc(int device, void** p, size_t bytes);   // device block cache of famsa_pack / famsa_free (famsa_pack.cu)
void cache_free(void* p);
void cache_trim();
}  // namespace famsa

#define FAMSA_CUDA(call)                                                     \
    do {                                                                     \
        cudaError_t e__ = (call);                                            \
        if (e__ != cudaSuccess) return famsa::cuda_fail(e__, #call);         \
    } while (0)
