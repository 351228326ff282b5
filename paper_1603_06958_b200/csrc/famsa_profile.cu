// famsa_profile.cu -- SURVEY.md 8(f) NEXT-4: sequence-versus-profile dynamic programming of FAMSA's stage III
// (PAPER.md:71-79, 107, 111-116, 133-139).  Boundary and the readings of the paper: include/famsa_profile.h,
// DESIGN.md P1-P9.
//
// Mapping: one warp per alignment (two alignments per warp, 16 lanes each, for sequences of <= 256 residues).  The
// SEQUENCE side (n2 <= 1024 residues) is spread over the lanes, J = 4, 8, ... 32 consecutive residues per lane, and for each of them the lane keeps the three states of the
// previous profile column (row) in registers: 3 J floats.  The rows are swept in a skewed wavefront: at step t
// lane l computes row t - l + 1, so what it needs from the left -- the three states of lane l-1's last residue
// in the same row -- was produced one step earlier and arrives by one __shfl_up per state; the value received
// for the previous row is kept as the diagonal.  Per cell: one shared-memory load of cost[row][residue] (the rows
// stream through a per-warp ring, one coalesced global load per step) and ~25 fp32 adds / compares / selects, one
// direction byte (2 bits per state).  All arithmetic is fp32 adds,
// subtractions and comparisons in the order the oracle's fp32 mode uses (products of nseq and a gap cost are
// formed once with __fmul_rn, nothing can contract into an FMA), so scores AND traceback decisions are
// bit-identical to it.  A second kernel (one warp per alignment, tile by tile) walks the direction bytes back.
// (Tried, r02: loading the lane's cost values one row ahead -- +16 registers at J = 16 -- was 1 % slower.)
// (Tried, r02: J in steps of 2 instead of 4 -- half the idle lane slots, but 16-bit direction stores for J = 2 mod 4
//  and twice as many, smaller launches: 245 against 262 GCUPS at 8192 alignments, 304 against 320 at 32768.)
#include <algorithm>
#include <cmath>
#include <mutex>
#include <vector>

#include "famsa_internal.h"
#include "famsa_profile.h"

namespace famsa {

constexpr float NEG = -3.0e38f;
constexpr int RING_STRIDE = 33;                              // per-alignment ring of cost rows in shared memory: 2 SEG rows of 33 floats
constexpr size_t RING_BYTES = 4 * 64 * RING_STRIDE * sizeof(float);   // 4 warps per CTA x (32 / SEG) alignments x 2 SEG rows
#ifndef SEQPROF_SEG16_MAX
#define SEQPROF_SEG16_MAX 256                                // sequences up to this length take 16 lanes (two alignments per warp);
                                                             // measured r02: 256 -> +7-8 % on batches of short sequences, 512 -> -20 % (J >= 20: 255 registers)
#endif

struct AlignDesc {
    int64_t cost_row0;       // first cost row of the profile
    int64_t seq0;            // first residue of the sequence
    int64_t dir0;            // byte offset of the direction bytes in the workspace (n1 + seg - 1 skewed rows of seg x J bytes)
    int64_t path_end;        // end of the path segment
    int32_t n1, n2, idx;     // columns, residues, index in the batch
    int16_t j, seg;          // residues per lane, lanes per alignment (32, or 16: two alignments share a warp)
};

__global__ void profile_costs_kernel(const uint32_t* __restrict__ counts, const float* __restrict__ subst, int64_t n_cols, float* __restrict__ cost) {
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n_cols * SYMS) return;
    const int64_t i = t / SYMS; const int c = (int)(t % SYMS);
    double s = 0.0;
#pragma unroll 8
    for (int d = 0; d < SYMS; ++d) s = __dadd_rn(s, __dmul_rn((double)counts[i * SYMS + d], (double)subst[d * SYMS + c]));
    cost[t] = (float)s;
}

template <int J, int SEG>
__global__ void __launch_bounds__(128) seqprof_kernel(const AlignDesc* __restrict__ desc, int n, const float* __restrict__ cost,
                                                      const uint8_t* __restrict__ seq, const float* __restrict__ gaps,
                                                      const int32_t* __restrict__ nseq, float* __restrict__ score,
                                                      uint8_t* __restrict__ final_state, uint8_t* __restrict__ ws, int want_dir) {
    // The residues-per-lane groups of one batch are launched back to back as programmatic dependents: a group
    // rarely fills the GPU (a batch of 8192 alignments splits into 8 groups), so the next group's CTAs start as soon
    // as this group's are all resident.  The groups are independent (disjoint outputs); every working warp ends with
    // griddepcontrol.wait, so a group cannot complete before its predecessor and the traceback kernel -- an
    // ordinary launch after the last group -- sees all of them.
    asm volatile("griddepcontrol.launch_dependents;");
    // SEG lanes per alignment: 32 (one alignment per warp) or 16 (two: short sequences would leave lanes idle and pay the
    // full 31-step skew; with 16 lanes the same registers hold twice the residues per lane, which also gives each lane
    // more independent work per step).  An idle second segment runs with n1 = 0: it takes part in the warp's shuffles
    // and barriers and never computes or stores.
    constexpr int APW = 32 / SEG, RROWS = 2 * SEG;
    const int warp = (int)((blockIdx.x * blockDim.x + threadIdx.x) >> 5), lane = threadIdx.x & 31;
    const int sl = lane & (SEG - 1), seg = lane / SEG;
    if (warp * APW >= n) return;
    const bool valid = warp * APW + seg < n;
    const AlignDesc d = desc[valid ? warp * APW + seg : n - 1];
    const int n1 = valid ? d.n1 : 0, n2 = d.n2, b = d.idx;
    const float To = gaps[4 * b], Te = gaps[4 * b + 1], Go = gaps[4 * b + 2], Ge = gaps[4 * b + 3];
    const float ns = (float)nseq[b];
    const float nTo = __fmul_rn(ns, To), nTe = __fmul_rn(ns, Te), nGo = __fmul_rn(ns, Go), nGe = __fmul_rn(ns, Ge);
    const int j0 = sl * J;                                   // this lane owns residues j0+1 .. j0+J (1-based)
    uint32_t yw[J / 4];                                      // their codes, 4 per word (code*4 = byte offset in a cost row)
#pragma unroll
    for (int q = 0; q < J / 4; ++q) {
        uint32_t w = 0;
#pragma unroll
        for (int r = 0; r < 4; ++r) { const int jj = j0 + 4 * q + r; w |= (uint32_t)(jj < n2 ? seq[d.seq0 + jj] : 0) << (8 * r); }
        yw[q] = w;
    }
    // row 0: residues before the first column are terminal gap columns, Y[0][j] = Y[0][j-1] - nseq T_e
    float yrun = 0.0f;
    for (int j = 1; j <= j0; ++j) yrun = j == 1 ? 0.0f - nTo : yrun - nTe;
    float dM = sl == 0 ? 0.0f : NEG, dX = NEG, dY = sl == 0 ? NEG : yrun;         // row 0 at residue j0: the first diagonal
    float Mp[J], Xp[J], Yp[J];
#pragma unroll
    for (int c = 0; c < J; ++c) { yrun = (j0 + c + 1) == 1 ? 0.0f - nTo : yrun - nTe; Mp[c] = NEG; Xp[c] = NEG; Yp[c] = yrun; }
    float x0 = 0.0f;                                         // lane 0: X[i][0], columns before the first residue
    float rM = NEG, rX = NEG, rY = NEG;                      // the row this lane finished last, at its last residue
    const float* crow = cost + d.cost_row0 * SYMS;
    // Cost rows go through a per-warp ring in shared memory: at one step the 32 lanes work on 32 DIFFERENT profile
    // columns, so a direct load of cost[column][residue] touches 32 cache lines per instruction and the L1 pipeline
    // -- not the ALU -- sets the pace (measured r02: 2.5 of 3 warps per scheduler waiting on the long scoreboard).
    // Instead the warp loads ONE new row per step with a single coalesced 128-byte load and the lanes read their
    // values from the ring; rows are 33 words apart, so the bank of (row r, symbol c) is (r + c) mod 32 and lanes on
    // different rows with the same residue do not collide systematically.
    extern __shared__ float ring_all[];
    float* ring = ring_all + ((threadIdx.x >> 5) * APW + seg) * (RROWS * RING_STRIDE);
#pragma unroll
    for (int q = 0; q < APW; ++q) ring[sl + q * SEG] = crow[sl + q * SEG];      // row 0 (every profile has one)
    __syncwarp();
    uint8_t* dir = ws + d.dir0;
    const int stride = SEG * J;
    int steps = n1 + SEG - 1;
    if (APW > 1) steps = max(steps, __shfl_xor_sync(0xffffffffu, steps, SEG));   // warp-uniform: the longer of the two profiles
    for (int t = 0; t < steps; ++t) {
        const int i = t - sl + 1;
        float next_row[APW];                                 // cost row t+1, used from the next step on
#pragma unroll
        for (int q = 0; q < APW; ++q) next_row[q] = t + 1 < n1 ? __ldg(crow + (size_t)(t + 1) * SYMS + sl + q * SEG) : 0.0f;
        float lM = __shfl_up_sync(0xffffffffu, rM, 1, SEG), lX = __shfl_up_sync(0xffffffffu, rX, 1, SEG), lY = __shfl_up_sync(0xffffffffu, rY, 1, SEG);
        if (i >= 1 && i <= n1) {
        if (sl == 0) { x0 = i == 1 ? 0.0f - To : x0 - Te; lM = NEG; lX = x0; lY = NEG; }
        const float goy = i == n1 ? nTo : nGo, gey = i == n1 ? nTe : nGe;
        const float* ci = ring + ((i - 1) & (RROWS - 1)) * RING_STRIDE;
        float cM = dM, cX = dX, cY = dY;                     // diagonal of the lane's first residue
        dM = lM; dX = lX; dY = lY;                           // ... and the next row's
        uint32_t dw[J / 4];
#pragma unroll
        for (int q = 0; q < J / 4; ++q) dw[q] = 0;
#pragma unroll
        for (int c = 0; c < J; ++c) {
            const int j = j0 + c + 1;
            const float gox = j == n2 ? To : Go, gex = j == n2 ? Te : Ge;
            const uint32_t code = (yw[c >> 2] >> (8 * (c & 3))) & 0xFFu;
            float bst = cM, v; uint32_t from = 0, dd;
            if (cX > bst) { bst = cX; from = 1; }
            if (cY > bst) { bst = cY; from = 2; }
            const float m = bst + ci[code]; dd = from;
            bst = Mp[c] - gox; from = 0;
            v = Xp[c] - gex; if (v > bst) { bst = v; from = 1; }
            v = Yp[c] - gox; if (v > bst) { bst = v; from = 2; }
            const float x = bst; dd |= from << 2;
            bst = lM - goy; from = 0;
            v = lX - goy; if (v > bst) { bst = v; from = 1; }
            v = lY - gey; if (v > bst) { bst = v; from = 2; }
            const float y = bst; dd |= from << 4;
            cM = Mp[c]; cX = Xp[c]; cY = Yp[c];
            Mp[c] = m; Xp[c] = x; Yp[c] = y;
            lM = m; lX = x; lY = y;
            dw[c >> 2] |= dd << (8 * (c & 3));
            if (i == n1 && j == n2) {                        // the end cell: score and the state the walk starts in
                float best = m; uint32_t st = 0;
                if (x > best) { best = x; st = 1; }
                if (y > best) { best = y; st = 2; }
                score[b] = best; final_state[b] = (uint8_t)st;
            }
        }
        rM = lM; rX = lX; rY = lY;
        // Direction bytes in a SKEWED layout: the bytes of (row i, lane l) go to workspace row t = i - 1 + l, so that
        // at one step all lanes of the alignment write into the same SEG x J-byte row (coalesced) instead of SEG different rows.
        if (want_dir) {
            uint8_t* out = dir + (size_t)t * stride + j0;
            if (J % 16 == 0) {
#pragma unroll
                for (int q = 0; q < J / 16; ++q) reinterpret_cast<uint4*>(out)[q] = make_uint4(dw[4 * q], dw[4 * q + 1], dw[4 * q + 2], dw[4 * q + 3]);
            } else if (J % 8 == 0) {
#pragma unroll
                for (int q = 0; q < J / 8; ++q) reinterpret_cast<uint2*>(out)[q] = make_uint2(dw[2 * q], dw[2 * q + 1]);
            } else {
#pragma unroll
                for (int q = 0; q < J / 4; ++q) reinterpret_cast<uint32_t*>(out)[q] = dw[q];
            }
        }
        }
#pragma unroll
        for (int q = 0; q < APW; ++q)                        // the slot's old row (t + 1 - 2 SEG) was last read at step t - SEG
            ring[((t + 1) & (RROWS - 1)) * RING_STRIDE + sl + q * SEG] = next_row[q];
        __syncwarp();
    }
    asm volatile("griddepcontrol.wait;" ::: "memory");
}

// Traceback: one WARP per alignment walks the direction bytes from (n1, n2) back to (0, 0); the operations are written
// right-aligned into the alignment's path segment.  The walk itself is a dependent chain (one thread), but its memory
// latency is not: the warp first loads the 32 x 32-cell tile of direction bytes whose lower right corner is the current
// cell (lane l: DP row i - l, eight aligned 32-bit words; a word never straddles a lane block of the skewed layout
// because J is a multiple of 4), lane 0 then walks inside the tile out of shared memory (at least 32, at most 63 steps),
// and the warp writes that stretch of the path out together.  One thread per alignment with a global load per step took
// 0.65 ms for 8192 alignments (long scoreboard: 19 warps per issue); see DESIGN.md 6.8 for the number now.
constexpr int TRACE_T = 32;
__global__ void __launch_bounds__(128) seqprof_trace_kernel(const AlignDesc* __restrict__ desc, int n, const uint8_t* __restrict__ final_state,
                                                            const uint8_t* __restrict__ ws, uint8_t* __restrict__ path, int32_t* __restrict__ path_len) {
    __shared__ uint32_t tile_all[4][TRACE_T][TRACE_T / 4 + 1];
    __shared__ uint8_t ops_all[4][2 * TRACE_T];
    const int warp = (int)((blockIdx.x * blockDim.x + threadIdx.x) >> 5), lane = threadIdx.x & 31;
    if (warp >= n) return;
    uint32_t (*tile)[TRACE_T / 4 + 1] = tile_all[threadIdx.x >> 5];
    uint8_t* ops = ops_all[threadIdx.x >> 5];
    const AlignDesc d = desc[warp];
    const uint8_t* dir = ws + d.dir0;
    const int stride = d.seg * d.j, J = d.j;
    int i = d.n1, j = d.n2, len = 0;
    uint32_t st = final_state[d.idx];
    uint8_t* out = path + d.path_end;                        // one past the next operation's place (the path is written backwards)
    while (i > 0 && j > 0) {                                 // warp-uniform: i, j, st are broadcast after every tile
        const int hi = ((j - 1) | 3) + 1, lo = max(0, hi - TRACE_T);      // zero-based columns [lo, hi), both multiples of 4
        const int ri = i - lane;                             // this lane's DP row
#pragma unroll
        for (int w = 0; w < TRACE_T / 4; ++w) {
            const int cz = lo + 4 * w;
            uint32_t v = 0;
            if (ri >= 1 && cz < hi) v = __ldg(reinterpret_cast<const uint32_t*>(dir + (size_t)(ri - 1 + cz / J) * stride + cz));
            tile[lane][w] = v;
        }
        __syncwarp();
        int steps = 0;
        if (lane == 0) {
            const int i_top = i;
            while (i > 0 && j > 0 && i_top - i < TRACE_T && j - 1 >= lo) {
                const uint32_t dd = (tile[i_top - i][(j - 1 - lo) >> 2] >> (8 * ((j - 1) & 3))) & 0xFFu;
                ops[steps++] = (uint8_t)st;
                if (st == 0) { st = dd & 3; --i; --j; }
                else if (st == 1) { st = (dd >> 2) & 3; --i; }
                else { st = (dd >> 4) & 3; --j; }
            }
        }
        __syncwarp();
        i = __shfl_sync(0xffffffffu, i, 0); j = __shfl_sync(0xffffffffu, j, 0);
        st = __shfl_sync(0xffffffffu, st, 0); steps = __shfl_sync(0xffffffffu, steps, 0);
        for (int q = lane; q < steps; q += 32) out[-1 - q] = ops[q];
        out -= steps; len += steps;
        __syncwarp();
    }
    if (lane == 0) {
        while (i > 0 || j > 0) {                             // along a border: runs of terminal gaps, no memory involved
            const uint32_t dd = i == 0 ? (j == 1 ? 0u : 2u) << 4 : (i == 1 ? 0u : 1u) << 2;
            *--out = (uint8_t)st; ++len;
            if (st == 0) { st = dd & 3; --i; --j; }
            else if (st == 1) { st = (dd >> 2) & 3; --i; }
            else { st = (dd >> 4) & 3; --j; }
        }
        path_len[d.idx] = len;
    }
}

// Pinned staging for the descriptors of a call: two buffers used alternately, each guarded by an event recorded
// after its copy, so that a call neither synchronises the stream (a cudaMemcpyAsync from pageable memory would) nor
// waits for more than the call before the previous one: consecutive batches overlap host preparation with the GPU.
struct DescStage { AlignDesc* p = nullptr; size_t cap = 0; cudaEvent_t ev = nullptr; bool used = false; };
static std::mutex g_desc_mu;
static DescStage g_desc[2];
static int g_desc_next = 0;

// lanes per alignment and residues per lane (a multiple of 4 with seg x J >= n2)
struct Shape { int seg, j; };
static Shape shape_of(int64_t n2) {
    if (n2 <= SEQPROF_SEG16_MAX) return Shape{16, (int)(4 * ((n2 + 63) / 64))};
    return Shape{32, (int)(4 * ((n2 + 127) / 128))};
}
static int64_t dir_bytes_of(int64_t n1, Shape sh) { return (n1 + sh.seg - 1) * sh.seg * sh.j; }
static int shape_class(Shape sh) { return (sh.seg == 32 ? 0 : 8) + 8 - sh.j / 4; }     // 16 classes; within a seg: heaviest J first

// One (seg, J) group of a batch: n alignments whose descriptors are consecutive.  Launched as a programmatic dependent of
// whatever precedes it in the stream (see seqprof_kernel).
static cudaError_t launch_seqprof_group(int seg, int j, const AlignDesc* d_desc, int n, const float* cost_dev, const uint8_t* seq_dev,
                                        const float* gaps_dev, const int32_t* nseq_dev, float* score_dev, uint8_t* final_state,
                                        uint8_t* ws, int want_dir, cudaStream_t st) {
    const int per_cta = 4 * (32 / seg);                      // 4 warps x alignments per warp
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)((n + per_cta - 1) / per_cta)); cfg.blockDim = dim3(128); cfg.dynamicSmemBytes = RING_BYTES; cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
#define SEQPROF_CASE(JJ) case JJ: return seg == 32 \
        ? cudaLaunchKernelEx(&cfg, seqprof_kernel<JJ, 32>, d_desc, n, cost_dev, seq_dev, gaps_dev, nseq_dev, score_dev, final_state, ws, want_dir) \
        : cudaLaunchKernelEx(&cfg, seqprof_kernel<JJ, 16>, d_desc, n, cost_dev, seq_dev, gaps_dev, nseq_dev, score_dev, final_state, ws, want_dir);
    switch (j) {
        SEQPROF_CASE(4) SEQPROF_CASE(8) SEQPROF_CASE(12) SEQPROF_CASE(16) SEQPROF_CASE(20) SEQPROF_CASE(24) SEQPROF_CASE(28) SEQPROF_CASE(32)
        default: return cudaErrorInvalidValue;
    }
#undef SEQPROF_CASE
}

}  // namespace famsa

using namespace famsa;

extern "C" double famsa_gap_scale(double k, double g_l, double g_d) { return 1.0 + std::log(k / g_l) / g_d; }

extern "C" int famsa_profile_costs(const uint32_t* counts_dev, const float* subst_dev, int64_t n_cols, float* cost_dev, void* cuda_stream) {
    if (n_cols < 0 || (n_cols > 0 && (!counts_dev || !subst_dev || !cost_dev))) { set_error("famsa_profile_costs: null pointer or n_cols < 0"); return FAMSA_EINVAL; }
    if (n_cols == 0) return FAMSA_OK;
    profile_costs_kernel<<<(unsigned)((n_cols * SYMS + 255) / 256), 256, 0, (cudaStream_t)cuda_stream>>>(counts_dev, subst_dev, n_cols, cost_dev);
    FAMSA_CUDA(cudaGetLastError());
    return FAMSA_OK;
}

static int seqprof_check(const int64_t* col_off, const int64_t* seq_off, int64_t n, const char* who) {
    if (n < 0 || !col_off || !seq_off) { set_error(std::string(who) + ": null offsets or n_align < 0"); return FAMSA_EINVAL; }
    if (col_off[0] < 0 || seq_off[0] < 0) { set_error(std::string(who) + ": negative offset"); return FAMSA_EINVAL; }
    for (int64_t b = 0; b < n; ++b) {
        const int64_t n1 = col_off[b + 1] - col_off[b], n2 = seq_off[b + 1] - seq_off[b];
        if (n1 < 1 || n2 < 1 || n2 > FAMSA_SEQPROF_MAX_SEQ || n1 > 0x7FFFFFF0LL) {
            set_error(std::string(who) + ": alignment " + std::to_string(b) + " has an empty profile, an empty sequence or more than " +
                      std::to_string(FAMSA_SEQPROF_MAX_SEQ) + " residues");
            return FAMSA_ELENGTH;
        }
    }
    return FAMSA_OK;
}

extern "C" int64_t famsa_seqprof_workspace(const int64_t* col_off_host, const int64_t* seq_off_host, int64_t n_align) {
    if (seqprof_check(col_off_host, seq_off_host, n_align, "famsa_seqprof_workspace") != FAMSA_OK) return -1;
    int64_t bytes = 0;
    for (int64_t b = 0; b < n_align; ++b)
        bytes += dir_bytes_of(col_off_host[b + 1] - col_off_host[b], shape_of(seq_off_host[b + 1] - seq_off_host[b]));
    return bytes + n_align;                                  // + one final-state byte per alignment
}

extern "C" int famsa_seqprof_align(const float* cost_dev, const int64_t* col_off_host, const uint8_t* seq_dev,
                                   const int64_t* seq_off_host, const float* gaps_dev, const int32_t* nseq_dev, int64_t n_align,
                                   float* score_dev, uint8_t* path_dev, int32_t* path_len_dev, void* workspace_dev, void* cuda_stream) {
    int rc = seqprof_check(col_off_host, seq_off_host, n_align, "famsa_seqprof_align");
    if (rc != FAMSA_OK) return rc;
    if (n_align == 0) return FAMSA_OK;
    if (n_align > 0x7FFFFFF0LL) { set_error("famsa_seqprof_align: too many alignments"); return FAMSA_EINVAL; }
    if (!cost_dev || !seq_dev || !gaps_dev || !nseq_dev || !score_dev || (path_dev && (!path_len_dev || !workspace_dev))) {
        set_error("famsa_seqprof_align: null pointer (path_dev needs path_len_dev and workspace_dev)"); return FAMSA_EINVAL;
    }
    if (reinterpret_cast<uintptr_t>(workspace_dev) & 15) { set_error("famsa_seqprof_align: workspace_dev must be 16-byte aligned"); return FAMSA_EINVAL; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    // descriptors, grouped by residues-per-lane variant (longest profiles first inside a group: the heavy warps start first)
    std::vector<AlignDesc> desc((size_t)n_align);
    std::vector<int64_t> order((size_t)n_align);
    int64_t dir_bytes = 0;
    for (int64_t b = 0; b < n_align; ++b) {
        AlignDesc& d = desc[(size_t)b];
        d.cost_row0 = col_off_host[b]; d.seq0 = seq_off_host[b];
        d.n1 = (int32_t)(col_off_host[b + 1] - col_off_host[b]); d.n2 = (int32_t)(seq_off_host[b + 1] - seq_off_host[b]);
        const Shape sh = shape_of(d.n2);
        d.idx = (int32_t)b; d.j = (int16_t)sh.j; d.seg = (int16_t)sh.seg;
        d.dir0 = dir_bytes; dir_bytes += dir_bytes_of(d.n1, sh);            // n1 + seg - 1 wavefront steps
        d.path_end = col_off_host[b + 1] + seq_off_host[b + 1];
        order[(size_t)b] = b;
    }
    std::stable_sort(order.begin(), order.end(), [&](int64_t p, int64_t q) {
        const AlignDesc &a = desc[(size_t)p], &c = desc[(size_t)q];
        if (a.j != c.j) return a.j > c.j;                       // heaviest group first, lighter groups fill its tail
        return a.seg != c.seg ? a.seg > c.seg : a.n1 > c.n1;
    });
    std::lock_guard<std::mutex> desc_lock(g_desc_mu);
    DescStage& stg = g_desc[g_desc_next]; g_desc_next ^= 1;
    if (!stg.ev) FAMSA_CUDA(cudaEventCreateWithFlags(&stg.ev, cudaEventDisableTiming));
    if (stg.used) FAMSA_CUDA(cudaEventSynchronize(stg.ev));              // the copy out of this buffer two calls ago
    if (stg.cap < (size_t)n_align) {
        if (stg.p) cudaFreeHost(stg.p);
        stg.p = nullptr; stg.cap = 0;
        if (cudaMallocHost((void**)&stg.p, sizeof(AlignDesc) * (size_t)n_align) != cudaSuccess) {
            cudaGetLastError(); set_error("famsa_seqprof_align: pinned allocation failed"); return FAMSA_ENOMEM;
        }
        stg.cap = (size_t)n_align;
    }
    AlignDesc* sorted = stg.p;
    for (int64_t b = 0; b < n_align; ++b) sorted[(size_t)b] = desc[(size_t)order[(size_t)b]];
    uint8_t* final_state = nullptr;
    uint8_t* ws = static_cast<uint8_t*>(workspace_dev);
    AlignDesc* d_desc = nullptr;
    uint8_t* own_state = nullptr;
    FAMSA_CUDA(cudaMallocAsync((void**)&d_desc, sizeof(AlignDesc) * (size_t)n_align, st));
    if (ws) final_state = ws + dir_bytes;
    else { FAMSA_CUDA(cudaMallocAsync((void**)&own_state, (size_t)n_align, st)); final_state = own_state; }
    FAMSA_CUDA(cudaMemcpyAsync(d_desc, sorted, sizeof(AlignDesc) * (size_t)n_align, cudaMemcpyHostToDevice, st));
    FAMSA_CUDA(cudaEventRecord(stg.ev, st));
    stg.used = true;
    const int want_dir = path_dev != nullptr;
    int64_t g0 = 0;
    while (g0 < n_align) {
        int64_t g1 = g0;
        while (g1 < n_align && sorted[(size_t)g1].j == sorted[(size_t)g0].j && sorted[(size_t)g1].seg == sorted[(size_t)g0].seg) ++g1;
        FAMSA_CUDA(launch_seqprof_group(sorted[(size_t)g0].seg, sorted[(size_t)g0].j, d_desc + g0, (int)(g1 - g0), cost_dev, seq_dev, gaps_dev,
                                        nseq_dev, score_dev, final_state, ws, want_dir, st));
        g0 = g1;
    }
    if (path_dev)
        seqprof_trace_kernel<<<(unsigned)((n_align + 3) / 4), 128, 0, st>>>(d_desc, (int)n_align, final_state, ws, path_dev, path_len_dev);
    FAMSA_CUDA(cudaGetLastError());
    FAMSA_CUDA(cudaFreeAsync(d_desc, st));
    if (own_state) FAMSA_CUDA(cudaFreeAsync(own_state, st));
    return FAMSA_OK;
}

// ---- famsa_seqprof_scores_static: the score-only alignment batch for callers that must not allocate ----------
// (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).  The same seqprof_kernel<J>
// instantiations as famsa_seqprof_align; what that call takes from cudaMallocAsync / cudaMallocHost -- the device copy
// of the alignment descriptors and one final-state byte per alignment -- lives in a file-scope device array of fixed
// size instead, and the host-side staging of the descriptors in a file-scope host array.  Every GPU that loads the
// library holds the device array (FAMSA_SEQPROF_STATIC_MAX x 49 bytes = 0.8 MB) until the process exits.
namespace famsa {

constexpr size_t STATIC_DESC_BYTES = sizeof(AlignDesc) * (size_t)FAMSA_SEQPROF_STATIC_MAX;
static __device__ __align__(256) unsigned char g_seqprof_scratch[STATIC_DESC_BYTES + (size_t)FAMSA_SEQPROF_STATIC_MAX];
// In HOST code `g_seqprof_scratch` is only a stand-in for the symbol, not a device address: the address a kernel may
// use comes from cudaGetSymbolAddress, taken once per device with that device current.
constexpr int STATIC_MAX_DEVICES = 64;
static std::mutex g_static_mu;                                    // guards the address table AND the host staging array
static unsigned char* g_static_dev_ptr[STATIC_MAX_DEVICES] = {};
static AlignDesc g_static_host_desc[FAMSA_SEQPROF_STATIC_MAX];    // host staging (static storage, pageable)

}  // namespace famsa

extern "C" int famsa_seqprof_scores_static(const float* cost_dev, const int64_t* col_off_host, const uint8_t* seq_dev,
                                           const int64_t* seq_off_host, const float* gaps_dev, const int32_t* nseq_dev,
                                           int64_t n_align, float* score_dev, void* cuda_stream) {
    if (n_align > FAMSA_SEQPROF_STATIC_MAX) {
        set_error("famsa_seqprof_scores_static: n_align exceeds FAMSA_SEQPROF_STATIC_MAX (16384 alignments per call): "
                  "split the batch, or use famsa_seqprof_align");
        return FAMSA_ERANGE;
    }
    int rc = seqprof_check(col_off_host, seq_off_host, n_align, "famsa_seqprof_scores_static");
    if (rc != FAMSA_OK) return rc;
    if (n_align == 0) return FAMSA_OK;
    if (!cost_dev || !seq_dev || !gaps_dev || !nseq_dev || !score_dev) { set_error("famsa_seqprof_scores_static: null pointer"); return FAMSA_EINVAL; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int device = -1;
    FAMSA_CUDA(cudaGetDevice(&device));
    if (device < 0 || device >= STATIC_MAX_DEVICES) { set_error("famsa_seqprof_scores_static: device ordinal out of range"); return FAMSA_ECUDA; }
    std::lock_guard<std::mutex> lock(g_static_mu);
    if (!g_static_dev_ptr[device]) {                                 // set-up, once per device, that device being current
        unsigned char* p = nullptr;
        FAMSA_CUDA(cudaGetSymbolAddress((void**)&p, g_seqprof_scratch));
        if (!p) { set_error("famsa_seqprof_scores_static: cudaGetSymbolAddress returned no address"); return FAMSA_ECUDA; }
        g_static_dev_ptr[device] = p;
    }
    AlignDesc* d_desc = reinterpret_cast<AlignDesc*>(g_static_dev_ptr[device]);
    uint8_t* final_state = g_static_dev_ptr[device] + STATIC_DESC_BYTES;
    // descriptors grouped by (lanes per alignment, residues per lane): a counting sort over the 16 classes into the static
    // host array (no heap allocation on this path)
    int64_t start[17] = {};                                          // 16 (seg, J) classes, see shape_class
    for (int64_t b = 0; b < n_align; ++b) start[shape_class(shape_of(seq_off_host[b + 1] - seq_off_host[b])) + 1]++;
    for (int c = 0; c < 16; ++c) start[c + 1] += start[c];
    int64_t fill[16];
    for (int c = 0; c < 16; ++c) fill[c] = start[c];
    for (int64_t b = 0; b < n_align; ++b) {
        const Shape sh = shape_of(seq_off_host[b + 1] - seq_off_host[b]);
        AlignDesc& d = g_static_host_desc[fill[shape_class(sh)]++];
        d.cost_row0 = col_off_host[b]; d.seq0 = seq_off_host[b];
        d.n1 = (int32_t)(col_off_host[b + 1] - col_off_host[b]); d.n2 = (int32_t)(seq_off_host[b + 1] - seq_off_host[b]);
        d.idx = (int32_t)b; d.j = (int16_t)sh.j; d.seg = (int16_t)sh.seg;
        d.dir0 = 0; d.path_end = 0;                                  // no traceback in this variant
    }
    // The array keeps the previous call's contents.  Nothing in it has to start at zero: every descriptor and every
    // final-state byte a call reads is written by that call first; the final-state bytes are cleared all the same, so
    // that no value of an earlier call can ever be mistaken for this one's.
    FAMSA_CUDA(cudaMemsetAsync(final_state, 0, (size_t)n_align, st));
    // pageable source: the runtime has staged the bytes when the call returns, so the host array is free again
    FAMSA_CUDA(cudaMemcpyAsync(d_desc, g_static_host_desc, sizeof(AlignDesc) * (size_t)n_align, cudaMemcpyHostToDevice, st));
    for (int c = 0; c < 16; ++c) {
        const int n = (int)(start[c + 1] - start[c]);
        if (n == 0) continue;
        FAMSA_CUDA(launch_seqprof_group(c < 8 ? 32 : 16, 32 - 4 * (c & 7), d_desc + start[c], n, cost_dev, seq_dev, gaps_dev, nseq_dev, score_dev,
                                        final_state, (uint8_t*)nullptr, 0, st));
    }
    return FAMSA_OK;
}
