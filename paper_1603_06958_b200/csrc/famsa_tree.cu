// famsa_tree.cu -- stage II consumer: single-linkage guide tree built incrementally from the streamed
// similarity row blocks in O(k) memory.  See include/famsa_lcs.h.
//
// State: the maximum spanning FOREST T of the similarity entries seen so far (<= k-1 edges).  Single
// linkage = the spanning tree's edges taken by decreasing similarity, so T is an O(k) summary from which
// the dendrogram follows, and MSF(E1 u E2) = MSF(MSF(E1) u E2): a row block [i0, i1) -- in any order --
// is merged in as follows, everything enqueued on the caller's stream, no host round trip:
//   1. round 0 of Boruvka on the BLOCK's own graph (vertices [0, i1), edges (v, u < v) for the block's rows
//      v): every vertex picks its best edge -- the best entry of its row and/or of its column.  These
//      candidates come out of the sweep's own epilogue (64-bit atomicMax keys, famsa_guide_forest) or out of
//      one pass over the block (famsa_tree_update on a caller's block).  Every component of the pick graph
//      contains a block row, so there are P <= rows <= 1024 components.
//   2. ONE pass over the block fills K[row][component] = the best edge from each block row into each OTHER
//      component (one CTA per row keeps the row's table in shared memory; monotone filter: a plain read of the
//      entry, an atomicMax only when it improves, so atomics are ~ entries x ln(columns)).  The picks of 1. plus, per pair of
//      components, the best entries of K are a sparse edge set S with MSF(T u block) = MSF(T u S): an edge
//      inside a component, or not the best of its component pair, closes a cycle of heavier edges.
//   3. a persistent cooperative kernel merges S into T by Boruvka rounds over (T's edges + S) with grid-wide
//      barriers between the phases, until a round hooks nothing.
// Every edge has a unique key (similarity descending, then (max, min) endpoint ascending), so each round's
// picks are edges of the one MSF under that order and only mutual picks form 2-cycles.
#include <cooperative_groups.h>
#include <cub/device/device_radix_sort.cuh>

#include <algorithm>
#include <cmath>
#include <new>

#include "famsa_internal.h"

namespace cg = cooperative_groups;

namespace famsa {

constexpr int TREE_SUB_ROWS = 1024;    // rows per internal update (bounds the component count P)
constexpr int KSTRIDE = 1024;          // row stride of the row x component table
constexpr uint32_t ERR_COMPONENTS = 1, ERR_SPARSE_FULL = 2, ERR_ROUNDS = 4;

// Device-resident scalars of a tree (one struct; the host reads it only when it needs a count).
struct TreeState {
    uint32_t m;          // edges of the current forest
    uint32_t ns;         // edges of the sparse candidate set S of the update in flight
    uint32_t P;          // components of the block graph after round 0
    uint32_t err;        // sticky ERR_* flags
    uint32_t rec;        // edges recorded by the merge in flight
    uint32_t rounds;     // Boruvka rounds run so far (all merges)
    uint32_t pad[2];
};

}  // namespace famsa

struct famsa_tree {
    int      device = 0;
    int      sm_count = 0;
    int64_t  k = 0;
    int64_t  rows = 0;                 // rows consumed so far (any order)
    bool     merged = false;           // sparse edges were merged in
    uint32_t *ta[2] = {nullptr, nullptr}, *tb[2] = {nullptr, nullptr};   // forest edges, a > b (double buffer)
    float    *tw[2] = {nullptr, nullptr};
    int      cur = 0;
    uint32_t *comp[2] = {nullptr, nullptr}, *parent = nullptr;           // merge kernel
    uint32_t *best_w = nullptr;                    // per component: float bits + 1 (0 = none)
    unsigned long long* best_id = nullptr;         // per component: (max << 32) | min of the chosen edge
    // block graph (round 0 + row x component table)
    unsigned long long *cand_row[2] = {nullptr, nullptr}, *cand_col[2] = {nullptr, nullptr};   // two slots: sweep n+1 fills one while update n reads the other
    unsigned long long *pick = nullptr;            // k
    uint32_t *bparent = nullptr, *rootidx = nullptr;                     // k each
    uint16_t *cid16 = nullptr;                     // k: compact component id of the block graph
    unsigned long long *ktab = nullptr;            // TREE_SUB_ROWS x KSTRIDE
    uint32_t *wab = nullptr;                       // KSTRIDE x KSTRIDE: best weight key per component pair
    uint32_t *sa = nullptr, *sb = nullptr; float* sw = nullptr;          // sparse set S
    size_t   s_cap = 0;
    famsa::TreeState* st = nullptr;                // device
    famsa::TreeState* h_st = nullptr;              // pinned
    int      merge_grid = 0;
    int64_t  launches = 0;
};

namespace famsa {

__device__ __forceinline__ unsigned long long cand_key(float w, uint32_t other) {
    const uint32_t b = __float_as_uint(w);
    if (b & 0x80000000u) return 0ull;                      // sign bit set (-0.0 included): not an edge
    return ((unsigned long long)(b + 1u) << 32) | (uint32_t)~other;      // max: higher similarity, then smaller `other`
}
__device__ __forceinline__ uint32_t key_other(unsigned long long key) { return ~(uint32_t)key; }
__device__ __forceinline__ uint32_t key_wbits1(unsigned long long key) { return (uint32_t)(key >> 32); }

// ---- round-0 candidates from a caller's block (famsa_tree_update): ONE pass, both directions -----------
// One CTA per block row v, 4 independent loads in flight per thread (measured r01: 1024 CTAs read a 1.7 GB block at
// 5.7 TB/s).  The row's best entry is reduced in the CTA; every entry is also a candidate of its COLUMN u, offered to
// cand_col[u] through the monotone filter (a plain read of the L2-resident key, an atomicMax only if it improves), as
// the sweep's epilogue does in the fused pipeline.  The caller zeroes cand_col[0, i1) first.
__global__ void __launch_bounds__(256) tree_cand_kernel(const float* __restrict__ sim, uint32_t i0, uint32_t i1, int64_t out_base,
                                                        unsigned long long* __restrict__ cand_row, unsigned long long* __restrict__ cand_col) {
    const uint32_t v = i0 + blockIdx.x;
    const float* row = sim + ((int64_t)v * (v - 1) / 2 - out_base);
    float bw = -1.0f; uint32_t bo = 0xFFFFFFFFu;
#pragma unroll 4
    for (uint32_t u = threadIdx.x; u < v; u += 256) {
        const float w = __ldg(row + u);
        if (w > bw) { bw = w; bo = u; }                    // u ascends per thread: the first of equals stays
        const unsigned long long ck = cand_key(w, v);
        if (ck > cand_col[u]) atomicMax(cand_col + u, ck);
    }
    unsigned long long key = bo == 0xFFFFFFFFu ? 0ull : cand_key(bw, bo);
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) key = max(key, __shfl_xor_sync(0xffffffffu, key, d));
    __shared__ unsigned long long sk[8];
    if ((threadIdx.x & 31) == 0) sk[threadIdx.x >> 5] = key;
    __syncthreads();
    if (threadIdx.x == 0) {
#pragma unroll
        for (int q = 1; q < 8; ++q) key = max(key, sk[q]);
        cand_row[v] = key;
    }
}

struct BlockArgs {
    uint32_t i0, i1;             // rows of the (sub-)block
    const unsigned long long *cand_row, *cand_col;
    unsigned long long* pick;
    uint32_t *bparent, *rootidx;
    uint16_t* cid16;
    unsigned long long* ktab;
    uint32_t* wab;
    uint32_t *sa, *sb; float* sw; uint32_t s_cap;
    TreeState* st;
};

// Round 0 on the block graph: every vertex x < i1 picks the better of its row and column candidates.
__global__ void tree_pick_kernel(BlockArgs a) {
    const uint32_t x = blockIdx.x * blockDim.x + threadIdx.x;
    if (x == 0) { a.st->P = 0; a.st->ns = 0; }
    if (x >= a.i1) return;
    const unsigned long long kr = x >= a.i0 ? a.cand_row[x] : 0ull;
    const unsigned long long kc = x + 1 < a.i1 ? a.cand_col[x] : 0ull;
    a.pick[x] = max(kr, kc);
}

// Hooking: x -> the other end of its pick; of a mutual pair the smaller index stays a root.  Every pick is an
// edge of the block graph's MSF (it is the best edge of a vertex) and is recorded once into S.
__global__ void tree_hook0_kernel(BlockArgs a) {
    const uint32_t x = blockIdx.x * blockDim.x + threadIdx.x;
    if (x >= a.i1) return;
    const unsigned long long key = a.pick[x];
    if (key == 0) { a.bparent[x] = x; return; }             // no edge at all (a one-row block of row 0)
    const uint32_t y = key_other(key);
    const bool mutual = a.pick[y] == ((key & 0xFFFFFFFF00000000ull) | (uint32_t)~x);
    if (mutual && x < y) { a.bparent[x] = x; return; }
    a.bparent[x] = y;
    const uint32_t pos = atomicAdd(&a.st->ns, 1u);
    if (pos < a.s_cap) { a.sa[pos] = max(x, y); a.sb[pos] = min(x, y); a.sw[pos] = __uint_as_float(key_wbits1(key) - 1u); }
    else atomicOr(&a.st->err, ERR_SPARSE_FULL);
}

// Component roots by pointer jumping (benign race: every write is an ancestor); roots get compact ids.
__global__ void tree_root0_kernel(BlockArgs a) {
    const uint32_t x = blockIdx.x * blockDim.x + threadIdx.x;
    if (x >= a.i1) return;
    uint32_t r = x;
    for (uint32_t p = a.bparent[r]; p != r; p = a.bparent[r]) {
        const uint32_t g = a.bparent[p];
        if (g != p) a.bparent[r] = g;
        r = p;
    }
    a.pick[x] = r;                                           // reuse: the root of x
    if (r == x) {
        const uint32_t id = atomicAdd(&a.st->P, 1u);
        if (id >= (uint32_t)KSTRIDE) atomicOr(&a.st->err, ERR_COMPONENTS);    // cannot happen: every component holds a block row
        a.rootidx[x] = id;
    }
}
__global__ void tree_cid_kernel(BlockArgs a) {
    const uint32_t x = blockIdx.x * blockDim.x + threadIdx.x;
    if (x >= a.i1) return;
    a.cid16[x] = (uint16_t)min(a.rootidx[(uint32_t)a.pick[x]], (uint32_t)KSTRIDE - 1);
}

// The one pass over the block: K[row][component b] = best edge from block row v into component b != comp(v).
// One CTA per row, so the row's table (P x 8 B <= 8 KB) is PRIVATE to the CTA: it lives in shared memory, an entry is
// read with a plain load and only an improving key goes to a shared-memory atomicMax (a stale read only costs a
// redundant atomic), and the CTA writes its P entries out once at the end -- no global atomics, no gathers from
// global memory.  HBM-bound: one read of the block + 2 B of (L2-resident) component id per entry.
__global__ void __launch_bounds__(256) tree_rowcomp_kernel(const float* __restrict__ sim, uint32_t i0, uint32_t i1, int64_t out_base, BlockArgs a) {
    __shared__ unsigned long long sk[KSTRIDE];
    const uint32_t P = a.st->P;
    if (P <= 1) return;                                     // the block graph is already connected
    for (uint32_t b = threadIdx.x; b < P; b += 256) sk[b] = 0ull;
    __syncthreads();
    const uint32_t v = i0 + blockIdx.x;
    const float* row = sim + ((int64_t)v * (v - 1) / 2 - out_base);
    const uint16_t ca = a.cid16[v];
    const uint16_t* __restrict__ cid = a.cid16;
    uint32_t u = threadIdx.x;
    for (; u + 7 * 256 < v; u += 8 * 256) {                 // 8 independent loads of each kind in flight
        float w[8]; uint16_t c[8];
#pragma unroll
        for (int q = 0; q < 8; ++q) { w[q] = __ldg(row + u + q * 256); c[q] = cid[u + q * 256]; }
#pragma unroll
        for (int q = 0; q < 8; ++q)
            if (c[q] != ca) {
                const unsigned long long key = cand_key(w[q], u + q * 256);
                if (key > sk[c[q]]) atomicMax(&sk[c[q]], key);
            }
    }
    for (; u < v; u += 256) {
        const float w = __ldg(row + u); const uint16_t c = cid[u];
        if (c != ca) {
            const unsigned long long key = cand_key(w, u);
            if (key > sk[c]) atomicMax(&sk[c], key);
        }
    }
    __syncthreads();
    unsigned long long* krow = a.ktab + (size_t)blockIdx.x * KSTRIDE;
    for (uint32_t b = threadIdx.x; b < P; b += 256) krow[b] = sk[b];
}

// S += the best entries of K per pair of components (ties keep several: harmless).
template <int PASS>
__global__ void tree_gather_kernel(BlockArgs a) {
    const uint32_t P = a.st->P;
    if (P <= 1) return;
    const uint32_t t = blockIdx.x * blockDim.x + threadIdx.x;
    const uint32_t vi = t / KSTRIDE, b = t % KSTRIDE;
    if (vi >= a.i1 - a.i0 || b >= P) return;
    const unsigned long long key = a.ktab[t];
    if (key == 0) return;
    const uint32_t v = a.i0 + vi, ca = a.cid16[v];
    uint32_t* wslot = &a.wab[min(ca, b) * KSTRIDE + max(ca, b)];
    if (PASS == 0) { atomicMax(wslot, key_wbits1(key)); return; }
    if (*wslot != key_wbits1(key)) return;
    const uint32_t u = key_other(key);
    const uint32_t pos = atomicAdd(&a.st->ns, 1u);
    if (pos < a.s_cap) { a.sa[pos] = v; a.sb[pos] = u; a.sw[pos] = __uint_as_float(key_wbits1(key) - 1u); }
    else atomicOr(&a.st->err, ERR_SPARSE_FULL);
}

// ---- the merge: MSF(T u S) by Boruvka rounds, one persistent cooperative kernel ------------------------
struct MergeArgs {
    uint32_t n;                                            // all k leaves
    const uint32_t *ta, *tb; const float* tw;              // current forest (st->m edges)
    const uint32_t *sa, *sb; const float* sw;              // sparse set S (st->ns edges)
    uint32_t *na, *nb; float* nw;                          // the new forest
    uint32_t *comp0, *comp1, *parent;
    uint32_t* best_w; unsigned long long* best_id;
    TreeState* st;
};

__device__ __forceinline__ unsigned long long edge_id(uint32_t x, uint32_t y) {
    return ((unsigned long long)max(x, y) << 32) | min(x, y);
}

__global__ void __launch_bounds__(256) tree_merge_kernel(MergeArgs a) {
    cg::grid_group grid = cg::this_grid();
    const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x, nth = gridDim.x * blockDim.x;
    const uint32_t m = a.st->m, ns = a.st->ns, items = m + ns;
    uint32_t* comp = a.comp0; uint32_t* comp_next = a.comp1;
    for (uint32_t x = tid; x < a.n; x += nth) comp[x] = x;
    grid.sync();                                           // (everyone has read st->m / st->ns before rec is reset)
    if (tid == 0) a.st->rec = 0;
    uint32_t recorded = 0, round = 0;
    for (;; ++round) {
        for (uint32_t x = tid; x < a.n; x += nth) { a.best_w[x] = 0; a.best_id[x] = ~0ull; }
        grid.sync();
        // per component: the highest similarity of an outgoing edge ...
        for (uint32_t e = tid; e < items; e += nth) {
            const uint32_t x = e < m ? a.ta[e] : a.sa[e - m], y = e < m ? a.tb[e] : a.sb[e - m];
            const uint32_t wb = __float_as_uint(e < m ? a.tw[e] : a.sw[e - m]);
            if (x == y || (wb & 0x80000000u)) continue;
            const uint32_t cx = comp[x], cy = comp[y];
            if (cx == cy) continue;
            atomicMax(&a.best_w[cx], wb + 1u); atomicMax(&a.best_w[cy], wb + 1u);
        }
        grid.sync();
        // ... and among the edges that reach it, the smallest edge id: the component's minimum-key outgoing edge
        for (uint32_t e = tid; e < items; e += nth) {
            const uint32_t x = e < m ? a.ta[e] : a.sa[e - m], y = e < m ? a.tb[e] : a.sb[e - m];
            const uint32_t wb = __float_as_uint(e < m ? a.tw[e] : a.sw[e - m]);
            if (x == y || (wb & 0x80000000u)) continue;
            const uint32_t cx = comp[x], cy = comp[y];
            if (cx == cy) continue;
            const unsigned long long id = edge_id(x, y);
            if (a.best_w[cx] == wb + 1u) atomicMin(&a.best_id[cx], id);
            if (a.best_w[cy] == wb + 1u) atomicMin(&a.best_id[cy], id);
        }
        grid.sync();
        // each component root hooks onto the component at the other end of its edge (mutual picks: the smaller
        // root stays) and records the edge once
        for (uint32_t c = tid; c < a.n; c += nth) {
            uint32_t p = c;
            if (comp[c] == c && a.best_w[c] != 0) {
                const unsigned long long id = a.best_id[c];
                const uint32_t hi = (uint32_t)(id >> 32), lo = (uint32_t)id;
                const uint32_t t = comp[comp[hi] == c ? lo : hi];
                if (!(a.best_id[t] == id && c < t)) {
                    p = t;
                    const uint32_t pos = atomicAdd(&a.st->rec, 1u);
                    a.na[pos] = hi; a.nb[pos] = lo; a.nw[pos] = __uint_as_float(a.best_w[c] - 1u);
                }
            }
            a.parent[c] = p;
        }
        grid.sync();
        const uint32_t rec = *(volatile uint32_t*)&a.st->rec;
        const bool done = rec == recorded;                   // a round that hooks nothing: done
        recorded = rec;
        if (done || round >= 63) break;
        for (uint32_t x = tid; x < a.n; x += nth) {
            uint32_t r = comp[x];
            for (uint32_t p = a.parent[r]; p != r; p = a.parent[r]) {     // pointer jumping (benign race: every
                const uint32_t g = a.parent[p];                            // write is an ancestor of r)
                if (g != p) a.parent[r] = g;
                r = p;
            }
            comp_next[x] = r;
        }
        grid.sync();
        uint32_t* s = comp; comp = comp_next; comp_next = s;
    }
    if (tid == 0) {
        a.st->m = recorded; a.st->ns = 0; a.st->rounds += round + 1;
        if (round >= 63) atomicOr(&a.st->err, ERR_ROUNDS);
    }
}

template <typename T>
static int tree_alloc(T** p, size_t n) {
    cudaError_t e = cudaMalloc((void**)p, std::max<size_t>(n, 1) * sizeof(T));
    if (e == cudaErrorMemoryAllocation) { cudaGetLastError(); set_error("famsa_tree: device allocation failed"); return FAMSA_ENOMEM; }
    if (e != cudaSuccess) return cuda_fail(e, "cudaMalloc");
    return FAMSA_OK;
}

static BlockArgs block_args(famsa_tree* t, int64_t i0, int64_t i1, int slot) {
    BlockArgs a;
    a.i0 = (uint32_t)i0; a.i1 = (uint32_t)i1;
    a.cand_row = t->cand_row[slot]; a.cand_col = t->cand_col[slot];
    a.pick = t->pick; a.bparent = t->bparent; a.rootidx = t->rootidx; a.cid16 = t->cid16;
    a.ktab = t->ktab; a.wab = t->wab;
    a.sa = t->sa; a.sb = t->sb; a.sw = t->sw; a.s_cap = (uint32_t)t->s_cap;
    a.st = t->st;
    return a;
}

// MSF(T u S) -> the other forest buffer; flips t->cur.  Enqueue only.
static int tree_merge(famsa_tree* t, cudaStream_t st) {
    const int cur = t->cur, nxt = cur ^ 1;
    MergeArgs a;
    a.n = (uint32_t)t->k;
    a.ta = t->ta[cur]; a.tb = t->tb[cur]; a.tw = t->tw[cur];
    a.sa = t->sa; a.sb = t->sb; a.sw = t->sw;
    a.na = t->ta[nxt]; a.nb = t->tb[nxt]; a.nw = t->tw[nxt];
    a.comp0 = t->comp[0]; a.comp1 = t->comp[1]; a.parent = t->parent;
    a.best_w = t->best_w; a.best_id = t->best_id; a.st = t->st;
    void* args[] = {&a};
    FAMSA_CUDA(cudaLaunchCooperativeKernel((const void*)tree_merge_kernel, dim3((unsigned)t->merge_grid), dim3(256), args, 0, st));
    t->launches++;
    t->cur = nxt;
    return FAMSA_OK;
}

// One (sub-)block of <= TREE_SUB_ROWS rows: candidates are in slot `slot` (fused == true: the sweep's
// epilogue put them there) or are computed from the block here.  Enqueue only.
int tree_consume(famsa_tree* t, int64_t i0, int64_t i1, const float* sim, int64_t out_base, int slot, bool fused, cudaStream_t st) {
    const BlockArgs a = block_args(t, i0, i1, slot);
    const unsigned gv = (unsigned)((i1 + 255) / 256);
    if (!fused) {
        FAMSA_CUDA(cudaMemsetAsync(t->cand_col[slot], 0, sizeof(unsigned long long) * (size_t)i1, st));
        tree_cand_kernel<<<(unsigned)(i1 - i0), 256, 0, st>>>(sim, a.i0, a.i1, out_base, t->cand_row[slot], t->cand_col[slot]);
        t->launches += 1;
    }
    tree_pick_kernel<<<gv, 256, 0, st>>>(a);
    tree_hook0_kernel<<<gv, 256, 0, st>>>(a);
    tree_root0_kernel<<<gv, 256, 0, st>>>(a);
    tree_cid_kernel<<<gv, 256, 0, st>>>(a);
    FAMSA_CUDA(cudaMemsetAsync(t->wab, 0, sizeof(uint32_t) * (size_t)KSTRIDE * KSTRIDE, st));
    tree_rowcomp_kernel<<<(unsigned)(i1 - i0), 256, 0, st>>>(sim, a.i0, a.i1, out_base, a);
    const unsigned gk = (unsigned)(((size_t)(i1 - i0) * KSTRIDE + 255) / 256);
    tree_gather_kernel<0><<<gk, 256, 0, st>>>(a);
    tree_gather_kernel<1><<<gk, 256, 0, st>>>(a);
    t->launches += 7;
    FAMSA_CUDA(cudaGetLastError());
    return tree_merge(t, st);
}

// Zero the candidate slot for rows [i0, i1) before the sweep's epilogue accumulates into it.
int tree_fused_begin(famsa_tree* t, int64_t i0, int64_t i1, int slot, cudaStream_t st) {
    FAMSA_CUDA(cudaMemsetAsync(t->cand_row[slot] + i0, 0, sizeof(unsigned long long) * (size_t)(i1 - i0), st));
    FAMSA_CUDA(cudaMemsetAsync(t->cand_col[slot], 0, sizeof(unsigned long long) * (size_t)i1, st));
    return FAMSA_OK;
}

// Wait for the tree's work and fetch its device scalars.
static int tree_read_state(famsa_tree* t) {
    FAMSA_CUDA(cudaSetDevice(t->device));
    FAMSA_CUDA(cudaDeviceSynchronize());
    FAMSA_CUDA(cudaMemcpy(t->h_st, t->st, sizeof(TreeState), cudaMemcpyDeviceToHost));
    if (t->h_st->err) {
        set_error(std::string("famsa_tree: the device reported") + ((t->h_st->err & ERR_ROUNDS) ? " no convergence after 64 Boruvka rounds" : "") +
                  ((t->h_st->err & ERR_SPARSE_FULL) ? " an overflow of the sparse candidate set" : "") +
                  ((t->h_st->err & ERR_COMPONENTS) ? " more block components than block rows" : ""));
        return FAMSA_EINVAL;
    }
    return FAMSA_OK;
}

}  // namespace famsa

using namespace famsa;

#define TREE_TRY(x) do { int rc__ = (x); if (rc__ != FAMSA_OK) { famsa_tree_free(t); return rc__; } } while (0)

extern "C" void famsa_tree_free(famsa_tree* t) {
    if (!t) return;
    cudaSetDevice(t->device);
    cudaDeviceSynchronize();
    for (int b = 0; b < 2; ++b) {
        cudaFree(t->ta[b]); cudaFree(t->tb[b]); cudaFree(t->tw[b]); cudaFree(t->comp[b]);
        cudaFree(t->cand_row[b]); cudaFree(t->cand_col[b]);
    }
    cudaFree(t->parent); cudaFree(t->best_w); cudaFree(t->best_id);
    cudaFree(t->pick); cudaFree(t->bparent); cudaFree(t->rootidx); cudaFree(t->cid16);
    cudaFree(t->ktab); cudaFree(t->wab); cudaFree(t->sa); cudaFree(t->sb); cudaFree(t->sw); cudaFree(t->st);
    if (t->h_st) cudaFreeHost(t->h_st);
    delete t;
}

extern "C" int famsa_tree_create(int64_t k, int device, famsa_tree** out) {
    if (!out) { set_error("famsa_tree_create: out is NULL"); return FAMSA_EINVAL; }
    *out = nullptr;
    if (k < 0 || k > 0x7FFFFFF0LL) { set_error("famsa_tree_create: bad k"); return FAMSA_EINVAL; }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) {
        cudaGetLastError(); set_error("famsa_tree_create: no such CUDA device (there is no CPU fallback)"); return FAMSA_ECUDA;
    }
    FAMSA_CUDA(cudaSetDevice(device));
    famsa_tree* t = new (std::nothrow) famsa_tree();
    if (!t) { set_error("famsa_tree_create: host allocation failed"); return FAMSA_ENOMEM; }
    t->device = device; t->k = k;
    int coop = 0, per_sm = 0;
    if (cudaDeviceGetAttribute(&t->sm_count, cudaDevAttrMultiProcessorCount, device) != cudaSuccess ||
        cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, device) != cudaSuccess ||
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, tree_merge_kernel, 256, 0) != cudaSuccess || per_sm < 1 || !coop) {
        cudaGetLastError(); famsa_tree_free(t); set_error("famsa_tree_create: the device cannot run the cooperative merge kernel"); return FAMSA_ECUDA;
    }
    t->merge_grid = t->sm_count;                           // one 256-thread CTA per SM: co-resident beside the sweep's CTAs
    const size_t n = (size_t)k;
    for (int b = 0; b < 2; ++b) {
        TREE_TRY(tree_alloc(&t->ta[b], n)); TREE_TRY(tree_alloc(&t->tb[b], n)); TREE_TRY(tree_alloc(&t->tw[b], n));
        TREE_TRY(tree_alloc(&t->comp[b], n)); TREE_TRY(tree_alloc(&t->cand_row[b], n)); TREE_TRY(tree_alloc(&t->cand_col[b], n));
    }
    TREE_TRY(tree_alloc(&t->parent, n)); TREE_TRY(tree_alloc(&t->best_w, n)); TREE_TRY(tree_alloc(&t->best_id, n));
    TREE_TRY(tree_alloc(&t->pick, n)); TREE_TRY(tree_alloc(&t->bparent, n)); TREE_TRY(tree_alloc(&t->rootidx, n)); TREE_TRY(tree_alloc(&t->cid16, n));
    TREE_TRY(tree_alloc(&t->ktab, (size_t)std::min<int64_t>(std::max<int64_t>(k, 1), TREE_SUB_ROWS) * KSTRIDE));
    TREE_TRY(tree_alloc(&t->wab, (size_t)KSTRIDE * KSTRIDE));
    t->s_cap = n + (size_t)std::min<int64_t>(std::max<int64_t>(k, 1), TREE_SUB_ROWS) * KSTRIDE;
    TREE_TRY(tree_alloc(&t->sa, t->s_cap)); TREE_TRY(tree_alloc(&t->sb, t->s_cap)); TREE_TRY(tree_alloc(&t->sw, t->s_cap));
    TREE_TRY(tree_alloc(&t->st, 1));
    if (cudaMemset(t->st, 0, sizeof(TreeState)) != cudaSuccess || cudaMallocHost((void**)&t->h_st, sizeof(TreeState)) != cudaSuccess) {
        cudaGetLastError(); famsa_tree_free(t); set_error("famsa_tree_create: state allocation failed"); return FAMSA_ENOMEM;
    }
    *out = t;
    return FAMSA_OK;
}

extern "C" int famsa_tree_update(famsa_tree* t, int64_t i0, int64_t i1, const float* sim_block, void* cuda_stream) {
    if (!t) { set_error("famsa_tree_update: tree is NULL"); return FAMSA_EINVAL; }
    if (i0 < 0 || i1 < i0 || i1 > t->k) { set_error("famsa_tree_update: bad row range"); return FAMSA_ERANGE; }
    if (i1 == i0) return FAMSA_OK;
    if (!sim_block && famsa_rows_pairs(i0, i1) > 0) { set_error("famsa_tree_update: sim_block is NULL"); return FAMSA_EINVAL; }
    FAMSA_CUDA(cudaSetDevice(t->device));
    const int64_t out_base = i0 * (i0 - 1) / 2;
    for (int64_t s0 = i0; s0 < i1; s0 += TREE_SUB_ROWS) {
        const int64_t s1 = std::min<int64_t>(s0 + TREE_SUB_ROWS, i1);
        if (famsa_rows_pairs(s0, s1) == 0) continue;       // row 0 alone: no entries
        int rc = tree_consume(t, s0, s1, sim_block, out_base, 0, false, (cudaStream_t)cuda_stream);
        if (rc != FAMSA_OK) return rc;
    }
    t->rows += i1 - i0;
    return FAMSA_OK;
}

extern "C" int famsa_tree_merge_edges(famsa_tree* t, const int64_t* a_host, const int64_t* b_host, const float* sim_host, int64_t m) {
    if (!t) { set_error("famsa_tree_merge_edges: tree is NULL"); return FAMSA_EINVAL; }
    if (m < 0 || (m > 0 && (!a_host || !b_host || !sim_host))) { set_error("famsa_tree_merge_edges: null input"); return FAMSA_EINVAL; }
    if (m == 0) return FAMSA_OK;
    FAMSA_CUDA(cudaSetDevice(t->device));
    std::vector<uint32_t> a(std::min<int64_t>(m, (int64_t)t->s_cap)), b(a.size());
    for (int64_t e0 = 0; e0 < m; e0 += (int64_t)t->s_cap) {                // S-sized slices, merged one after the other
        const int64_t n = std::min<int64_t>(m - e0, (int64_t)t->s_cap);
        for (int64_t e = 0; e < n; ++e) {
            const int64_t x = a_host[e0 + e], y = b_host[e0 + e]; const float w = sim_host[e0 + e];
            if (x < 0 || x >= t->k || y < 0 || y >= t->k || !(w >= 0.0f) || std::signbit(w)) {
                set_error("famsa_tree_merge_edges: edge " + std::to_string(e0 + e) + " has a leaf out of range or a negative (-0.0 included) / NaN similarity");
                return FAMSA_ERANGE;
            }
            a[e] = (uint32_t)x; b[e] = (uint32_t)y;
        }
        FAMSA_CUDA(cudaDeviceSynchronize());                               // S is free (no update in flight)
        const uint32_t ns = (uint32_t)n;
        FAMSA_CUDA(cudaMemcpy(t->sa, a.data(), 4ull * n, cudaMemcpyHostToDevice));
        FAMSA_CUDA(cudaMemcpy(t->sb, b.data(), 4ull * n, cudaMemcpyHostToDevice));
        FAMSA_CUDA(cudaMemcpy(t->sw, sim_host + e0, 4ull * n, cudaMemcpyHostToDevice));
        FAMSA_CUDA(cudaMemcpy(&t->st->ns, &ns, sizeof(ns), cudaMemcpyHostToDevice));
        int rc = tree_merge(t, nullptr);
        if (rc != FAMSA_OK) return rc;
        FAMSA_CUDA(cudaDeviceSynchronize());
    }
    t->merged = true;
    return FAMSA_OK;
}

extern "C" int64_t famsa_tree_edge_count(const famsa_tree* t) {
    if (!t) return 0;
    if (tree_read_state(const_cast<famsa_tree*>(t)) != FAMSA_OK) return -1;
    return t->h_st->m;
}

extern "C" int famsa_tree_edges(famsa_tree* t, int64_t* a_host, int64_t* b_host, float* sim_host) {
    if (!t) { set_error("famsa_tree_edges: tree is NULL"); return FAMSA_EINVAL; }
    int rc = tree_read_state(t);
    if (rc != FAMSA_OK) return rc;
    const int64_t m = t->h_st->m;
    if (m == 0) return FAMSA_OK;
    if (!a_host || !b_host || !sim_host) { set_error("famsa_tree_edges: null output"); return FAMSA_EINVAL; }
    std::vector<uint32_t> a(m), b(m);
    FAMSA_CUDA(cudaMemcpy(a.data(), t->ta[t->cur], sizeof(uint32_t) * m, cudaMemcpyDeviceToHost));
    FAMSA_CUDA(cudaMemcpy(b.data(), t->tb[t->cur], sizeof(uint32_t) * m, cudaMemcpyDeviceToHost));
    FAMSA_CUDA(cudaMemcpy(sim_host, t->tw[t->cur], sizeof(float) * m, cudaMemcpyDeviceToHost));
    for (int64_t e = 0; e < m; ++e) { a_host[e] = a[e]; b_host[e] = b[e]; }
    return FAMSA_OK;
}

namespace famsa {

__global__ void tree_sortkeys_kernel(uint32_t m, const uint32_t* ta, const uint32_t* tb, unsigned long long* id_key, uint32_t* idx) {
    const uint32_t e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= m) return;
    id_key[e] = ((unsigned long long)ta[e] << 32) | tb[e];
    idx[e] = e;
}
__global__ void tree_wkeys_kernel(uint32_t m, const float* tw, const uint32_t* idx, uint32_t* w_key) {
    const uint32_t e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e < m) w_key[e] = ~__float_as_uint(tw[idx[e]]);     // ascending key == descending similarity
}
__global__ void tree_uf_init_kernel(uint32_t k, uint32_t* uf, unsigned long long* info) {
    const uint32_t x = blockIdx.x * blockDim.x + threadIdx.x;
    if (x < k) { uf[x] = x; info[x] = ((unsigned long long)x << 32) | 1u; }   // (cluster id, size)
}

// The dendrogram from the sorted tree edges: Kruskal's union-find in edge order, which is sequential in the
// unions but not in the memory latency.  One CTA works through the edges in batches of DG_B:
//   A (all threads)  the roots of both endpoints of the batch's edges, found in the union-find as it stood
//                    before the batch (read-only walks, all in flight at once: the L2 latency of the finds,
//                    which made the one-lane version 0.8 us per merge, is paid once per batch; the endpoints
//                    of the NEXT batch are fetched before this batch's serial phase);
//   B (all threads)  equal roots among the 2 x DG_B slots are identified through a small shared-memory hash
//                    table (canonical slot = smallest slot with that root);
//   C (one thread)   the batch's unions in edge order on a LOCAL union-find over the slots, in shared memory,
//                    with the next edge's slots and the (speculative) set records loaded ahead;
//   D (all threads)  the local result goes back to the global arrays: every root of the batch points to its
//                    final root, the final roots carry (cluster id, size), the endpoints are compressed.
// Cluster ids and sizes are < 2^32 (k <= 2^31 - 16), so (id, size) is one 64-bit word.
constexpr int DG_B = 512, DG_H = 2048, DG_HBITS = 11;    // batch, hash-table size (2^DG_HBITS >= 4 x slots / 2); measured
                                                          // r02: the per-batch costs (finds, hash, write-back) are ~60 % of a 128-edge batch
__global__ void __launch_bounds__(DG_B) tree_dendrogram_kernel(uint32_t k, const uint32_t* __restrict__ order, const uint32_t* __restrict__ ta,
                                                               const uint32_t* __restrict__ tb, const float* __restrict__ tw,
                                                               uint32_t* uf, unsigned long long* info,
                                                               long long* out_a, long long* out_b, float* out_w, long long* out_size) {
    __shared__ uint32_t s_root[2 * DG_B];                  // global root of each slot (2q, 2q+1 = the endpoints of edge q)
    __shared__ uint32_t s_vert[2 * DG_B];                  // the endpoints themselves
    __shared__ __align__(4) uint16_t s_canon[2 * DG_B + 2];   // smallest slot with the same root (+2: read-ahead slack)
    __shared__ uint16_t s_par[2 * DG_B];                   // local union-find over canonical slots
    __shared__ uint16_t s_hidx[2 * DG_B];
    __shared__ uint2 s_info[2 * DG_B];                     // (.x = size, .y = cluster id) of a local root
    __shared__ uint32_t h_key[DG_H], h_slot[DG_H];          // hash table of phase B; afterwards reused:
    uint32_t* const s_cnt = h_key;                          //   [2 DG_B] references to each canonical slot in this batch
    uint32_t* const s_oa = h_slot; uint32_t* const s_ob = h_slot + DG_B; uint32_t* const s_os = h_slot + 2 * DG_B;   // merge outputs
    uint16_t* const s_hub = s_hidx;                         //   [DG_B] the edge's hub slot (0xFFFF: none)
    static_assert(2 * DG_B <= DG_H && 3 * DG_B <= DG_H, "aliases fit");
    const uint32_t tid = threadIdx.x, m = k - 1;
    uint32_t nx = 0, ny = 0; float nw = 0.0f;              // this thread's edge of the next batch
    if (tid < m) { const uint32_t e = order[tid]; nx = ta[e]; ny = tb[e]; nw = tw[e]; }
    for (uint32_t t0 = 0; t0 < m; t0 += DG_B) {
        const uint32_t nb = min((uint32_t)DG_B, m - t0);
        for (uint32_t h = tid; h < DG_H; h += DG_B) { h_key[h] = 0xFFFFFFFFu; h_slot[h] = 0xFFFFFFFFu; }
        // A: roots as of the start of the batch
        if (tid < nb) {
            uint32_t x = nx, y = ny;
            out_w[t0 + tid] = nw;
            s_vert[2 * tid] = x; s_vert[2 * tid + 1] = y;
            uint32_t px = __ldcg(uf + x), py = __ldcg(uf + y);
            while (px != x || py != y) {                   // the two walks advance together
                if (px != x) { x = px; px = __ldcg(uf + x); }
                if (py != y) { y = py; py = __ldcg(uf + y); }
            }
            s_root[2 * tid] = x; s_root[2 * tid + 1] = y;
        }
        if (t0 + DG_B + tid < m) { const uint32_t e = order[t0 + DG_B + tid]; nx = ta[e]; ny = tb[e]; nw = tw[e]; }   // in flight during B-D
        __syncthreads();
        // B: canonical slots through the hash table; the canonical ones load their root's (id, size)
        for (uint32_t s = tid; s < 2 * nb; s += DG_B) {
            const uint32_t r = s_root[s];
            uint32_t h = (r * 2654435761u) >> (32 - DG_HBITS);
            for (;;) {
                const uint32_t old = atomicCAS(&h_key[h], 0xFFFFFFFFu, r);
                if (old == 0xFFFFFFFFu || old == r) break;
                h = (h + 1) & (DG_H - 1);
            }
            atomicMin(&h_slot[h], s);
            s_hidx[s] = (uint16_t)h;
            s_par[s] = (uint16_t)s;
        }
        __syncthreads();
        uint32_t my_c[2];                                   // (2 slots per thread: 2 nb <= 2 DG_B)
        for (uint32_t s = tid, n = 0; s < 2 * nb; s += DG_B, ++n) {
            const uint32_t c = h_slot[s_hidx[s]];
            my_c[n] = c;
            if (c == s) { const unsigned long long v = __ldcg(info + s_root[s]); s_info[s] = make_uint2((uint32_t)v, (uint32_t)(v >> 32)); }
        }
        __syncthreads();                                    // the hash table is free from here on
        for (uint32_t s = tid, n = 0; s < 2 * nb; s += DG_B, ++n) { s_canon[s] = (uint16_t)my_c[n]; s_cnt[s] = 0; }
        __syncthreads();
        for (uint32_t s = tid; s < 2 * nb; s += DG_B) atomicAdd(&s_cnt[s_canon[s]], 1u);
        __syncthreads();
        // Classification.  A canonical slot referenced more than once in the batch is a HUB (in single linkage: the growing
        // cluster that the next edges chain onto).  If no edge joins two hubs, the batch falls apart into independent
        // pieces -- free edges (both sets referenced once) and one chain per hub, whose k-th edge only needs the running
        // (id, size) of its hub -- and phase C runs in parallel; otherwise one thread does the batch's unions in order.
        bool bad = false;
        if (tid < nb) {
            const uint32_t cx = s_canon[2 * tid], cy = s_canon[2 * tid + 1];
            const bool hx = s_cnt[cx] > 1, hy = s_cnt[cy] > 1;
            bad = (hx && hy) || cx == cy;
            s_hub[tid] = (uint16_t)(hx ? cx : (hy ? cy : 0xFFFFu));
        }
        const bool serial = __syncthreads_or(bad);
        // C: the unions, in edge order.  One thread, so what counts is the length of its dependent instruction
        // chain per edge: 32-bit (id, size) halves, results to shared memory (phase D writes them out, widened).
        if (!serial) {
            const uint32_t id0 = k + t0;
            if (tid < nb && s_hub[tid] == 0xFFFFu) {        // a free edge: nothing else in the batch touches its two sets
                const uint32_t x = s_canon[2 * tid], y = s_canon[2 * tid + 1];
                const uint2 ix = s_info[x], iy = s_info[y];
                const uint32_t sz = ix.x + iy.x;
                s_oa[tid] = min(ix.y, iy.y); s_ob[tid] = max(ix.y, iy.y); s_os[tid] = sz;
                const bool keep_x = ix.x >= iy.x;
                s_par[keep_x ? y : x] = (uint16_t)(keep_x ? x : y);
                s_info[keep_x ? x : y] = make_uint2(sz, id0 + tid);
            }
            for (uint32_t h = tid; h < 2 * nb; h += DG_B) { // one thread per hub walks the hub's edges in order
                if (s_canon[h] != h || s_cnt[h] < 2) continue;
                uint2 run = s_info[h];                      // the hub's running (size, id)
                for (uint32_t q0 = 0; q0 < nb; q0 += 4) {   // four edges at a time: their loads do not depend on `run`
                    uint32_t hub[4], oth[4]; uint2 io[4];
#pragma unroll
                    for (int r = 0; r < 4; ++r) {
                        const uint32_t q = min(q0 + r, nb - 1);
                        hub[r] = q0 + r < nb ? s_hub[q] : 0xFFFFu;
                        const uint32_t c0 = s_canon[2 * q], c1 = s_canon[2 * q + 1];
                        oth[r] = c0 == h ? c1 : c0;
                    }
#pragma unroll
                    for (int r = 0; r < 4; ++r) io[r] = s_info[oth[r]];
#pragma unroll
                    for (int r = 0; r < 4; ++r)
                        if (hub[r] == h) {
                            const uint32_t q = q0 + r, sz = run.x + io[r].x;
                            s_oa[q] = min(run.y, io[r].y); s_ob[q] = max(run.y, io[r].y); s_os[q] = sz;
                            s_par[oth[r]] = (uint16_t)h;
                            run = make_uint2(sz, id0 + q);
                        }
                }
                s_info[h] = run;
            }
        } else if (tid == 0) {
            const uint32_t* canon2 = reinterpret_cast<const uint32_t*>(s_canon);
            uint32_t cc = canon2[0];
            const uint32_t id0 = k + t0;
            for (uint32_t q = 0; q < nb; ++q) {
                const uint32_t cnext = canon2[q + 1];      // read ahead (slack entry past the batch)
                const uint32_t sx = cc & 0xFFFFu, sy = cc >> 16;
                uint32_t x = sx, y = sy;
                uint32_t px = s_par[x], py = s_par[y];
                uint2 ix = s_info[x], iy = s_info[y];      // valid if x, y are local roots (the common case); .x = size, .y = id
                if (px != x) { do { x = px; px = s_par[x]; } while (px != x); ix = s_info[x]; s_par[sx] = (uint16_t)x; }
                if (py != y) { do { y = py; py = s_par[y]; } while (py != y); iy = s_info[y]; s_par[sy] = (uint16_t)y; }
                const uint32_t sz = ix.x + iy.x;
                s_oa[q] = min(ix.y, iy.y); s_ob[q] = max(ix.y, iy.y); s_os[q] = sz;
                const bool keep_x = ix.x >= iy.x;            // the larger set stays the root
                const uint32_t root = keep_x ? x : y, child = keep_x ? y : x;
                s_par[child] = (uint16_t)root;
                s_info[root] = make_uint2(sz, id0 + q);
                cc = cnext;
            }
        }
        __syncthreads();
        if (tid < nb) { out_a[t0 + tid] = s_oa[tid]; out_b[t0 + tid] = s_ob[tid]; out_size[t0 + tid] = s_os[tid]; }
        // D: back to the global union-find
        for (uint32_t s = tid; s < 2 * nb; s += DG_B) {
            uint32_t f = s_canon[s];
            while (s_par[f] != f) f = s_par[f];            // read-only walk
            const uint32_t rf = s_root[f];
            if (s_canon[s] == s) {
                uf[s_root[s]] = rf;
                if (f == s) info[rf] = ((unsigned long long)s_info[s].y << 32) | s_info[s].x;
            }
            uf[s_vert[s]] = rf;                            // full compression of the queried leaves
        }
        __syncthreads();
    }
}

}  // namespace famsa

extern "C" int famsa_tree_finish(famsa_tree* t, int64_t* id_a_host, int64_t* id_b_host, float* sim_host, int64_t* size_host) {
    if (!t) { set_error("famsa_tree_finish: tree is NULL"); return FAMSA_EINVAL; }
    if (t->k < 2) return FAMSA_OK;
    int rc = tree_read_state(t);
    if (rc != FAMSA_OK) return rc;
    if ((int64_t)t->h_st->m != t->k - 1 || (!t->merged && t->rows < t->k)) {
        set_error("famsa_tree_finish: the forest has " + std::to_string(t->h_st->m) + " of " + std::to_string(t->k - 1) +
                  " edges: not every row has been consumed or merged in"); return FAMSA_ERANGE;
    }
    if (!id_a_host || !id_b_host || !sim_host || !size_host) { set_error("famsa_tree_finish: null output"); return FAMSA_EINVAL; }
    const uint32_t k = (uint32_t)t->k, m = k - 1;
    const int cur = t->cur;
    // one scratch allocation, carved up (256-byte aligned pieces)
    size_t off = 0;
    auto carve = [&](size_t bytes) { const size_t o = off; off += (bytes + 255) & ~(size_t)255; return o; };
    size_t b1 = 0, b2 = 0;
    FAMSA_CUDA(cub::DeviceRadixSort::SortPairs(nullptr, b1, (unsigned long long*)nullptr, (unsigned long long*)nullptr, (uint32_t*)nullptr, (uint32_t*)nullptr, (int)m));
    FAMSA_CUDA(cub::DeviceRadixSort::SortPairs(nullptr, b2, (uint32_t*)nullptr, (uint32_t*)nullptr, (uint32_t*)nullptr, (uint32_t*)nullptr, (int)m));
    const size_t o_idk = carve(8ull * m), o_idk2 = carve(8ull * m), o_wk = carve(4ull * m), o_wk2 = carve(4ull * m);
    const size_t o_idx = carve(4ull * m), o_idx2 = carve(4ull * m), o_order = carve(4ull * m), o_uf = carve(4ull * k), o_info = carve(8ull * k);
    const size_t o_oa = carve(8ull * m), o_ob = carve(8ull * m), o_osz = carve(8ull * m), o_ow = carve(4ull * m), o_cub = carve(std::max(b1, b2));
    uint8_t* base = nullptr;
    if (cache_alloc(t->device, (void**)&base, off) != cudaSuccess) { cudaGetLastError(); set_error("famsa_tree_finish: device allocation failed"); return FAMSA_ENOMEM; }
    struct Guard { uint8_t* p; ~Guard() { cudaDeviceSynchronize(); cache_free(p); } } guard{base};   // scratch from the block cache (famsa_trim releases it)
    unsigned long long *idk = (unsigned long long*)(base + o_idk), *idk2 = (unsigned long long*)(base + o_idk2), *info = (unsigned long long*)(base + o_info);
    uint32_t *wk = (uint32_t*)(base + o_wk), *wk2 = (uint32_t*)(base + o_wk2), *idx = (uint32_t*)(base + o_idx), *idx2 = (uint32_t*)(base + o_idx2);
    uint32_t *order = (uint32_t*)(base + o_order), *uf = (uint32_t*)(base + o_uf);
    long long *oa = (long long*)(base + o_oa), *ob = (long long*)(base + o_ob), *osz = (long long*)(base + o_osz);
    float* ow = (float*)(base + o_ow);
    void* cubtmp = base + o_cub;
    const unsigned g = (m + 255) / 256;
    tree_sortkeys_kernel<<<g, 256>>>(m, t->ta[cur], t->tb[cur], idk, idx);
    FAMSA_CUDA(cub::DeviceRadixSort::SortPairs(cubtmp, b1, idk, idk2, idx, idx2, (int)m));      // two stable passes: by edge id,
    tree_wkeys_kernel<<<g, 256>>>(m, t->tw[cur], idx2, wk);
    FAMSA_CUDA(cub::DeviceRadixSort::SortPairs(cubtmp, b2, wk, wk2, idx2, order, (int)m));       // then by similarity
    tree_uf_init_kernel<<<(k + 255) / 256, 256>>>(k, uf, info);
    tree_dendrogram_kernel<<<1, DG_B>>>(k, order, t->ta[cur], t->tb[cur], t->tw[cur], uf, info, oa, ob, ow, osz);
    t->launches += 10;
    FAMSA_CUDA(cudaGetLastError());
    static_assert(sizeof(long long) == sizeof(int64_t), "int64_t");
    FAMSA_CUDA(cudaMemcpy(id_a_host, oa, 8ull * m, cudaMemcpyDeviceToHost));
    FAMSA_CUDA(cudaMemcpy(id_b_host, ob, 8ull * m, cudaMemcpyDeviceToHost));
    FAMSA_CUDA(cudaMemcpy(size_host, osz, 8ull * m, cudaMemcpyDeviceToHost));
    FAMSA_CUDA(cudaMemcpy(sim_host, ow, 4ull * m, cudaMemcpyDeviceToHost));
    return FAMSA_OK;
}

extern "C" int famsa_guide_forest(famsa_ctx* ctx, int64_t block_rows, int64_t part, int64_t parts, famsa_tree** out) {
    if (!out) { set_error("famsa_guide_forest: out is NULL"); return FAMSA_EINVAL; }
    *out = nullptr;
    if (!ctx) { set_error("famsa_guide_forest: ctx is NULL"); return FAMSA_EINVAL; }
    if (block_rows < 0 || parts < 1 || part < 0 || part >= parts) { set_error("famsa_guide_forest: bad block_rows / part / parts"); return FAMSA_EINVAL; }
    if (block_rows == 0) block_rows = TREE_SUB_ROWS;
    if (block_rows > TREE_SUB_ROWS) { set_error("famsa_guide_forest: block_rows must be <= 1024"); return FAMSA_EINVAL; }
    const int64_t k = ctx->k;
    FAMSA_CUDA(cudaSetDevice(ctx->device));
    famsa_tree* t = nullptr;
    int rc = famsa_tree_create(k, ctx->device, &t);
    if (rc != FAMSA_OK) return rc;
    const int64_t nb_all = (k + block_rows - 1) / block_rows;
    std::vector<int64_t> mine;                             // this part's row blocks: part, part + parts, ...
    for (int64_t b = part; b < nb_all; b += parts) mine.push_back(b);
    const int64_t nb = (int64_t)mine.size();
    if (k < 2 || nb == 0) { *out = t; return FAMSA_OK; }
    auto rows_of = [&](int64_t n, int64_t& i0, int64_t& i1) { i0 = mine[n] * block_rows; i1 = std::min(i0 + block_rows, k); };
    int64_t i0, i1;
    int64_t max_pairs = 1;                                 // (the last block may be short: take the max)
    for (int64_t n = 0; n < nb; ++n) { rows_of(n, i0, i1); max_pairs = std::max(max_pairs, famsa_rows_pairs(i0, i1)); }
    float* buf[2] = {nullptr, nullptr};
    cudaStream_t sa = nullptr, sb = nullptr;
    cudaEvent_t ev_swept[2] = {nullptr, nullptr}, ev_merged[2] = {nullptr, nullptr};
    auto cleanup = [&](bool keep_tree) {
        cudaDeviceSynchronize();
        cudaFree(buf[0]); cudaFree(buf[1]);
        if (sa) cudaStreamDestroy(sa);
        if (sb) cudaStreamDestroy(sb);
        for (int q = 0; q < 2; ++q) { if (ev_swept[q]) cudaEventDestroy(ev_swept[q]); if (ev_merged[q]) cudaEventDestroy(ev_merged[q]); }
        if (!keep_tree) famsa_tree_free(t);
    };
#define GT_CUDA(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) { int r__ = (e__ == cudaErrorMemoryAllocation) ? FAMSA_ENOMEM : FAMSA_ECUDA; \
        famsa::cuda_fail(e__, #call); cleanup(false); return r__; } } while (0)
#define GT_TRY(x) do { int r__ = (x); if (r__ != FAMSA_OK) { cleanup(false); return r__; } } while (0)
    GT_CUDA(cudaMalloc((void**)&buf[0], std::max<int64_t>(max_pairs, 1) * sizeof(float)));
    GT_CUDA(cudaMalloc((void**)&buf[1], std::max<int64_t>(max_pairs, 1) * sizeof(float)));
    int prio_lo = 0, prio_hi = 0;
    GT_CUDA(cudaDeviceGetStreamPriorityRange(&prio_lo, &prio_hi));
    GT_CUDA(cudaStreamCreateWithPriority(&sa, cudaStreamNonBlocking, prio_lo));
    GT_CUDA(cudaStreamCreateWithPriority(&sb, cudaStreamNonBlocking, prio_hi));   // the tree's small kernels go first when SM resources free up
    for (int q = 0; q < 2; ++q) {
        GT_CUDA(cudaEventCreateWithFlags(&ev_swept[q], cudaEventDisableTiming));
        GT_CUDA(cudaEventCreateWithFlags(&ev_merged[q], cudaEventDisableTiming));
    }
    // Pipeline, all enqueued without a host round trip: stream sa sweeps block n into buffer n & 1 (its epilogue
    // also leaves the round-0 candidates in candidate slot n & 1), stream sb merges block n into the forest;
    // the sweep of block n + 2 waits for the merge of block n (same buffer and slot).
    for (int64_t n = 0; n < nb; ++n) {
        const int q = (int)(n & 1);
        rows_of(n, i0, i1);
        if (n >= 2) GT_CUDA(cudaStreamWaitEvent(sa, ev_merged[q], 0));
        if (famsa_rows_pairs(i0, i1) > 0) {
            GT_TRY(famsa::tree_fused_begin(t, i0, i1, q, sa));
            famsa::TreeCand tc{t->cand_row[q], t->cand_col[q]};
            GT_TRY(famsa::sweep_rows(ctx, i0, i1, nullptr, buf[q], nullptr, &tc, sa));
        }
        GT_CUDA(cudaEventRecord(ev_swept[q], sa));
        GT_CUDA(cudaStreamWaitEvent(sb, ev_swept[q], 0));
        if (famsa_rows_pairs(i0, i1) > 0) GT_TRY(famsa::tree_consume(t, i0, i1, buf[q], i0 * (i0 - 1) / 2, q, true, sb));
        t->rows += i1 - i0;
        GT_CUDA(cudaEventRecord(ev_merged[q], sb));
    }
    cleanup(true);
    ctx->launches += t->launches;
    *out = t;
    return FAMSA_OK;
#undef GT_CUDA
#undef GT_TRY
}

extern "C" int famsa_guide_tree(famsa_ctx* ctx, int64_t block_rows, int64_t* id_a_host, int64_t* id_b_host,
                                float* sim_host, int64_t* size_host) {
    famsa_tree* t = nullptr;
    int rc = famsa_guide_forest(ctx, block_rows, 0, 1, &t);
    if (rc != FAMSA_OK) return rc;
    const int64_t before = t->launches;
    rc = famsa_tree_finish(t, id_a_host, id_b_host, sim_host, size_host);
    ctx->launches += t->launches - before;
    famsa_tree_free(t);
    return rc;
}
