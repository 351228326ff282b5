// famsa_tree.cu -- stage II consumer: single-linkage guide tree built incrementally from the streamed
// similarity row blocks in O(k) memory.  See include/famsa_lcs.h.
//
// State: the maximum spanning FOREST T of the similarity entries seen so far (<= k-1 edges).  Single
// linkage = the spanning tree's edges taken by decreasing similarity, so T is an O(k) summary from which
// the dendrogram follows, and MSF(E1 u E2) = MSF(MSF(E1) u E2): a row block [i0, i1) -- in any order --
// is merged in by Boruvka rounds over (T's edges) + (the block's dense entries (v, u < v)); the forests
// of several ranks are merged the same way from their edge lists (famsa_tree_merge_edges).
// Every edge has a unique key (similarity descending, then (max, min) endpoint ascending), so each
// round's picks are edges of the one MSF under that order and only mutual picks form 2-cycles.
// A round is data-parallel: two streaming passes over the block (best edge per new row, best edge
// per column), then O(k) per-component reductions with 32/64-bit atomics, hooking and relabelling.
#include <cub/device/device_radix_sort.cuh>

#include <algorithm>
#include <cmath>
#include <new>

#include "famsa_internal.h"

struct famsa_tree {
    int      device = 0;
    int64_t  k = 0;
    int64_t  rows = 0;                 // rows consumed so far (any order)
    int64_t  max_row_end = 0;          // largest i1 seen: leaves 0..max_row_end-1 are one component
    int64_t  m = 0;                    // edges of the current forest
    bool     merged = false;           // sparse edges were merged in: components above max_row_end may exist
    uint32_t *ta[2] = {nullptr, nullptr}, *tb[2] = {nullptr, nullptr};   // tree edges, a > b (double buffer)
    float    *tw[2] = {nullptr, nullptr};
    int      cur = 0;
    uint32_t *comp[2] = {nullptr, nullptr}, *parent = nullptr;
    float    *cand_w[2] = {nullptr, nullptr};      // [0] as row owner (new vertices), [1] as column owner
    uint32_t *cand_o[2] = {nullptr, nullptr};
    uint32_t *best_w = nullptr;                    // per component: float bits + 1 (0 = none)
    unsigned long long* best_id = nullptr;         // per component: (max << 32) | min of the chosen edge
    uint32_t *counters = nullptr;                  // [0] edges recorded, [1] roots
    uint32_t *h_counters = nullptr;                // pinned
    int64_t  launches = 0, rounds = 0;
};

namespace famsa {

constexpr float NO_EDGE = -1.0f;       // similarities are >= 0

__device__ __forceinline__ bool better(float w, uint32_t o, float bw, uint32_t bo) {
    return w > bw || (w == bw && o < bo);
}

// Best edge of each NEW vertex v (a row of the block) to a different component, over columns u < v.
// A CTA takes ROW_R consecutive rows: one load of comp[u] serves all of them and each thread keeps
// ROW_R x 4 independent loads in flight.  Measured on a 1.7 GB block: ROW_R = 1 (1024 CTAs) reads 5.7 TB/s,
// ROW_R = 4 (256 CTAs) only 2.9 TB/s -- the CTA count matters more than sharing comp[u]; ROW_R = 1 is used.
// HBM-bound: one pass over the block.
template <int ROW_R>
__global__ void __launch_bounds__(256) tree_row_kernel(const float* __restrict__ sim, uint32_t i0, uint32_t i1, int64_t out_base,
                                                       const uint32_t* __restrict__ comp, float* __restrict__ cw, uint32_t* __restrict__ co) {
    const uint32_t v0 = i0 + blockIdx.x * ROW_R;
    const float* row[ROW_R]; uint32_t cv[ROW_R], vv[ROW_R];
    float bw[ROW_R]; uint32_t bo[ROW_R];
#pragma unroll
    for (int r = 0; r < ROW_R; ++r) {
        const uint32_t v = min(v0 + r, i1 - 1);            // rows past the block repeat its last row (not stored)
        vv[r] = v0 + r < i1 ? v : 0;                       // ... with an empty column range
        row[r] = sim + ((int64_t)v * (v - 1) / 2 - out_base);
        cv[r] = comp[v]; bw[r] = NO_EDGE; bo[r] = 0xFFFFFFFFu;
    }
    uint32_t vmax = 0;
#pragma unroll
    for (int r = 0; r < ROW_R; ++r) vmax = max(vmax, vv[r]);
#pragma unroll 4
    for (uint32_t u = threadIdx.x; u < vmax; u += 256) {
        const uint32_t c = comp[u];
        float w[ROW_R];
#pragma unroll
        for (int r = 0; r < ROW_R; ++r) w[r] = u < vv[r] ? __ldg(row[r] + u) : NO_EDGE;   // all loads first: ROW_R in flight
#pragma unroll
        for (int r = 0; r < ROW_R; ++r)
            if (c != cv[r] && w[r] > bw[r]) { bw[r] = w[r]; bo[r] = u; }                  // u ascends per thread: first of equals stays
    }
    __shared__ float sw[ROW_R][8];
    __shared__ uint32_t so[ROW_R][8];
#pragma unroll
    for (int r = 0; r < ROW_R; ++r) {
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) {
            const float ow = __shfl_xor_sync(0xffffffffu, bw[r], d);
            const uint32_t oo = __shfl_xor_sync(0xffffffffu, bo[r], d);
            if (better(ow, oo, bw[r], bo[r])) { bw[r] = ow; bo[r] = oo; }
        }
        if ((threadIdx.x & 31) == 0) { sw[r][threadIdx.x >> 5] = bw[r]; so[r][threadIdx.x >> 5] = bo[r]; }
    }
    __syncthreads();
    if (threadIdx.x < ROW_R && v0 + threadIdx.x < i1) {
        const int r = threadIdx.x;
        float w = sw[r][0]; uint32_t o = so[r][0];
        for (int q = 1; q < 8; ++q)
            if (better(sw[r][q], so[r][q], w, o)) { w = sw[r][q]; o = so[r][q]; }
        cw[v0 + r] = w; co[v0 + r] = o;
    }
}

// Best edge of each vertex u < i1-1 (a column) to a different component, over the block's rows v > u.
// A CTA covers 64 consecutive columns with 8 row slices (threadIdx.y): consecutive threads read
// consecutive floats of a row (coalesced), each thread keeps several independent loads in flight, and
// the 8 slices of a column are combined in shared memory.  HBM-bound: one pass over the block.
constexpr int COL_X = 64, COL_Y = 8;
__global__ void __launch_bounds__(COL_X * COL_Y) tree_col_kernel(const float* __restrict__ sim, uint32_t i0, uint32_t i1, int64_t out_base,
                                                                 const uint32_t* __restrict__ comp, float* __restrict__ cw, uint32_t* __restrict__ co) {
    __shared__ uint32_t scomp[1024];
    __shared__ float sw[COL_Y][COL_X];
    __shared__ uint32_t so[COL_Y][COL_X];
    const uint32_t tid = threadIdx.y * COL_X + threadIdx.x;
    const uint32_t u = blockIdx.x * COL_X + threadIdx.x;
    const bool live = u + 1 < i1;
    const uint32_t cu = live ? comp[u] : 0;
    float bw = NO_EDGE; uint32_t bo = 0xFFFFFFFFu;
    for (uint32_t t0 = i0; t0 < i1; t0 += 1024) {           // the block's rows, 1024 at a time
        const uint32_t t1 = min(t0 + 1024, i1);
        __syncthreads();
        for (uint32_t t = tid; t0 + t < t1; t += COL_X * COL_Y) scomp[t] = comp[t0 + t];
        __syncthreads();
        if (live) {
            // rows v = first + threadIdx.y, + COL_Y, ...  (first = the first row of this pass below column u)
            const uint32_t first = max(t0, u + 1);
#pragma unroll 4
            for (uint32_t v = first + threadIdx.y; v < t1; v += COL_Y) {
                if (scomp[v - t0] != cu) {
                    const float w = __ldg(sim + ((int64_t)v * (v - 1) / 2 - out_base + u));
                    if (w > bw) { bw = w; bo = v; }          // v ascends within a slice: the first of equal weights stays
                }
            }
        }
    }
    sw[threadIdx.y][threadIdx.x] = bw; so[threadIdx.y][threadIdx.x] = bo;
    __syncthreads();
    if (threadIdx.y == 0 && live) {
#pragma unroll
        for (int q = 1; q < COL_Y; ++q)
            if (better(sw[q][threadIdx.x], so[q][threadIdx.x], bw, bo)) { bw = sw[q][threadIdx.x]; bo = so[q][threadIdx.x]; }
        cw[u] = bw; co[u] = bo;
    }
}

}  // namespace famsa

namespace famsa {

struct TreeArgs {
    uint32_t n;                 // all k leaves
    uint32_t i0, i1;            // rows of the dense block (i0 == i1: none)
    uint32_t m;                 // edges of the current forest
    uint32_t xm;                // extra sparse edges (famsa_tree_merge_edges)
    const uint32_t *xa, *xb; const float* xw;
    const uint32_t *ta, *tb; const float* tw;            // current forest
    uint32_t *na, *nb; float* nw;                        // new tree being recorded
    const uint32_t* comp; uint32_t* comp_next; uint32_t* parent;
    const float *cw_row, *cw_col; const uint32_t *co_row, *co_col;
    uint32_t* best_w; unsigned long long* best_id;
    uint32_t* counters;
};

__device__ __forceinline__ unsigned long long edge_id(uint32_t x, uint32_t y) {
    return ((unsigned long long)max(x, y) << 32) | min(x, y);
}

__global__ void tree_reset_kernel(TreeArgs a, int first) {
    const uint32_t x = blockIdx.x * blockDim.x + threadIdx.x;
    if (x < a.n) {
        a.best_w[x] = 0; a.best_id[x] = ~0ull;
        if (first) const_cast<uint32_t*>(a.comp)[x] = x;
    }
    if (x == 0) { a.counters[1] = 0; if (first) a.counters[0] = 0; }
}

// Items: [0, n) row candidates, [n, 2n) column candidates, [2n, 2n+m) forest edges, then xm extra edges.
// PASS 0: per component, the highest similarity of an outgoing edge.  PASS 1: among the edges that
// reach it, the smallest edge id.  Together: the component's minimum-key outgoing edge.
template <int PASS>
__global__ void tree_best_kernel(TreeArgs a) {
    const uint32_t t = blockIdx.x * blockDim.x + threadIdx.x;
    uint32_t x, y; float w;
    bool both = false;
    if (t < a.n) {
        if (t < a.i0 || t >= a.i1) return;
        x = t; w = a.cw_row[t]; y = a.co_row[t];
    } else if (t < 2 * a.n) {
        x = t - a.n;
        if (a.i1 == a.i0 || x + 1 >= a.i1) return;
        w = a.cw_col[x]; y = a.co_col[x];
    } else if (t < 2 * a.n + a.m) {
        const uint32_t e = t - 2 * a.n;
        x = a.ta[e]; y = a.tb[e]; w = a.tw[e];
        if (a.comp[x] == a.comp[y]) return;
        both = true;
    } else if (t < 2 * a.n + a.m + a.xm) {
        const uint32_t e = t - 2 * a.n - a.m;
        x = a.xa[e]; y = a.xb[e]; w = a.xw[e];
        if (x == y || a.comp[x] == a.comp[y]) return;
        both = true;
    } else {
        return;
    }
    if (__float_as_uint(w) & 0x80000000u) return;           // NO_EDGE, or any sign-bit-set weight (-0.0 included)
    const uint32_t key = __float_as_uint(w) + 1u;          // similarities >= +0: bit order == value order
    const uint32_t cx = a.comp[x];
    if (PASS == 0) {
        atomicMax(&a.best_w[cx], key);
        if (both) atomicMax(&a.best_w[a.comp[y]], key);
    } else {
        const unsigned long long id = edge_id(x, y);
        if (a.best_w[cx] == key) atomicMin(&a.best_id[cx], id);
        if (both) { const uint32_t cy = a.comp[y]; if (a.best_w[cy] == key) atomicMin(&a.best_id[cy], id); }
    }
}

// Each component root hooks onto the component at the other end of its edge (mutual picks: the
// smaller root stays) and records the edge once.
__global__ void tree_hook_kernel(TreeArgs a) {
    const uint32_t c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= a.n) return;
    if (a.comp[c] != c) { a.parent[c] = c; return; }        // not a representative
    const uint32_t key = a.best_w[c];
    if (key == 0) { a.parent[c] = c; return; }              // no outgoing edge: the last component
    const unsigned long long id = a.best_id[c];
    const uint32_t hi = (uint32_t)(id >> 32), lo = (uint32_t)id;
    const uint32_t other = a.comp[hi] == c ? lo : hi;
    const uint32_t t = a.comp[other];
    const bool mutual = a.best_id[t] == id;
    if (mutual && c < t) { a.parent[c] = c; return; }       // t hooks onto c and records the edge
    a.parent[c] = t;
    const uint32_t pos = atomicAdd(&a.counters[0], 1u);
    a.na[pos] = hi; a.nb[pos] = lo; a.nw[pos] = __uint_as_float(key - 1u);
}

__global__ void tree_relabel_kernel(TreeArgs a) {
    const uint32_t x = blockIdx.x * blockDim.x + threadIdx.x;
    if (x >= a.n) return;
    uint32_t r = a.comp[x];
    for (uint32_t p = a.parent[r]; p != r; p = a.parent[r]) {      // hooks form a forest of depth >= 1: climb with
        const uint32_t g = a.parent[p];                            // pointer jumping (benign race: every write is an
        if (g != p) a.parent[r] = g;                               // ancestor of r), so chains halve as they are walked
        r = p;
    }
    a.comp_next[x] = r;
    if (r == x) atomicAdd(&a.counters[1], 1u);              // x is a root of the new partition
}

template <typename T>
static int tree_alloc(T** p, size_t n) {
    cudaError_t e = cudaMalloc((void**)p, std::max<size_t>(n, 1) * sizeof(T));
    if (e == cudaErrorMemoryAllocation) { cudaGetLastError(); set_error("famsa_tree: device allocation failed"); return FAMSA_ENOMEM; }
    if (e != cudaSuccess) return cuda_fail(e, "cudaMalloc");
    return FAMSA_OK;
}

}  // namespace famsa

using namespace famsa;

#define TREE_TRY(x) do { int rc__ = (x); if (rc__ != FAMSA_OK) { famsa_tree_free(t); return rc__; } } while (0)

extern "C" void famsa_tree_free(famsa_tree* t) {
    if (!t) return;
    cudaSetDevice(t->device);
    for (int b = 0; b < 2; ++b) {
        cudaFree(t->ta[b]); cudaFree(t->tb[b]); cudaFree(t->tw[b]); cudaFree(t->comp[b]);
        cudaFree(t->cand_w[b]); cudaFree(t->cand_o[b]);
    }
    cudaFree(t->parent); cudaFree(t->best_w); cudaFree(t->best_id); cudaFree(t->counters);
    if (t->h_counters) cudaFreeHost(t->h_counters);
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
    const size_t n = (size_t)k;
    for (int b = 0; b < 2; ++b) {
        TREE_TRY(tree_alloc(&t->ta[b], n)); TREE_TRY(tree_alloc(&t->tb[b], n)); TREE_TRY(tree_alloc(&t->tw[b], n));
        TREE_TRY(tree_alloc(&t->comp[b], n)); TREE_TRY(tree_alloc(&t->cand_w[b], n)); TREE_TRY(tree_alloc(&t->cand_o[b], n));
    }
    TREE_TRY(tree_alloc(&t->parent, n)); TREE_TRY(tree_alloc(&t->best_w, n)); TREE_TRY(tree_alloc(&t->best_id, n));
    TREE_TRY(tree_alloc(&t->counters, 2));
    if (cudaMallocHost((void**)&t->h_counters, 2 * sizeof(uint32_t)) != cudaSuccess) {
        cudaGetLastError(); famsa_tree_free(t); set_error("famsa_tree_create: pinned allocation failed"); return FAMSA_ENOMEM;
    }
    *out = t;
    return FAMSA_OK;
}

namespace famsa {

// Boruvka rounds over (current forest) + (dense block rows [i0, i1), if any) + (xm extra edges).
static int tree_rounds(famsa_tree* t, int64_t i0, int64_t i1, const float* sim_block,
                       const uint32_t* xa, const uint32_t* xb, const float* xw, uint32_t xm, cudaStream_t st) {
    const int cur = t->cur, nxt = cur ^ 1;
    TreeArgs a;
    a.n = (uint32_t)t->k; a.i0 = (uint32_t)i0; a.i1 = (uint32_t)i1; a.m = (uint32_t)t->m;
    a.xa = xa; a.xb = xb; a.xw = xw; a.xm = xm;
    a.ta = t->ta[cur]; a.tb = t->tb[cur]; a.tw = t->tw[cur];
    a.na = t->ta[nxt]; a.nb = t->tb[nxt]; a.nw = t->tw[nxt];
    a.parent = t->parent;
    a.cw_row = t->cand_w[0]; a.co_row = t->cand_o[0]; a.cw_col = t->cand_w[1]; a.co_col = t->cand_o[1];
    a.best_w = t->best_w; a.best_id = t->best_id; a.counters = t->counters;
    const bool dense = i1 > i0 && i1 >= 2;
    const int64_t out_base = i0 * (i0 - 1) / 2;
    const unsigned gv = (unsigned)((a.n + 255) / 256);
    const unsigned gi = (unsigned)((2ull * a.n + a.m + a.xm + 255) / 256);
    // a dense row v links every u < v, so after any dense update leaves 0..max_row_end-1 are ONE component
    // and the leaves above are singletons: the round that reaches that count is the last one.  Without a
    // dense block (merge of sparse edges) the loop ends on the first round that hooks nothing.
    const int64_t max_end = std::max<int64_t>(t->max_row_end, dense ? i1 : 0);
    const uint32_t roots_done = max_end >= 2 ? (uint32_t)(1 + t->k - max_end) : (uint32_t)t->k;
    int cb = 0;                                            // which comp buffer holds the current labels
    uint32_t hooked = 0;
    for (int round = 0; round < 64; ++round) {
        a.comp = t->comp[cb]; a.comp_next = t->comp[cb ^ 1];
        tree_reset_kernel<<<gv, 256, 0, st>>>(a, round == 0);
        if (dense) {
            tree_row_kernel<1><<<(unsigned)(i1 - i0), 256, 0, st>>>(sim_block, a.i0, a.i1, out_base, a.comp, t->cand_w[0], t->cand_o[0]);
            tree_col_kernel<<<(unsigned)((a.i1 - 1 + COL_X - 1) / COL_X), dim3(COL_X, COL_Y), 0, st>>>(sim_block, a.i0, a.i1, out_base, a.comp, t->cand_w[1], t->cand_o[1]);
            t->launches += 2;
        }
        tree_best_kernel<0><<<gi, 256, 0, st>>>(a);
        tree_best_kernel<1><<<gi, 256, 0, st>>>(a);
        tree_hook_kernel<<<gv, 256, 0, st>>>(a);
        tree_relabel_kernel<<<gv, 256, 0, st>>>(a);
        FAMSA_CUDA(cudaMemcpyAsync(t->h_counters, t->counters, 2 * sizeof(uint32_t), cudaMemcpyDeviceToHost, st));
        FAMSA_CUDA(cudaStreamSynchronize(st));
        t->launches += 5; t->rounds++;
        cb ^= 1;
        const bool progress = t->h_counters[0] != hooked;
        hooked = t->h_counters[0];
        if (!progress || (!t->merged && xm == 0 && t->h_counters[1] == roots_done)) break;
    }
    FAMSA_CUDA(cudaGetLastError());
    if (hooked + t->h_counters[1] != (uint32_t)t->k || (!t->merged && xm == 0 && t->h_counters[1] != roots_done)) {
        set_error("famsa_tree: Boruvka did not converge (NaN similarities?)"); return FAMSA_EINVAL;
    }
    t->cur = nxt; t->m = hooked; t->max_row_end = max_end;
    return FAMSA_OK;
}

}  // namespace famsa

extern "C" int famsa_tree_update(famsa_tree* t, int64_t i0, int64_t i1, const float* sim_block, void* cuda_stream) {
    if (!t) { set_error("famsa_tree_update: tree is NULL"); return FAMSA_EINVAL; }
    if (i0 < 0 || i1 < i0 || i1 > t->k) { set_error("famsa_tree_update: bad row range"); return FAMSA_ERANGE; }
    if (i1 == i0) return FAMSA_OK;
    if (!sim_block && famsa_rows_pairs(i0, i1) > 0) { set_error("famsa_tree_update: sim_block is NULL"); return FAMSA_EINVAL; }
    FAMSA_CUDA(cudaSetDevice(t->device));
    if (famsa_rows_pairs(i0, i1) > 0) {
        int rc = tree_rounds(t, i0, i1, sim_block, nullptr, nullptr, nullptr, 0, (cudaStream_t)cuda_stream);
        if (rc != FAMSA_OK) return rc;
    }
    t->rows += i1 - i0;
    return FAMSA_OK;
}

extern "C" int famsa_tree_merge_edges(famsa_tree* t, const int64_t* a_host, const int64_t* b_host, const float* sim_host, int64_t m) {
    if (!t) { set_error("famsa_tree_merge_edges: tree is NULL"); return FAMSA_EINVAL; }
    if (m < 0 || (m > 0 && (!a_host || !b_host || !sim_host))) { set_error("famsa_tree_merge_edges: null input"); return FAMSA_EINVAL; }
    if (m == 0) return FAMSA_OK;
    if (m > 0x7FFFFFF0LL) { set_error("famsa_tree_merge_edges: too many edges"); return FAMSA_EINVAL; }
    FAMSA_CUDA(cudaSetDevice(t->device));
    std::vector<uint32_t> a(m), b(m);
    for (int64_t e = 0; e < m; ++e) {
        if (a_host[e] < 0 || a_host[e] >= t->k || b_host[e] < 0 || b_host[e] >= t->k || !(sim_host[e] >= 0.0f) || std::signbit(sim_host[e])) {
            set_error("famsa_tree_merge_edges: edge " + std::to_string(e) + " has a leaf out of range or a negative (-0.0 included) / NaN similarity");
            return FAMSA_ERANGE;
        }
        a[e] = (uint32_t)a_host[e]; b[e] = (uint32_t)b_host[e];
    }
    uint32_t *xa = nullptr, *xb = nullptr; float* xw = nullptr;
    cudaError_t e1 = cudaMalloc((void**)&xa, 4ull * m), e2 = cudaMalloc((void**)&xb, 4ull * m), e3 = cudaMalloc((void**)&xw, 4ull * m);
    int rc = FAMSA_OK;
    if (e1 != cudaSuccess || e2 != cudaSuccess || e3 != cudaSuccess) {
        cudaGetLastError(); set_error("famsa_tree_merge_edges: device allocation failed"); rc = FAMSA_ENOMEM;
    } else if (cudaMemcpy(xa, a.data(), 4ull * m, cudaMemcpyHostToDevice) != cudaSuccess ||
               cudaMemcpy(xb, b.data(), 4ull * m, cudaMemcpyHostToDevice) != cudaSuccess ||
               cudaMemcpy(xw, sim_host, 4ull * m, cudaMemcpyHostToDevice) != cudaSuccess) {
        rc = famsa::cuda_fail(cudaGetLastError(), "famsa_tree_merge_edges: copy");
    } else {
        rc = tree_rounds(t, 0, 0, nullptr, xa, xb, xw, (uint32_t)m, nullptr);
        if (rc == FAMSA_OK) t->merged = true;
    }
    cudaFree(xa); cudaFree(xb); cudaFree(xw);
    return rc;
}

extern "C" int64_t famsa_tree_edge_count(const famsa_tree* t) { return t ? t->m : 0; }

extern "C" int famsa_tree_edges(famsa_tree* t, int64_t* a_host, int64_t* b_host, float* sim_host) {
    if (!t) { set_error("famsa_tree_edges: tree is NULL"); return FAMSA_EINVAL; }
    const int64_t m = t->m;
    if (m == 0) return FAMSA_OK;
    if (!a_host || !b_host || !sim_host) { set_error("famsa_tree_edges: null output"); return FAMSA_EINVAL; }
    FAMSA_CUDA(cudaSetDevice(t->device));
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

// The dendrogram from the sorted tree edges: a union-find pass, inherently sequential (O(k alpha(k))
// L2-resident steps, once per tree).  One warp: all lanes stage a batch of edges in shared memory and
// write the batch's merges back (coalesced), lane 0 runs the union-find of the batch in between, so the
// serial path touches global memory only for the union-find arrays themselves.
constexpr int DG_BATCH = 1024;
__global__ void __launch_bounds__(32) tree_dendrogram_kernel(uint32_t k, const uint32_t* order, const uint32_t* ta, const uint32_t* tb, const float* tw,
                                                             uint32_t* uf, long long* cid, long long* csize,
                                                             long long* out_a, long long* out_b, float* out_w, long long* out_size) {
    __shared__ uint32_t sa[DG_BATCH], sb[DG_BATCH];
    __shared__ long long oa[DG_BATCH], ob[DG_BATCH], os[DG_BATCH];
    const uint32_t lane = threadIdx.x, m = k - 1;
    for (uint32_t x = lane; x < k; x += 32) { uf[x] = x; cid[x] = x; csize[x] = 1; }
    __syncwarp();
    for (uint32_t t0 = 0; t0 < m; t0 += DG_BATCH) {
        const uint32_t nb = min((uint32_t)DG_BATCH, m - t0);
        for (uint32_t q = lane; q < nb; q += 32) {
            const uint32_t e = order[t0 + q];
            sa[q] = ta[e]; sb[q] = tb[e]; out_w[t0 + q] = tw[e];
        }
        __syncwarp();
        if (lane == 0) {
            for (uint32_t q = 0; q < nb; ++q) {
                uint32_t ra = sa[q], rb = sb[q];
                uint32_t pa = uf[ra], pb = uf[rb];                  // the two finds advance together
                while (pa != ra || pb != rb) {
                    if (pa != ra) { const uint32_t g = uf[pa]; uf[ra] = g; ra = g; pa = uf[ra]; }
                    if (pb != rb) { const uint32_t g = uf[pb]; uf[rb] = g; rb = g; pb = uf[rb]; }
                }
                const long long ia = cid[ra], ib = cid[rb];
                const long long za = csize[ra], zb = csize[rb];
                oa[q] = ia < ib ? ia : ib; ob[q] = ia < ib ? ib : ia; os[q] = za + zb;
                if (za < zb) { const uint32_t s = ra; ra = rb; rb = s; }
                uf[rb] = ra; csize[ra] = za + zb; cid[ra] = (long long)k + t0 + q;
            }
        }
        __syncwarp();
        for (uint32_t q = lane; q < nb; q += 32) { out_a[t0 + q] = oa[q]; out_b[t0 + q] = ob[q]; out_size[t0 + q] = os[q]; }
        __syncwarp();
    }
}

}  // namespace famsa

extern "C" int famsa_tree_finish(famsa_tree* t, int64_t* id_a_host, int64_t* id_b_host, float* sim_host, int64_t* size_host) {
    if (!t) { set_error("famsa_tree_finish: tree is NULL"); return FAMSA_EINVAL; }
    if (t->k < 2) return FAMSA_OK;
    if (t->m != t->k - 1 || (!t->merged && t->rows < t->k)) {
        set_error("famsa_tree_finish: the forest has " + std::to_string(t->m) + " of " + std::to_string(t->k - 1) +
                  " edges: not every row has been consumed or merged in"); return FAMSA_ERANGE;
    }
    if (!id_a_host || !id_b_host || !sim_host || !size_host) { set_error("famsa_tree_finish: null output"); return FAMSA_EINVAL; }
    FAMSA_CUDA(cudaSetDevice(t->device));
    const uint32_t k = (uint32_t)t->k, m = k - 1;
    const int cur = t->cur;
    struct Tmp { std::vector<void*> p; ~Tmp() { for (void* q : p) cudaFree(q); } } tmp;
    auto dalloc = [&](void** p, size_t bytes) { cudaError_t e = cudaMalloc(p, std::max<size_t>(bytes, 16)); if (e == cudaSuccess) tmp.p.push_back(*p); return e; };
    unsigned long long *idk = nullptr, *idk2 = nullptr; uint32_t *wk = nullptr, *wk2 = nullptr, *idx = nullptr, *idx2 = nullptr, *order = nullptr, *uf = nullptr;
    long long *cid = nullptr, *csize = nullptr, *oa = nullptr, *ob = nullptr, *osz = nullptr; float* ow = nullptr; void* cubtmp = nullptr;
    FAMSA_CUDA(dalloc((void**)&idk, 8ull * m)); FAMSA_CUDA(dalloc((void**)&idk2, 8ull * m));
    FAMSA_CUDA(dalloc((void**)&wk, 4ull * m)); FAMSA_CUDA(dalloc((void**)&wk2, 4ull * m));
    FAMSA_CUDA(dalloc((void**)&idx, 4ull * m)); FAMSA_CUDA(dalloc((void**)&idx2, 4ull * m)); FAMSA_CUDA(dalloc((void**)&order, 4ull * m));
    FAMSA_CUDA(dalloc((void**)&uf, 4ull * k)); FAMSA_CUDA(dalloc((void**)&cid, 8ull * k)); FAMSA_CUDA(dalloc((void**)&csize, 8ull * k));
    FAMSA_CUDA(dalloc((void**)&oa, 8ull * m)); FAMSA_CUDA(dalloc((void**)&ob, 8ull * m)); FAMSA_CUDA(dalloc((void**)&osz, 8ull * m));
    FAMSA_CUDA(dalloc((void**)&ow, 4ull * m));
    const unsigned g = (m + 255) / 256;
    tree_sortkeys_kernel<<<g, 256>>>(m, t->ta[cur], t->tb[cur], idk, idx);
    size_t b1 = 0, b2 = 0;                                  // two stable passes: by edge id, then by similarity
    FAMSA_CUDA(cub::DeviceRadixSort::SortPairs(nullptr, b1, idk, idk2, idx, idx2, (int)m));
    FAMSA_CUDA(cub::DeviceRadixSort::SortPairs(nullptr, b2, wk, wk2, idx2, order, (int)m));
    FAMSA_CUDA(dalloc(&cubtmp, std::max(b1, b2)));
    FAMSA_CUDA(cub::DeviceRadixSort::SortPairs(cubtmp, b1, idk, idk2, idx, idx2, (int)m));
    tree_wkeys_kernel<<<g, 256>>>(m, t->tw[cur], idx2, wk);
    FAMSA_CUDA(cub::DeviceRadixSort::SortPairs(cubtmp, b2, wk, wk2, idx2, order, (int)m));
    tree_dendrogram_kernel<<<1, 32>>>(k, order, t->ta[cur], t->tb[cur], t->tw[cur], uf, cid, csize, oa, ob, ow, osz);
    t->launches += 9;
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
    if (block_rows == 0) block_rows = 1024;
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
    cudaEvent_t ev[2] = {nullptr, nullptr};
    auto cleanup = [&](bool keep_tree) {
        cudaDeviceSynchronize();
        cudaFree(buf[0]); cudaFree(buf[1]);
        if (sa) cudaStreamDestroy(sa);
        if (sb) cudaStreamDestroy(sb);
        if (ev[0]) cudaEventDestroy(ev[0]);
        if (ev[1]) cudaEventDestroy(ev[1]);
        if (!keep_tree) famsa_tree_free(t);
    };
#define GT_CUDA(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) { int r__ = (e__ == cudaErrorMemoryAllocation) ? FAMSA_ENOMEM : FAMSA_ECUDA; \
        famsa::cuda_fail(e__, #call); cleanup(false); return r__; } } while (0)
#define GT_TRY(x) do { int r__ = (x); if (r__ != FAMSA_OK) { cleanup(false); return r__; } } while (0)
    GT_CUDA(cudaMalloc((void**)&buf[0], std::max<int64_t>(max_pairs, 1) * sizeof(float)));
    GT_CUDA(cudaMalloc((void**)&buf[1], std::max<int64_t>(max_pairs, 1) * sizeof(float)));
    GT_CUDA(cudaStreamCreateWithFlags(&sa, cudaStreamNonBlocking));
    GT_CUDA(cudaStreamCreateWithFlags(&sb, cudaStreamNonBlocking));
    GT_CUDA(cudaEventCreateWithFlags(&ev[0], cudaEventDisableTiming));
    GT_CUDA(cudaEventCreateWithFlags(&ev[1], cudaEventDisableTiming));
    rows_of(0, i0, i1);
    if (famsa_rows_pairs(i0, i1) > 0) GT_TRY(famsa::sweep_rows(ctx, i0, i1, nullptr, buf[0], nullptr, sa));
    GT_CUDA(cudaEventRecord(ev[0], sa));
    for (int64_t n = 0; n < nb; ++n) {
        if (n + 1 < nb) {                                  // sweep the next block while this one is merged
            int64_t n0, n1;
            rows_of(n + 1, n0, n1);
            GT_TRY(famsa::sweep_rows(ctx, n0, n1, nullptr, buf[(n + 1) & 1], nullptr, sa));
            GT_CUDA(cudaEventRecord(ev[(n + 1) & 1], sa));
        }
        rows_of(n, i0, i1);
        GT_CUDA(cudaStreamWaitEvent(sb, ev[n & 1], 0));
        GT_TRY(famsa_tree_update(t, i0, i1, buf[n & 1], sb));
    }
    ctx->launches += t->launches;
    cleanup(true);
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
