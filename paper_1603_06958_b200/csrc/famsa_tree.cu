// famsa_tree.cu -- stage II consumer: single-linkage guide tree built incrementally from the streamed
// similarity row blocks in O(k) memory.  See include/famsa_lcs.h.
//
// State: the maximum spanning tree T of the complete similarity graph over the rows consumed so far
// (n-1 edges).  Single linkage = T's edges taken by decreasing similarity, so T is an O(k) summary
// from which the dendrogram follows, and MST(G + new rows) = MST(T + new rows): a row block [i0, i1)
// is merged in by Boruvka rounds over the graph (T's edges) + (the block's dense entries (v, u < v)).
// Every edge has a unique key (similarity descending, then (max, min) endpoint ascending), so each
// round's picks are edges of the one MST under that order and only mutual picks form 2-cycles.
// A round is data-parallel: two streaming passes over the block (best edge per new row, best edge
// per column), then O(k) per-component reductions with 32/64-bit atomics, hooking and relabelling.
#include <cub/device/device_radix_sort.cuh>

#include <algorithm>
#include <new>

#include "famsa_internal.h"

struct famsa_tree {
    int      device = 0;
    int64_t  k = 0;
    int64_t  rows = 0;                 // rows consumed so far; T has max(rows-1, 0) edges
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
__global__ void __launch_bounds__(256) tree_row_kernel(const float* __restrict__ sim, uint32_t i0, uint32_t i1, int64_t out_base,
                                                       const uint32_t* __restrict__ comp, float* __restrict__ cw, uint32_t* __restrict__ co) {
    const uint32_t v = i0 + blockIdx.x;
    const float* row = sim + ((int64_t)v * (v - 1) / 2 - out_base);
    const uint32_t cv = comp[v];
    float bw = NO_EDGE; uint32_t bo = 0xFFFFFFFFu;
    for (uint32_t u = threadIdx.x; u < v; u += 256) {
        if (comp[u] != cv) {
            const float w = __ldg(row + u);
            if (better(w, u, bw, bo)) { bw = w; bo = u; }
        }
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        const float ow = __shfl_xor_sync(0xffffffffu, bw, d);
        const uint32_t oo = __shfl_xor_sync(0xffffffffu, bo, d);
        if (better(ow, oo, bw, bo)) { bw = ow; bo = oo; }
    }
    __shared__ float sw[8];
    __shared__ uint32_t so[8];
    if ((threadIdx.x & 31) == 0) { sw[threadIdx.x >> 5] = bw; so[threadIdx.x >> 5] = bo; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int q = 1; q < 8; ++q)
            if (better(sw[q], so[q], bw, bo)) { bw = sw[q]; bo = so[q]; }
        cw[v] = bw; co[v] = bo;
    }
}

// Best edge of each vertex u < i1-1 (a column) to a different component, over the block's rows v > u.
__global__ void __launch_bounds__(256) tree_col_kernel(const float* __restrict__ sim, uint32_t i0, uint32_t i1, int64_t out_base,
                                                       const uint32_t* __restrict__ comp, float* __restrict__ cw, uint32_t* __restrict__ co) {
    __shared__ uint32_t scomp[1024];
    const uint32_t u = blockIdx.x * 256 + threadIdx.x;
    const bool live = u + 1 < i1;
    const uint32_t cu = live ? comp[u] : 0;
    float bw = NO_EDGE; uint32_t bo = 0xFFFFFFFFu;
    for (uint32_t t0 = i0; t0 < i1; t0 += 1024) {           // the block's rows, 1024 at a time
        const uint32_t t1 = min(t0 + 1024, i1);
        __syncthreads();
        for (uint32_t t = threadIdx.x; t0 + t < t1; t += 256) scomp[t] = comp[t0 + t];
        __syncthreads();
        if (live) {
            uint32_t v = max(t0, u + 1);
            int64_t off = (int64_t)v * (v - 1) / 2 - out_base + u;
            for (; v < t1; ++v) {
                if (scomp[v - t0] != cu) {
                    const float w = __ldg(sim + off);
                    if (w > bw) { bw = w; bo = v; }          // v ascends: the first of equal weights stays
                }
                off += v;
            }
        }
    }
    if (live) { cw[u] = bw; co[u] = bo; }
}

}  // namespace famsa

namespace famsa {

struct TreeArgs {
    uint32_t n;                 // vertices after this update (= i1)
    uint32_t i0, i1;
    uint32_t m;                 // old tree edges (i0 - 1, or 0)
    const uint32_t *ta, *tb; const float* tw;            // old tree
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

// Items: [0, n) row candidates, [n, 2n) column candidates, [2n, 2n+m) old tree edges.
// PASS 0: per component, the highest similarity of an outgoing edge.  PASS 1: among the edges that
// reach it, the smallest edge id.  Together: the component's minimum-key outgoing edge.
template <int PASS>
__global__ void tree_best_kernel(TreeArgs a) {
    const uint32_t t = blockIdx.x * blockDim.x + threadIdx.x;
    uint32_t x, y; float w;
    bool both = false;
    if (t < a.n) {
        if (t < a.i0) return;
        x = t; w = a.cw_row[t]; y = a.co_row[t];
    } else if (t < 2 * a.n) {
        x = t - a.n;
        if (x + 1 >= a.i1) return;
        w = a.cw_col[x]; y = a.co_col[x];
    } else if (t < 2 * a.n + a.m) {
        const uint32_t e = t - 2 * a.n;
        x = a.ta[e]; y = a.tb[e]; w = a.tw[e];
        if (a.comp[x] == a.comp[y]) return;
        both = true;
    } else {
        return;
    }
    if (w < 0.0f) return;                                   // NO_EDGE
    const uint32_t key = __float_as_uint(w) + 1u;          // similarities >= 0: bit order == value order
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
    while (a.parent[r] != r) r = a.parent[r];
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

extern "C" int famsa_tree_update(famsa_tree* t, int64_t i0, int64_t i1, const float* sim_block, void* cuda_stream) {
    if (!t) { set_error("famsa_tree_update: tree is NULL"); return FAMSA_EINVAL; }
    if (i0 != t->rows || i1 < i0 || i1 > t->k) {
        set_error("famsa_tree_update: rows must arrive in order: expected i0 = " + std::to_string(t->rows)); return FAMSA_ERANGE;
    }
    if (i1 == i0) return FAMSA_OK;
    if (!sim_block && famsa_rows_pairs(i0, i1) > 0) { set_error("famsa_tree_update: sim_block is NULL"); return FAMSA_EINVAL; }
    FAMSA_CUDA(cudaSetDevice(t->device));
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int cur = t->cur, nxt = cur ^ 1;
    TreeArgs a;
    a.n = (uint32_t)i1; a.i0 = (uint32_t)i0; a.i1 = (uint32_t)i1; a.m = i0 > 0 ? (uint32_t)(i0 - 1) : 0;
    a.ta = t->ta[cur]; a.tb = t->tb[cur]; a.tw = t->tw[cur];
    a.na = t->ta[nxt]; a.nb = t->tb[nxt]; a.nw = t->tw[nxt];
    a.parent = t->parent;
    a.cw_row = t->cand_w[0]; a.co_row = t->cand_o[0]; a.cw_col = t->cand_w[1]; a.co_col = t->cand_o[1];
    a.best_w = t->best_w; a.best_id = t->best_id; a.counters = t->counters;
    const int64_t out_base = i0 * (i0 - 1) / 2;
    const unsigned gv = (unsigned)((a.n + 255) / 256);
    const unsigned gi = (unsigned)((2ull * a.n + a.m + 255) / 256);
    int cb = 0;                                            // which comp buffer holds the current labels
    if (a.n >= 2) {
        for (int round = 0; round < 64; ++round) {
            a.comp = t->comp[cb]; a.comp_next = t->comp[cb ^ 1];
            tree_reset_kernel<<<gv, 256, 0, st>>>(a, round == 0);
            tree_row_kernel<<<(unsigned)(i1 - i0), 256, 0, st>>>(sim_block, a.i0, a.i1, out_base, a.comp, t->cand_w[0], t->cand_o[0]);
            tree_col_kernel<<<(unsigned)((a.i1 - 1 + 255) / 256), 256, 0, st>>>(sim_block, a.i0, a.i1, out_base, a.comp, t->cand_w[1], t->cand_o[1]);
            tree_best_kernel<0><<<gi, 256, 0, st>>>(a);
            tree_best_kernel<1><<<gi, 256, 0, st>>>(a);
            tree_hook_kernel<<<gv, 256, 0, st>>>(a);
            tree_relabel_kernel<<<gv, 256, 0, st>>>(a);
            FAMSA_CUDA(cudaMemcpyAsync(t->h_counters, t->counters, 2 * sizeof(uint32_t), cudaMemcpyDeviceToHost, st));
            FAMSA_CUDA(cudaStreamSynchronize(st));
            t->launches += 7; t->rounds++;
            cb ^= 1;
            if (t->h_counters[1] <= 1) break;
        }
        FAMSA_CUDA(cudaGetLastError());
        if (t->h_counters[1] != 1 || t->h_counters[0] != a.n - 1) {
            set_error("famsa_tree_update: Boruvka did not converge (NaN similarities?)"); return FAMSA_EINVAL;
        }
    }
    t->cur = nxt; t->rows = i1;
    return FAMSA_OK;
}

extern "C" int famsa_tree_edges(famsa_tree* t, int64_t* a_host, int64_t* b_host, float* sim_host) {
    if (!t) { set_error("famsa_tree_edges: tree is NULL"); return FAMSA_EINVAL; }
    const int64_t m = t->rows > 0 ? t->rows - 1 : 0;
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

__global__ void tree_sortkeys_kernel(uint32_t m, const uint32_t* ta, const uint32_t* tb, const float* tw,
                                     unsigned long long* id_key, uint32_t* w_key, uint32_t* idx) {
    const uint32_t e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= m) return;
    id_key[e] = ((unsigned long long)ta[e] << 32) | tb[e];
    idx[e] = e;
    (void)tw; (void)w_key;
}
__global__ void tree_wkeys_kernel(uint32_t m, const float* tw, const uint32_t* idx, uint32_t* w_key) {
    const uint32_t e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e < m) w_key[e] = ~__float_as_uint(tw[idx[e]]);     // ascending key == descending similarity
}

// The dendrogram from the sorted tree edges: a union-find pass, inherently sequential (one thread;
// O(k alpha(k)) L2-resident steps, once per tree).
__global__ void tree_dendrogram_kernel(uint32_t k, const uint32_t* order, const uint32_t* ta, const uint32_t* tb, const float* tw,
                                       uint32_t* uf, long long* cid, long long* csize,
                                       long long* out_a, long long* out_b, float* out_w, long long* out_size) {
    if (blockIdx.x != 0 || threadIdx.x != 0) return;
    for (uint32_t x = 0; x < k; ++x) { uf[x] = x; cid[x] = x; csize[x] = 1; }
    for (uint32_t t = 0; t + 1 < k; ++t) {
        const uint32_t e = order[t];
        uint32_t ra = ta[e], rb = tb[e];
        while (uf[ra] != ra) { uf[ra] = uf[uf[ra]]; ra = uf[ra]; }
        while (uf[rb] != rb) { uf[rb] = uf[uf[rb]]; rb = uf[rb]; }
        const long long ia = cid[ra], ib = cid[rb];
        out_a[t] = ia < ib ? ia : ib; out_b[t] = ia < ib ? ib : ia; out_w[t] = tw[e];
        if (csize[ra] < csize[rb]) { const uint32_t s = ra; ra = rb; rb = s; }
        uf[rb] = ra; csize[ra] += csize[rb]; cid[ra] = (long long)k + t;
        out_size[t] = csize[ra];
    }
}

}  // namespace famsa

extern "C" int famsa_tree_finish(famsa_tree* t, int64_t* id_a_host, int64_t* id_b_host, float* sim_host, int64_t* size_host) {
    if (!t) { set_error("famsa_tree_finish: tree is NULL"); return FAMSA_EINVAL; }
    if (t->rows != t->k) { set_error("famsa_tree_finish: only " + std::to_string(t->rows) + " of " + std::to_string(t->k) + " rows consumed"); return FAMSA_ERANGE; }
    if (t->k < 2) return FAMSA_OK;
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
    tree_sortkeys_kernel<<<g, 256>>>(m, t->ta[cur], t->tb[cur], t->tw[cur], idk, wk, idx);
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

extern "C" int famsa_guide_tree(famsa_ctx* ctx, int64_t block_rows, int64_t* id_a_host, int64_t* id_b_host,
                                float* sim_host, int64_t* size_host) {
    if (!ctx) { set_error("famsa_guide_tree: ctx is NULL"); return FAMSA_EINVAL; }
    if (block_rows < 0) { set_error("famsa_guide_tree: block_rows < 0"); return FAMSA_EINVAL; }
    if (block_rows == 0) block_rows = 1024;
    const int64_t k = ctx->k;
    if (k < 2) return FAMSA_OK;
    FAMSA_CUDA(cudaSetDevice(ctx->device));
    famsa_tree* t = nullptr;
    int rc = famsa_tree_create(k, ctx->device, &t);
    if (rc != FAMSA_OK) return rc;
    const int64_t nb = (k + block_rows - 1) / block_rows;
    const int64_t max_pairs = famsa_rows_pairs(std::max<int64_t>(k - block_rows, 0), k);
    float* buf[2] = {nullptr, nullptr};
    cudaStream_t sa = nullptr, sb = nullptr;
    cudaEvent_t ev[2] = {nullptr, nullptr};
    auto cleanup = [&]() {
        cudaDeviceSynchronize();
        cudaFree(buf[0]); cudaFree(buf[1]);
        if (sa) cudaStreamDestroy(sa);
        if (sb) cudaStreamDestroy(sb);
        if (ev[0]) cudaEventDestroy(ev[0]);
        if (ev[1]) cudaEventDestroy(ev[1]);
        famsa_tree_free(t);
    };
#define GT_CUDA(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) { int r__ = (e__ == cudaErrorMemoryAllocation) ? FAMSA_ENOMEM : FAMSA_ECUDA; \
        famsa::cuda_fail(e__, #call); cleanup(); return r__; } } while (0)
#define GT_TRY(x) do { int r__ = (x); if (r__ != FAMSA_OK) { cleanup(); return r__; } } while (0)
    GT_CUDA(cudaMalloc((void**)&buf[0], std::max<int64_t>(max_pairs, 1) * sizeof(float)));
    GT_CUDA(cudaMalloc((void**)&buf[1], std::max<int64_t>(max_pairs, 1) * sizeof(float)));
    GT_CUDA(cudaStreamCreateWithFlags(&sa, cudaStreamNonBlocking));
    GT_CUDA(cudaStreamCreateWithFlags(&sb, cudaStreamNonBlocking));
    GT_CUDA(cudaEventCreateWithFlags(&ev[0], cudaEventDisableTiming));
    GT_CUDA(cudaEventCreateWithFlags(&ev[1], cudaEventDisableTiming));
    auto rows_of = [&](int64_t b, int64_t& i0, int64_t& i1) { i0 = b * block_rows; i1 = std::min(i0 + block_rows, k); };
    int64_t i0, i1;
    rows_of(0, i0, i1);
    if (famsa_rows_pairs(i0, i1) > 0) GT_TRY(famsa::sweep_rows(ctx, i0, i1, nullptr, buf[0], sa));
    GT_CUDA(cudaEventRecord(ev[0], sa));
    for (int64_t b = 0; b < nb; ++b) {
        if (b + 1 < nb) {                                  // sweep the next block while this one is merged
            int64_t n0, n1;
            rows_of(b + 1, n0, n1);
            GT_TRY(famsa::sweep_rows(ctx, n0, n1, nullptr, buf[(b + 1) & 1], sa));
            GT_CUDA(cudaEventRecord(ev[(b + 1) & 1], sa));
        }
        rows_of(b, i0, i1);
        GT_CUDA(cudaStreamWaitEvent(sb, ev[b & 1], 0));
        GT_TRY(famsa_tree_update(t, i0, i1, buf[b & 1], sb));
    }
    rc = famsa_tree_finish(t, id_a_host, id_b_host, sim_host, size_host);
    ctx->launches += t->launches;
    cleanup();
    return rc;
#undef GT_CUDA
#undef GT_TRY
}
