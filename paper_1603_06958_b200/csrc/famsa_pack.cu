// famsa_pack.cu -- steps a1-a3 of the path on the device: encode, length sort, residue-stream
// and match-table build ("bit-parallel approach": per-symbol match bit-vectors of
// the sequence that carries V).  One-off, O(sum |S|).  See include/famsa_lcs.h.
#include <cub/device/device_radix_sort.cuh>

#include <algorithm>
#include <chrono>
#include <cstdio>
#include <cstring>
#include <new>

#include "famsa_internal.h"

namespace famsa {

static thread_local std::string g_err;
void set_error(const std::string& msg) { g_err = msg; }
int cuda_fail(cudaError_t e, const char* what) {
    g_err = std::string(what) + ": " + cudaGetErrorString(e);
    cudaGetLastError();
    return FAMSA_ECUDA;
}

// ---- a1: encode.  byte < 25 is a code; letters map to ACDEFGHIKLMNPQRSTVWY BZXUO, J -> X,
// case folded (R9/R10).  First bad position -> atomicMin.
__device__ __forceinline__ int encode_byte(uint8_t c) {
    if (c < 25) return c;
    c &= 0xDF;                                  // fold case ('a'..'z' -> 'A'..'Z')
    if (c < 'A' || c > 'Z') return -1;
    //                       A  B   C  D  E  F  G  H  I  J   K  L  M   N   O   P   Q   R   S   T   U   V   W   X   Y   Z
    const int8_t tab[26] = { 0, 20, 1, 2, 3, 4, 5, 6, 7, 22, 8, 9, 10, 11, 24, 12, 13, 14, 15, 16, 23, 17, 18, 22, 19, 21 };
    return tab[c - 'A'];
}

__global__ void encode_kernel(const uint8_t* __restrict__ raw, uint8_t* __restrict__ codes,
                              int64_t n, unsigned long long* first_bad) {
    int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (; p < n; p += stride) {
        uint8_t c = raw[p];
        // a byte in 'a'..'z' folds onto a letter; '@', '[', '{' etc. must not
        bool letter_or_code = c < 25 || (c >= 'A' && c <= 'Z') || (c >= 'a' && c <= 'z');
        int e = letter_or_code ? encode_byte(c) : -1;
        if (e < 0) { atomicMin(first_bad, (unsigned long long)p); e = 31; }
        codes[p] = (uint8_t)e;
    }
}

// ---- a2: sort keys.  key = MAX_LEN - len (ascending key == descending length); a stable
// radix sort keeps ties in ascending original index (R15).
__global__ void sortkey_kernel(const int64_t* __restrict__ offsets, int64_t k,
                               uint32_t* keys, uint32_t* idx) {
    int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (s < k) {
        keys[s] = (uint32_t)(FAMSA_MAX_LEN - (offsets[s + 1] - offsets[s]));
        idx[s] = (uint32_t)s;
    }
}

// ---- residue streams: one thread per 16-byte chunk of one lane.
__global__ void stream_kernel(const uint8_t* __restrict__ codes, const int64_t* __restrict__ offsets,
                              const uint32_t* __restrict__ perm, const uint32_t* __restrict__ len,
                              const uint32_t* __restrict__ goff, int64_t k, int64_t n_groups,
                              uint8_t* __restrict__ stream) {
    // grid: x = group, threads loop over (chunk, lane)
    int64_t g = blockIdx.x;
    if (g >= n_groups) return;
    uint32_t base = goff[g], nch = goff[g + 1] - base;
    for (uint32_t t = threadIdx.x; t < nch * GROUP; t += blockDim.x) {
        uint32_t c = t / GROUP, lane = t % GROUP;
        int64_t s = g * GROUP + lane;
        uint32_t L = s < k ? len[s] : 0;
        const uint8_t* src = s < k ? codes + offsets[perm[s]] : nullptr;
        uint32_t w[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            uint32_t v = 0;
#pragma unroll
            for (int r = 0; r < 4; ++r) {
                uint32_t p = c * CHUNK + q * 4 + r;
                uint32_t b = p < L ? (uint32_t)src[p] * 4u : (uint32_t)PAD_BYTE;
                v |= b << (8 * r);
            }
            w[q] = v;
        }
        reinterpret_cast<uint4*>(stream)[((size_t)base + c) * GROUP + lane] = make_uint4(w[0], w[1], w[2], w[3]);
    }
}

// ---- a3: match tables.  One warp per (sequence, stored word): lane r holds residue 32*w + r,
// symbol c's word is the ballot of (code == c); lane c stores it -> one coalesced 128-byte row.
// Words past the sequence end (padding inside a block, or the odd stride word) are all-zero.
__global__ void table_kernel(const uint8_t* __restrict__ codes, const int64_t* __restrict__ offsets,
                             const uint32_t* __restrict__ perm, const uint32_t* __restrict__ len,
                             const uint32_t* __restrict__ toff, const uint32_t* __restrict__ twords,
                             int64_t k, uint32_t* __restrict__ tables) {
    // grid.x = sequence; warps of the block loop over that sequence's stored rows.
    int64_t s = blockIdx.x;
    if (s >= k) return;
    uint32_t L = len[s];
    const uint8_t* src = codes + offsets[perm[s]];
    uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
    uint32_t rows = twords[s];                 // stored rows = nblk * wst
    uint32_t wb = twords[k + s], wst = twords[2 * k + s];
    for (uint32_t row = warp; row < rows; row += nwarp) {
        uint32_t blk = row / wst, wi = row % wst;
        uint32_t code = 255;
        if (wi < wb) {
            uint32_t p = (blk * wb + wi) * 32 + lane;
            if (p < L) code = src[p];
        }
        uint32_t mine = 0;
#pragma unroll
        for (int c = 0; c < SYMS; ++c) {
            uint32_t m = __ballot_sync(0xffffffffu, code == (uint32_t)c);
            if (lane == (uint32_t)c) mine = m;
        }
        tables[((size_t)toff[s] + row) * SYMS + lane] = mine;
    }
}

// ---- device block cache: famsa_pack / famsa_free in a loop (the end-to-end path of a streaming caller) would
// otherwise pay ~10 cudaMalloc + cudaFree of up to 0.5 GB each per call, whose latency varies between 1 and 50 ms
// with the state of the process' address space (measured r02).  Freed blocks are kept (up to CACHE_LIMIT bytes per
// process) and handed to the next allocation of about the same size on the same device; famsa_trim() releases them.
struct CachedBlock { int device; void* p; size_t bytes; };
static std::mutex g_cache_mu;
static std::vector<CachedBlock> g_cache;                 // idle blocks
static std::vector<CachedBlock> g_live;                  // blocks handed out (to know their size when they come back)
static size_t g_cache_bytes = 0;
constexpr size_t CACHE_LIMIT = (size_t)6 << 30;

cudaError_t cache_alloc(int device, void** p, size_t bytes) {
    bytes = (std::max<size_t>(bytes, 1) + 255) & ~(size_t)255;
    {
        std::lock_guard<std::mutex> lk(g_cache_mu);
        int best = -1;
        for (size_t n = 0; n < g_cache.size(); ++n) {
            const CachedBlock& b = g_cache[n];
            if (b.device == device && b.bytes >= bytes && b.bytes <= bytes + bytes / 8 + 4096 &&
                (best < 0 || b.bytes < g_cache[best].bytes)) best = (int)n;
        }
        if (best >= 0) {
            *p = g_cache[best].p;
            g_live.push_back(g_cache[best]); g_cache_bytes -= g_cache[best].bytes;
            g_cache.erase(g_cache.begin() + best);
            return cudaSuccess;
        }
    }
    cudaError_t e = cudaMalloc(p, bytes);
    if (e == cudaErrorMemoryAllocation) { cudaGetLastError(); cache_trim(); e = cudaMalloc(p, bytes); }   // the cache must never cause an OOM
    if (e == cudaSuccess) { std::lock_guard<std::mutex> lk(g_cache_mu); g_live.push_back(CachedBlock{device, *p, bytes}); }
    return e;
}

// The caller guarantees that nothing on the device still uses the block (famsa_free synchronises the device first).
void cache_free(void* p) {
    if (!p) return;
    CachedBlock b{-1, nullptr, 0};
    {
        std::lock_guard<std::mutex> lk(g_cache_mu);
        for (size_t n = 0; n < g_live.size(); ++n)
            if (g_live[n].p == p) { b = g_live[n]; g_live.erase(g_live.begin() + n); break; }
        if (b.p && g_cache_bytes + b.bytes <= CACHE_LIMIT) { g_cache.push_back(b); g_cache_bytes += b.bytes; return; }
    }
    cudaFree(p);
}

void cache_trim() {
    std::vector<CachedBlock> all;
    { std::lock_guard<std::mutex> lk(g_cache_mu); all.swap(g_cache); g_cache_bytes = 0; }
    int cur = 0; cudaGetDevice(&cur);
    for (const CachedBlock& b : all) { cudaSetDevice(b.device); cudaFree(b.p); }
    cudaSetDevice(cur);
}

template <typename T>
static cudaError_t dalloc(int device, T** p, size_t n) { return cache_alloc(device, (void**)p, std::max<size_t>(n, 1) * sizeof(T)); }

}  // namespace famsa

using namespace famsa;

extern "C" void famsa_free(famsa_ctx* ctx) {
    if (!ctx) return;
    cudaSetDevice(ctx->device);
    if (ctx->stg) famsa::staging_release(ctx->stg);       // drains the host path's streams, then back to the pool
    if (ctx->s_direct) { cudaStreamSynchronize(ctx->s_direct); cudaStreamDestroy(ctx->s_direct); }
    for (famsa::HostChunkTimers& t : ctx->direct_timers) for (cudaEvent_t e : t.ev) if (e) cudaEventDestroy(e);
    cudaDeviceSynchronize();                              // as cudaFree would: nothing may still read the packed set
    famsa::cache_free(ctx->d_stream); famsa::cache_free(ctx->d_tables); famsa::cache_free(ctx->d_len);
    famsa::cache_free(ctx->d_toff); famsa::cache_free(ctx->d_goff);
    delete ctx;
}

static int pack_impl(const uint8_t* seqs, const int64_t* offsets, int64_t k, int device, famsa_ctx* ctx);

extern "C" int famsa_pack(const uint8_t* seqs, const int64_t* offsets, int64_t k, int device,
                          famsa_ctx** out) {
    if (!out) { set_error("famsa_pack: out is NULL"); return FAMSA_EINVAL; }
    *out = nullptr;
    if (k < 0 || !offsets || (k > 0 && !seqs && offsets[k] > 0)) {
        set_error("famsa_pack: null pointer or k < 0"); return FAMSA_EINVAL;
    }
    if (offsets[0] != 0) { set_error("famsa_pack: offsets[0] != 0"); return FAMSA_EINVAL; }
    for (int64_t s = 0; s < k; ++s) {
        int64_t L = offsets[s + 1] - offsets[s];
        if (L < 0) { set_error("famsa_pack: offsets decrease at " + std::to_string(s)); return FAMSA_EINVAL; }
        if (L == 0 || L > FAMSA_MAX_LEN) {
            set_error("famsa_pack: sequence " + std::to_string(s) + " has length " + std::to_string(L));
            return FAMSA_ELENGTH;
        }
    }
    if (k > 0x7FFFFFF0LL) { set_error("famsa_pack: k too large (at most 2^31 - 16 sequences)"); return FAMSA_EINVAL; }
    famsa_ctx* ctx = new (std::nothrow) famsa_ctx();
    if (!ctx) { set_error("famsa_pack: host allocation failed"); return FAMSA_ENOMEM; }
    int rc;
    try {
        rc = pack_impl(seqs, offsets, k, device, ctx);
    } catch (const std::bad_alloc&) {
        set_error("famsa_pack: host allocation failed"); rc = FAMSA_ENOMEM;
    }
    if (rc != FAMSA_OK) { famsa_free(ctx); return rc; }
    *out = ctx;
    return FAMSA_OK;
}

namespace {
struct DevTmp {                       // pack_impl's scratch: ONE device allocation carved up (a cudaMalloc / cudaFree pair
    uint8_t* base = nullptr;          // per piece cost famsa_pack ~2 ms), freed on every exit path
    size_t cap = 0, used = 0;
    std::vector<void*> extra;         // pieces that did not fit the reservation (never with the sizes pack_impl reserves)
    int device = 0;
    ~DevTmp() { cudaDeviceSynchronize(); famsa::cache_free(base); for (void* p : extra) famsa::cache_free(p); }
    static size_t padded(size_t bytes) { return (std::max<size_t>(bytes, 1) + 255) & ~(size_t)255; }
    int reserve(size_t bytes) {
        cudaError_t e = famsa::cache_alloc(device, (void**)&base, std::max<size_t>(bytes, 256));
        if (e == cudaErrorMemoryAllocation) { cudaGetLastError(); famsa::set_error("famsa_pack: device allocation failed"); return FAMSA_ENOMEM; }
        if (e != cudaSuccess) return famsa::cuda_fail(e, "cudaMalloc");
        cap = std::max<size_t>(bytes, 256);
        return FAMSA_OK;
    }
    template <typename T> int alloc(T** p, size_t n) {
        const size_t bytes = padded(n * sizeof(T));
        if (used + bytes <= cap) { *p = reinterpret_cast<T*>(base + used); used += bytes; return FAMSA_OK; }
        cudaError_t e = famsa::dalloc(device, p, n);
        if (e == cudaErrorMemoryAllocation) { cudaGetLastError(); famsa::set_error("famsa_pack: device allocation failed"); return FAMSA_ENOMEM; }
        if (e != cudaSuccess) return famsa::cuda_fail(e, "cudaMalloc");
        extra.push_back(*p);
        return FAMSA_OK;
    }
};
template <typename T> int ctx_alloc(int device, T** p, size_t n) {
    cudaError_t e = famsa::dalloc(device, p, n);
    if (e == cudaErrorMemoryAllocation) { cudaGetLastError(); famsa::set_error("famsa_pack: device allocation failed"); return FAMSA_ENOMEM; }
    if (e != cudaSuccess) return famsa::cuda_fail(e, "cudaMalloc");
    return FAMSA_OK;
}
}  // namespace

#define FAMSA_TRY(x) do { int rc__ = (x); if (rc__ != FAMSA_OK) return rc__; } while (0)

static int pack_impl(const uint8_t* seqs, const int64_t* offsets, int64_t k, int device, famsa_ctx* ctx) {
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) {
        cudaGetLastError();
        set_error("famsa_pack: no CUDA device " + std::to_string(device) + " (there is no CPU fallback)");
        return FAMSA_ECUDA;
    }
    FAMSA_CUDA(cudaSetDevice(device));
    int cc_major = 0, cc_minor = 0, sm_count = 0;            // (cudaGetDeviceProperties costs ~1 ms per call: attributes instead)
    FAMSA_CUDA(cudaDeviceGetAttribute(&cc_major, cudaDevAttrComputeCapabilityMajor, device));
    FAMSA_CUDA(cudaDeviceGetAttribute(&cc_minor, cudaDevAttrComputeCapabilityMinor, device));
    FAMSA_CUDA(cudaDeviceGetAttribute(&sm_count, cudaDevAttrMultiProcessorCount, device));
    if (cc_major != 10) {
        set_error("famsa_pack: device is sm_" + std::to_string(cc_major * 10 + cc_minor) +
                  ", this library is built for sm_100a only");
        return FAMSA_ECUDA;
    }
    ctx->device = device; ctx->sm_count = sm_count; ctx->k = k;
    ctx->n_groups = (k + GROUP - 1) / GROUP;
    const int64_t total = offsets[k];
    using clk = std::chrono::steady_clock;
    auto ms_since = [](clk::time_point t) { return std::chrono::duration<double, std::milli>(clk::now() - t).count(); };
    clk::time_point t_phase = clk::now();
    DevTmp tmp;
    tmp.device = device;
    cudaStream_t st = nullptr;           // legacy default stream; pack synchronises before returning
    size_t cub_bytes = 0;
    if (k > 0) FAMSA_CUDA(cub::DeviceRadixSort::SortPairs(nullptr, cub_bytes, (uint32_t*)nullptr, (uint32_t*)nullptr, (uint32_t*)nullptr,
                                                         (uint32_t*)nullptr, (int)k, 0, 16, st));
    FAMSA_TRY(tmp.reserve(2 * DevTmp::padded((size_t)total) + DevTmp::padded(8 * ((size_t)k + 1)) + DevTmp::padded(8) +
                          4 * DevTmp::padded(4 * (size_t)k) + DevTmp::padded(cub_bytes) + DevTmp::padded(12 * (size_t)k)));

    // ---- a1 encode
    uint8_t *d_raw = nullptr, *d_codes = nullptr; int64_t* d_off = nullptr; unsigned long long* d_bad = nullptr;
    FAMSA_TRY(tmp.alloc(&d_raw, (size_t)total));
    FAMSA_TRY(tmp.alloc(&d_codes, (size_t)total));
    FAMSA_TRY(tmp.alloc(&d_off, (size_t)k + 1));
    FAMSA_TRY(tmp.alloc(&d_bad, 1));
    if (total) FAMSA_CUDA(cudaMemcpyAsync(d_raw, seqs, (size_t)total, cudaMemcpyHostToDevice, st));
    FAMSA_CUDA(cudaMemcpyAsync(d_off, offsets, sizeof(int64_t) * (size_t)(k + 1), cudaMemcpyHostToDevice, st));
    FAMSA_CUDA(cudaMemsetAsync(d_bad, 0xFF, sizeof(unsigned long long), st));
    if (total) {
        int grid = (int)std::min<int64_t>((total + 255) / 256, (int64_t)ctx->sm_count * 16);
        encode_kernel<<<grid, 256, 0, st>>>(d_raw, d_codes, total, d_bad);
        ctx->launches++;
    }
    unsigned long long bad = ~0ull;
    FAMSA_CUDA(cudaMemcpyAsync(&bad, d_bad, sizeof(bad), cudaMemcpyDeviceToHost, st));
    FAMSA_CUDA(cudaStreamSynchronize(st));
    if (bad != ~0ull) {
        set_error("famsa_pack: byte " + std::to_string((int)seqs[bad]) + " at position " + std::to_string(bad) +
                  " is neither a residue code (< 25) nor an amino-acid letter");
        return FAMSA_ESYMBOL;
    }
    ctx->pack_ms[0] = ms_since(t_phase); t_phase = clk::now();

    // ---- a2 length sort (descending, stable)
    uint32_t *d_key = nullptr, *d_key2 = nullptr, *d_idx = nullptr, *d_perm = nullptr;
    FAMSA_TRY(tmp.alloc(&d_key, (size_t)k)); FAMSA_TRY(tmp.alloc(&d_key2, (size_t)k));
    FAMSA_TRY(tmp.alloc(&d_idx, (size_t)k)); FAMSA_TRY(tmp.alloc(&d_perm, (size_t)k));
    ctx->perm.resize(k); ctx->len.resize(k);
    if (k > 0) {
        sortkey_kernel<<<(unsigned)((k + 255) / 256), 256, 0, st>>>(d_off, k, d_key, d_idx);
        ctx->launches++;
        void* d_cub = nullptr;
        FAMSA_TRY(tmp.alloc((uint8_t**)&d_cub, cub_bytes));
        FAMSA_CUDA(cub::DeviceRadixSort::SortPairs(d_cub, cub_bytes, d_key, d_key2, d_idx, d_perm, (int)k, 0, 16, st));
        ctx->launches += 3;               // cub: histogram + onesweep passes (>= 3 kernels for 16 bits)
        std::vector<uint32_t> hperm(k), hkey(k);
        FAMSA_CUDA(cudaMemcpyAsync(hperm.data(), d_perm, sizeof(uint32_t) * k, cudaMemcpyDeviceToHost, st));
        FAMSA_CUDA(cudaMemcpyAsync(hkey.data(), d_key2, sizeof(uint32_t) * k, cudaMemcpyDeviceToHost, st));
        FAMSA_CUDA(cudaStreamSynchronize(st));
        for (int64_t s = 0; s < k; ++s) { ctx->perm[s] = hperm[s]; ctx->len[s] = FAMSA_MAX_LEN - hkey[s]; }
    }
    ctx->max_len = k ? ctx->len[0] : 0;
    ctx->large_cw = ctx->max_len > (uint32_t)CW_SMALL * 32;
    ctx->pack_ms[1] = ms_since(t_phase); t_phase = clk::now();

    // ---- host plan: table offsets, block plans, buckets, group offsets, length prefix sums
    ctx->toff.resize(k); ctx->goff.resize(ctx->n_groups + 1); ctx->len_prefix.resize(k + 1);
    std::vector<uint32_t> twords(3 * (size_t)k);
    uint64_t rows_total = 0;
    ctx->len_prefix[0] = 0.0;
    for (int64_t s = 0; s < k; ++s) {
        BlockPlan p = plan_blocks(ctx->len[s], ctx->large_cw);
        if (rows_total > 0xFFFFFFFFull - 5000) { set_error("famsa_pack: match tables exceed 2^32 rows"); return FAMSA_ENOMEM; }
        ctx->toff[s] = (uint32_t)rows_total;
        twords[s] = (uint32_t)(p.nblk * p.wst); twords[k + s] = (uint32_t)p.wb; twords[2 * k + s] = (uint32_t)p.wst;
        rows_total += (uint64_t)p.nblk * p.wst;
        if (ctx->buckets.empty() || ctx->buckets.back().nblk != p.nblk || ctx->buckets.back().wb != p.wb)
            ctx->buckets.push_back(Bucket{s, s + 1, p.nblk, p.wb});
        else
            ctx->buckets.back().r1 = s + 1;
        ctx->len_prefix[s + 1] = ctx->len_prefix[s] + (double)ctx->len[s];
    }
    uint64_t chunks_total = 0;
    for (int64_t g = 0; g < ctx->n_groups; ++g) {
        ctx->goff[g] = (uint32_t)chunks_total;
        chunks_total += (ctx->len[g * GROUP] + CHUNK - 1) / CHUNK;     // first of the group is its longest
        if (chunks_total > 0xFFFFFFF0ull) { set_error("famsa_pack: residue stream too large"); return FAMSA_ENOMEM; }
    }
    ctx->goff[ctx->n_groups] = (uint32_t)chunks_total;
    ctx->stream_bytes = (size_t)chunks_total * GROUP * CHUNK;
    ctx->table_bytes = (size_t)rows_total * ROW_BYTES;

    ctx->pack_ms[2] = ms_since(t_phase); t_phase = clk::now();

    // ---- device-resident set
    uint32_t* d_twords = nullptr;
    FAMSA_TRY(tmp.alloc(&d_twords, twords.size()));
    FAMSA_TRY(ctx_alloc(device, &ctx->d_stream, ctx->stream_bytes + 512));
    FAMSA_TRY(ctx_alloc(device, &ctx->d_tables, ctx->table_bytes / 4 + 64));
    FAMSA_TRY(ctx_alloc(device, &ctx->d_len, (size_t)k));
    FAMSA_TRY(ctx_alloc(device, &ctx->d_toff, (size_t)k));
    FAMSA_TRY(ctx_alloc(device, &ctx->d_goff, (size_t)ctx->n_groups + 1));
    if (k > 0) {
        FAMSA_CUDA(cudaMemcpyAsync(ctx->d_len, ctx->len.data(), sizeof(uint32_t) * k, cudaMemcpyHostToDevice, st));
        FAMSA_CUDA(cudaMemcpyAsync(ctx->d_toff, ctx->toff.data(), sizeof(uint32_t) * k, cudaMemcpyHostToDevice, st));
        FAMSA_CUDA(cudaMemcpyAsync(d_twords, twords.data(), sizeof(uint32_t) * twords.size(), cudaMemcpyHostToDevice, st));
    }
    FAMSA_CUDA(cudaMemcpyAsync(ctx->d_goff, ctx->goff.data(), sizeof(uint32_t) * (ctx->n_groups + 1), cudaMemcpyHostToDevice, st));
    if (k > 0) {
        stream_kernel<<<(unsigned)ctx->n_groups, 256, 0, st>>>(d_codes, d_off, d_perm, ctx->d_len, ctx->d_goff, k,
                                                               ctx->n_groups, ctx->d_stream);
        table_kernel<<<(unsigned)k, 128, 0, st>>>(d_codes, d_off, d_perm, ctx->d_len, ctx->d_toff, d_twords, k, ctx->d_tables);
        ctx->launches += 2;
    }
    FAMSA_CUDA(cudaGetLastError());
    FAMSA_CUDA(cudaStreamSynchronize(st));
    ctx->pack_ms[3] = ms_since(t_phase);
    return FAMSA_OK;
}

extern "C" int famsa_pack_profile(const famsa_ctx* ctx, double* ms4) {
    if (!ctx || !ms4) { set_error("famsa_pack_profile: null argument"); return FAMSA_EINVAL; }
    for (int q = 0; q < 4; ++q) ms4[q] = ctx->pack_ms[q];
    return FAMSA_OK;
}

// ---- small accessors -----------------------------------------------------------------------
extern "C" int64_t famsa_rows_pairs(int64_t i0, int64_t i1) {
    if (i0 < 0 || i0 > i1) return -1;
    return i1 * (i1 - 1) / 2 - i0 * (i0 - 1) / 2;
}

extern "C" int famsa_rows_cells(const famsa_ctx* ctx, int64_t i0, int64_t i1, double* cells) {
    if (!ctx || !cells) { set_error("famsa_rows_cells: null argument"); return FAMSA_EINVAL; }
    if (i0 < 0 || i0 > i1 || i1 > ctx->k) { set_error("famsa_rows_cells: bad row range"); return FAMSA_ERANGE; }
    double c = 0.0;
    for (int64_t i = i0; i < i1; ++i) c += (double)ctx->len[i] * ctx->len_prefix[i];
    *cells = c;
    return FAMSA_OK;
}

extern "C" int famsa_k(const famsa_ctx* ctx, int64_t* k) {
    if (!ctx || !k) { set_error("famsa_k: null argument"); return FAMSA_EINVAL; }
    *k = ctx->k; return FAMSA_OK;
}

extern "C" int famsa_perm(const famsa_ctx* ctx, int64_t* perm_host) {
    if (!ctx || (!perm_host && ctx->k)) { set_error("famsa_perm: null argument"); return FAMSA_EINVAL; }
    if (ctx->k) memcpy(perm_host, ctx->perm.data(), sizeof(int64_t) * ctx->k);
    return FAMSA_OK;
}

extern "C" int famsa_lengths(const famsa_ctx* ctx, uint32_t* len_host) {
    if (!ctx || (!len_host && ctx->k)) { set_error("famsa_lengths: null argument"); return FAMSA_EINVAL; }
    if (ctx->k) memcpy(len_host, ctx->len.data(), sizeof(uint32_t) * ctx->k);
    return FAMSA_OK;
}

extern "C" int famsa_codes(const famsa_ctx* ctx, int64_t s, uint8_t* codes_host) {
    if (!ctx || !codes_host) { set_error("famsa_codes: null argument"); return FAMSA_EINVAL; }
    if (s < 0 || s >= ctx->k) { set_error("famsa_codes: sequence index out of range"); return FAMSA_ERANGE; }
    FAMSA_CUDA(cudaSetDevice(ctx->device));
    int64_t g = s / GROUP, lane = s % GROUP;
    uint32_t L = ctx->len[s], nch = (L + CHUNK - 1) / CHUNK;
    std::vector<uint8_t> buf((size_t)nch * CHUNK);
    // lane's chunks are 512 bytes apart: a strided 2-D copy
    FAMSA_CUDA(cudaMemcpy2D(buf.data(), CHUNK, ctx->d_stream + (size_t)ctx->goff[g] * 512 + lane * CHUNK, 512,
                            CHUNK, nch, cudaMemcpyDeviceToHost));
    for (uint32_t p = 0; p < L; ++p) codes_host[p] = buf[p] >> 2;
    return FAMSA_OK;
}

extern "C" int famsa_match(const famsa_ctx* ctx, int64_t s, int c, uint32_t* words_host) {
    if (!ctx || !words_host) { set_error("famsa_match: null argument"); return FAMSA_EINVAL; }
    if (s < 0 || s >= ctx->k || c < 0 || c >= SYMS) { set_error("famsa_match: index out of range"); return FAMSA_ERANGE; }
    FAMSA_CUDA(cudaSetDevice(ctx->device));
    BlockPlan p = plan_blocks(ctx->len[s], ctx->large_cw);
    uint32_t rows = (uint32_t)(p.nblk * p.wst), ws = (ctx->len[s] + 31) / 32;
    std::vector<uint32_t> col(rows);
    FAMSA_CUDA(cudaMemcpy2D(col.data(), 4, ctx->d_tables + (size_t)ctx->toff[s] * SYMS + c, ROW_BYTES, 4, rows,
                            cudaMemcpyDeviceToHost));
    for (uint32_t w = 0; w < ws; ++w) words_host[w] = col[(w / p.wb) * p.wst + (w % p.wb)];
    return FAMSA_OK;
}

extern "C" int64_t famsa_launch_count(const famsa_ctx* ctx) { return ctx ? ctx->launches.load() : 0; }

extern "C" const char* famsa_strerror(int code) {
    switch (code) {
        case FAMSA_OK: return "ok";
        case FAMSA_EINVAL: return "invalid argument";
        case FAMSA_ESYMBOL: return "byte is neither a residue code nor an amino-acid letter";
        case FAMSA_ELENGTH: return "sequence is empty or longer than 65535";
        case FAMSA_ERANGE: return "row range out of bounds";
        case FAMSA_ENOMEM: return "out of memory";
        case FAMSA_ECUDA: return "CUDA error or no sm_100 device";
        default: return "unknown error";
    }
}

extern "C" const char* famsa_last_error(void) { return famsa::g_err.c_str(); }
