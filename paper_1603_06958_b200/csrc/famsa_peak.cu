// famsa_peak.cu -- measures the roofline denominator: the chip's INT32 ALU-pipe issue rate.
// MEASURED_PEAKS.json carries no integer peak, so the library measures one:
// 8 word-steps per thread and step, each LOP3 -> IADD3.X -> LOP3 (+ one LOP3 that keeps the mask
// live), the adds linked by the hardware carry exactly as in the sweep so that ptxas cannot move
// them to the FMA pipe as IMAD.IADD; no shared-memory load; all SMs, 32 warps per SM.
#include "famsa_internal.h"

namespace famsa {

constexpr int PEAK_CHAINS = 8;
constexpr int PEAK_ITERS = 4096;
constexpr int PEAK_UNROLL = 8;     // triples per chain per loop iteration

__global__ void __launch_bounds__(256) alu_peak_kernel(uint32_t* out, uint32_t seed, long long* cycles) {
    uint32_t v[PEAK_CHAINS], m[PEAK_CHAINS];
#pragma unroll
    for (int c = 0; c < PEAK_CHAINS; ++c) {
        v[c] = seed ^ (threadIdx.x * 2654435761u + c * 40503u);
        m[c] = (seed >> 3) + blockIdx.x * 97u + c;
    }
    { uint32_t z = 0; asm volatile("add.cc.u32 %0, %0, %0;" : "+r"(z)); }      // define the carry flag
    long long t0 = clock64();
#pragma unroll 1
    for (int it = 0; it < PEAK_ITERS; ++it) {
#pragma unroll
        for (int u = 0; u < PEAK_UNROLL; ++u) {
#pragma unroll
            for (int c = 0; c < PEAK_CHAINS; ++c) {
                uint32_t x = v[c] & m[c];                 // LOP3
                uint32_t s;                               // IADD3 / IADD3.X: the carry keeps it on the ALU pipe
                asm volatile("addc.cc.u32 %0, %1, %2;" : "=r"(s) : "r"(v[c]), "r"(x));   // carry never dies
                v[c] = s | (v[c] & ~m[(c + 1) % PEAK_CHAINS]);   // LOP3
                m[c] ^= s;                                // keeps m live and loop-variant (LOP3)
            }
        }
    }
    long long t1 = clock64();
    uint32_t acc = 0;
#pragma unroll
    for (int c = 0; c < PEAK_CHAINS; ++c) acc ^= v[c] + m[c];
    out[blockIdx.x * blockDim.x + threadIdx.x] = acc;
    if (threadIdx.x == 0) cycles[blockIdx.x] = t1 - t0;
}


// ---- the sweep's instruction mix: per word-step LDS.32 + LOP3 + IADD3.X + LOP3, one PRMT per residue,
// V (10 words) in registers, the table rows in shared memory in the sweep's [word][symbol] layout (bank =
// symbol, so no residue mix conflicts), pseudo-random residues, no global traffic.  The achieved ALU-pipe
// rate is the ceiling of this mix: what is left between it and 64 is the SM's issue behaviour with one
// shared-memory load per three ALU instructions, not something a sweep kernel can recover.
constexpr int MIX_W = 10;
constexpr int MIX_ITERS = 2000;
constexpr int MIX_THREADS = 128;
constexpr int MIX_CTAS_PER_SM = 10;    // 40 warps per SM

template <int I> struct MixLoad {
    static __device__ __forceinline__ void run(uint32_t (&m)[MIX_W], uint32_t addr) {
        asm("ld.shared.u32 %0, [%1+%2];" : "=r"(m[I]) : "r"(addr), "n"(I * ROW_BYTES));
        MixLoad<I + 1>::run(m, addr);
    }
};
template <> struct MixLoad<MIX_W> { static __device__ __forceinline__ void run(uint32_t (&)[MIX_W], uint32_t) {} };

__global__ void __launch_bounds__(MIX_THREADS) mix_peak_kernel(uint32_t* out, uint32_t seed, long long* cycles) {
    __shared__ __align__(256) uint32_t tab[SYMS * MIX_W + 64];
    for (int t = threadIdx.x; t < SYMS * MIX_W + 64; t += MIX_THREADS) tab[t] = seed * (t + 1) * 2654435761u;
    __syncthreads();
    uint32_t V[MIX_W];
#pragma unroll
    for (int w = 0; w < MIX_W; ++w) V[w] = ~0u;
    const uint32_t sbase = (uint32_t)__cvta_generic_to_shared(tab);
    uint32_t bw = seed ^ threadIdx.x * 0x01010101u;
    const long long t0 = clock64();
#pragma unroll 1
    for (int it = 0; it < MIX_ITERS; ++it) {
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const uint32_t addr = __byte_perm(bw & 0x7c7c7c7cu, sbase, 0x7650 + r);   // PRMT, as residue_addr() in the sweep
            uint32_t m[MIX_W], s[MIX_W];
            MixLoad<0>::run(m, addr);
#pragma unroll
            for (int w = 0; w < MIX_W; ++w) {
                const uint32_t u = V[w] & m[w];
                if (w == 0) asm volatile("add.cc.u32 %0, %1, %2;" : "=r"(s[w]) : "r"(V[w]), "r"(u));
                else        asm volatile("addc.cc.u32 %0, %1, %2;" : "=r"(s[w]) : "r"(V[w]), "r"(u));
            }
#pragma unroll
            for (int w = 0; w < MIX_W; ++w) V[w] = s[w] | (V[w] & ~m[w]);
        }
        bw = bw * 1664525u + 1013904223u;
    }
    const long long t1 = clock64();
    uint32_t acc = 0;
#pragma unroll
    for (int w = 0; w < MIX_W; ++w) acc += __popc(~V[w]);
    out[blockIdx.x * MIX_THREADS + threadIdx.x] = acc;
    if (threadIdx.x == 0) cycles[blockIdx.x] = t1 - t0;
}

}  // namespace famsa

using namespace famsa;

extern "C" int famsa_alu_peak(int device, double* instr_per_s, double* instr_per_clk_sm, double* sm_mhz) {
    if (!instr_per_s || !instr_per_clk_sm || !sm_mhz) { set_error("famsa_alu_peak: null argument"); return FAMSA_EINVAL; }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) {
        cudaGetLastError(); set_error("famsa_alu_peak: no such CUDA device"); return FAMSA_ECUDA;
    }
    FAMSA_CUDA(cudaSetDevice(device));
    cudaDeviceProp prop;
    FAMSA_CUDA(cudaGetDeviceProperties(&prop, device));
    const int threads = 256, ctas_per_sm = 4, grid = prop.multiProcessorCount * ctas_per_sm;
    uint32_t* d_out = nullptr; long long* d_cyc = nullptr;
    FAMSA_CUDA(cudaMalloc((void**)&d_out, sizeof(uint32_t) * grid * threads));
    FAMSA_CUDA(cudaMalloc((void**)&d_cyc, sizeof(long long) * grid));
    cudaEvent_t e0, e1;
    FAMSA_CUDA(cudaEventCreate(&e0)); FAMSA_CUDA(cudaEventCreate(&e1));
    float best_ms = 1e30f;
    for (int rep = 0; rep < 6; ++rep) {           // first reps warm the clocks
        FAMSA_CUDA(cudaEventRecord(e0, 0));
        alu_peak_kernel<<<grid, threads>>>(d_out, 0x9E3779B9u + rep, d_cyc);
        FAMSA_CUDA(cudaEventRecord(e1, 0));
        FAMSA_CUDA(cudaEventSynchronize(e1));
        float ms = 0; FAMSA_CUDA(cudaEventElapsedTime(&ms, e0, e1));
        if (rep >= 2 && ms < best_ms) best_ms = ms;
    }
    FAMSA_CUDA(cudaGetLastError());
    std::vector<long long> cyc(grid);
    FAMSA_CUDA(cudaMemcpy(cyc.data(), d_cyc, sizeof(long long) * grid, cudaMemcpyDeviceToHost));
    long long cmax = 0; for (long long c : cyc) cmax = c > cmax ? c : cmax;
    cudaFree(d_out); cudaFree(d_cyc); cudaEventDestroy(e0); cudaEventDestroy(e1);
    // 4 ALU instructions per chain step (3 LOP3 + 1 IADD3)
    const double instr = 4.0 * PEAK_CHAINS * PEAK_UNROLL * (double)PEAK_ITERS * threads * (double)grid;
    const double sec = best_ms * 1e-3;
    *instr_per_s = instr / sec;
    // every SM runs ctas_per_sm CTAs concurrently for ~the whole kernel: cmax cycles elapsed per SM
    *sm_mhz = (double)cmax / sec * 1e-6;
    *instr_per_clk_sm = instr / prop.multiProcessorCount / (double)cmax;
    return FAMSA_OK;
}

extern "C" int famsa_mix_peak(int device, double* alu_instr_per_clk_sm, double* sm_mhz) {
    if (!alu_instr_per_clk_sm || !sm_mhz) { set_error("famsa_mix_peak: null argument"); return FAMSA_EINVAL; }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) {
        cudaGetLastError(); set_error("famsa_mix_peak: no such CUDA device"); return FAMSA_ECUDA;
    }
    FAMSA_CUDA(cudaSetDevice(device));
    cudaDeviceProp prop;
    FAMSA_CUDA(cudaGetDeviceProperties(&prop, device));
    const int grid = prop.multiProcessorCount * MIX_CTAS_PER_SM;
    uint32_t* d_out = nullptr; long long* d_cyc = nullptr;
    FAMSA_CUDA(cudaMalloc((void**)&d_out, sizeof(uint32_t) * grid * MIX_THREADS));
    FAMSA_CUDA(cudaMalloc((void**)&d_cyc, sizeof(long long) * grid));
    cudaEvent_t e0, e1;
    FAMSA_CUDA(cudaEventCreate(&e0)); FAMSA_CUDA(cudaEventCreate(&e1));
    float best_ms = 1e30f;
    for (int rep = 0; rep < 5; ++rep) {
        FAMSA_CUDA(cudaEventRecord(e0, 0));
        mix_peak_kernel<<<grid, MIX_THREADS>>>(d_out, 12345u + rep, d_cyc);
        FAMSA_CUDA(cudaEventRecord(e1, 0));
        FAMSA_CUDA(cudaEventSynchronize(e1));
        float ms = 0; FAMSA_CUDA(cudaEventElapsedTime(&ms, e0, e1));
        if (rep >= 2 && ms < best_ms) best_ms = ms;
    }
    FAMSA_CUDA(cudaGetLastError());
    std::vector<long long> cyc(grid);
    FAMSA_CUDA(cudaMemcpy(cyc.data(), d_cyc, sizeof(long long) * grid, cudaMemcpyDeviceToHost));
    long long cmax = 0; for (long long c : cyc) cmax = c > cmax ? c : cmax;
    cudaFree(d_out); cudaFree(d_cyc); cudaEventDestroy(e0); cudaEventDestroy(e1);
    // all MIX_CTAS_PER_SM CTAs of an SM are resident together: cmax cycles for the SM's whole share
    const double wordsteps_per_sm = (double)MIX_ITERS * 4 * MIX_W * MIX_THREADS * MIX_CTAS_PER_SM;
    *alu_instr_per_clk_sm = 3.0 * wordsteps_per_sm / (double)cmax;
    *sm_mhz = (double)cmax / (best_ms * 1e-3) * 1e-6;
    return FAMSA_OK;
}
