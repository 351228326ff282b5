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
