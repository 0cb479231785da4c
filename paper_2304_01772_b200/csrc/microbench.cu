// microbench.cu — the second, tighter roofline denominator of SURVEY.md section 8(d): the stand-alone rate of the
// algorithmic work of the sweep ("Philox plus compare", BASELINE.json north star) measured on the device the handle
// would run on, registers only: Philox-4x32-10 with host-precomputed round keys, its four output words each compared
// against a threshold and folded into a mask.  No lattice, no memory traffic, no class look-up.  bench.py reports the
// sweep kernels against the nominal INT32 peak (the headline fraction) and against this measured rate.
#include "../../include/spin.h"
#include "spin_internal.cuh"

namespace spin {
namespace {

template <int kCalls>
__global__ void __launch_bounds__(256) philox_compare_kernel(uint32_t* out, int outer, RoundKeys rk, uint32_t thr) {
    uint32_t acc = 0;
    const uint32_t g = (blockIdx.x * blockDim.x + threadIdx.x) * kCalls;
    for (int o = 0; o < outer; ++o) {
#pragma unroll
        for (int c = 0; c < kCalls; ++c) {
            // the counter words depend on the running mask, so no product can be hoisted out of the loop
            uint32_t r[4];
            philox4x32_10(rk, g + c + (acc & 2u), acc & 1u, (uint32_t)o + (acc & 4u), 0x11000000u, r);
            asm volatile("{\n\t.reg .pred p;\n\tsetp.ls.u32 p, %1, %2;\n\t@p xor.b32 %0, %0, 0xFE;\n\t}" : "+r"(acc) : "r"(r[0]), "r"(thr));
            asm volatile("{\n\t.reg .pred p;\n\tsetp.ls.u32 p, %1, %2;\n\t@p xor.b32 %0, %0, 0xFE00;\n\t}" : "+r"(acc) : "r"(r[1]), "r"(thr));
            asm volatile("{\n\t.reg .pred p;\n\tsetp.ls.u32 p, %1, %2;\n\t@p xor.b32 %0, %0, 0xFE0000;\n\t}" : "+r"(acc) : "r"(r[2]), "r"(thr));
            asm volatile("{\n\t.reg .pred p;\n\tsetp.ls.u32 p, %1, %2;\n\t@p xor.b32 %0, %0, 0xFE000000;\n\t}" : "+r"(acc) : "r"(r[3]), "r"(thr));
        }
    }
    if (acc == 0x12345679u) out[0] = acc;   // never true in practice; keeps the chain alive
}

}  // namespace
}  // namespace spin

extern "C" int spin_measure_philox_compare_rate(double* words_per_ns) {
    using namespace spin;
    if (!words_per_ns) return SPIN_ERR_INVALID;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
        return SPIN_ERR_CUDA;
    uint32_t* d = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (cudaMalloc(&d, 64) != cudaSuccess) return SPIN_ERR_CUDA;
    int rc = SPIN_OK;
    RoundKeys rk;
    uint32_t k0 = 1u, k1 = 0u;
    for (int r = 0; r < 10; ++r) { rk.k0[r] = k0; rk.k1[r] = k1; k0 += kPhiloxW0; k1 += kPhiloxW1; }
    const int threads = 256, blocks = sms * 8, outer = 2000, calls = 4;   // 8 warps per SM sub-partition, 4 calls in flight
    float best = 1e30f;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) rc = SPIN_ERR_CUDA;
    for (int rep = 0; rep < 7 && rc == SPIN_OK; ++rep) {
        cudaEventRecord(e0, 0);
        philox_compare_kernel<calls><<<blocks, threads>>>(d, outer, rk, 0x2c0b21d7u);
        cudaEventRecord(e1, 0);
        if (cudaEventSynchronize(e1) != cudaSuccess || cudaGetLastError() != cudaSuccess) { rc = SPIN_ERR_CUDA; break; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep >= 2 && ms < best) best = ms;   // two warm-up launches
    }
    if (rc == SPIN_OK) *words_per_ns = 4.0 * (double)blocks * threads * outer * calls / ((double)best * 1e6);
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    cudaFree(d);
    return rc;
}
