// int_rates.cu — register-only microbenchmarks that fix the ALU roofline denominators of the sweep kernels on
// the box they run on: issue rate per SM per clock of the integer
// instructions the Metropolis path is made of, and the standalone Philox-4x32-10 (+4 compares) rate.
// Standalone program: prints a markdown table.  Not part of libspin.so and not used by the sweep path.
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o int_rates int_rates.cu && ./int_rates
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#define CK(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) { printf("CUDA error %s at %d\n", cudaGetErrorString(e_), __LINE__); return 1; } } while (0)

constexpr int kChains = 8;     // independent dependency chains per thread
constexpr int kInner = 64;     // unrolled ops per chain per outer iteration

enum Op { OP_LOP3, OP_IADD3, OP_IMAD, OP_WIDE, OP_HI, OP_HI_LO, OP_PRMT, OP_SETP_XOR, OP_WIDE_LOP3, OP_SHF, OP_WIDE_2LOP3, OP_WIDE_LOP3_ADD, OP_WIDE_LOP3_SETP, OP_L2I, OP_L2R, OP_L3R, OP_L3I, OP_ADD3R, OP_SETP_DEP, OP_VOTE, OP_LDS, OP_LDS_U8, OP_SEL, OP_DP4A, OP_PLOP_IMM, OP_CARRY, OP_COUNT };
static const char* kOpName[OP_COUNT] = {
    "LOP3 (3-input xor)", "IADD3", "IMAD (mad.lo.u32)", "IMAD.WIDE.U32 (mul.wide.u32)", "IMAD.HI.U32 (mul.hi.u32)",
    "mul.hi.u32 + mul.lo.u32 pair", "PRMT", "ISETP + predicated LOP3", "IMAD.WIDE.U32 + LOP3 (one Philox half-round)",
    "SHF (funnel shift)", "IMAD.WIDE.U32 + 2 LOP3", "IMAD.WIDE.U32 + LOP3 + IADD3", "IMAD.WIDE.U32 + LOP3 + ISETP + predicated LOP3",
    "LOP3 reg ^ imm", "LOP3 reg ^ reg", "LOP3 reg ^ reg ^ reg", "LOP3 reg ^ reg ^ imm", "IADD3 reg + reg + reg",
    "ISETP (data dependent) + predicated LOP3 imm", "VOTE.ballot + LOP3", "LDS (32-bit, data-dependent address)",
    "LDS.U8 (data-dependent address)", "ISETP + SEL", "IDP4A (dp4a.s32.u32 with accumulate)",
    "ISETP (uniform threshold) + predicated LOP3 reg | imm (2 ops; the per-site pair of the bit-sliced kernels)",
    "IADD3 carry-out + IADD3.X shift-in (add.cc / addc: compare bit shifted into a mask, 2 ops)"};
static const int kOpsPerStep[OP_COUNT] = {1, 1, 1, 1, 1, 2, 1, 2, 2, 1, 3, 3, 4, 1, 1, 1, 1, 1, 2, 2, 1, 1, 2, 1, 2, 2};

template <int kOp>
__device__ __forceinline__ void step(uint32_t& a, uint32_t& b, uint32_t k) {
    if (kOp == OP_LOP3) { asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a) : "r"(b), "r"(k)); }
    else if (kOp == OP_IADD3) { asm volatile("add.u32 %0, %0, %1;" : "+r"(a) : "r"(b)); }
    else if (kOp == OP_IMAD) { asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(a) : "r"(k), "r"(b)); }
    else if (kOp == OP_WIDE) {
        uint64_t p; asm volatile("mul.wide.u32 %0, %1, %2;" : "=l"(p) : "r"(a), "r"(k));
        asm volatile("mov.b64 {%0, %1}, %2;" : "=r"(b), "=r"(a) : "l"(p));
    }
    else if (kOp == OP_HI) { asm volatile("mul.hi.u32 %0, %0, %1;" : "+r"(a) : "r"(k)); }
    else if (kOp == OP_HI_LO) {
        uint32_t h; asm volatile("mul.hi.u32 %0, %1, %2;" : "=r"(h) : "r"(a), "r"(k));
        asm volatile("mul.lo.u32 %0, %1, %2;" : "=r"(b) : "r"(a), "r"(k)); a = h;
    }
    else if (kOp == OP_PRMT) { asm volatile("prmt.b32 %0, %0, %1, 0x4321;" : "+r"(a) : "r"(b)); }
    else if (kOp == OP_SETP_XOR) {
        asm volatile("{\n\t.reg .pred p;\n\tsetp.ls.u32 p, %1, %2;\n\t@p xor.b32 %0, %0, 0xFE;\n\t}" : "+r"(a) : "r"(b), "r"(k));
    }
    else if (kOp == OP_WIDE_LOP3) {
        uint64_t p; uint32_t lo, hi; asm volatile("mul.wide.u32 %0, %1, %2;" : "=l"(p) : "r"(a), "r"(k));
        asm volatile("mov.b64 {%0, %1}, %2;" : "=r"(lo), "=r"(hi) : "l"(p));
        asm volatile("lop3.b32 %0, %1, %2, %3, 0x96;" : "=r"(a) : "r"(hi), "r"(b), "r"(k)); b = lo;
    }
    else if (kOp == OP_WIDE_2LOP3 || kOp == OP_WIDE_LOP3_ADD || kOp == OP_WIDE_LOP3_SETP) {
        uint64_t p; uint32_t lo, hi; asm volatile("mul.wide.u32 %0, %1, %2;" : "=l"(p) : "r"(a), "r"(k));
        asm volatile("mov.b64 {%0, %1}, %2;" : "=r"(lo), "=r"(hi) : "l"(p));
        asm volatile("lop3.b32 %0, %1, %2, %3, 0x96;" : "=r"(a) : "r"(hi), "r"(b), "r"(k));
        if (kOp == OP_WIDE_2LOP3) asm volatile("lop3.b32 %0, %1, %2, %3, 0x96;" : "=r"(b) : "r"(lo), "r"(b), "r"(k));
        else if (kOp == OP_WIDE_LOP3_ADD) asm volatile("add.u32 %0, %1, %2;" : "=r"(b) : "r"(lo), "r"(b));
        else asm volatile("{\n\t.reg .pred p;\n\tsetp.ls.u32 p, %1, %2;\n\t@p xor.b32 %0, %0, 0xFE;\n\t}" : "+r"(b) : "r"(lo), "r"(k));
    }
    else if (kOp == OP_L2I) { asm volatile("xor.b32 %0, %0, 0x9E3779B9;" : "+r"(a)); }
    else if (kOp == OP_L2R) { asm volatile("xor.b32 %0, %0, %1;" : "+r"(a) : "r"(b)); }
    else if (kOp == OP_L3R) { asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a) : "r"(b), "r"(k)); }   // k is per-thread here
    else if (kOp == OP_L3I) { asm volatile("lop3.b32 %0, %0, %1, 0x9E3779B9, 0x96;" : "+r"(a) : "r"(b)); }
    else if (kOp == OP_ADD3R) { asm volatile("{\n\t.reg .u32 t;\n\tadd.u32 t, %0, %1;\n\tadd.u32 %0, t, %2;\n\t}" : "+r"(a) : "r"(b), "r"(k)); }
    else if (kOp == OP_SETP_DEP) {
        asm volatile("{\n\t.reg .pred p;\n\tsetp.ls.u32 p, %0, %1;\n\t@p xor.b32 %0, %0, 0xFE01;\n\t@!p add.u32 %0, %0, 0x1234567;\n\t}" : "+r"(a) : "r"(b));
    }
    else if (kOp == OP_VOTE) {
        asm volatile("{\n\t.reg .pred p;\n\t.reg .b32 t;\n\tsetp.ls.u32 p, %0, %1;\n\tvote.sync.ballot.b32 t, p, 0xffffffff;\n\txor.b32 %0, %0, t;\n\t}" : "+r"(a) : "r"(b));
    }
    else if (kOp == OP_LDS) { asm volatile("ld.shared.u32 %0, [%0];" : "+r"(a)); }
    else if (kOp == OP_LDS_U8) { asm volatile("ld.shared.u8 %0, [%0];" : "+r"(a)); }
    else if (kOp == OP_SEL) {
        asm volatile("{\n\t.reg .pred p;\n\tsetp.ls.u32 p, %0, %1;\n\tselp.b32 %0, %1, %2, p;\n\t}" : "+r"(a) : "r"(b), "r"(k));
    }
    else if (kOp == OP_DP4A) { asm volatile("dp4a.s32.u32 %0, %1, %2, %0;" : "+r"(a) : "r"(b), "r"(k)); }
    else if (kOp == OP_PLOP_IMM) {
        // a plays the random word (changes every step), b collects the predicate bits
        asm volatile("{\n\t.reg .pred p;\n\tsetp.ls.u32 p, %1, %2;\n\t@p or.b32 %0, %0, 0x10;\n\t}" : "+r"(b) : "r"(a), "r"(k));
        asm volatile("add.u32 %0, %0, %1;" : "+r"(a) : "r"(b));
    }
    else if (kOp == OP_CARRY) {
        asm volatile("{\n\t.reg .u32 t;\n\tadd.cc.u32 t, %1, %2;\n\taddc.u32 %0, %0, %0;\n\t}" : "+r"(b) : "r"(a), "r"(k));
        asm volatile("add.u32 %0, %0, %1;" : "+r"(a) : "r"(b));
    }
    else if (kOp == OP_SHF) { asm volatile("shf.l.wrap.b32 %0, %0, %1, 7;" : "+r"(a) : "r"(b)); }
}

template <int kOp>
__global__ void __launch_bounds__(256) op_kernel(uint32_t* out, int outer, uint32_t k) {
    uint32_t a[kChains], b[kChains];
    __shared__ uint32_t sm[256];
    if (kOp == OP_LDS || kOp == OP_LDS_U8) {
        // every word holds a 4-aligned byte offset < 256 (so does every byte, for the U8 form): pointer chasing
        sm[threadIdx.x] = (kOp == OP_LDS) ? ((threadIdx.x * 37u + 11u) & 63u) * 4u : 0x04040404u * ((threadIdx.x * 5u + 3u) & 63u);
        __syncthreads();
    }
#pragma unroll
    for (int c = 0; c < kChains; ++c) {
        a[c] = threadIdx.x * 2654435761u + c; b[c] = blockIdx.x + 77u * c;
        if (kOp == OP_LDS || kOp == OP_LDS_U8) a[c] = (uint32_t)__cvta_generic_to_shared(sm) + ((threadIdx.x + c) & 63u) * 4u;
    }
    const uint32_t kk = (kOp == OP_L3R) ? (k ^ threadIdx.x) : k;   // a vector register for the 3-register form
    for (int o = 0; o < outer; ++o) {
#pragma unroll
        for (int i = 0; i < kInner; ++i) {
#pragma unroll
            for (int c = 0; c < kChains; ++c) step<kOp>(a[c], b[c], kk);
        }
    }
    uint32_t s = 0;
#pragma unroll
    for (int c = 0; c < kChains; ++c) s ^= a[c] ^ b[c];
    if (s == 0x12345678u) out[0] = s;   // never true in practice; keeps the chains alive
}

// Philox-4x32-10 with host-precomputed round keys, then 4 compares folded into one word (the algorithmic work of
// 4 Ising updates: "Philox plus compare").  kCalls independent calls per iteration.  kVariant selects how the
// multipliers / round keys reach the instructions: 0 = immediates + uniform registers (what nvcc does by default),
// 1 = multipliers in vector registers, 2 = round keys in vector registers, 3 = both.
struct Keys { uint32_t k0[10], k1[10]; };
template <int kCalls, int kVariant>
__global__ void __launch_bounds__(256) philox_kernel(uint32_t* out, int outer, Keys rk, uint32_t thr) {
    uint32_t acc = 0;
    uint32_t g = (blockIdx.x * blockDim.x + threadIdx.x) * kCalls;
    uint32_t m0 = 0xD2511F53u, m1 = 0xCD9E8D57u;
    const volatile uint32_t* vec = out + 8 + (threadIdx.x & 1);   // per-thread loads: values live in vector registers
    if (kVariant & 1) { m0 = vec[0]; m1 = vec[2]; }
    uint32_t k0[10], k1[10];
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        k0[r] = rk.k0[r]; k1[r] = rk.k1[r];
        if (kVariant & 2) { k0[r] = vec[4 + 4 * r]; k1[r] = vec[6 + 4 * r]; }
    }
    for (int o = 0; o < outer; ++o) {
#pragma unroll
        for (int c = 0; c < kCalls; ++c) {
            uint32_t c0 = g + c + (acc & 2u), c1 = acc & 1u, c2 = o + (acc & 4u), c3 = 0x11000000u;   // thread-dependent: no hoisting
#pragma unroll
            for (int r = 0; r < 10; ++r) {
                const uint64_t p0 = (uint64_t)m0 * c0, p1 = (uint64_t)m1 * c2;
                const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0[r], n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1[r];
                c1 = (uint32_t)p1; c3 = (uint32_t)p0; c0 = n0; c2 = n2;
            }
            asm volatile("{\n\t.reg .pred p;\n\tsetp.ls.u32 p, %1, %2;\n\t@p xor.b32 %0, %0, 0xFE;\n\t}" : "+r"(acc) : "r"(c0), "r"(thr));
            asm volatile("{\n\t.reg .pred p;\n\tsetp.ls.u32 p, %1, %2;\n\t@p xor.b32 %0, %0, 0xFE00;\n\t}" : "+r"(acc) : "r"(c1), "r"(thr));
            asm volatile("{\n\t.reg .pred p;\n\tsetp.ls.u32 p, %1, %2;\n\t@p xor.b32 %0, %0, 0xFE0000;\n\t}" : "+r"(acc) : "r"(c2), "r"(thr));
            asm volatile("{\n\t.reg .pred p;\n\tsetp.ls.u32 p, %1, %2;\n\t@p xor.b32 %0, %0, 0xFE000000;\n\t}" : "+r"(acc) : "r"(c3), "r"(thr));
        }
    }
    if (acc == 0x12345679u) out[1] = acc;
}

static int g_sms = 0;
static double g_mhz = 0;

template <typename F>
static int time_kernel(F launch, double* ms_out) {
    cudaEvent_t e0, e1;
    CK(cudaEventCreate(&e0)); CK(cudaEventCreate(&e1));
    launch(); launch();
    CK(cudaDeviceSynchronize());
    float best = 1e30f;
    for (int rep = 0; rep < 5; ++rep) {
        CK(cudaEventRecord(e0)); launch(); CK(cudaEventRecord(e1)); CK(cudaEventSynchronize(e1));
        float ms; CK(cudaEventElapsedTime(&ms, e0, e1)); if (ms < best) best = ms;
    }
    CK(cudaGetLastError());
    *ms_out = best;
    return 0;
}

template <int kOp>
static int run_op(uint32_t* d, int warps_per_smsp) {
    const int threads = 256, blocks = g_sms * warps_per_smsp * 4 * 32 / threads, outer = 400;
    double ms;
    if (time_kernel([&] { op_kernel<kOp><<<blocks, threads>>>(d, outer, 0xD2511F53u); }, &ms)) return 1;
    const double steps = (double)blocks * threads * outer * kInner * kChains;
    const double per_s = steps * kOpsPerStep[kOp] / (ms * 1e-3);
    printf("| %s | %d | %.2f | %.2f | %.1f |\n", kOpName[kOp], warps_per_smsp, per_s / 1e12,
           per_s / (g_sms * g_mhz * 1e6), 32.0 * 4.0 / (per_s / kOpsPerStep[kOp] / (g_sms * g_mhz * 1e6)));
    return 0;
}

template <int kCalls, int kVariant>
static int run_philox(uint32_t* d, int warps_per_smsp) {
    const int threads = 256, blocks = g_sms * warps_per_smsp * 4 * 32 / threads, outer = 2000;
    Keys rk; uint32_t k0 = 1, k1 = 0;
    for (int r = 0; r < 10; ++r) { rk.k0[r] = k0; rk.k1[r] = k1; k0 += 0x9E3779B9u; k1 += 0xBB67AE85u; }
    double ms;
    if (time_kernel([&] { philox_kernel<kCalls, kVariant><<<blocks, threads>>>(d, outer, rk, 0x2c0b21d7u); }, &ms)) return 1;
    const double calls = (double)blocks * threads * outer * kCalls;
    printf("| Philox-4x32-10 + 4 compares, %d calls in flight per thread, operand variant %d | %d | %.1f words/ns | %.2f Tint32op/s (44 ops/call) | %.1f cyc/call/SMSP |\n",
           kCalls, kVariant, warps_per_smsp, 4.0 * calls / (ms * 1e6), 44.0 * calls / (ms * 1e-3) / 1e12,
           (ms * 1e-3) * g_mhz * 1e6 / (calls / 32.0 / (g_sms * 4.0)));
    return 0;
}

int main(int argc, char** argv) {
    const bool only_philox = argc > 1;   // any argument: only the half-round and Philox kernels (for ncu captures)
    cudaDeviceProp p; CK(cudaGetDeviceProperties(&p, 0));
    int khz = 0; CK(cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, 0));
    g_sms = p.multiProcessorCount; g_mhz = khz / 1e3;
    printf("# integer issue rates, %s, %d SMs, max SM clock %.0f MHz (rates per clock assume the max clock)\n\n", p.name, g_sms, g_mhz);
    uint32_t* d; CK(cudaMalloc(&d, 4096));
    {   // out[8..]: multipliers and round keys for the "vector register" operand variants (each value stored twice)
        uint32_t h[1024] = {0}; uint32_t a = 1, b = 0;
        h[8] = h[9] = 0xD2511F53u; h[10] = h[11] = 0xCD9E8D57u;
        for (int r = 0; r < 10; ++r) { h[12 + 4 * r] = h[13 + 4 * r] = a; h[14 + 4 * r] = h[15 + 4 * r] = b; a += 0x9E3779B9u; b += 0xBB67AE85u; }
        CK(cudaMemcpy(d, h, sizeof(h), cudaMemcpyHostToDevice));
    }
    printf("| instruction | warps/SMSP | T op/s | lanes/SM/clk | cycles per warp instruction per SMSP |\n|---|---|---|---|---|\n");
    for (int w : {4, 8}) {
        if (only_philox) { if (run_op<OP_WIDE_LOP3>(d, w) || run_op<OP_WIDE_2LOP3>(d, w) || run_op<OP_WIDE_LOP3_ADD>(d, w) || run_op<OP_WIDE_LOP3_SETP>(d, w)) return 1; continue; }
        if (run_op<OP_LOP3>(d, w) || run_op<OP_IADD3>(d, w) || run_op<OP_IMAD>(d, w) || run_op<OP_WIDE>(d, w) ||
            run_op<OP_HI>(d, w) || run_op<OP_HI_LO>(d, w) || run_op<OP_PRMT>(d, w) || run_op<OP_SHF>(d, w) ||
            run_op<OP_SETP_XOR>(d, w) || run_op<OP_WIDE_LOP3>(d, w) || run_op<OP_WIDE_2LOP3>(d, w) || run_op<OP_WIDE_LOP3_ADD>(d, w) || run_op<OP_WIDE_LOP3_SETP>(d, w) || run_op<OP_L2I>(d, w) || run_op<OP_L2R>(d, w) || run_op<OP_L3R>(d, w) || run_op<OP_L3I>(d, w) || run_op<OP_ADD3R>(d, w) || run_op<OP_SETP_DEP>(d, w) || run_op<OP_VOTE>(d, w) || run_op<OP_SEL>(d, w) || run_op<OP_LDS>(d, w) || run_op<OP_LDS_U8>(d, w) || run_op<OP_DP4A>(d, w) || run_op<OP_PLOP_IMM>(d, w) || run_op<OP_CARRY>(d, w)) return 1;
    }
    printf("\n| kernel | warps/SMSP | rate | | |\n|---|---|---|---|---|\n");
    for (int w : {4, 8}) {
        if (run_philox<1, 0>(d, w) || run_philox<2, 0>(d, w) || run_philox<4, 0>(d, w) || run_philox<2, 1>(d, w) || run_philox<2, 2>(d, w) || run_philox<2, 3>(d, w)) return 1;
    }
    return 0;
}
