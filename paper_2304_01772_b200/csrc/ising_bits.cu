// ising_bits.cu — rows a2/a3 for the Ising model in the bit-packed (multi-spin coded) layout
// [B][2][L][L/64] uint32, bit b of word w = same-colour site k = 32 w + b of that row, bit set = spin -1.
// Same rule, same Philox words as the int8 kernels (Alg. 1 + checkerboard).
// One thread per word = 32 sites = 8 Philox calls.  The neighbour count is a bit-sliced full adder; the
// 4-bit class index of every site is assembled nibble-parallel (8 sites per LOP3) and looked up through shared
// memory, so the per-site work is two byte-addressed loads + compare + select.
#include "spin_internal.cuh"

namespace spin {

namespace {

__device__ __forceinline__ uint32_t sel(uint32_t m, uint32_t a, uint32_t b) { return (a & m) | (b & ~m); }

constexpr int kRowsLong = 8;    // rows per thread when the launch fills the GPU several times over
constexpr int kRowsMid = 4;     // under about one wave of 8-row blocks
constexpr int kRowsShort = 2;   // latency-bound shapes: short threads, four times as many
constexpr int kThreads = 128;
constexpr int kMinBlocks = kIsingBitsBlocksPerSm;   // resident blocks per SM (spin_internal.cuh)

// One word = 32 sites = 8 Philox calls.  up / dn / ct: other-colour words of rows i-1, i+1, i; sd: the side
// neighbours (ct shifted by one site, with the bit of the adjacent word).  The class nibbles of the 32 sites are
// assembled nibble-parallel into t[0..3] (site 4c+e in nibble c of t[e], bit order rotated by e), stored to a
// per-thread shared-memory slot, and read back a byte (two sites) at a time; a constant byte table turns that byte
// into 4 * class of its low / high nibble, which is the address of the threshold: per site LDS.U8, LDS, ISETP and a
// select, no extraction arithmetic (the LSU has the headroom, the integer issue slots do not).
template <int kOff>
__device__ __forceinline__ uint32_t slot_load_u8(uint32_t saddr) {
    uint32_t v;
    asm volatile("ld.shared.u8 %0, [%1+%2];" : "=r"(v) : "r"(saddr), "n"(kOff));
    return v;
}

template <int kOff>
__device__ __forceinline__ void slot_store_u32(uint32_t saddr, uint32_t v) {
    asm volatile("st.shared.u32 [%0+%1], %2;" :: "r"(saddr), "n"(kOff), "r"(v));
}

constexpr int kAuxBytes = 2048;            // [e][half][byte] -> 4 * class

template <bool kHasNever, int kC, int kE>
__device__ __forceinline__ void site_step(uint32_t& flip, uint32_t v, uint32_t r, const uint32_t* stab,
                                          const uint8_t* sT, uint32_t never) {
    const uint32_t c4 = sT[(kE * 2 + (kC & 1)) * 256 + v];
    const uint32_t U = *(const uint32_t*)((const char*)stab + c4);
    bool acc = r <= U;
    if (kHasNever) acc = acc && !((never >> (c4 >> 2)) & 1u);
    if (acc) flip |= 1u << (4 * kC + kE);
}

template <bool kHasNever, int kC>
__device__ __forceinline__ void group_step(uint32_t& flip, const uint32_t r[4], const uint32_t v[4], const uint32_t* stab,
                                           const uint8_t* sT, uint32_t never) {
    site_step<kHasNever, kC, 0>(flip, v[0], r[0], stab, sT, never);
    site_step<kHasNever, kC, 1>(flip, v[1], r[1], stab, sT, never);
    site_step<kHasNever, kC, 2>(flip, v[2], r[2], stab, sT, never);
    site_step<kHasNever, kC, 3>(flip, v[3], r[3], stab, sT, never);
}

// Two Philox groups (sites 8p .. 8p+7) share one byte of each t[e].
template <bool kHasNever, int kP>
__device__ __forceinline__ void pair_step(const PhiloxCtx& a, uint32_t& flip, uint32_t g0, uint32_t c1,
                                          const uint32_t* stab, const uint8_t* sT, uint32_t never, uint32_t slot) {
    uint32_t v[4];
    v[0] = slot_load_u8<0 * kThreads * 4 + kP>(slot);
    v[1] = slot_load_u8<1 * kThreads * 4 + kP>(slot);
    v[2] = slot_load_u8<2 * kThreads * 4 + kP>(slot);
    v[3] = slot_load_u8<3 * kThreads * 4 + kP>(slot);
    uint32_t r[4];
    philox4x32_10(a.rk, g0 + 2 * kP, c1, a.c2, a.c3, r);
    group_step<kHasNever, 2 * kP>(flip, r, v, stab, sT, never);
    philox4x32_10(a.rk, g0 + 2 * kP + 1, c1, a.c2, a.c3, r);
    group_step<kHasNever, 2 * kP + 1>(flip, r, v, stab, sT, never);
}

template <bool kHasNever>
__device__ __forceinline__ uint32_t update_word(const PhiloxCtx& a, uint32_t own, uint32_t up, uint32_t dn, uint32_t ct,
                                                uint32_t sd, uint32_t g0, uint32_t c1, const uint32_t* stab,
                                                const uint8_t* sT, uint32_t never, uint32_t slot) {
    // bit-sliced count of -1 neighbours: nd = P0 + 2 P1 + 4 P2
    const uint32_t s1 = up ^ dn ^ ct;
    const uint32_t k1 = (up & dn) | (ct & (up | dn));
    const uint32_t P0 = s1 ^ sd;
    const uint32_t k2 = s1 & sd;
    const uint32_t P1 = k1 ^ k2;
    const uint32_t P2 = k1 & k2;
    const uint32_t P1a = P1 << 1, P1b = P1 >> 3, P2a = P2 << 2, P2b = P2 >> 2, Da = own << 3, Db = own >> 1;
    slot_store_u32<0 * kThreads * 4>(slot, sel(0x11111111u, P0, sel(0x22222222u, P1a, sel(0x44444444u, P2a, Da))));
    slot_store_u32<1 * kThreads * 4>(slot, sel(0x11111111u, Db, sel(0x22222222u, P0, sel(0x44444444u, P1a, P2a))));
    slot_store_u32<2 * kThreads * 4>(slot, sel(0x11111111u, P2b, sel(0x22222222u, Db, sel(0x44444444u, P0, P1a))));
    slot_store_u32<3 * kThreads * 4>(slot, sel(0x11111111u, P1b, sel(0x22222222u, P2b, sel(0x44444444u, Db, P0))));
    uint32_t flip = 0u;
    pair_step<kHasNever, 0>(a, flip, g0, c1, stab, sT, never, slot);
    pair_step<kHasNever, 1>(a, flip, g0, c1, stab, sT, never, slot);
    pair_step<kHasNever, 2>(a, flip, g0, c1, stab, sT, never, slot);
    pair_step<kHasNever, 3>(a, flip, g0, c1, stab, sT, never, slot);
    return own ^ flip;
}

// Row-marching: one thread owns word x of kRows consecutive rows (same skeleton as ising_int8.cu: the three
// other-colour words it needs stay in registers, running pointers, two rows per rolled iteration because the side
// of the horizontal neighbour alternates, programmatic dependent launch).
// kBonds: +-J couplings (SweepArgs::bonds): the neighbour words are XORed with the sign planes of the bonds that
// join them to the row's sites, so the adder counts neighbours whose bond-weighted spin is -1; nothing else changes.
template <int kColour, bool kHasNever, int kRows, bool kBonds>
__device__ __forceinline__ void march_rows(const SweepArgs& a, const PhiloxCtx& pc, const uint32_t* stab, const uint8_t* sT, uint32_t never,
                                           uint32_t slot, int b, int rb, int x) {
    const int L = a.L, WW = L >> 6;                       // words per colour-row
    const size_t half = (size_t)L * WW;
    const int i0 = rb * kRows;
    uint32_t* pOwn = (uint32_t*)a.lattice + ((size_t)b * 2 + kColour) * half + (size_t)i0 * WW + x;
    const uint32_t* oth = (const uint32_t*)a.lattice + ((size_t)b * 2 + (1 - kColour)) * half;
    const int xNext = (x == WW - 1) ? 0 : x + 1, xPrev = (x == 0) ? WW - 1 : x - 1;
    const int iu = i0 == 0 ? L - 1 : i0 - 1;
    const int iLast = (i0 + kRows == L) ? 0 : i0 + kRows;
    const uint32_t* pOth = oth + (size_t)(i0 + 2) * WW + x;
    const uint32_t* pOthLast = oth + (size_t)iLast * WW + x;
    // even rows of the block have parity kColour (side neighbour k+1 iff parity 1), odd rows 1 - kColour
    const uint32_t* pEdgeEven = oth + (size_t)i0 * WW + (kColour ? xNext : xPrev);
    const uint32_t* pEdgeOdd = oth + (size_t)(i0 + 1) * WW + (kColour ? xPrev : xNext);
    const size_t rowStride = (size_t)WW;
    uint32_t wU = __ldg(oth + (size_t)iu * WW + x);
    uint32_t wC = __ldg(pOth - 2 * rowStride);
    uint32_t wD = __ldg(pOth - rowStride);
    uint32_t own = *pOwn;
    uint32_t edge = __ldg(pEdgeEven);
    uint32_t g0 = (uint32_t)i0 * (uint32_t)(L >> 3) + 8u * (uint32_t)x;   // (i*(L/2) + 32x) >> 2
    const uint32_t c1 = (uint32_t)b + a.replica_offset;
    // bond sign planes of this colour: plane p of row i, word x at pB[p * half + i * WW + x]
    const uint32_t* pB = kBonds ? a.bonds + ((size_t)b * 2 + kColour) * 4 * half + (size_t)i0 * WW + x : nullptr;
#pragma unroll 1
    for (int rr = 0; rr < kRows; rr += 2) {
        const bool more = rr + 2 < kRows;
        if (!more && a.pdl_trigger == kPdlLastRows) pdl_launch_dependents();
        const uint32_t n1 = __ldg(more ? pOth : pOthLast);
        const uint32_t own1 = *(pOwn + rowStride);
        const uint32_t edge1 = __ldg(pEdgeOdd);
        uint32_t bu = 0u, bd = 0u, bc = 0u, bs = 0u, bu1 = 0u, bd1 = 0u, bc1 = 0u, bs1 = 0u;
        if (kBonds) {
            bu = __ldg(pB); bd = __ldg(pB + half); bc = __ldg(pB + 2 * half); bs = __ldg(pB + 3 * half);
            bu1 = __ldg(pB + rowStride); bd1 = __ldg(pB + half + rowStride);
            bc1 = __ldg(pB + 2 * half + rowStride); bs1 = __ldg(pB + 3 * half + rowStride);
            pB += 2 * rowStride;
        }
        uint32_t sd = kColour ? ((wC >> 1) | (edge << 31)) : ((wC << 1) | (edge >> 31));
        *pOwn = update_word<kHasNever>(pc, own, wU ^ bu, wD ^ bd, wC ^ bc, sd ^ bs, g0, c1, stab, sT, never, slot);
        uint32_t n2 = n1, own2 = own1, edge2 = edge1;
        if (more) {
            n2 = __ldg(pOth + rowStride);
            own2 = *(pOwn + 2 * rowStride);
            edge2 = __ldg(pEdgeEven + 2 * rowStride);
        }
        sd = kColour ? ((wD << 1) | (edge1 >> 31)) : ((wD >> 1) | (edge1 << 31));
        *(pOwn + rowStride) = update_word<kHasNever>(pc, own1, wC ^ bu1, n1 ^ bd1, wD ^ bc1, sd ^ bs1, g0 + (uint32_t)(L >> 3),
                                                     c1, stab, sT, never, slot);
        wU = wD;
        wC = n1;
        wD = n2;
        own = own2;
        edge = edge2;
        pOth += 2 * rowStride;
        pOwn += 2 * rowStride;
        pEdgeEven += 2 * rowStride;
        pEdgeOdd += 2 * rowStride;
        g0 += (uint32_t)(L >> 2);
    }
}

template <int kColour, int kRows, bool kBonds, bool kDevT>
__global__ void __launch_bounds__(kThreads, kMinBlocks) ising_bits_kernel(SweepArgs a, int bpr) {
    __shared__ uint32_t stab[16];                          // U[class], class = d * 8 + nd
    __shared__ __align__(16) uint8_t sT[kAuxBytes];        // [e][half][byte] -> 4 * class
    __shared__ uint32_t sidx[4 * kThreads];                // per-thread slot: word e of thread t at sidx[e * 128 + t]
    if (a.pdl_trigger == kPdlAtStart) pdl_launch_dependents();
    const int b = blockIdx.x / bpr;
    const int blk = blockIdx.x - b * bpr;
    for (int k = threadIdx.x; k < kAuxBytes / 16; k += blockDim.x) ((uint4*)sT)[k] = ((const uint4*)a.aux)[k];   // constant
    pdl_wait();
    uint32_t c2, c3;
    sweep_counter_words<kDevT>(a, c2, c3);
    const PhiloxCtx pc = {a.rk, c2, c3};
    const uint32_t* tab = a.tables + (size_t)b * kTableStride;
    const uint32_t never = tab[kTabNever];
    for (int m = threadIdx.x; m < 16; m += blockDim.x) stab[m] = tab[m];
    __syncthreads();
    const uint32_t slot = (uint32_t)__cvta_generic_to_shared(&sidx[threadIdx.x]);
    const int WW = a.L >> 6;
    const int u = blk * blockDim.x + threadIdx.x;
    if (u >= (a.L / kRows) * WW) return;                  // ragged last block of a replica (after the barrier)
    const int rb = u / WW, x = u - rb * WW;
    if (never) march_rows<kColour, true, kRows, kBonds>(a, pc, stab, sT, never, slot, b, rb, x);
    else march_rows<kColour, false, kRows, kBonds>(a, pc, stab, sT, never, slot, b, rb, x);
}

// ---- shared-memory-resident kernel ("a 1024^2 replica is 128 KiB as bits and fits one CTA"): one CTA per
// replica keeps both colours in shared memory and runs every sweep of a call in one launch, half-sweeps separated by
// __syncthreads(): zero HBM traffic per sweep.  One thread per 32-site word per pass; the side of the horizontal
// neighbour depends on the row parity and is handled with selects (no divergence).  The kernels are ALU-bound, so this
// only removes launch gaps; with one CTA per replica it needs a batch of at least the SM count to match the streaming
// kernels and is used on request (SPIN_POLICY_RESIDENT), not by AUTO.
constexpr int kBitsResThreads = 256;

__global__ void __launch_bounds__(kBitsResThreads) ising_bits_resident_kernel(ResidentArgs a, const uint8_t* __restrict__ aux) {
    extern __shared__ __align__(16) uint32_t blat[];          // [2][L][L/64] words
    __shared__ uint32_t stab[16];
    __shared__ __align__(16) uint8_t sT[kAuxBytes];
    __shared__ uint32_t sidx[4 * kBitsResThreads];            // word e of thread t at [(t >> 7) * 512 + e * 128 + (t & 127)]
    const int L = a.L, WW = L >> 6, half = L * WW;
    const int b = blockIdx.x;
    uint32_t* g = (uint32_t*)a.lattice + (size_t)b * 2 * half;
    for (int k = threadIdx.x; k < 2 * half; k += blockDim.x) blat[k] = g[k];
    for (int k = threadIdx.x; k < kAuxBytes / 16; k += blockDim.x) ((uint4*)sT)[k] = ((const uint4*)aux)[k];
    const uint32_t* tab = a.tables + (size_t)b * kTableStride;
    if (threadIdx.x < 16) stab[threadIdx.x] = tab[threadIdx.x];
    const uint32_t never = tab[kTabNever];
    __syncthreads();
    const uint32_t slot = (uint32_t)__cvta_generic_to_shared(&sidx[(threadIdx.x >> 7) * 512 + (threadIdx.x & 127)]);
    const uint32_t c1 = (uint32_t)b + a.replica_offset;
    SweepArgs sa;                                             // update_word reads rk, c2, c3 from here
    sa.rk = a.rk;
    for (long long s = 0; s < a.n_sweeps; ++s) {
        const unsigned long long t = a.t0 + (unsigned long long)s;
        sa.c2 = (uint32_t)(t & 0xFFFFFFFFull);
        for (int colour = 0; colour < 2; ++colour) {
            sa.c3 = (uint32_t)((t >> 32) & 0xFFFFFFull) | ((uint32_t)colour << 24) | (kDomainIsing << 28);
            uint32_t* own1 = blat + colour * half;
            const uint32_t* oth1 = blat + (1 - colour) * half;
            for (int w = threadIdx.x; w < half; w += blockDim.x) {
                const int i = w / WW, x = w - i * WW;
                const int iu = i == 0 ? L - 1 : i - 1, id = i == L - 1 ? 0 : i + 1;
                const bool par = ((i + colour) & 1) != 0;     // side neighbour of site k: k+1 if par else k-1
                const uint32_t ct = oth1[w];
                const uint32_t ew = oth1[i * WW + (par ? (x == WW - 1 ? 0 : x + 1) : (x == 0 ? WW - 1 : x - 1))];
                const uint32_t sd = par ? ((ct >> 1) | (ew << 31)) : ((ct << 1) | (ew >> 31));
                const uint32_t g0 = (uint32_t)i * (uint32_t)(L >> 3) + 8u * (uint32_t)x;
                uint32_t res;
                if (never) res = update_word<true>(PhiloxCtx{sa.rk, sa.c2, sa.c3}, own1[w], oth1[iu * WW + x], oth1[id * WW + x], ct, sd, g0, c1, stab, sT, never, slot);
                else res = update_word<false>(PhiloxCtx{sa.rk, sa.c2, sa.c3}, own1[w], oth1[iu * WW + x], oth1[id * WW + x], ct, sd, g0, c1, stab, sT, never, slot);
                own1[w] = res;
            }
            __syncthreads();
        }
    }
    for (int k = threadIdx.x; k < 2 * half; k += blockDim.x) g[k] = blat[k];
}

}  // namespace

bool ising_bits_resident_fits(int L) { return L % 64 == 0 && (size_t)L * L / 8 <= 200 * 1024; }

int launch_ising_bits_resident(const ResidentArgs& a, const uint8_t* aux, cudaStream_t s) {
    if (cudaFuncSetAttribute(ising_bits_resident_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024) != cudaSuccess) {
        cudaGetLastError();
        return 0;
    }
    ising_bits_resident_kernel<<<(unsigned)a.batch, kBitsResThreads, (size_t)a.L * a.L / 8, s>>>(a, aux);
    return 1;
}

// Host side of the constant lookup table: entry [e][half][v] = 4 * class of the low (half 0) / high (half 1) nibble
// of v, where the nibble of a site 4c+e holds (D, P2, P1, P0) rotated by e bits (see update_word).
uint8_t* ising_bits_make_aux_table() {
    {
        uint8_t h[kAuxBytes];
        for (int e = 0; e < 4; ++e)
            for (int half = 0; half < 2; ++half)
                for (int v = 0; v < 256; ++v) {
                    const int nib = half ? (v >> 4) : (v & 15);
                    const int b0 = nib & 1, b1 = (nib >> 1) & 1, b2 = (nib >> 2) & 1, b3 = (nib >> 3) & 1;
                    int D, P0, P1, P2;
                    switch (e) {
                        case 0: P0 = b0; P1 = b1; P2 = b2; D = b3; break;
                        case 1: D = b0; P0 = b1; P1 = b2; P2 = b3; break;
                        case 2: P2 = b0; D = b1; P0 = b2; P1 = b3; break;
                        default: P1 = b0; P2 = b1; D = b2; P0 = b3; break;
                    }
                    h[(e * 2 + half) * 256 + v] = (uint8_t)(4 * (D * 8 + P2 * 4 + P1 * 2 + P0));
                }
        uint8_t* p = nullptr;
        if (cudaMalloc(&p, kAuxBytes) != cudaSuccess) return nullptr;
        if (cudaMemcpy(p, h, kAuxBytes, cudaMemcpyHostToDevice) != cudaSuccess) { cudaFree(p); return nullptr; }
        return p;
    }
}

// The instantiation for (rows per thread, colour, +-J couplings); kDevT: sweep index from device memory (graph nodes).
template <bool kDevT>
static void (*pick_bits_kernel(int rows, int colour, bool bonds))(SweepArgs, int) {
    if (rows == kRowsShort) {
        if (bonds) return colour == 0 ? ising_bits_kernel<0, kRowsShort, true, kDevT> : ising_bits_kernel<1, kRowsShort, true, kDevT>;
        return colour == 0 ? ising_bits_kernel<0, kRowsShort, false, kDevT> : ising_bits_kernel<1, kRowsShort, false, kDevT>;
    }
    if (rows == kRowsMid) {
        if (bonds) return colour == 0 ? ising_bits_kernel<0, kRowsMid, true, kDevT> : ising_bits_kernel<1, kRowsMid, true, kDevT>;
        return colour == 0 ? ising_bits_kernel<0, kRowsMid, false, kDevT> : ising_bits_kernel<1, kRowsMid, false, kDevT>;
    }
    if (bonds) return colour == 0 ? ising_bits_kernel<0, kRowsLong, true, kDevT> : ising_bits_kernel<1, kRowsLong, true, kDevT>;
    return colour == 0 ? ising_bits_kernel<0, kRowsLong, false, kDevT> : ising_bits_kernel<1, kRowsLong, false, kDevT>;
}

int launch_ising_bits_half_sweep(const SweepArgs& a, cudaStream_t s) {
    // rows per thread and release point: measured crossovers of this kernel (148 x kMinBlocks block slots); the
    // smallest launches do best when the next one is released as soon as a thread has its first rows in registers
    const int perReplica8 = (a.L / kRowsLong) * (a.L >> 6);
    const long long threads8 = (long long)perReplica8 * a.batch * (a.plan_scale > 0 ? a.plan_scale : 1);
    RowsPlan plan = plan_rows(threads8, perReplica8, 148 * kMinBlocks, 0.3, 0.75, false);
    if (plan.rows == kRowsShort && threads8 < 148ll * kMinBlocks * 128 / 10) plan.trigger = kPdlLastRows;
    const int perReplica = (a.L / plan.rows) * (a.L >> 6);
    const int tpb = pick_block(perReplica);               // the last block of a replica may be ragged
    const int bpr = (perReplica + tpb - 1) / tpb;
    const unsigned grid = (unsigned)((long long)bpr * a.batch);
    SweepArgs args = a;
    args.pdl_trigger = plan.trigger;
    const bool bonds = a.bonds != nullptr;
    void (*k)(SweepArgs, int) = a.t_dev ? pick_bits_kernel<true>(plan.rows, a.colour, bonds) : pick_bits_kernel<false>(plan.rows, a.colour, bonds);
    launch_pdl(k, grid, (unsigned)tpb, s, args, bpr);
    return 1;
}

}  // namespace spin
