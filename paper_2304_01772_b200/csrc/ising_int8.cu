// ising_int8.cu — rows a2/a3: one colour's Metropolis half-sweep of the Ising model, int8 spins in the
// checkerboard-split layout [B][2][L][L/2] (Alg. 1 + checkerboard; Eq. 1-2,
// PAPER.md:99-115).  Integer only: neighbour count, class index, one Philox word per site (one call per 4
// consecutive same-colour sites), one unsigned compare against the replica's threshold table, flip.
#include "spin_internal.cuh"

#include <cmath>

namespace spin {

namespace {

// Class index used on the device: d*8 + nd, d = 1 iff own spin is -1, nd = number of -1 neighbours.
__device__ __forceinline__ bool accept_slow(uint32_t r, const uint32_t* tab, int idx) {
    return (r <= tab[idx]) && !((tab[kTabNever] >> idx) & 1u);
}

// ---- generic kernel: any even L.  One thread per Philox group (4 consecutive same-colour sites, which may
// span rows when L/2 is not a multiple of 4).  Byte loads; used for L % 32 != 0.
__global__ void ising_int8_generic_kernel(SweepArgs a) {
    pdl_wait();   // launched with programmatic stream serialisation: the previous half-sweep must have completed
    const int L = a.L, W = L >> 1;
    const long long half = (long long)L * W;          // sites of one colour
    const long long groups = (half + 3) >> 2;
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= groups * a.batch) return;
    const int b = (int)(gid / groups);
    const uint32_t g = (uint32_t)(gid % groups);
    const uint32_t* tab = a.tables + (size_t)b * kTableStride;
    int8_t* own = (int8_t*)a.lattice + ((size_t)b * 2 + a.colour) * half;
    const int8_t* oth = (const int8_t*)a.lattice + ((size_t)b * 2 + (1 - a.colour)) * half;
    uint32_t r[4];
    philox4x32_10(a.rk, g, (uint32_t)b + a.replica_offset, a.c2, a.c3, r);
#pragma unroll
    for (int e = 0; e < 4; ++e) {
        const long long n = 4ll * g + e;
        if (n >= half) break;
        const int i = (int)(n / W), k = (int)(n % W);
        const int p = (i + a.colour) & 1;
        const int iu = i == 0 ? L - 1 : i - 1, id = i == L - 1 ? 0 : i + 1;
        const int ks = p ? (k == W - 1 ? 0 : k + 1) : (k == 0 ? W - 1 : k - 1);
        const int s = own[n];
        const int nd = (oth[(size_t)iu * W + k] < 0) + (oth[(size_t)id * W + k] < 0) + (oth[(size_t)i * W + k] < 0) +
                       (oth[(size_t)i * W + ks] < 0);
        const int idx = (s < 0 ? 8 : 0) + nd;
        if (accept_slow(r[e], tab, idx)) own[n] = (int8_t)(-s);
    }
}

// ---- row-marching kernel: L % 32 == 0.
// Measured on B200 (profiles/r1_microbench.md): LOP3 / PRMT / SHF / IMAD issue at 64 lanes/SM/clk, IMAD.WIDE at 32,
// two-operand IADD3 / ISETP at 128, LDS at 32.  An IMAD.WIDE + LOP3 pair (one Philox half-round) completes in 4.1
// cycles per SM sub-partition, but every further instruction adds its own issue time, and the kernel runs at the
// same speed with 20 or 32 resident warps per SM: it is bound by the number of integer instructions per site, not by
// latency or memory.  The design therefore minimises integer instructions and pushes byte extraction onto the LSU:
//   * one thread owns a strip of 16 consecutive same-colour sites (one 128-bit word) and marches down kRows rows,
//     keeping the three other-colour rows it needs in registers, already masked to "4 if spin is -1" per byte
//     (one LOP3 per loaded word, reused as up / centre / down of three rows and for the shifted side word);
//   * per 4-site word the class byte offset 4*nd + 32*d is two IADD3 (up+centre+down, + side + own&0x20);
//   * the four offset bytes are written to a per-thread shared-memory slot (STS) and read back one byte at a
//     time (LDS.U8) straight into the address of the threshold LDS: no extraction instruction;
//   * per site: one ISETP (r <= U) and one predicated LOP3 (flip), nothing else.
// Loads of the next rows are issued before the current row is computed, through running pointers (no per-load index
// arithmetic); the loop is rolled two rows per iteration (the side-neighbour parity alternates) so that the body
// (about 540 instructions) stays resident in the instruction caches.  Launched with programmatic dependent launch:
// the next half-sweep's blocks are scheduled while this one drains.
constexpr int kRowsLong = 8;    // rows per thread when the launch fills the GPU several times over
constexpr int kRowsMid = 4;     // ... about one wave of 8-row blocks or less: more, shorter blocks
constexpr int kRowsShort = 2;   // ... and when even those leave SMs idle (latency-bound shapes)
constexpr int kMinBlocks = kIsingInt8BlocksPerSm;   // resident blocks per SM (spin_internal.cuh)
constexpr int kRowsThreads = 128;

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

// One site: threshold fetch (LDS with the class byte as address), compare, and a predicated add of the byte's flip
// pattern into the word's flip mask (a two-operand add issues at twice the rate of a logic op; the bytes are disjoint).
template <bool kHasNever, int kE>
__device__ __forceinline__ void site_step(uint32_t& fm, uint32_t o, uint32_t r, const uint32_t* stab) {
    const uint32_t U = *(const uint32_t*)((const char*)stab + o);
    if (kHasNever) {
        const bool acc = (r <= U) && !((stab[kTabNever] >> (o >> 2)) & 1u);
        if (acc) fm += 0xFEu << (8 * kE);
    } else if (kE == 0) {
        // the first site of a word defines the mask (one select, no zero-initialisation)
        asm("{\n\t.reg .pred p;\n\tsetp.ls.u32 p, %1, %2;\n\tselp.b32 %0, %3, 0, p;\n\t}"
            : "=r"(fm) : "r"(r), "r"(U), "n"(0xFEu));
    } else {
        // kept in PTX so that it stays one ISETP + one predicated IADD
        asm("{\n\t.reg .pred p;\n\tsetp.ls.u32 p, %1, %2;\n\t@p add.u32 %0, %0, %3;\n\t}"
            : "+r"(fm) : "r"(r), "r"(U), "n"(0xFEu << (8 * kE)));
    }
}

// One 4-site word.  t = byte offsets 4*nd + 32*d of its four sites; kJ = index of the word in the strip.
template <bool kHasNever, int kJ>
__device__ __forceinline__ uint32_t update_word(uint32_t own, uint32_t t, const uint32_t r[4], const uint32_t* stab,
                                                uint32_t slot) {
    slot_store_u32<kJ * kRowsThreads * 4>(slot, t);
    const uint32_t o0 = slot_load_u8<kJ * kRowsThreads * 4 + 0>(slot);
    const uint32_t o1 = slot_load_u8<kJ * kRowsThreads * 4 + 1>(slot);
    const uint32_t o2 = slot_load_u8<kJ * kRowsThreads * 4 + 2>(slot);
    const uint32_t o3 = slot_load_u8<kJ * kRowsThreads * 4 + 3>(slot);
    uint32_t fm = 0u;                      // 0xFE in the bytes that flip
    site_step<kHasNever, 0>(fm, o0, r[0], stab);
    site_step<kHasNever, 1>(fm, o1, r[1], stab);
    site_step<kHasNever, 2>(fm, o2, r[2], stab);
    site_step<kHasNever, 3>(fm, o3, r[3], stab);
    return own ^ fm;
}

// One row of one strip.  um / cm / dm: masked (4 per -1 spin) other-colour words of rows i-1, i, i+1;
// kParity = 1: the side neighbour of site k is other[i][k+1], else other[i][k-1]; `edge` is the masked 32-bit
// word holding the 17th byte (next strip's first word, or previous strip's last word).
template <bool kHasNever, int kParity>
__device__ __forceinline__ uint4 update_row(const RoundKeys& rk, uint32_t c2, uint32_t c3, uint4 own, const uint4& um,
                                            const uint4& cm, const uint4& dm, uint32_t edge, uint32_t g0, uint32_t c1,
                                            const uint32_t* stab, uint32_t slot, uint4* tout = nullptr) {
    uint32_t s0, s1, s2, s3;
    if (kParity) {
        s0 = __byte_perm(cm.x, cm.y, 0x4321);
        s1 = __byte_perm(cm.y, cm.z, 0x4321);
        s2 = __byte_perm(cm.z, cm.w, 0x4321);
        s3 = __byte_perm(cm.w, edge, 0x4321);
    } else {
        s0 = __byte_perm(edge, cm.x, 0x6543);
        s1 = __byte_perm(cm.x, cm.y, 0x6543);
        s2 = __byte_perm(cm.y, cm.z, 0x6543);
        s3 = __byte_perm(cm.z, cm.w, 0x6543);
    }
    const uint32_t kOwn = 0x20202020u;   // bit 5 of a +-1 byte is set iff the spin is -1: contributes 32*d
    const uint32_t t0 = (um.x + cm.x + dm.x) + s0 + (own.x & kOwn);
    const uint32_t t1 = (um.y + cm.y + dm.y) + s1 + (own.y & kOwn);
    const uint32_t t2 = (um.z + cm.z + dm.z) + s2 + (own.z & kOwn);
    const uint32_t t3 = (um.w + cm.w + dm.w) + s3 + (own.w & kOwn);
    if (tout) *tout = make_uint4(t0, t1, t2, t3);   // bytes 4 * nd + 32 * d (fused measurement)
    uint32_t r0[4], r1[4], r2[4], r3[4];
    philox4x32_10(rk, g0 + 0, c1, c2, c3, r0);
    philox4x32_10(rk, g0 + 1, c1, c2, c3, r1);
    philox4x32_10(rk, g0 + 2, c1, c2, c3, r2);
    philox4x32_10(rk, g0 + 3, c1, c2, c3, r3);
    uint4 res;
    res.x = update_word<kHasNever, 0>(own.x, t0, r0, stab, slot);
    res.y = update_word<kHasNever, 1>(own.y, t1, r1, stab, slot);
    res.z = update_word<kHasNever, 2>(own.z, t2, r2, stab, slot);
    res.w = update_word<kHasNever, 3>(own.w, t3, r3, stab, slot);
    return res;
}

// Loads of lattice words.  The two-launches-per-sweep kernels read the other colour through the read-only path (it is
// constant during a launch); the persistent kernel below runs many half-sweeps in one launch, so everything another
// SM may have written since this SM last read it must bypass the (non-coherent) L1: ld.global.cg.
template <bool kCoherent> __device__ __forceinline__ uint4 ld4(const uint4* p) { return kCoherent ? __ldcg(p) : __ldg(p); }
template <bool kCoherent> __device__ __forceinline__ uint32_t ld1(const uint32_t* p) { return kCoherent ? __ldcg(p) : __ldg(p); }
template <bool kCoherent> __device__ __forceinline__ uint4 ldown(const uint4* p) { return kCoherent ? __ldcg(p) : *p; }

__device__ __forceinline__ uint4 mask4(const uint4& v) {
    const uint32_t m = 0x04040404u;      // 4 per -1 spin
    return make_uint4(v.x & m, v.y & m, v.z & m, v.w & m);
}

// Sums for the fused E / M reduction (kMeasure, colour-1 launches), kept as packed byte counters so that a row costs a few
// full-rate logic / add instructions (IDP4A shares the pipe of the Philox multiplies, which is the kernel's bottleneck):
//   cS  += 4 per -1 spin of the updated strip `res`            (bit 2 of a +-1 byte)
//   cC  += the masked centre word (4 per -1 colour-0 spin: every colour-0 site is the centre word of exactly one strip)
//   cB[j] += 4 nd of the sites of word j whose NEW spin is -1   (t & res & 0x1C: t = 4 nd + 32 d, res = 0xFF / 0x01)
// A byte grows by at most 16 per row (cB) or 16 per row over the four words (cS, cC): no overflow for <= 8 rows.
// With nS, nC, nB the byte sums: number of -1 colour-1 spins = nS / 4, of -1 colour-0 spins = nC / 4,
// sum over colour-1 sites of 4 nd = 4 nC (every colour-0 site is a neighbour of four colour-1 sites), so
//   sum s = N/2 - nS/2,   sum s * 4 nd = 4 nC - 2 nB,   E_int = -(4 sum s - (sum s * 4 nd) / 2),   M = N - (nS + nC) / 2.
struct MeasureCounters {
    uint32_t cS, cC;
    uint4 cB;
};
__device__ __forceinline__ void measure_row(const uint4& res, const uint4& t, const uint4& cm, MeasureCounters& mc) {
    const uint32_t m = 0x04040404u, k = 0x1C1C1C1Cu;
    mc.cS += ((res.x & m) + (res.y & m)) + ((res.z & m) + (res.w & m));
    mc.cC += (cm.x + cm.y) + (cm.z + cm.w);
    mc.cB.x += t.x & res.x & k;
    mc.cB.y += t.y & res.y & k;
    mc.cB.z += t.z & res.z & k;
    mc.cB.w += t.w & res.w & k;
}

template <int kColour, bool kHasNever, int kRows, bool kPersist = false, bool kMeasure = false>
__device__ __forceinline__ void march_rows(const SweepArgs& a, uint32_t c2, uint32_t c3, const uint32_t* stab, uint32_t slot,
                                           int b, int rb, int x, MeasureCounters* mc = nullptr) {
    const int L = a.L, W = L >> 1, W16 = W >> 4, W4 = W >> 2;
    const size_t half = (size_t)L * W;
    const int i0 = rb * kRows;
    int8_t* ownBase = (int8_t*)a.lattice + ((size_t)b * 2 + kColour) * half;
    const int8_t* oth = (const int8_t*)a.lattice + ((size_t)b * 2 + (1 - kColour)) * half;
    const uint4* oth4 = (const uint4*)oth;
    const uint32_t* oth1 = (const uint32_t*)oth;
    // word index of the edge word inside a row: next strip's first word / previous strip's last word (periodic)
    const uint32_t eNext = (x == W16 - 1) ? 0u : 4u * x + 4u;
    const uint32_t ePrev = (x == 0) ? (uint32_t)W4 - 1u : 4u * x - 1u;
    const int iu = i0 == 0 ? L - 1 : i0 - 1;
    const int iLast = (i0 + kRows == L) ? 0 : i0 + kRows;       // the only prefetched row that can wrap
    // Running pointers, advanced by one row stride per row: no per-load index arithmetic inside the unrolled rows.
    const size_t rowStride = (size_t)W16;                        // in uint4
    const size_t edgeStride2 = 2 * (size_t)W4;                   // two rows, in uint32
    const uint4* pOth = oth4 + (size_t)(i0 + 2) * W16 + x;       // next other-colour row to prefetch
    const uint4* pOthLast = oth4 + (size_t)iLast * W16 + x;
    uint4* pOwn = (uint4*)ownBase + (size_t)i0 * W16 + x;
    // even rows of the block have parity kColour, odd rows 1 - kColour (i0 is even)
    const uint32_t* pEdgeEven = oth1 + (size_t)i0 * W4 + (kColour ? eNext : ePrev);
    const uint32_t* pEdgeOdd = oth1 + (size_t)(i0 + 1) * W4 + (kColour ? ePrev : eNext);
    uint4 wU = mask4(ld4<kPersist>(oth4 + (size_t)iu * W16 + x));     // masked other-colour rows i-1, i, i+1
    uint4 wC = mask4(ld4<kPersist>(pOth - 2 * rowStride));
    uint4 wD = mask4(ld4<kPersist>(pOth - rowStride));
    uint4 own = ldown<kPersist>(pOwn);
    uint32_t edge = ld1<kPersist>(pEdgeEven) & 0x04040404u;
    uint32_t g0 = (uint32_t)i0 * (uint32_t)W4 + 4u * (uint32_t)x;
    const uint32_t c1 = (uint32_t)b + a.replica_offset;
    if (!kPersist && !kMeasure) __syncthreads();   // the block's threshold table (filled by the caller) is first read below: the loads
                                      // above are already in flight while the block waits for it
    // Two rows per iteration (the side-neighbour parity alternates); the four iterations of an 8-row thread are
    // unrolled so that the register window rotates by renaming instead of moves (measured: +2.5 % over the rolled loop).
#pragma unroll 4
    for (int rr = 0; rr < kRows; rr += 2) {
        const bool more = rr + 2 < kRows;
        // inputs of the odd row i+1: other-colour row i+2 (the only one that can wrap), own row i+1, its edge word
        const uint4 n1 = ld4<kPersist>(more ? pOth : pOthLast);
        const uint4 own1 = ldown<kPersist>(pOwn + rowStride);
        const uint32_t edge1 = ld1<kPersist>(pEdgeOdd);
        // inputs of the next even row i+2: other-colour row i+3, own row i+2, its edge word
        uint4 n2 = n1, own2 = own1;
        uint32_t edge2 = edge1;
        if (more) {
            n2 = ld4<kPersist>(pOth + rowStride);
            own2 = ldown<kPersist>(pOwn + 2 * rowStride);
            edge2 = ld1<kPersist>(pEdgeEven + edgeStride2);
        }
        uint4 tw;
        uint4 res = update_row<kHasNever, kColour>(a.rk, c2, c3, own, wU, wC, wD, edge, g0, c1, stab, slot, kMeasure ? &tw : nullptr);
        *pOwn = res;
        if (kMeasure) measure_row(res, tw, wC, *mc);
        const uint4 n1m = mask4(n1);
        res = update_row<kHasNever, 1 - kColour>(a.rk, c2, c3, own1, wC, wD, n1m, edge1 & 0x04040404u,
                                                 g0 + (uint32_t)W4, c1, stab, slot, kMeasure ? &tw : nullptr);
        *(pOwn + rowStride) = res;
        if (kMeasure) measure_row(res, tw, wD, *mc);
        wU = wD;
        wC = n1m;
        wD = mask4(n2);
        own = own2;
        edge = edge2 & 0x04040404u;
        pOth += 2 * rowStride;
        pOwn += 2 * rowStride;
        pEdgeEven += edgeStride2;
        pEdgeOdd += edgeStride2;
        g0 += 2u * (uint32_t)W4;
    }
}

// One block covers blockDim.x consecutive strips-times-row-blocks of one replica; bpr = blocks per replica.
template <int kColour, int kRows, bool kDevT>
__global__ void __launch_bounds__(kRowsThreads, kMinBlocks) ising_int8_rows_kernel(SweepArgs a, int bpr) {
    __shared__ uint32_t stab[kTableStride];
    __shared__ uint32_t sidx[4 * kRowsThreads];   // per-thread slot: word j of thread t at sidx[j * 128 + t]
    if (a.pdl_trigger == kPdlAtStart) pdl_launch_dependents();
    const int b = blockIdx.x / bpr;
    const int blk = blockIdx.x - b * bpr;
    pdl_wait();
    uint32_t c2, c3;
    sweep_counter_words<kDevT>(a, c2, c3);
    const uint32_t never = a.tables[(size_t)b * kTableStride + kTabNever];   // block-uniform
    for (int k = threadIdx.x; k < kTableStride; k += blockDim.x) stab[k] = a.tables[(size_t)b * kTableStride + k];
    const int W16 = a.L >> 5;
    const int u = blk * blockDim.x + threadIdx.x;
    // ragged last block of a replica: the spare threads have done their share of the table fill and leave (an
    // exited thread counts as arrived at the barrier inside march_rows)
    if (u >= (a.L / kRows) * W16) return;
    const int rb = u / W16, x = u - rb * W16;
    const uint32_t slot = (uint32_t)__cvta_generic_to_shared(&sidx[threadIdx.x]);
    if (never) march_rows<kColour, true, kRows>(a, c2, c3, stab, slot, b, rb, x);
    else march_rows<kColour, false, kRows>(a, c2, c3, stab, slot, b, rb, x);
}

// Colour-1 half-sweep with the E / M reduction fused in (spin_sweep_measure on the streaming path): the same marching
// code; every thread also sums measure_row() over its rows, the block adds its three sums to a.measure_acc[b][0..2]
// (nS, nC, nB), and launch_ising_measure_finalize turns them into E and M once the launch is complete.
template <int kRows>
__global__ void __launch_bounds__(kRowsThreads, kMinBlocks) ising_int8_rows_measure_kernel(SweepArgs a, int bpr) {
    __shared__ uint32_t stab[kTableStride];
    __shared__ uint32_t sidx[4 * kRowsThreads];
    __shared__ int ssum[3 * (kRowsThreads / 32)];
    if (a.pdl_trigger == kPdlAtStart) pdl_launch_dependents();
    const int b = blockIdx.x / bpr;
    const int blk = blockIdx.x - b * bpr;
    pdl_wait();
    const uint32_t never = a.tables[(size_t)b * kTableStride + kTabNever];   // block-uniform
    for (int k = threadIdx.x; k < kTableStride; k += blockDim.x) stab[k] = a.tables[(size_t)b * kTableStride + k];
    const int W16 = a.L >> 5;
    const int u = blk * blockDim.x + threadIdx.x;
    MeasureCounters mc = {0u, 0u, make_uint4(0u, 0u, 0u, 0u)};
    __syncthreads();                       // the table; here and not inside march_rows: the spare threads of a ragged last
                                           // block stay for the block sum, and a barrier may not sit in divergent code
    if (u < (a.L / kRows) * W16) {
        const int rb = u / W16, x = u - rb * W16;
        const uint32_t slot = (uint32_t)__cvta_generic_to_shared(&sidx[threadIdx.x]);
        if (never) march_rows<1, true, kRows, false, true>(a, a.c2, a.c3, stab, slot, b, rb, x, &mc);
        else march_rows<1, false, kRows, false, true>(a, a.c2, a.c3, stab, slot, b, rb, x, &mc);
    }
    // byte sums nS, nC, nB of the thread (unsigned bytes, one IDP4A per counter word)
    int msum[3];
    msum[0] = __dp4a(mc.cS, 0x01010101u, 0u);
    msum[1] = __dp4a(mc.cC, 0x01010101u, 0u);
    msum[2] = __dp4a(mc.cB.x, 0x01010101u, __dp4a(mc.cB.y, 0x01010101u, __dp4a(mc.cB.z, 0x01010101u, __dp4a(mc.cB.w, 0x01010101u, 0u))));
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        msum[0] += __shfl_xor_sync(0xFFFFFFFFu, msum[0], o);
        msum[1] += __shfl_xor_sync(0xFFFFFFFFu, msum[1], o);
        msum[2] += __shfl_xor_sync(0xFFFFFFFFu, msum[2], o);
    }
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    if (lane == 0) { ssum[3 * w] = msum[0]; ssum[3 * w + 1] = msum[1]; ssum[3 * w + 2] = msum[2]; }
    __syncthreads();
    if (threadIdx.x < 3) {
        long long t = 0;
        for (int k = 0; k < (int)((blockDim.x + 31) >> 5); ++k) t += ssum[3 * k + threadIdx.x];
        atomicAdd((unsigned long long*)a.measure_acc + 3 * (size_t)b + threadIdx.x, (unsigned long long)t);
    }
}

// r[0..2] = the byte sums (nS, nC, nB) of one replica (measure_row) -> E_int, M; moments as accumulate_moments_kernel
// (observe.cu); the sums are cleared.
__device__ __forceinline__ void measure_finalize_replica(long long* r, long long sites, long long* E_out, long long* M_out,
                                                         long long* m) {
    const long long nS = r[0], nC = r[1], nB = r[2];
    r[0] = 0; r[1] = 0; r[2] = 0;
    const long long sum1 = sites / 2 - nS / 2;                  // sum of the colour-1 spins
    const long long e = -(4 * sum1 - (4 * nC - 2 * nB) / 2);
    const long long mag = sites - (nS + nC) / 2;
    if (E_out) *E_out = e;
    if (M_out) *M_out = mag;
    if (m) {
        const unsigned long long ae = e < 0 ? (unsigned long long)(-e) : (unsigned long long)e;
        const unsigned long long lo = ae * ae, hi = __umul64hi(ae, ae);
        const unsigned long long old_lo = (unsigned long long)m[2];
        const unsigned long long new_lo = old_lo + lo;
        m[0] += 1;
        m[1] += e;
        m[2] = (long long)new_lo;
        m[3] = (long long)((unsigned long long)m[3] + hi + (new_lo < old_lo ? 1ull : 0ull));
        m[4] += mag;
        m[5] += mag < 0 ? -mag : mag;
        m[6] += mag * mag;
        m[7] += e * mag;
    }
}

// After the last sweep of a measured call (the sweeps before it are finalised by the next sweep's colour-0 launch).
__global__ void ising_measure_finalize_kernel(long long* acc, int batch, long long sites, long long* E_out, long long* M_out,
                                              long long* moments) {
    pdl_wait();
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= batch) return;
    measure_finalize_replica(acc + 3 * (size_t)b, sites, E_out ? E_out + b : nullptr, M_out ? M_out + b : nullptr,
                             moments ? moments + 8 * (size_t)b : nullptr);
}

// Colour-0 half-sweep of a measured run: ising_int8_rows_kernel<0, kRows> plus the finalisation of the previous sweep's sums
// by the first thread of every replica's first block (its colour-1 launch is complete once pdl_wait returns, and the next
// colour-1 launch, which adds to the same sums, starts after this one).
template <int kRows>
__global__ void __launch_bounds__(kRowsThreads, kMinBlocks) ising_int8_rows_fin_kernel(SweepArgs a, int bpr) {
    __shared__ uint32_t stab[kTableStride];
    __shared__ uint32_t sidx[4 * kRowsThreads];
    if (a.pdl_trigger == kPdlAtStart) pdl_launch_dependents();
    const int b = blockIdx.x / bpr;
    const int blk = blockIdx.x - b * bpr;
    pdl_wait();
    if (blk == 0 && threadIdx.x == 0 && a.fin_pending)
        measure_finalize_replica(a.measure_acc + 3 * (size_t)b, (long long)a.L * a.L, a.fin_E ? a.fin_E + b : nullptr,
                                 a.fin_M ? a.fin_M + b : nullptr, a.fin_mom ? a.fin_mom + 8 * (size_t)b : nullptr);
    const uint32_t never = a.tables[(size_t)b * kTableStride + kTabNever];   // block-uniform
    for (int k = threadIdx.x; k < kTableStride; k += blockDim.x) stab[k] = a.tables[(size_t)b * kTableStride + k];
    const int W16 = a.L >> 5;
    const int u = blk * blockDim.x + threadIdx.x;
    if (u >= (a.L / kRows) * W16) return;
    const int rb = u / W16, x = u - rb * W16;
    const uint32_t slot = (uint32_t)__cvta_generic_to_shared(&sidx[threadIdx.x]);
    if (never) march_rows<0, true, kRows>(a, a.c2, a.c3, stab, slot, b, rb, x);
    else march_rows<0, false, kRows>(a, a.c2, a.c3, stab, slot, b, rb, x);
}

// ---- persistent kernel for launch-bound shapes (lattices too big for one CTA's shared memory, too small for a
// half-sweep to hide a kernel launch: the paper's own Table III sizes).  All sweeps of a call run in
// ONE cooperative launch: the grid is what fits on the GPU at once, every block loops over its share of the
// (replica, row block, strip) work items with the same march_rows code, and the half-sweeps are separated by a grid-wide
// barrier (one atomic arrive + an acquire spin per block, ~1 us) instead of a kernel boundary (~2.7 us with PDL).  The
// lattice stays in L2.  Work items are assigned statically (item v -> block v % gridDim), so a word is always written
// by the same block.  Only tables without never-classes take this path (the host falls back to streaming otherwise).
__device__ __forceinline__ void grid_barrier(unsigned int* counter, unsigned int& target) {
    __syncthreads();
    if (threadIdx.x == 0) {
        target += gridDim.x;
        __threadfence();                                   // this block's lattice writes are visible before it arrives
        atomicAdd(counter, 1u);
        unsigned int seen;
        do {
            asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(counter) : "memory");
        } while ((int)(seen - target) < 0);
    }
    __syncthreads();
}

template <int kRows>
__global__ void __launch_bounds__(kRowsThreads, kMinBlocks) ising_int8_persistent_kernel(SweepArgs a, int bpr, int items,
                                                                                         unsigned long long t0,
                                                                                         long long n_sweeps,
                                                                                         unsigned int* counter) {
    __shared__ uint32_t stab[kTableStride];
    __shared__ uint32_t sidx[4 * kRowsThreads];
    const uint32_t slot = (uint32_t)__cvta_generic_to_shared(&sidx[threadIdx.x]);
    const int W16 = a.L >> 5;
    const int perReplica = (a.L / kRows) * W16;
    unsigned int target = 0u;
    int loaded = -1;                                        // replica whose table is in stab
    for (long long s = 0; s < n_sweeps; ++s) {
        const unsigned long long t = t0 + (unsigned long long)s;
        a.c2 = (uint32_t)(t & 0xFFFFFFFFull);
#pragma unroll 1
        for (int colour = 0; colour < 2; ++colour) {
            a.c3 = (uint32_t)((t >> 32) & 0xFFFFFFull) | ((uint32_t)colour << 24) | (kDomainIsing << 28);
            for (int v = blockIdx.x; v < items; v += gridDim.x) {
                const int b = v / bpr, blk = v - b * bpr;
                if (b != loaded) {                          // block-uniform
                    __syncthreads();
                    for (int k = threadIdx.x; k < kTableStride; k += blockDim.x) stab[k] = a.tables[(size_t)b * kTableStride + k];
                    __syncthreads();
                    loaded = b;
                }
                const int u = blk * blockDim.x + threadIdx.x;
                if (u < perReplica) {
                    const int rb = u / W16, x = u - rb * W16;
                    if (colour == 0) march_rows<0, false, kRows, true>(a, a.c2, a.c3, stab, slot, b, rb, x);
                    else march_rows<1, false, kRows, true>(a, a.c2, a.c3, stab, slot, b, rb, x);
                }
            }
            grid_barrier(counter, target);
        }
    }
}

// ---- temporally blocked tile kernel (launch-bound shapes, L % 8 == 0).  The counter-based random numbers make every
// update a pure function of (seed, replica, site, sweep, colour) and of the neighbouring spins, so a CTA can advance a
// TILE of one replica by several sweeps on its own if it also carries a halo: each half-sweep the outermost valid ring
// of the halo becomes stale (its outside neighbours are not there), so 2 * sweeps halo rows / columns keep the interior
// exact.  The halo sites are updated redundantly by the neighbouring tiles with identical results.  One launch =
// `sweeps` full sweeps for every tile: the launch gap (~2.7 us per half-sweep on the streaming path) is paid once per
// `sweeps` sweeps, and a one-replica lattice is spread over all SMs instead of one.
// Region in shared memory: rows r <-> global row (i0 - HR + r) mod L, words wx <-> global k = (k0 - HK + 4 wx) mod (L/2),
// both colours.  One thread per 4-site word (= one Philox group) per half-sweep; region-edge words use clamped
// neighbours (their results are stale by construction and never reach the interior).
template <bool kHasNever>
__device__ __forceinline__ void tiled_half_sweep(const TiledArgs& a, int colour, uint32_t c2, uint32_t c3, uint32_t* own1,
                                                 const uint32_t* oth1, int SR, int SWX, int iBase, int kBase,
                                                 const uint32_t* stab, uint32_t slot, uint32_t c1, int rLo, int rHi) {
    const int L = a.L, W = L >> 1, W4 = W >> 2;
    const uint32_t m = 0x04040404u;
    for (int task = rLo * SWX + threadIdx.x; task < rHi * SWX; task += blockDim.x) {   // rows [rLo, rHi): see the kernel
        const int r = task / SWX, wx = task - r * SWX;
        int gi = iBase + r;                                    // iBase in [0, L): at most two wraps for regions <= 2 L
        gi = gi >= L ? gi - L : gi;
        gi = gi >= L ? gi - L : gi;
        int gk = kBase + 4 * wx;
        gk = gk >= W ? gk - W : gk;
        gk = gk >= W ? gk - W : gk;
        const bool par = ((gi + colour) & 1) != 0;             // side neighbour of site k: k+1 if par else k-1
        const int ru = r == 0 ? 0 : r - 1, rd = r == SR - 1 ? r : r + 1;
        const int xs = par ? (wx == SWX - 1 ? wx : wx + 1) : (wx == 0 ? 0 : wx - 1);
        const uint32_t um = oth1[ru * SWX + wx] & m, cm = oth1[task] & m, dm = oth1[rd * SWX + wx] & m;
        const uint32_t nb = oth1[r * SWX + xs] & m;
        const uint32_t sd = __byte_perm(par ? cm : nb, par ? nb : cm, par ? 0x4321u : 0x6543u);
        const uint32_t own = own1[task];
        const uint32_t n4 = um + cm + dm + sd;                  // 4 x number of -1 neighbours per byte
        uint32_t rw[4];
        philox4x32_10(a.rk, (uint32_t)gi * (uint32_t)W4 + (uint32_t)(gk >> 2), c1, c2, c3, rw);
        own1[task] = update_word<kHasNever, 0>(own, n4 + (own & 0x20202020u), rw, stab, slot);
    }
}

constexpr int kTiledThreads = 1024;

// kOneWord: the region has at most blockDim.x words per colour, so every thread owns ONE word for the whole launch and
// its coordinates, neighbour offsets and Philox group are computed once; a half-sweep is then one latency chain per
// thread between two barriers (these shapes are latency-bound: the fewer dependent rounds per half-sweep the better).
// Otherwise the words are dealt out round-robin every half-sweep (tiled_half_sweep).
template <bool kOneWord>
__global__ void __launch_bounds__(kTiledThreads) ising_int8_tiled_kernel(TiledArgs a) {
    extern __shared__ __align__(16) uint32_t tsm[];
    __shared__ uint32_t stab[kTableStride];
    __shared__ uint32_t sidx[kTiledThreads];
    const int L = a.L, W = L >> 1;
    const int SR = a.TR + 2 * a.HR, SWX = (a.TK + 2 * a.HK) >> 2;
    const int perReplica = a.tilesR * a.tilesK;
    const int b = blockIdx.x / perReplica, tile = blockIdx.x - b * perReplica;
    const int tr = tile / a.tilesK, tk = tile - tr * a.tilesK;
    const int i0 = tr * a.TR, k0 = tk * a.TK;
    int iBase = (i0 - a.HR) % L, kBase = (k0 - a.HK) % W;
    iBase = iBase < 0 ? iBase + L : iBase;
    kBase = kBase < 0 ? kBase + W : kBase;
    uint32_t* reg0 = tsm;                                      // colour 0: [SR][SWX] words
    uint32_t* reg1 = tsm + SR * SWX;
    const size_t half = (size_t)L * W;
    const uint32_t* g0 = (const uint32_t*)((const int8_t*)a.src + (size_t)b * 2 * half);
    const uint32_t* g1 = (const uint32_t*)((const int8_t*)a.src + (size_t)b * 2 * half + half);
    const int W4 = W >> 2;
    pdl_wait();
    for (int k = threadIdx.x; k < kTableStride; k += blockDim.x) stab[k] = a.tables[(size_t)b * kTableStride + k];
    for (int task = threadIdx.x; task < SR * SWX; task += blockDim.x) {
        const int r = task / SWX, wx = task - r * SWX;
        int gi = iBase + r;
        gi = gi >= L ? gi - L : gi;
        gi = gi >= L ? gi - L : gi;
        int gk = kBase + 4 * wx;
        gk = gk >= W ? gk - W : gk;
        gk = gk >= W ? gk - W : gk;
        const size_t gw = (size_t)gi * W4 + (gk >> 2);
        reg0[task] = __ldcg(g0 + gw);
        reg1[task] = __ldcg(g1 + gw);
    }
    __syncthreads();
    const uint32_t slot = (uint32_t)__cvta_generic_to_shared(&sidx[threadIdx.x]);
    const uint32_t c1 = (uint32_t)b + a.replica_offset;
    const bool never = stab[kTabNever] != 0u;
    // the thread's own word (kOneWord)
    const int task = threadIdx.x;
    const bool mine = task < SR * SWX;
    int oU = 0, oD = 0, oNext = 0, oPrev = 0, dr = 0;          // dr: distance of the thread's row from the tile's interior rows
    uint32_t group = 0u, par0 = 0u;
    if (kOneWord && mine) {
        const int r = task / SWX, wx = task - r * SWX;
        int gi = iBase + r;
        gi = gi >= L ? gi - L : gi;
        gi = gi >= L ? gi - L : gi;
        int gk = kBase + 4 * wx;
        gk = gk >= W ? gk - W : gk;
        gk = gk >= W ? gk - W : gk;
        oU = (r == 0 ? 0 : r - 1) * SWX + wx;
        oD = (r == SR - 1 ? r : r + 1) * SWX + wx;
        dr = r < a.HR ? a.HR - r : (r >= a.HR + a.TR ? r - (a.HR + a.TR - 1) : 0);
        oNext = r * SWX + (wx == SWX - 1 ? wx : wx + 1);
        oPrev = r * SWX + (wx == 0 ? 0 : wx - 1);
        group = (uint32_t)gi * (uint32_t)W4 + (uint32_t)(gk >> 2);
        par0 = (uint32_t)gi & 1u;
    }
    for (int s = 0; s < a.sweeps; ++s) {
        const unsigned long long t = a.t0 + (unsigned long long)s;
        const uint32_t c2 = (uint32_t)(t & 0xFFFFFFFFull);
        const uint32_t c3lo = (uint32_t)((t >> 32) & 0xFFFFFFull) | (kDomainIsing << 28);
        for (int colour = 0; colour < 2; ++colour) {
            const uint32_t c3 = c3lo | ((uint32_t)colour << 24);
            uint32_t* own1 = colour ? reg1 : reg0;
            const uint32_t* oth1 = colour ? reg0 : reg1;
            // a site can still reach the interior by the end of the launch only if it is within `reach` sites of it: rows
            // farther out are not updated any more (their values are stale by then anyway)
            const int reach = 2 * (a.sweeps - s) - 1 - colour;
            if (kOneWord) {
                if (mine && dr <= reach) {
                    const uint32_t m = 0x04040404u;
                    const bool par = ((par0 + (uint32_t)colour) & 1u) != 0u;   // side neighbour of site k: k+1 if par else k-1
                    const uint32_t um = oth1[oU] & m, cm = oth1[task] & m, dm = oth1[oD] & m;
                    const uint32_t nb = oth1[par ? oNext : oPrev] & m;
                    const uint32_t sd = __byte_perm(par ? cm : nb, par ? nb : cm, par ? 0x4321u : 0x6543u);
                    const uint32_t own = own1[task];
                    uint32_t rw[4];
                    philox4x32_10(a.rk, group, c1, c2, c3, rw);
                    const uint32_t tcls = um + cm + dm + sd + (own & 0x20202020u);
                    own1[task] = never ? update_word<true, 0>(own, tcls, rw, stab, slot) : update_word<false, 0>(own, tcls, rw, stab, slot);
                }
            } else if (never) tiled_half_sweep<true>(a, colour, c2, c3, own1, oth1, SR, SWX, iBase, kBase, stab, slot, c1, max(0, a.HR - reach), min(SR, a.HR + a.TR + reach));
            else tiled_half_sweep<false>(a, colour, c2, c3, own1, oth1, SR, SWX, iBase, kBase, stab, slot, c1, max(0, a.HR - reach), min(SR, a.HR + a.TR + reach));
            __syncthreads();
        }
    }
    // write back the interior (clipped at the lattice edge for the last tile row / column)
    const int rows = min(a.TR, L - i0), wcols = min(a.TK, W - k0) >> 2;
    uint32_t* o0 = (uint32_t*)((int8_t*)a.dst + (size_t)b * 2 * half);
    uint32_t* o1 = (uint32_t*)((int8_t*)a.dst + (size_t)b * 2 * half + half);
    for (int task2 = threadIdx.x; task2 < rows * wcols; task2 += blockDim.x) {
        const int rr = task2 / wcols, ww = task2 - rr * wcols;
        const int sidxw = (a.HR + rr) * SWX + (a.HK >> 2) + ww;
        const size_t gw = (size_t)(i0 + rr) * W4 + ((k0 >> 2) + ww);
        o0[gw] = reg0[sidxw];
        o1[gw] = reg1[sidxw];
    }
}

// ---- shared-memory-resident kernel: L % 32 == 0 and the replica (L^2 bytes) fits one CTA's shared memory.
// One CTA per replica runs every sweep of the call: both colours stay in shared memory, the half-sweeps are
// separated by __syncthreads() (a colour only reads the other colour), the Philox counter words of sweep t are
// formed in the kernel, and after each sweep the exact E_int and M of the replica are reduced from shared memory
// (same byte-SIMD bond count as observe.cu), written to the traces and accumulated into the moments by thread 0.
// Per row strip the work is the same update_row as the HBM kernel.
constexpr int kResThreads = 256;
constexpr size_t kResMaxLatticeBytes = 196608;   // 3 CTAs of L = 256 per SM; one CTA up to L = 416


// Rows of one parity at a time: the side of the horizontal neighbour depends on (row + colour) & 1, and a warp spans
// several rows when L/32 < 32, so mixing parities in one pass would make every warp execute both variants.
// kMeasure: also accumulate, from the updated strip and the neighbour sums already in registers, sS = sum of the new
// spins and sSN = sum of (new spin) x (4 x number of -1 neighbours) (IDP4A on the +-1 bytes): after the colour-1 pass
// every bond has been seen from its colour-1 end with final values, so E_int = -(4 sS1 - sSN1 / 2), M = sS0 + sS1.
// Three block sums with one pair of barriers (valid in thread 0 only).
__device__ __forceinline__ void block_sum3(int& a, int& b, int& c, int* scratch) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        a += __shfl_xor_sync(0xFFFFFFFFu, a, o);
        b += __shfl_xor_sync(0xFFFFFFFFu, b, o);
        c += __shfl_xor_sync(0xFFFFFFFFu, c, o);
    }
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    __syncthreads();                       // scratch may still be read from the previous sweep
    if (lane == 0) { scratch[3 * w] = a; scratch[3 * w + 1] = b; scratch[3 * w + 2] = c; }
    __syncthreads();
    if (threadIdx.x == 0) {
        const int nw = (blockDim.x + 31) >> 5;
        a = b = c = 0;
        for (int k = 0; k < nw; ++k) { a += scratch[3 * k]; b += scratch[3 * k + 1]; c += scratch[3 * k + 2]; }
    }
}

template <bool kHasNever, int kParity, bool kMeasure>
__device__ __forceinline__ void resident_rows(const ResidentArgs& a, int colour, uint32_t c2, uint32_t c3, uint8_t* lat,
                                              const uint32_t* stab, uint32_t slot, uint32_t c1, int& sS, int& sSN) {
    const int L = a.L, W = L >> 1, W16 = W >> 4, W4 = W >> 2;
    uint4* own4 = (uint4*)(lat + (size_t)colour * L * W);
    const uint4* oth4 = (const uint4*)(lat + (size_t)(1 - colour) * L * W);
    const uint32_t* oth1 = (const uint32_t*)oth4;
    const int rowPar = (kParity + colour) & 1;                  // rows i with (i + colour) & 1 == kParity
    const int units = (L >> 1) * W16;
    for (int v = threadIdx.x; v < units; v += blockDim.x) {
        const int ih = v / W16, x = v - ih * W16;
        const int i = 2 * ih + rowPar, u = i * W16 + x;
        const int iu = i == 0 ? L - 1 : i - 1, id = i == L - 1 ? 0 : i + 1;
        const uint4 um = mask4(oth4[iu * W16 + x]), cm = mask4(oth4[u]), dm = mask4(oth4[id * W16 + x]);
        const uint4 own = own4[u];
        const uint32_t g0 = (uint32_t)u * 4u;                   // (i * W + 16 x) >> 2
        const int ew = kParity ? ((x == W16 - 1) ? 0 : 4 * x + 4) : ((x == 0) ? W4 - 1 : 4 * x - 1);
        const uint32_t edge = oth1[i * W4 + ew] & 0x04040404u;
        const uint4 res = update_row<kHasNever, kParity>(a.rk, c2, c3, own, um, cm, dm, edge, g0, c1, stab, slot);
        own4[u] = res;
        if (kMeasure) {
            const int ones = 0x01010101;
            sS += __dp4a((int)res.x, ones, __dp4a((int)res.y, ones, __dp4a((int)res.z, ones, __dp4a((int)res.w, ones, 0))));
            if (colour == 1) {
                uint32_t s0, s1, s2, s3;
                if (kParity) {
                    s0 = __byte_perm(cm.x, cm.y, 0x4321); s1 = __byte_perm(cm.y, cm.z, 0x4321);
                    s2 = __byte_perm(cm.z, cm.w, 0x4321); s3 = __byte_perm(cm.w, edge, 0x4321);
                } else {
                    s0 = __byte_perm(edge, cm.x, 0x6543); s1 = __byte_perm(cm.x, cm.y, 0x6543);
                    s2 = __byte_perm(cm.y, cm.z, 0x6543); s3 = __byte_perm(cm.z, cm.w, 0x6543);
                }
                // bytes 4 * nd <= 16: dp4a with the bytes of the new spins as signed, the counts as unsigned
                int t = 0;
                asm("dp4a.s32.u32 %0, %1, %2, %0;" : "+r"(t) : "r"(res.x), "r"(um.x + cm.x + dm.x + s0));
                asm("dp4a.s32.u32 %0, %1, %2, %0;" : "+r"(t) : "r"(res.y), "r"(um.y + cm.y + dm.y + s1));
                asm("dp4a.s32.u32 %0, %1, %2, %0;" : "+r"(t) : "r"(res.z), "r"(um.z + cm.z + dm.z + s2));
                asm("dp4a.s32.u32 %0, %1, %2, %0;" : "+r"(t) : "r"(res.w), "r"(um.w + cm.w + dm.w + s3));
                sSN += t;
            }
        }
    }
}

// Tiny lattices (L <= 64): one thread per 4-site word (= one Philox group) instead of per 16-site strip, so that a
// half-sweep of a 32 x 32 replica is one short pass of 128 threads rather than two passes of 16 busy lanes.  The row
// parity (which side the horizontal neighbour is on) is handled with selects on the PRMT operands: no divergence.
template <bool kHasNever, bool kMeasure>
__device__ __forceinline__ void resident_words(const ResidentArgs& a, int colour, uint32_t c2, uint32_t c3, uint8_t* lat,
                                               const uint32_t* stab, uint32_t slot, uint32_t c1, int& sS, int& sSN) {
    const int L = a.L, W = L >> 1, W4 = W >> 2;
    uint32_t* own1 = (uint32_t*)(lat + (size_t)colour * L * W);
    const uint32_t* oth1 = (const uint32_t*)(lat + (size_t)(1 - colour) * L * W);
    const int words = L * W4;
    const uint32_t m = 0x04040404u;
    for (int w = threadIdx.x; w < words; w += blockDim.x) {
        const int i = w / W4, x = w - i * W4;
        const int iu = i == 0 ? L - 1 : i - 1, id = i == L - 1 ? 0 : i + 1;
        const bool par = ((i + colour) & 1) != 0;              // side neighbour of site k: k+1 if par else k-1
        const uint32_t um = oth1[iu * W4 + x] & m, cm = oth1[w] & m, dm = oth1[id * W4 + x] & m;
        const int xs = par ? (x == W4 - 1 ? 0 : x + 1) : (x == 0 ? W4 - 1 : x - 1);
        const uint32_t nb = oth1[i * W4 + xs] & m;
        const uint32_t sd = __byte_perm(par ? cm : nb, par ? nb : cm, par ? 0x4321u : 0x6543u);
        const uint32_t own = own1[w];
        const uint32_t n4 = um + cm + dm + sd;                  // 4 x number of -1 neighbours per byte
        uint32_t r[4];
        philox4x32_10(a.rk, (uint32_t)w, c1, c2, c3, r);       // word index = Philox group (n >> 2)
        const uint32_t res = update_word<kHasNever, 0>(own, n4 + (own & 0x20202020u), r, stab, slot);
        own1[w] = res;
        if (kMeasure) {
            sS = __dp4a((int)res, 0x01010101, sS);
            if (colour == 1) asm("dp4a.s32.u32 %0, %1, %2, %0;" : "+r"(sSN) : "r"(res), "r"(n4));
        }
    }
}

template <bool kHasNever, bool kMeasure>
__device__ __forceinline__ void resident_half_sweep(const ResidentArgs& a, int colour, uint32_t c2, uint32_t c3,
                                                    uint8_t* lat, const uint32_t* stab, uint32_t slot, uint32_t c1,
                                                    int& sS, int& sSN) {
    if (a.L <= 64) {      // block-uniform
        resident_words<kHasNever, kMeasure>(a, colour, c2, c3, lat, stab, slot, c1, sS, sSN);
        return;
    }
    resident_rows<kHasNever, 0, kMeasure>(a, colour, c2, c3, lat, stab, slot, c1, sS, sSN);
    resident_rows<kHasNever, 1, kMeasure>(a, colour, c2, c3, lat, stab, slot, c1, sS, sSN);
}

__global__ void __launch_bounds__(kResThreads) ising_int8_resident_kernel(ResidentArgs a) {
    extern __shared__ __align__(16) uint8_t smem[];
    const int L = a.L;
    const size_t latBytes = (size_t)L * L;
    uint8_t* lat = smem;
    uint32_t* stab = (uint32_t*)(smem + latBytes);
    uint32_t* sidx = stab + kTableStride;                       // per-thread slots, word j of thread t at [j * 256 + t]
    int* scratch = (int*)(sidx + 4 * kResThreads);
    const int b = blockIdx.x;
    uint4* g4 = (uint4*)((uint8_t*)a.lattice + (size_t)b * latBytes);
    for (int k = threadIdx.x; k < (int)(latBytes >> 4); k += blockDim.x) ((uint4*)lat)[k] = g4[k];
    for (int k = threadIdx.x; k < kTableStride; k += blockDim.x) stab[k] = a.tables[(size_t)b * kTableStride + k];
    __syncthreads();
    // update_word addresses word j of a thread at slot + j * 128 words: one 512-word region per 128 threads
    const uint32_t slot = (uint32_t)__cvta_generic_to_shared(&sidx[(threadIdx.x >> 7) * 512 + (threadIdx.x & 127)]);
    const uint32_t c1 = (uint32_t)b + a.replica_offset;
    const bool never = stab[kTabNever] != 0u;
    long long mom[8];
    if (a.moments && threadIdx.x == 0)
        for (int k = 0; k < 8; ++k) mom[k] = a.moments[(size_t)b * 8 + k];
    for (long long s = 0; s < a.n_sweeps; ++s) {
        const unsigned long long t = a.t0 + (unsigned long long)s;
        const uint32_t c2 = (uint32_t)(t & 0xFFFFFFFFull);
        const uint32_t c3lo = (uint32_t)((t >> 32) & 0xFFFFFFull) | (kDomainIsing << 28);
        int sS0 = 0, sS1 = 0, sSN = 0;      // this thread's share of sum s (colour 0, colour 1) and of sum s * 4 nd
        for (int colour = 0; colour < 2; ++colour) {
            const uint32_t c3 = c3lo | ((uint32_t)colour << 24);
            int& sS = colour ? sS1 : sS0;
            if (never) {
                if (a.measure) resident_half_sweep<true, true>(a, colour, c2, c3, lat, stab, slot, c1, sS, sSN);
                else resident_half_sweep<true, false>(a, colour, c2, c3, lat, stab, slot, c1, sS, sSN);
            } else {
                if (a.measure) resident_half_sweep<false, true>(a, colour, c2, c3, lat, stab, slot, c1, sS, sSN);
                else resident_half_sweep<false, false>(a, colour, c2, c3, lat, stab, slot, c1, sS, sSN);
            }
            __syncthreads();
        }
        if (a.measure) {
            // Every bond has exactly one colour-1 end, and after the colour-1 pass both ends are final:
            // sum_bonds s s' = sum over colour-1 sites of s * nn, nn = 4 - 2 nd = 4 - (4 nd) / 2.
            int totS0 = sS0, totS1 = sS1, totSN = sSN;
            block_sum3(totS0, totS1, totSN, scratch);
            if (threadIdx.x == 0) {
                const long long e = -(4ll * totS1 - (long long)totSN / 2), mag = (long long)totS0 + totS1;
                if (a.E_trace) a.E_trace[(size_t)s * a.batch + b] = e;
                if (a.M_trace) a.M_trace[(size_t)s * a.batch + b] = mag;
                if (a.moments) {
                    const unsigned long long ae = e < 0 ? (unsigned long long)(-e) : (unsigned long long)e;
                    const unsigned long long lo = ae * ae, hi = __umul64hi(ae, ae);
                    const unsigned long long old_lo = (unsigned long long)mom[2], new_lo = old_lo + lo;
                    mom[0] += 1;
                    mom[1] += e;
                    mom[2] = (long long)new_lo;
                    mom[3] = (long long)((unsigned long long)mom[3] + hi + (new_lo < old_lo ? 1ull : 0ull));
                    mom[4] += mag;
                    mom[5] += mag < 0 ? -mag : mag;
                    mom[6] += mag * mag;
                    mom[7] += e * mag;
                }
            }
        }
    }
    if (a.moments && threadIdx.x == 0)
        for (int k = 0; k < 8; ++k) a.moments[(size_t)b * 8 + k] = mom[k];
    for (int k = threadIdx.x; k < (int)(latBytes >> 4); k += blockDim.x) g4[k] = ((uint4*)lat)[k];
}

}  // namespace

const char* ising_int8_variant(int L) { return (L % 32 == 0) ? "ising_int8_rows128" : "ising_int8_generic"; }

int launch_ising_int8_half_sweep(const SweepArgs& a, cudaStream_t s) {
    if (a.L % 32 == 0) {
        // rows per thread and release point: measured crossovers of this kernel (148 x kMinBlocks block slots)
        const int perReplica8 = (a.L / kRowsLong) * (a.L >> 5);
        // (as one of two replica groups every launch has half the blocks: 2-row threads stay ahead up to 0.6 waves)
        const bool grouped = a.plan_scale > 1;
        const RowsPlan plan = plan_rows((long long)perReplica8 * a.batch * (grouped ? a.plan_scale : 1), perReplica8, 148 * kMinBlocks,
                                        grouped ? 0.6 : 0.25, 1.2, true);
        const int perReplica = (a.L / plan.rows) * (a.L >> 5);    // strips x row blocks of one colour
        const int tpb = pick_block(perReplica);               // the last block of a replica may be ragged
        const int bpr = (perReplica + tpb - 1) / tpb;
        const unsigned grid = (unsigned)((long long)bpr * a.batch);
        SweepArgs args = a;
        args.pdl_trigger = plan.trigger;
        void (*k)(SweepArgs, int);
        if (a.measure_acc && a.colour == 1) {
            k = plan.rows == kRowsShort ? ising_int8_rows_measure_kernel<kRowsShort>
                : plan.rows == kRowsMid ? ising_int8_rows_measure_kernel<kRowsMid> : ising_int8_rows_measure_kernel<kRowsLong>;
        } else if (a.measure_acc) {
            k = plan.rows == kRowsShort ? ising_int8_rows_fin_kernel<kRowsShort>
                : plan.rows == kRowsMid ? ising_int8_rows_fin_kernel<kRowsMid> : ising_int8_rows_fin_kernel<kRowsLong>;
        } else if (a.t_dev) {
            if (plan.rows == kRowsShort) k = a.colour == 0 ? ising_int8_rows_kernel<0, kRowsShort, true> : ising_int8_rows_kernel<1, kRowsShort, true>;
            else if (plan.rows == kRowsMid) k = a.colour == 0 ? ising_int8_rows_kernel<0, kRowsMid, true> : ising_int8_rows_kernel<1, kRowsMid, true>;
            else k = a.colour == 0 ? ising_int8_rows_kernel<0, kRowsLong, true> : ising_int8_rows_kernel<1, kRowsLong, true>;
        } else if (plan.rows == kRowsShort) k = a.colour == 0 ? ising_int8_rows_kernel<0, kRowsShort, false> : ising_int8_rows_kernel<1, kRowsShort, false>;
        else if (plan.rows == kRowsMid) k = a.colour == 0 ? ising_int8_rows_kernel<0, kRowsMid, false> : ising_int8_rows_kernel<1, kRowsMid, false>;
        else k = a.colour == 0 ? ising_int8_rows_kernel<0, kRowsLong, false> : ising_int8_rows_kernel<1, kRowsLong, false>;
        launch_pdl(k, grid, (unsigned)tpb, s, args, bpr);
    } else {
        const long long half = (long long)a.L * (a.L >> 1);
        const long long total = ((half + 3) >> 2) * a.batch;
        launch_pdl(ising_int8_generic_kernel, (unsigned)((total + 127) / 128), 128u, s, a);
    }
    return 1;
}

}  // namespace spin

namespace spin {

int launch_ising_measure_finalize(long long* acc, int batch, long long sites, long long* E_out, long long* M_out,
                                  long long* moments, cudaStream_t s) {
    launch_pdl(ising_measure_finalize_kernel, (unsigned)((batch + 127) / 128), 128u, s, acc, batch, sites, E_out, M_out, moments);
    return 1;
}

static size_t resident_smem_bytes(int L) {
    return (size_t)L * L + sizeof(uint32_t) * (kTableStride + 4 * kResThreads) + sizeof(int) * 32;
}

bool ising_int8_resident_fits(int L) { return L % 32 == 0 && (size_t)L * L <= kResMaxLatticeBytes; }

// Cooperative launch of the persistent kernel: n_sweeps sweeps from t0 in one launch.  counter: one zeroed device
// word.  Returns the number of kernels launched (1), or 0 when the shape does not qualify / the launch is refused (the
// caller then uses the streaming path).
int launch_ising_int8_persistent(const SweepArgs& a, unsigned long long t0, long long n_sweeps, unsigned int* counter,
                                 cudaStream_t s) {
    if (a.L % 32 != 0) return 0;
    const long long longThreads = (long long)(a.L / kRowsLong) * (a.L >> 5) * a.batch;
    const bool shortRows = longThreads < 148ll * 4 * kRowsThreads || (a.L / kRowsLong) * (a.L >> 5) < kRowsThreads / 2;
    const int rows = shortRows ? kRowsShort : kRowsLong;
    const int perReplica = (a.L / rows) * (a.L >> 5);
    const int tpb = pick_block(perReplica);
    int bpr = (perReplica + tpb - 1) / tpb;
    int items = bpr * a.batch;
    void (*kern)(SweepArgs, int, int, unsigned long long, long long, unsigned int*) =
        shortRows ? ising_int8_persistent_kernel<kRowsShort> : ising_int8_persistent_kernel<kRowsLong>;
    int dev = 0, sms = 0, perSm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&perSm, kern, tpb, 0) != cudaSuccess || perSm < 1) {
        cudaGetLastError();
        return 0;
    }
    int grid = sms * perSm;
    if (grid > items) grid = items;
    SweepArgs args = a;
    void* params[] = {&args, &bpr, &items, &t0, &n_sweeps, &counter};
    if (cudaMemsetAsync(counter, 0, sizeof(unsigned int), s) != cudaSuccess ||
        cudaLaunchCooperativeKernel((void*)kern, dim3((unsigned)grid), dim3((unsigned)tpb), params, 0, s) != cudaSuccess) {
        cudaGetLastError();
        return 0;
    }
    return 1;
}

// Tile geometry for the tiled kernel: about one tile per SM (148 on a B200) over the whole batch, tiles as square as
// the word granularity allows, 4 sweeps per launch (halo 8) when a tile has at least 32 rows, else 2 (halo 4).
struct TileGeom {
    int TR, TK, HR, HK, tilesR, tilesK, sweeps;
    size_t smem;
};

// At most one tile per SM over the whole batch (a second tile on an SM doubles that SM's time and every launch waits for
// the slowest tile: 153 tiles ran 1 x 640^2 at 149 flips/ns, 144 tiles at 220), and among those grids the one whose
// region (tile + halo) has the fewest words per colour: that is the work per half-sweep of every SM.  4 sweeps per launch
// (halo 8) whenever such a region wraps around the lattice at most once, else 2 (halo 4): measured, 4 beats 2, 3, 5, 6
// and 8 on every shape AUTO sends here (profiles/r2_pdl_placement.md).
static bool tile_geometry(int batch, int L, TileGeom& g) {
    if (L % 8 != 0 || L < 16) return false;
    const int W = L >> 1;
    int perReplica = 148 / batch;                               // tiles allowed per replica
    if (perReplica < 1) perReplica = 1;
    for (int sweeps = 4; sweeps >= 2; sweeps -= 2) {
        // staleness moves one SITE per half-sweep: 2 * sweeps rows, and 2 * sweeps actual columns = `sweeps` same-colour
        // columns (k indexes every other column), rounded up to a whole 4-site word
        const int HR = 2 * sweeps, HK = (sweeps + 3) / 4 * 4;
        long long bestWords = -1;
        for (int tilesK = 1; tilesK <= perReplica && tilesK <= (W + 15) / 16; ++tilesK) {
            const int TK = ((W + tilesK - 1) / tilesK + 3) / 4 * 4;
            if ((W + TK - 1) / TK != tilesK) continue;          // rounding merged two columns of tiles
            for (int tilesR = 1; tilesR * tilesK <= perReplica && tilesR <= (L + 7) / 8; ++tilesR) {
                const int TR = (L + tilesR - 1) / tilesR;
                if (TR < 8 || (L + TR - 1) / TR != tilesR) continue;
                if (TR + 2 * HR > 2 * L || TK + 2 * HK > 2 * W) continue;   // the region may wrap around the lattice at most once
                const long long words = (long long)(TR + 2 * HR) * ((TK + 2 * HK) >> 2);
                if ((size_t)words * 8 > 200 * 1024) continue;
                if (bestWords < 0 || words < bestWords) {
                    bestWords = words;
                    g.TR = TR; g.TK = TK; g.tilesR = tilesR; g.tilesK = tilesK; g.sweeps = sweeps; g.HR = HR; g.HK = HK;
                    g.smem = (size_t)words * 8;
                }
            }
        }
        if (bestWords >= 0) return true;
    }
    return false;
}

bool ising_int8_tiled_fits(int batch, int L) {
    TileGeom g;
    return tile_geometry(batch, L, g);
}

int launch_ising_int8_tiled(const SweepArgs& a, void* shadow, unsigned long long t0, long long n_sweeps, cudaStream_t s) {
    TileGeom g;
    if (!tile_geometry(a.batch, a.L, g) || !shadow) return 0;
    if (cudaFuncSetAttribute(ising_int8_tiled_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024) != cudaSuccess ||
        cudaFuncSetAttribute(ising_int8_tiled_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024) != cudaSuccess) {
        cudaGetLastError();
        return 0;
    }
    TiledArgs t;
    t.tables = a.tables; t.batch = a.batch; t.L = a.L; t.replica_offset = a.replica_offset;
    t.TR = g.TR; t.TK = g.TK; t.HR = g.HR; t.HK = g.HK; t.tilesR = g.tilesR; t.tilesK = g.tilesK; t.rk = a.rk;
    const unsigned grid = (unsigned)((long long)g.tilesR * g.tilesK * a.batch);
    const long long words = (long long)(g.TR + 2 * g.HR) * ((g.TK + 2 * g.HK) >> 2);
    const bool oneWord = words <= kTiledThreads;                // one word per thread for the whole launch
    const unsigned tpb = oneWord ? (unsigned)((words + 31) / 32 * 32) : (unsigned)kTiledThreads;
    void* cur = a.lattice;
    void* other = shadow;
    int launches = 0;
    for (long long done = 0; done < n_sweeps; done += g.sweeps) {
        t.src = cur; t.dst = other; t.t0 = t0 + (unsigned long long)done;
        t.sweeps = (int)(n_sweeps - done < g.sweeps ? n_sweeps - done : g.sweeps);
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(grid, 1, 1);
        cfg.blockDim = dim3(tpb, 1, 1);
        cfg.dynamicSmemBytes = g.smem;
        cfg.stream = s;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        if (oneWord) cudaLaunchKernelEx(&cfg, ising_int8_tiled_kernel<true>, t);
        else cudaLaunchKernelEx(&cfg, ising_int8_tiled_kernel<false>, t);
        ++launches;
        void* tmp = cur; cur = other; other = tmp;
    }
    if (cur != a.lattice)                                       // an odd number of launches: the result is in the shadow
        cudaMemcpyAsync(a.lattice, cur, (size_t)a.batch * a.L * a.L, cudaMemcpyDeviceToDevice, s);
    return launches;
}

// Opt the resident kernel in to more than 48 KiB of dynamic shared memory on the CURRENT device (called once per
// handle at creation: the attribute is per device, and cheap to set again).
cudaError_t ising_int8_resident_configure() {
    return cudaFuncSetAttribute(ising_int8_resident_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                (int)(kResMaxLatticeBytes + sizeof(uint32_t) * (kTableStride + 4 * kResThreads) + 128));
}

int launch_ising_int8_resident(const ResidentArgs& a, cudaStream_t s) {
    const size_t smem = resident_smem_bytes(a.L);
    const int units = a.L <= 64 ? a.L * (a.L >> 3) : a.L * (a.L >> 5);   // words (tiny lattices) or strips per colour
    int tpb = kResThreads;
    while (tpb > 32 && tpb / 2 >= units) tpb >>= 1;           // L = 32: 128 words -> 128 threads
    ising_int8_resident_kernel<<<(unsigned)a.batch, tpb, smem, s>>>(a);
    return 1;
}

}  // namespace spin
