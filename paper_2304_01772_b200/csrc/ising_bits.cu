// ising_bits.cu — rows a2/a3 for the Ising model in the bit-packed (multi-spin coded) layout
// [B][2][L][L/64] uint32, bit b of word w = same-colour site k = 32 w + b of that row, bit set = spin -1.
// Same rule, same Philox words as the int8 kernels (Alg. 1 + checkerboard).
// One thread per word = 32 sites = 8 Philox calls.  The neighbour count is a bit-sliced full adder; the
// 4-bit class index of every site is assembled nibble-parallel (8 sites per LOP3), so the per-site work is
// extract + LDS + compare + predicated OR.
#include "spin_internal.cuh"

namespace spin {

namespace {

__device__ __forceinline__ uint32_t sel(uint32_t m, uint32_t a, uint32_t b) { return (a & m) | (b & ~m); }

// Per-e nibble tables: the 4 sites of a nibble (e = 0..3) see the class bits (D, P2, P1, P0) at different
// nibble positions; decode_class turns a nibble value back into the standard class index d*8 + nd.
__device__ __forceinline__ int decode_class(int e, int nib) {
    const int b0 = nib & 1, b1 = (nib >> 1) & 1, b2 = (nib >> 2) & 1, b3 = (nib >> 3) & 1;
    int D, P0, P1, P2;
    switch (e) {
        case 0: P0 = b0; P1 = b1; P2 = b2; D = b3; break;
        case 1: D = b0; P0 = b1; P1 = b2; P2 = b3; break;
        case 2: P2 = b0; D = b1; P0 = b2; P1 = b3; break;
        default: P1 = b0; P2 = b1; D = b2; P0 = b3; break;
    }
    return D * 8 + P2 * 4 + P1 * 2 + P0;
}

constexpr int kRowsLong = 8;    // rows per thread when the launch fills the GPU several times over
constexpr int kRowsShort = 2;   // latency-bound shapes: short threads, four times as many
constexpr int kThreads = 128;
#ifndef BITS_MINB
#define BITS_MINB 8
#endif

// One word = 32 sites = 8 Philox calls.  up / dn / ct: other-colour words of rows i-1, i+1, i; sd: the side
// neighbours (ct shifted by one site, with the bit of the adjacent word).  stab[e][nibble] holds U for the class
// whose bits sit in that nibble order; the nibble of site 4c+e is read pre-scaled (x4) so that it is the byte offset
// of the threshold: per site SHF + LOP3 (extract), LDS, ISETP, predicated OR.
template <bool kHasNever>
__device__ __forceinline__ uint32_t update_word(const SweepArgs& a, uint32_t own, uint32_t up, uint32_t dn, uint32_t ct,
                                                uint32_t sd, uint32_t g0, uint32_t c1, const uint32_t (*stab)[16],
                                                const uint32_t* snever) {
    // bit-sliced count of -1 neighbours: nd = P0 + 2 P1 + 4 P2
    const uint32_t s1 = up ^ dn ^ ct;
    const uint32_t k1 = (up & dn) | (ct & (up | dn));
    const uint32_t P0 = s1 ^ sd;
    const uint32_t k2 = s1 & sd;
    const uint32_t P1 = k1 ^ k2;
    const uint32_t P2 = k1 & k2;
    const uint32_t P1a = P1 << 1, P1b = P1 >> 3, P2a = P2 << 2, P2b = P2 >> 2, Da = own << 3, Db = own >> 1;
    uint32_t t[4];
    t[0] = sel(0x11111111u, P0, sel(0x22222222u, P1a, sel(0x44444444u, P2a, Da)));
    t[1] = sel(0x11111111u, Db, sel(0x22222222u, P0, sel(0x44444444u, P1a, P2a)));
    t[2] = sel(0x11111111u, P2b, sel(0x22222222u, Db, sel(0x44444444u, P0, P1a)));
    t[3] = sel(0x11111111u, P1b, sel(0x22222222u, P2b, sel(0x44444444u, Db, P0)));
    uint32_t flip = 0u;
#pragma unroll
    for (int c = 0; c < 8; ++c) {
        uint32_t r[4];
        philox4x32_10(a.rk, g0 + c, c1, a.c2, a.c3, r);
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            // byte offset 4 * nibble of site 4c+e
            const uint32_t o4 = (c == 0 ? (t[e] << 2) : (t[e] >> (4 * c - 2))) & 0x3Cu;
            bool acc = r[e] <= *(const uint32_t*)((const char*)stab[e] + o4);
            if (kHasNever) acc = acc && !((snever[e] >> (o4 >> 2)) & 1u);
            if (acc) flip |= 1u << (4 * c + e);
        }
    }
    return own ^ flip;
}

// Row-marching: one thread owns word x of kRows consecutive rows (same skeleton as ising_int8.cu: the three
// other-colour words it needs stay in registers, running pointers, two rows per rolled iteration because the side
// of the horizontal neighbour alternates, programmatic dependent launch).
template <int kColour, bool kHasNever, int kRows>
__device__ __forceinline__ void march_rows(const SweepArgs& a, const uint32_t (*stab)[16], const uint32_t* snever, int b,
                                           int rb, int x) {
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
#pragma unroll 1
    for (int rr = 0; rr < kRows; rr += 2) {
        const bool more = rr + 2 < kRows;
        const uint32_t n1 = __ldg(more ? pOth : pOthLast);
        const uint32_t own1 = *(pOwn + rowStride);
        const uint32_t edge1 = __ldg(pEdgeOdd);
        uint32_t sd = kColour ? ((wC >> 1) | (edge << 31)) : ((wC << 1) | (edge >> 31));
        *pOwn = update_word<kHasNever>(a, own, wU, wD, wC, sd, g0, c1, stab, snever);
        uint32_t n2 = n1, own2 = own1, edge2 = edge1;
        if (more) {
            n2 = __ldg(pOth + rowStride);
            own2 = *(pOwn + 2 * rowStride);
            edge2 = __ldg(pEdgeEven + 2 * rowStride);
        }
        sd = kColour ? ((wD << 1) | (edge1 >> 31)) : ((wD >> 1) | (edge1 << 31));
        *(pOwn + rowStride) = update_word<kHasNever>(a, own1, wC, n1, wD, sd, g0 + (uint32_t)(L >> 3), c1, stab, snever);
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

template <int kColour, int kRows>
__global__ void __launch_bounds__(kThreads, BITS_MINB) ising_bits_kernel(SweepArgs a, int bpr) {
    __shared__ uint32_t stab[4][16];
    __shared__ uint32_t snever[4];
    pdl_launch_dependents();
    const int b = blockIdx.x / bpr;
    const int blk = blockIdx.x - b * bpr;
    pdl_wait();
    const uint32_t* tab = a.tables + (size_t)b * kTableStride;
    const uint32_t never = tab[kTabNever];
    for (int m = threadIdx.x; m < 64; m += blockDim.x) {
        const int e = m >> 4, nib = m & 15;
        stab[e][nib] = tab[decode_class(e, nib)];
    }
    if (threadIdx.x < 4) {
        uint32_t m = 0u;
        for (int nib = 0; nib < 16; ++nib) m |= ((never >> decode_class(threadIdx.x, nib)) & 1u) << nib;
        snever[threadIdx.x] = m;
    }
    __syncthreads();
    const int WW = a.L >> 6;
    const int u = blk * blockDim.x + threadIdx.x;         // < (L / kRows) * WW by construction
    const int rb = u / WW, x = u - rb * WW;
    if (never) march_rows<kColour, true, kRows>(a, stab, snever, b, rb, x);
    else march_rows<kColour, false, kRows>(a, stab, snever, b, rb, x);
}

}  // namespace

int launch_ising_bits_half_sweep(const SweepArgs& a, cudaStream_t s) {
    const long long longThreads = (long long)(a.L / kRowsLong) * (a.L >> 6) * a.batch;
    const bool shortRows = longThreads < 148ll * 64;      // the per-block table set-up makes short threads pay off only for tiny launches
    const int rows = shortRows ? kRowsShort : kRowsLong;
    const int perReplica = (a.L / rows) * (a.L >> 6);
    int tpb = kThreads;
    while (perReplica % tpb) tpb >>= 1;
    const int bpr = perReplica / tpb;
    const unsigned grid = (unsigned)((long long)bpr * a.batch);
    if (shortRows) {
        if (a.colour == 0) launch_pdl(ising_bits_kernel<0, kRowsShort>, grid, (unsigned)tpb, s, a, bpr);
        else launch_pdl(ising_bits_kernel<1, kRowsShort>, grid, (unsigned)tpb, s, a, bpr);
    } else {
        if (a.colour == 0) launch_pdl(ising_bits_kernel<0, kRowsLong>, grid, (unsigned)tpb, s, a, bpr);
        else launch_pdl(ising_bits_kernel<1, kRowsLong>, grid, (unsigned)tpb, s, a, bpr);
    }
    return 1;
}

}  // namespace spin
