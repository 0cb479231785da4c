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
            const uint32_t o = (t[e] >> (4 * c)) & 0xFu;
            bool acc = r[e] <= stab[e][o];
            if (kHasNever) acc = acc && !((snever[e] >> o) & 1u);
            if (acc) flip |= 1u << (4 * c + e);
        }
    }
    return own ^ flip;
}

__global__ void __launch_bounds__(128) ising_bits_kernel(SweepArgs a, int bpr) {
    __shared__ uint32_t stab[4][16];
    __shared__ uint32_t snever[4];
    const int b = blockIdx.x / bpr;
    const int blk = blockIdx.x - b * bpr;
    const uint32_t* tab = a.tables + (size_t)b * kTableStride;
    const uint32_t never = tab[kTabNever];
    if (threadIdx.x < 64) {
        const int e = threadIdx.x >> 4, nib = threadIdx.x & 15;
        stab[e][nib] = tab[decode_class(e, nib)];
    }
    if (threadIdx.x < 4) {
        uint32_t m = 0u;
        for (int nib = 0; nib < 16; ++nib) m |= ((never >> decode_class(threadIdx.x, nib)) & 1u) << nib;
        snever[threadIdx.x] = m;
    }
    __syncthreads();
    const int L = a.L, WW = L >> 6;                       // words per colour-row
    const int u = blk * blockDim.x + threadIdx.x;         // < L * WW by construction
    const int i = u / WW, x = u - i * WW;
    const size_t half = (size_t)L * WW;
    uint32_t* ownp = (uint32_t*)a.lattice + ((size_t)b * 2 + a.colour) * half + (size_t)i * WW + x;
    const uint32_t* oth = (const uint32_t*)a.lattice + ((size_t)b * 2 + (1 - a.colour)) * half;
    const int iu = i == 0 ? L - 1 : i - 1, id = i == L - 1 ? 0 : i + 1;
    const uint32_t own = *ownp;
    const uint32_t up = __ldg(oth + (size_t)iu * WW + x);
    const uint32_t dn = __ldg(oth + (size_t)id * WW + x);
    const uint32_t ct = __ldg(oth + (size_t)i * WW + x);
    uint32_t sd;
    if ((i + a.colour) & 1) {   // side neighbour of site k is other[i][k+1]
        const uint32_t nx = __ldg(oth + (size_t)i * WW + (x == WW - 1 ? 0 : x + 1));
        sd = (ct >> 1) | (nx << 31);
    } else {                    // other[i][k-1]
        const uint32_t pv = __ldg(oth + (size_t)i * WW + (x == 0 ? WW - 1 : x - 1));
        sd = (ct << 1) | (pv >> 31);
    }
    const uint32_t g0 = (uint32_t)i * (uint32_t)(L >> 3) + 8u * (uint32_t)x;   // (i*(L/2) + 32x) >> 2
    const uint32_t c1 = (uint32_t)b + a.replica_offset;
    uint32_t res;
    if (never) res = update_word<true>(a, own, up, dn, ct, sd, g0, c1, stab, snever);
    else res = update_word<false>(a, own, up, dn, ct, sd, g0, c1, stab, snever);
    *ownp = res;
}

}  // namespace

int launch_ising_bits_half_sweep(const SweepArgs& a, cudaStream_t s) {
    const int perReplica = a.L * (a.L >> 6);
    int tpb = 128;
    while (perReplica % tpb) tpb >>= 1;
    const int bpr = perReplica / tpb;
    ising_bits_kernel<<<(unsigned)((long long)bpr * a.batch), tpb, 0, s>>>(a, bpr);
    return 1;
}

}  // namespace spin
