// ising_int8.cu — rows a2/a3: one colour's Metropolis half-sweep of the Ising model, int8 spins in the
// checkerboard-split layout [B][2][L][L/2] (Alg. 1 + checkerboard; Eq. 1-2,
// PAPER.md:99-115).  Integer only: neighbour count, class index, one Philox word per site (one call per 4
// consecutive same-colour sites), one unsigned compare against the replica's threshold table, flip.
#include "spin_internal.cuh"

namespace spin {

namespace {

// Class index used on the device: d*8 + nd, d = 1 iff own spin is -1, nd = number of -1 neighbours.
__device__ __forceinline__ bool accept_slow(uint32_t r, const uint32_t* tab, int idx) {
    return (r <= tab[idx]) && !((tab[kTabNever] >> idx) & 1u);
}

// ---- generic kernel: any even L.  One thread per Philox group (4 consecutive same-colour sites, which may
// span rows when L/2 is not a multiple of 4).  Byte loads; used for L % 32 != 0.
__global__ void ising_int8_generic_kernel(SweepArgs a) {
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

// ---- vectorised kernel: L % 32 == 0.  One thread per 16 consecutive same-colour sites of a row (one 128-bit
// word): 4 coalesced 128-bit loads (own, up, centre, down of the other colour), one byte for the 17th
// neighbour, 4 Philox calls, byte-SIMD neighbour counts, one LDS + compare + predicated XOR per site.
template <bool kHasNever>
__device__ __forceinline__ uint32_t update_word(uint32_t own, uint32_t up, uint32_t dn, uint32_t ct, uint32_t sd,
                                                const uint32_t r[4], const uint32_t* stab) {
    // bit 1 of a +-1 byte is set iff the spin is -1
    const uint32_t m = 0x02020202u;
    const uint32_t sum2 = (up & m) + (dn & m) + (ct & m) + (sd & m);   // 2*nd per byte (0..8)
    const uint32_t off = (sum2 << 1) + ((own & m) << 4);               // byte offset 4*(d*8 + nd)
#pragma unroll
    for (int e = 0; e < 4; ++e) {
        const uint32_t o = (off >> (8 * e)) & 0xFFu;
        const uint32_t U = *(const uint32_t*)((const char*)stab + o);
        bool acc = r[e] <= U;
        if (kHasNever) acc = acc && !((stab[kTabNever] >> (o >> 2)) & 1u);
        if (acc) own ^= 0xFEu << (8 * e);
    }
    return own;
}

template <bool kHasNever>
__device__ __forceinline__ void update_vec(SweepArgs& a, const uint32_t* stab, int b, int i, int x) {
    const int L = a.L, W = L >> 1, W16 = W >> 4;
    const size_t half = (size_t)L * W;
    uint4* ownp = (uint4*)((int8_t*)a.lattice + ((size_t)b * 2 + a.colour) * half) + (size_t)i * W16 + x;
    const int8_t* oth = (const int8_t*)a.lattice + ((size_t)b * 2 + (1 - a.colour)) * half;
    const int iu = i == 0 ? L - 1 : i - 1, id = i == L - 1 ? 0 : i + 1;
    const uint4 own = *ownp;
    const uint4 up = __ldg((const uint4*)(oth + (size_t)iu * W) + x);
    const uint4 dn = __ldg((const uint4*)(oth + (size_t)id * W) + x);
    const uint4 ct = __ldg((const uint4*)(oth + (size_t)i * W) + x);
    const int p = (i + a.colour) & 1;
    uint32_t s0, s1, s2, s3;
    if (p) {  // side neighbour of site k is other[i][k+1]
        const int kn = (x == W16 - 1) ? 0 : 16 * x + 16;
        const uint32_t nx = (uint32_t)(uint8_t)__ldg(oth + (size_t)i * W + kn);
        s0 = __byte_perm(ct.x, ct.y, 0x4321);
        s1 = __byte_perm(ct.y, ct.z, 0x4321);
        s2 = __byte_perm(ct.z, ct.w, 0x4321);
        s3 = __byte_perm(ct.w, nx, 0x4321);
    } else {  // side neighbour of site k is other[i][k-1]
        const int kp = (x == 0) ? W - 1 : 16 * x - 1;
        const uint32_t pv = (uint32_t)(uint8_t)__ldg(oth + (size_t)i * W + kp);
        s0 = __byte_perm(pv, ct.x, 0x6540);
        s1 = __byte_perm(ct.x, ct.y, 0x6543);
        s2 = __byte_perm(ct.y, ct.z, 0x6543);
        s3 = __byte_perm(ct.z, ct.w, 0x6543);
    }
    const uint32_t g0 = (uint32_t)i * (uint32_t)(W >> 2) + 4u * (uint32_t)x;
    const uint32_t c1 = (uint32_t)b + a.replica_offset;
    uint4 res;
    uint32_t r[4];
    philox4x32_10(a.rk, g0 + 0, c1, a.c2, a.c3, r);
    res.x = update_word<kHasNever>(own.x, up.x, dn.x, ct.x, s0, r, stab);
    philox4x32_10(a.rk, g0 + 1, c1, a.c2, a.c3, r);
    res.y = update_word<kHasNever>(own.y, up.y, dn.y, ct.y, s1, r, stab);
    philox4x32_10(a.rk, g0 + 2, c1, a.c2, a.c3, r);
    res.z = update_word<kHasNever>(own.z, up.z, dn.z, ct.z, s2, r, stab);
    philox4x32_10(a.rk, g0 + 3, c1, a.c2, a.c3, r);
    res.w = update_word<kHasNever>(own.w, up.w, dn.w, ct.w, s3, r, stab);
    *ownp = res;
}

// One block covers blockDim.x consecutive 128-bit words of one replica; bpr = blocks per replica.
__global__ void __launch_bounds__(256) ising_int8_vec_kernel(SweepArgs a, int bpr) {
    __shared__ uint32_t stab[kTableStride];
    const int b = blockIdx.x / bpr;
    const int blk = blockIdx.x - b * bpr;
    if (threadIdx.x < kTableStride) stab[threadIdx.x] = a.tables[(size_t)b * kTableStride + threadIdx.x];
    __syncthreads();
    const int W16 = a.L >> 5;
    const int u = blk * blockDim.x + threadIdx.x;          // < L * W16 by construction
    const int i = u / W16, x = u - i * W16;
    if (stab[kTabNever]) update_vec<true>(a, stab, b, i, x);
    else update_vec<false>(a, stab, b, i, x);
}

}  // namespace

const char* ising_int8_variant(int L) { return (L % 32 == 0) ? "ising_int8_vec128" : "ising_int8_generic"; }

int launch_ising_int8_half_sweep(const SweepArgs& a, cudaStream_t s) {
    if (a.L % 32 == 0) {
        const int perReplica = a.L * (a.L >> 5);            // 128-bit words of one colour
        int tpb = 256;
        while (perReplica % tpb) tpb >>= 1;                  // L = 32 -> 32 threads
        const int bpr = perReplica / tpb;
        ising_int8_vec_kernel<<<(unsigned)((long long)bpr * a.batch), tpb, 0, s>>>(a, bpr);
    } else {
        const long long half = (long long)a.L * (a.L >> 1);
        const long long total = ((half + 3) >> 2) * a.batch;
        ising_int8_generic_kernel<<<(unsigned)((total + 127) / 128), 128, 0, s>>>(a);
    }
    return 1;
}

}  // namespace spin
