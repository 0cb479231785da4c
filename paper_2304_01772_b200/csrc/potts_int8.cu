// potts_int8.cu — rows a2/a3 for the q-state Potts model, uint8 states in the checkerboard-split layout
// [B][2][L][L/2] (Eq. 5-6 and the "one of the q-1 other states" proposal; Alg. 1,
// PAPER.md:127-138).  One Philox call feeds 2 sites (proposal word + acceptance word).  q is per replica.
#include "spin_internal.cuh"

namespace spin {

namespace {

__device__ __forceinline__ bool accept_slow(uint32_t r, const uint32_t* tab, int idx) {
    return (r <= tab[idx]) && !((tab[kTabNever] >> idx) & 1u);
}

// ---- generic kernel: any even L, one thread per Philox group (2 consecutive same-colour sites).
__global__ void potts_int8_generic_kernel(SweepArgs a) {
    const int L = a.L, W = L >> 1;
    const long long half = (long long)L * W;
    const long long groups = (half + 1) >> 1;
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= groups * a.batch) return;
    const int b = (int)(gid / groups);
    const uint32_t g = (uint32_t)(gid % groups);
    const uint32_t* tab = a.tables + (size_t)b * kTableStride;
    const uint32_t q = tab[kTabQ];
    uint8_t* own = (uint8_t*)a.lattice + ((size_t)b * 2 + a.colour) * half;
    const uint8_t* oth = (const uint8_t*)a.lattice + ((size_t)b * 2 + (1 - a.colour)) * half;
    uint32_t r[4];
    philox4x32_10(a.rk, g, (uint32_t)b + a.replica_offset, a.c2, a.c3, r);
#pragma unroll
    for (int e = 0; e < 2; ++e) {
        const long long n = 2ll * g + e;
        if (n >= half) break;
        const int i = (int)(n / W), k = (int)(n % W);
        const int p = (i + a.colour) & 1;
        const int iu = i == 0 ? L - 1 : i - 1, id = i == L - 1 ? 0 : i + 1;
        const int ks = p ? (k == W - 1 ? 0 : k + 1) : (k == 0 ? W - 1 : k - 1);
        const uint32_t old = own[n];
        uint32_t nw = old + 1u + __umulhi(r[2 * e], q - 1u);
        if (nw >= q) nw -= q;
        const uint32_t nb[4] = {oth[(size_t)iu * W + k], oth[(size_t)id * W + k], oth[(size_t)i * W + k],
                                oth[(size_t)i * W + ks]};
        int dn = 0;
#pragma unroll
        for (int t = 0; t < 4; ++t) dn += (int)(nb[t] == nw) - (int)(nb[t] == old);
        if (accept_slow(r[2 * e + 1], tab, dn + 4)) own[n] = (uint8_t)nw;
    }
}

// ---- vectorised kernel: L % 32 == 0, one thread per 16 consecutive same-colour sites (8 Philox calls).
// Byte-SIMD throughout: states are < 128, so for x = a ^ b (per byte < 128) bit 7 of x + 0x7F is "a != b".
// The 4 "differs from old" bits and the 4 "differs from new" bits of a site are gathered into one byte that
// indexes a 256-entry shared table holding U[dn + 4] (dn = n_new - n_old = #(!= old) - #(!= new)).
__device__ __forceinline__ uint32_t neq_bits(uint32_t v, uint32_t u, uint32_t d, uint32_t c, uint32_t s) {
    const uint32_t k = 0x7F7F7F7Fu;
    const uint32_t a0 = (v ^ u) + k, a1 = ((v ^ d) + k) >> 1, a2 = ((v ^ c) + k) >> 2, a3 = ((v ^ s) + k) >> 3;
    // bit 7 from a0, bit 6 from a1, bit 5 from a2, bit 4 from a3 (low nibble is garbage, masked by the caller)
    uint32_t t = (a2 & 0x20202020u) | (a3 & ~0x20202020u);
    t = (a1 & 0x40404040u) | (t & ~0x40404040u);
    t = (a0 & 0x80808080u) | (t & ~0x80808080u);
    return t;
}

template <bool kHasNever>
__device__ __forceinline__ uint32_t update_word(uint32_t own, uint32_t up, uint32_t dn, uint32_t ct, uint32_t sd,
                                                const uint32_t r0[4], const uint32_t r1[4], uint32_t q,
                                                const uint32_t* stab, const uint32_t* snever) {
    // proposal (O6): new = old + 1 + floor(r_prop (q-1) / 2^32), minus q if >= q
    const uint32_t qm1 = q - 1u;
    const uint32_t d = __umulhi(r0[0], qm1) | (__umulhi(r0[2], qm1) << 8) | (__umulhi(r1[0], qm1) << 16) |
                       (__umulhi(r1[2], qm1) << 24);
    uint32_t nw = own + 0x01010101u + d;                              // <= 2q-2 per byte
    const uint32_t ge = ((nw + (0x80u - q) * 0x01010101u) >> 7) & 0x01010101u;   // 1 where nw >= q
    nw -= ge * q;
    const uint32_t mo = neq_bits(own, up, dn, ct, sd);
    const uint32_t mn = neq_bits(nw, up, dn, ct, sd);
    const uint32_t idx = (mo & 0xF0F0F0F0u) | ((mn >> 4) & 0x0F0F0F0Fu);
    const uint32_t racc[4] = {r0[1], r0[3], r1[1], r1[3]};
#pragma unroll
    for (int e = 0; e < 4; ++e) {
        const uint32_t o = (idx >> (8 * e)) & 0xFFu;
        bool acc = racc[e] <= stab[o];
        if (kHasNever) acc = acc && !((snever[o >> 5] >> (o & 31u)) & 1u);
        if (acc) own = __byte_perm(own, nw, 0x3210 ^ ((0x4 + e) << (4 * e)) ^ (e << (4 * e)));
    }
    return own;
}

template <bool kHasNever>
__device__ __forceinline__ void update_vec(SweepArgs& a, const uint32_t* stab, const uint32_t* snever, uint32_t q,
                                           int b, int i, int x) {
    const int L = a.L, W = L >> 1, W16 = W >> 4;
    const size_t half = (size_t)L * W;
    uint4* ownp = (uint4*)((uint8_t*)a.lattice + ((size_t)b * 2 + a.colour) * half) + (size_t)i * W16 + x;
    const uint8_t* oth = (const uint8_t*)a.lattice + ((size_t)b * 2 + (1 - a.colour)) * half;
    const int iu = i == 0 ? L - 1 : i - 1, id = i == L - 1 ? 0 : i + 1;
    const uint4 own = *ownp;
    const uint4 up = __ldg((const uint4*)(oth + (size_t)iu * W) + x);
    const uint4 dn = __ldg((const uint4*)(oth + (size_t)id * W) + x);
    const uint4 ct = __ldg((const uint4*)(oth + (size_t)i * W) + x);
    const int p = (i + a.colour) & 1;
    uint32_t s0, s1, s2, s3;
    if (p) {
        const int kn = (x == W16 - 1) ? 0 : 16 * x + 16;
        const uint32_t nx = (uint32_t)__ldg(oth + (size_t)i * W + kn);
        s0 = __byte_perm(ct.x, ct.y, 0x4321);
        s1 = __byte_perm(ct.y, ct.z, 0x4321);
        s2 = __byte_perm(ct.z, ct.w, 0x4321);
        s3 = __byte_perm(ct.w, nx, 0x4321);
    } else {
        const int kp = (x == 0) ? W - 1 : 16 * x - 1;
        const uint32_t pv = (uint32_t)__ldg(oth + (size_t)i * W + kp);
        s0 = __byte_perm(pv, ct.x, 0x6540);
        s1 = __byte_perm(ct.x, ct.y, 0x6543);
        s2 = __byte_perm(ct.y, ct.z, 0x6543);
        s3 = __byte_perm(ct.z, ct.w, 0x6543);
    }
    // same-colour index n = i*W + 16x + ...; Philox group = n >> 1
    const uint32_t g0 = (uint32_t)i * (uint32_t)(W >> 1) + 8u * (uint32_t)x;
    const uint32_t c1 = (uint32_t)b + a.replica_offset;
    uint4 res;
    uint32_t r0[4], r1[4];
    philox4x32_10(a.rk, g0 + 0, c1, a.c2, a.c3, r0);
    philox4x32_10(a.rk, g0 + 1, c1, a.c2, a.c3, r1);
    res.x = update_word<kHasNever>(own.x, up.x, dn.x, ct.x, s0, r0, r1, q, stab, snever);
    philox4x32_10(a.rk, g0 + 2, c1, a.c2, a.c3, r0);
    philox4x32_10(a.rk, g0 + 3, c1, a.c2, a.c3, r1);
    res.y = update_word<kHasNever>(own.y, up.y, dn.y, ct.y, s1, r0, r1, q, stab, snever);
    philox4x32_10(a.rk, g0 + 4, c1, a.c2, a.c3, r0);
    philox4x32_10(a.rk, g0 + 5, c1, a.c2, a.c3, r1);
    res.z = update_word<kHasNever>(own.z, up.z, dn.z, ct.z, s2, r0, r1, q, stab, snever);
    philox4x32_10(a.rk, g0 + 6, c1, a.c2, a.c3, r0);
    philox4x32_10(a.rk, g0 + 7, c1, a.c2, a.c3, r1);
    res.w = update_word<kHasNever>(own.w, up.w, dn.w, ct.w, s3, r0, r1, q, stab, snever);
    *ownp = res;
}

__global__ void __launch_bounds__(256) potts_int8_vec_kernel(SweepArgs a, int bpr) {
    __shared__ uint32_t stab[256];
    __shared__ uint32_t snever[8];
    const int b = blockIdx.x / bpr;
    const int blk = blockIdx.x - b * bpr;
    const uint32_t* tab = a.tables + (size_t)b * kTableStride;
    const uint32_t never = tab[kTabNever];
    if (threadIdx.x < 8) snever[threadIdx.x] = 0u;
    __syncthreads();
    for (int m = threadIdx.x; m < 256; m += blockDim.x) {
        // high nibble: "neighbour != old" bits, low nibble: "neighbour != new" bits
        const int cls = __popc(m >> 4) - __popc(m & 15) + 4;
        stab[m] = tab[cls];
        if ((never >> cls) & 1u) atomicOr(&snever[m >> 5], 1u << (m & 31));
    }
    __syncthreads();
    const uint32_t q = tab[kTabQ];
    const int W16 = a.L >> 5;
    const int u = blk * blockDim.x + threadIdx.x;
    const int i = u / W16, x = u - i * W16;
    if (never) update_vec<true>(a, stab, snever, q, b, i, x);
    else update_vec<false>(a, stab, snever, q, b, i, x);
}

}  // namespace

const char* potts_int8_variant(int L) { return (L % 32 == 0) ? "potts_int8_vec128" : "potts_int8_generic"; }

int launch_potts_int8_half_sweep(const SweepArgs& a, cudaStream_t s) {
    if (a.L % 32 == 0) {
        const int perReplica = a.L * (a.L >> 5);
        int tpb = 256;
        while (perReplica % tpb) tpb >>= 1;
        const int bpr = perReplica / tpb;
        potts_int8_vec_kernel<<<(unsigned)((long long)bpr * a.batch), tpb, 0, s>>>(a, bpr);
    } else {
        const long long half = (long long)a.L * (a.L >> 1);
        const long long total = ((half + 1) >> 1) * a.batch;
        potts_int8_generic_kernel<<<(unsigned)((total + 127) / 128), 128, 0, s>>>(a);
    }
    return 1;
}

}  // namespace spin
