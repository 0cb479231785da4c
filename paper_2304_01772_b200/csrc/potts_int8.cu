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
    pdl_wait();   // launched with programmatic stream serialisation: the previous half-sweep must have completed
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

// ---- row-marching kernel: L % 32 == 0.  Same skeleton as the Ising int8 kernel (ising_int8.cu): one thread owns a
// strip of 16 consecutive same-colour sites (8 Philox calls per row) and marches down kRows rows with the three
// other-colour rows it needs in registers, running pointers, a rolled two-row loop and programmatic dependent launch.
// Byte-SIMD throughout: states are < 128, so for x = a ^ b (per byte < 128) bit 7 of x + 0x7F is "a != b".
// The 4 "differs from old" bits and the 4 "differs from new" bits of a site are gathered into one byte that
// indexes a 256-entry shared table holding U[dn + 4] (dn = n_new - n_old = #(!= old) - #(!= new)); the four index
// bytes of a word go through a per-thread shared-memory slot (STS, then LDS.U8 straight into the table address).
constexpr int kRowsLong = 8;    // rows per thread when the launch fills the GPU several times over
constexpr int kRowsMid = 4;     // under about one and a half waves of 8-row blocks
constexpr int kRowsShort = 2;   // latency-bound shapes: short threads, four times as many
constexpr int kRowsThreads = 128;
constexpr int kMinBlocks = kPottsBlocksPerSm;   // resident blocks per SM (spin_internal.cuh)

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

// kSmallQ (q <= 16, states < 16): x = a ^ b < 16, so x + 0x3F / 0x1F / 0x0F raise bit 6 / 5 / 4 iff x != 0 and leave the
// higher bits clear: the four indicator bits land in place without shifts.
template <bool kSmallQ>
__device__ __forceinline__ uint32_t neq_bits(uint32_t v, uint32_t u, uint32_t d, uint32_t c, uint32_t s) {
    const uint32_t k = 0x7F7F7F7Fu;
    uint32_t a0, a1, a2, a3;
    if (kSmallQ) {
        a0 = (v ^ u) + k; a1 = (v ^ d) + 0x3F3F3F3Fu; a2 = (v ^ c) + 0x1F1F1F1Fu; a3 = (v ^ s) + 0x0F0F0F0Fu;
    } else {
        a0 = (v ^ u) + k; a1 = ((v ^ d) + k) >> 1; a2 = ((v ^ c) + k) >> 2; a3 = ((v ^ s) + k) >> 3;
    }
    if (kSmallQ) {
        // High nibbles: a0 = 1000 / 0111, a1 = 0100 / 0011, a2 = 0010 / 0001, a3 = 0001 / 0000 (differs / equal).  Their
        // XOR is a one-to-one code of the four indicator bits (the toggles 1111, 0111, 0011, 0001 are independent), so
        // two 3-input XORs replace the three bit-selects; the pattern table decodes it (small_q_count below).
        return a0 ^ a1 ^ a2 ^ a3;
    }
    // bit 7 from a0, bit 6 from a1, bit 5 from a2, bit 4 from a3 (low nibble is garbage, masked by the caller)
    uint32_t t = (a2 & 0x20202020u) | (a3 & ~0x20202020u);
    t = (a1 & 0x40404040u) | (t & ~0x40404040u);
    t = (a0 & 0x80808080u) | (t & ~0x80808080u);
    return t;
}

// Number of differing neighbours encoded in a nibble: plain indicator bits (general path) or the XOR code of the
// shift-free path: n ^ 0101 = i0 1111 ^ i1 0111 ^ i2 0011 ^ i3 0001, so (i0..i3) is its Gray code.
__device__ __forceinline__ int nibble_count(int n, bool small_q) {
    if (!small_q) return __popc(n);
    const int b = n ^ 5;
    return __popc((b ^ (b >> 1)) & 15);
}

// One site: threshold fetch (the index byte scales into the table address), compare, replace the byte by the proposal.
template <bool kHasNever, int kE>
__device__ __forceinline__ void site_step(uint32_t& acc_mask, uint32_t o, uint32_t r, const uint32_t* stab,
                                          const uint32_t* snever) {
    // two byte-addressed loads (no address arithmetic): pattern byte -> 4 * class -> U[class]
    const uint32_t c4 = ((const uint8_t*)(stab + 16))[o];
    bool acc = r <= *(const uint32_t*)((const char*)stab + c4);
    if (kHasNever) acc = acc && !((snever[0] >> (c4 >> 2)) & 1u);
    if (kHasNever) {
        if (acc) acc_mask |= 0xFFu << (8 * kE);
    } else {
        // kept in PTX so that it stays one ISETP + one predicated add (the bytes are disjoint; a two-operand add
        // issues at twice the rate of a logic op or a PRMT)
        asm("{\n\t.reg .pred p;\n\tsetp.ls.u32 p, %1, %2;\n\t@p add.u32 %0, %0, %3;\n\t}"
            : "+r"(acc_mask) : "r"(r), "r"(*(const uint32_t*)((const char*)stab + c4)), "n"(0xFFu << (8 * kE)));
    }
}

// One site with a field on the state label (kField): the threshold depends on the class AND on new - old.  ftab: the
// replica's [9][255] entries (always << 32) | T (accept iff always or r < T: a threshold of 0 never accepts, so there is no
// never-mask on this path); df = new - old + 127 of the site.
template <int kE>
__device__ __forceinline__ void site_step_field(uint32_t& acc_mask, uint32_t o, uint32_t df, uint32_t r, const uint32_t* stab,
                                                const unsigned long long* ftab) {
    const uint32_t c4 = ((const uint8_t*)(stab + 16))[o];             // 4 * (dn + 4)
    const unsigned long long ent = __ldg(ftab + (c4 >> 2) * 255u + df);
    if ((uint32_t)(ent >> 32) != 0u || r < (uint32_t)ent) acc_mask |= 0xFFu << (8 * kE);
}

// One 4-site word: r0 feeds sites 0, 1 (proposal words r0[0], r0[2]; acceptance words r0[1], r0[3]), r1 sites 2, 3.
// kPow2: q - 1 is a power of two 2^k <= 8 (q = 2, 3, 5, 9): floor(r (q-1) / 2^32) is the top k bits of r, so the four
// proposal offsets of a word come from the top bytes of the four words with three PRMT, a shift and a mask
// (dshift = 8 - k, dmask = (2^k - 1) per byte) instead of four IMAD.HI (half-rate) and three merges.
template <bool kHasNever, bool kSmallQ, bool kPow2, int kJ, bool kField = false>
__device__ __forceinline__ uint32_t update_word(uint32_t own, uint32_t up, uint32_t dn, uint32_t ct, uint32_t sd,
                                                const uint32_t r0[4], const uint32_t r1[4], uint32_t q, uint32_t geAdd,
                                                uint32_t dshift, uint32_t dmask,
                                                const uint32_t* stab, const uint32_t* snever, uint32_t slot,
                                                const unsigned long long* ftab = nullptr) {
    // proposal (O6): new = old + 1 + floor(r_prop (q-1) / 2^32), minus q if >= q
    const uint32_t qm1 = q - 1u;
    uint32_t d;
    if (kPow2) {
        const uint32_t t01 = __byte_perm(r0[0], r0[2], 0x0073), t23 = __byte_perm(r1[0], r1[2], 0x0073);
        d = (__byte_perm(t01, t23, 0x5410) >> dshift) & dmask;
    } else {
        d = __umulhi(r0[0], qm1) | (__umulhi(r0[2], qm1) << 8) | (__umulhi(r1[0], qm1) << 16) | (__umulhi(r1[2], qm1) << 24);
    }
    uint32_t nw = own + 0x01010101u + d;                              // <= 2q-2 per byte
    const uint32_t ge = ((nw + geAdd) >> 7) & 0x01010101u;            // 1 where nw >= q (geAdd = (0x80 - q) per byte)
    nw -= ge * q;
    const uint32_t mo = neq_bits<kSmallQ>(own, up, dn, ct, sd);
    const uint32_t mn = neq_bits<kSmallQ>(nw, up, dn, ct, sd);
    const uint32_t idx = (mo & 0xF0F0F0F0u) | ((mn >> 4) & 0x0F0F0F0Fu);
    slot_store_u32<kJ * kRowsThreads * 4>(slot, idx);
    const uint32_t o0 = slot_load_u8<kJ * kRowsThreads * 4 + 0>(slot);
    const uint32_t o1 = slot_load_u8<kJ * kRowsThreads * 4 + 1>(slot);
    const uint32_t o2 = slot_load_u8<kJ * kRowsThreads * 4 + 2>(slot);
    const uint32_t o3 = slot_load_u8<kJ * kRowsThreads * 4 + 3>(slot);
    uint32_t am = 0u;                                                 // 0xFF in the bytes whose proposal is accepted
    if (kField) {
        const uint32_t df = (nw + 0x7F7F7F7Fu) - own;                 // new - old + 127 per byte (states <= 126: no carries)
        site_step_field<0>(am, o0, df & 0xFFu, r0[1], stab, ftab);
        site_step_field<1>(am, o1, (df >> 8) & 0xFFu, r0[3], stab, ftab);
        site_step_field<2>(am, o2, (df >> 16) & 0xFFu, r1[1], stab, ftab);
        site_step_field<3>(am, o3, df >> 24, r1[3], stab, ftab);
        return (own & ~am) | (nw & am);
    }
    site_step<kHasNever, 0>(am, o0, r0[1], stab, snever);
    site_step<kHasNever, 1>(am, o1, r0[3], stab, snever);
    site_step<kHasNever, 2>(am, o2, r1[1], stab, snever);
    site_step<kHasNever, 3>(am, o3, r1[3], stab, snever);
    return (own & ~am) | (nw & am);
}

// One row of one strip.  up / ct / dn: other-colour words of rows i-1, i, i+1; kParity = 1: the side neighbour of
// site k is other[i][k+1], else other[i][k-1]; `edge` is the 32-bit word holding the 17th byte.
template <bool kHasNever, bool kSmallQ, bool kPow2, int kParity, bool kField = false>
__device__ __forceinline__ uint4 update_row(const PhiloxCtx& a, uint4 own, const uint4& up, const uint4& ct,
                                            const uint4& dn, uint32_t edge, uint32_t g0, uint32_t c1, uint32_t q,
                                            uint32_t geAdd, uint32_t dshift, uint32_t dmask, const uint32_t* stab,
                                            const uint32_t* snever, uint32_t slot, const unsigned long long* ftab = nullptr) {
    uint32_t s0, s1, s2, s3;
    if (kParity) {
        s0 = __byte_perm(ct.x, ct.y, 0x4321);
        s1 = __byte_perm(ct.y, ct.z, 0x4321);
        s2 = __byte_perm(ct.z, ct.w, 0x4321);
        s3 = __byte_perm(ct.w, edge, 0x4321);
    } else {
        s0 = __byte_perm(edge, ct.x, 0x6543);
        s1 = __byte_perm(ct.x, ct.y, 0x6543);
        s2 = __byte_perm(ct.y, ct.z, 0x6543);
        s3 = __byte_perm(ct.z, ct.w, 0x6543);
    }
    uint4 res;
    uint32_t r0[4], r1[4];
    philox4x32_10(a.rk, g0 + 0, c1, a.c2, a.c3, r0);
    philox4x32_10(a.rk, g0 + 1, c1, a.c2, a.c3, r1);
    res.x = update_word<kHasNever, kSmallQ, kPow2, 0, kField>(own.x, up.x, dn.x, ct.x, s0, r0, r1, q, geAdd, dshift, dmask, stab, snever, slot, ftab);
    philox4x32_10(a.rk, g0 + 2, c1, a.c2, a.c3, r0);
    philox4x32_10(a.rk, g0 + 3, c1, a.c2, a.c3, r1);
    res.y = update_word<kHasNever, kSmallQ, kPow2, 1, kField>(own.y, up.y, dn.y, ct.y, s1, r0, r1, q, geAdd, dshift, dmask, stab, snever, slot, ftab);
    philox4x32_10(a.rk, g0 + 4, c1, a.c2, a.c3, r0);
    philox4x32_10(a.rk, g0 + 5, c1, a.c2, a.c3, r1);
    res.z = update_word<kHasNever, kSmallQ, kPow2, 2, kField>(own.z, up.z, dn.z, ct.z, s2, r0, r1, q, geAdd, dshift, dmask, stab, snever, slot, ftab);
    philox4x32_10(a.rk, g0 + 6, c1, a.c2, a.c3, r0);
    philox4x32_10(a.rk, g0 + 7, c1, a.c2, a.c3, r1);
    res.w = update_word<kHasNever, kSmallQ, kPow2, 3, kField>(own.w, up.w, dn.w, ct.w, s3, r0, r1, q, geAdd, dshift, dmask, stab, snever, slot, ftab);
    return res;
}

template <int kColour, bool kHasNever, bool kSmallQ, bool kPow2, int kRows, bool kField = false>
__device__ __forceinline__ void march_rows(const SweepArgs& a, const PhiloxCtx& pc, const uint32_t* stab, const uint32_t* snever, uint32_t q,
                                           uint32_t slot, int b, int rb, int x, const unsigned long long* ftab = nullptr) {
    const int L = a.L, W = L >> 1, W16 = W >> 4, W4 = W >> 2;
    const size_t half = (size_t)L * W;
    const int i0 = rb * kRows;
    uint8_t* ownBase = (uint8_t*)a.lattice + ((size_t)b * 2 + kColour) * half;
    const uint8_t* oth = (const uint8_t*)a.lattice + ((size_t)b * 2 + (1 - kColour)) * half;
    const uint4* oth4 = (const uint4*)oth;
    const uint32_t* oth1 = (const uint32_t*)oth;
    const uint32_t eNext = (x == W16 - 1) ? 0u : 4u * x + 4u;    // word index of the edge word inside a row
    const uint32_t ePrev = (x == 0) ? (uint32_t)W4 - 1u : 4u * x - 1u;
    const int iu = i0 == 0 ? L - 1 : i0 - 1;
    const int iLast = (i0 + kRows == L) ? 0 : i0 + kRows;        // the only prefetched row that can wrap
    const size_t rowStride = (size_t)W16;                         // in uint4
    const size_t edgeStride2 = 2 * (size_t)W4;                    // two rows, in uint32
    const uint4* pOth = oth4 + (size_t)(i0 + 2) * W16 + x;
    const uint4* pOthLast = oth4 + (size_t)iLast * W16 + x;
    uint4* pOwn = (uint4*)ownBase + (size_t)i0 * W16 + x;
    // even rows of the block have parity kColour, odd rows 1 - kColour (i0 is even)
    const uint32_t* pEdgeEven = oth1 + (size_t)i0 * W4 + (kColour ? eNext : ePrev);
    const uint32_t* pEdgeOdd = oth1 + (size_t)(i0 + 1) * W4 + (kColour ? ePrev : eNext);
    uint4 wU = __ldg(oth4 + (size_t)iu * W16 + x);               // other-colour rows i-1, i, i+1
    uint4 wC = __ldg(pOth - 2 * rowStride);
    uint4 wD = __ldg(pOth - rowStride);
    uint4 own = *pOwn;
    uint32_t edge = __ldg(pEdgeEven);
    uint32_t g0 = (uint32_t)i0 * (uint32_t)(W >> 1) + 8u * (uint32_t)x;   // Philox group = n >> 1
    const uint32_t c1 = (uint32_t)b + a.replica_offset;
    const uint32_t geAdd = (0x80u - q) * 0x01010101u;
    // q - 1 = 2^k: offsets are the top k bits of the proposal words
    const uint32_t kbits = 31u - (uint32_t)__clz((int)(q - 1u));
    const uint32_t dshift = 8u - kbits, dmask = ((1u << kbits) - 1u) * 0x01010101u;
    // rolled: with the q - 1 = 2^k variant next to the general small-q one, two unrolled bodies no longer fit the
    // instruction cache when replicas with different q share a launch (C4: 529 unrolled vs 538 rolled updates/ns)
#pragma unroll 1
    for (int rr = 0; rr < kRows; rr += 2) {
        const bool more = rr + 2 < kRows;
        const uint4 n1 = __ldg(more ? pOth : pOthLast);
        const uint4 own1 = *(pOwn + rowStride);
        const uint32_t edge1 = __ldg(pEdgeOdd);
        uint4 res = update_row<kHasNever, kSmallQ, kPow2, kColour, kField>(pc, own, wU, wC, wD, edge, g0, c1, q, geAdd, dshift, dmask, stab, snever, slot, ftab);
        *pOwn = res;
        uint4 n2 = n1, own2 = own1;
        uint32_t edge2 = edge1;
        if (more) {
            n2 = __ldg(pOth + rowStride);
            own2 = *(pOwn + 2 * rowStride);
            edge2 = __ldg(pEdgeEven + edgeStride2);
        }
        res = update_row<kHasNever, kSmallQ, kPow2, 1 - kColour, kField>(pc, own1, wC, wD, n1, edge1, g0 + (uint32_t)(W >> 1), c1, q, geAdd,
                                                                         dshift, dmask, stab, snever, slot, ftab);
        *(pOwn + rowStride) = res;
        wU = wD;
        wC = n1;
        wD = n2;
        own = own2;
        edge = edge2;
        pOth += 2 * rowStride;
        pOwn += 2 * rowStride;
        pEdgeEven += edgeStride2;
        pEdgeOdd += edgeStride2;
        g0 += (uint32_t)W;
    }
}

// One block covers blockDim.x consecutive strips-times-row-blocks of one replica; bpr = blocks per replica.
template <int kColour, int kRows, bool kDevT>
__global__ void __launch_bounds__(kRowsThreads, kMinBlocks) potts_int8_rows_kernel(SweepArgs a, int bpr) {
    __shared__ uint32_t stab[16 + 64];            // U[dn + 4] in [0..8]; from word 16: 256-byte pattern -> 4 * class table
    __shared__ uint32_t snever[1];
    __shared__ uint32_t sidx[4 * kRowsThreads];   // per-thread slot: word j of thread t at sidx[j * 128 + t]
    if (a.pdl_trigger == kPdlAtStart) pdl_launch_dependents();
    const int b = blockIdx.x / bpr;
    const int blk = blockIdx.x - b * bpr;
    pdl_wait();
    uint32_t c2, c3;
    sweep_counter_words<kDevT>(a, c2, c3);
    const PhiloxCtx pc = {a.rk, c2, c3};
    const uint32_t* tab = a.tables + (size_t)b * kTableStride;
    const uint32_t never = tab[kTabNever];
    for (int m = threadIdx.x; m < 16; m += blockDim.x) stab[m] = tab[m];
    if (threadIdx.x == 0) snever[0] = never;
    const uint32_t q = tab[kTabQ];
    const bool small_q = !never && q <= 16u;                // the variant this block runs (see the dispatch below)
    for (int m = threadIdx.x; m < 256; m += blockDim.x) {
        // high nibble: "neighbour != old" code, low nibble: "neighbour != new" code
        const int cls = nibble_count(m >> 4, small_q) - nibble_count(m & 15, small_q) + 4;
        ((uint8_t*)(stab + 16))[m] = (uint8_t)(4 * cls);
    }
    __syncthreads();
    const int W16 = a.L >> 5;
    const int u = blk * blockDim.x + threadIdx.x;
    if (u >= (a.L / kRows) * W16) return;                  // ragged last block of a replica (after the barrier)
    const int rb = u / W16, x = u - rb * W16;
    const uint32_t slot = (uint32_t)__cvta_generic_to_shared(&sidx[threadIdx.x]);
    if (never) march_rows<kColour, true, false, false, kRows>(a, pc, stab, snever, q, slot, b, rb, x);
    else if (q <= 16u && ((q - 1u) & (q - 2u)) == 0u) march_rows<kColour, false, true, true, kRows>(a, pc, stab, snever, q, slot, b, rb, x);
    else if (q <= 16u) march_rows<kColour, false, true, false, kRows>(a, pc, stab, snever, q, slot, b, rb, x);   // shift-free indicators
    else march_rows<kColour, false, false, false, kRows>(a, pc, stab, snever, q, slot, b, rb, x);
}

// Half-sweep with a field on the state label (Eq. 5 of the paper with its field term): the same marching
// code; the acceptance entry of a site comes from the replica's [9][255] table in global memory (L1-resident: a replica
// touches at most 9 x (2 q - 1) entries), indexed by the class and by new - old.
template <int kColour, int kRows>
__global__ void __launch_bounds__(kRowsThreads, kMinBlocks) potts_int8_rows_field_kernel(SweepArgs a, int bpr) {
    __shared__ uint32_t stab[16 + 64];            // from word 16: 256-byte pattern -> 4 * class table (words 0..15 unused)
    __shared__ uint32_t snever[1];
    __shared__ uint32_t sidx[4 * kRowsThreads];
    if (a.pdl_trigger == kPdlAtStart) pdl_launch_dependents();
    const int b = blockIdx.x / bpr;
    const int blk = blockIdx.x - b * bpr;
    pdl_wait();
    const PhiloxCtx pc = {a.rk, a.c2, a.c3};
    const uint32_t q = a.tables[(size_t)b * kTableStride + kTabQ];
    if (threadIdx.x == 0) snever[0] = 0u;
    for (int m = threadIdx.x; m < 256; m += blockDim.x) {
        const int cls = nibble_count(m >> 4, false) - nibble_count(m & 15, false) + 4;
        ((uint8_t*)(stab + 16))[m] = (uint8_t)(4 * cls);
    }
    __syncthreads();
    const int W16 = a.L >> 5;
    const int u = blk * blockDim.x + threadIdx.x;
    if (u >= (a.L / kRows) * W16) return;
    const int rb = u / W16, x = u - rb * W16;
    const uint32_t slot = (uint32_t)__cvta_generic_to_shared(&sidx[threadIdx.x]);
    march_rows<kColour, false, false, false, kRows, true>(a, pc, stab, snever, q, slot, b, rb, x, a.potts_tab2 + (size_t)b * 9 * 255);
}

}  // namespace

const char* potts_int8_variant(int L) { return (L % 32 == 0) ? "potts_int8_rows128" : "potts_int8_generic"; }

// The instantiation for (rows per thread, colour); kDevT: sweep index from device memory (graph nodes).
template <bool kDevT>
static void (*pick_potts_kernel(int rows, int colour))(SweepArgs, int) {
    if (rows == kRowsShort) return colour == 0 ? potts_int8_rows_kernel<0, kRowsShort, kDevT> : potts_int8_rows_kernel<1, kRowsShort, kDevT>;
    if (rows == kRowsMid) return colour == 0 ? potts_int8_rows_kernel<0, kRowsMid, kDevT> : potts_int8_rows_kernel<1, kRowsMid, kDevT>;
    return colour == 0 ? potts_int8_rows_kernel<0, kRowsLong, kDevT> : potts_int8_rows_kernel<1, kRowsLong, kDevT>;
}

int launch_potts_int8_half_sweep(const SweepArgs& a, cudaStream_t s) {
    if (a.L % 32 == 0) {
        // rows per thread and release point: measured crossovers of this kernel (148 x kMinBlocks block slots)
        const int perReplica8 = (a.L / kRowsLong) * (a.L >> 5);
        const bool grouped = a.plan_scale > 1;                 // one of two replica groups: half the blocks per launch
        const RowsPlan plan = plan_rows((long long)perReplica8 * a.batch * (grouped ? a.plan_scale : 1), perReplica8, 148 * kMinBlocks,
                                        grouped ? 0.55 : 0.3, grouped ? 1.2 : 1.5, false);
        const int perReplica = (a.L / plan.rows) * (a.L >> 5);    // strips x row blocks of one colour
        const int tpb = pick_block(perReplica);               // the last block of a replica may be ragged
        const int bpr = (perReplica + tpb - 1) / tpb;
        const unsigned grid = (unsigned)((long long)bpr * a.batch);
        SweepArgs args = a;
        args.pdl_trigger = plan.trigger;
        void (*k)(SweepArgs, int) = a.t_dev ? pick_potts_kernel<true>(plan.rows, a.colour) : pick_potts_kernel<false>(plan.rows, a.colour);
        if (a.potts_tab2) {
            if (plan.rows == kRowsShort) k = a.colour == 0 ? potts_int8_rows_field_kernel<0, kRowsShort> : potts_int8_rows_field_kernel<1, kRowsShort>;
            else if (plan.rows == kRowsMid) k = a.colour == 0 ? potts_int8_rows_field_kernel<0, kRowsMid> : potts_int8_rows_field_kernel<1, kRowsMid>;
            else k = a.colour == 0 ? potts_int8_rows_field_kernel<0, kRowsLong> : potts_int8_rows_field_kernel<1, kRowsLong>;
        }
        launch_pdl(k, grid, (unsigned)tpb, s, args, bpr);
    } else {
        const long long half = (long long)a.L * (a.L >> 1);
        const long long total = ((half + 1) >> 1) * a.batch;
        launch_pdl(potts_int8_generic_kernel, (unsigned)((total + 127) / 128), 128u, s, a);
    }
    return 1;
}

}  // namespace spin
