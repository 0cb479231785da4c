// init_layout.cu — row a0 (initial lattice from Philox, O3) and the natural <-> checkerboard-split
// layout conversions used by spin_get_spins / spin_set_spins.  None of this is on the hot loop.
#include "spin_internal.cuh"

namespace spin {

namespace {

// Position of natural site (i, j) in the colour-split layouts.
__device__ __forceinline__ size_t int8_index(int b, int L, int i, int j) {
    const int c = (i + j) & 1;
    const int W = L >> 1;
    return (((size_t)b * 2 + c) * L + i) * W + (j >> 1);
}

// O3: one thread per Philox group of 4 consecutive natural sites p = 4g .. 4g+3.
// int8 layout: scattered byte stores (init is not hot).
__global__ void init_int8_kernel(InitArgs a, int potts) {
    const long long N = (long long)a.L * a.L;
    const long long groups = (N + 3) >> 2;
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= groups * a.batch) return;
    const int b = (int)(gid / groups);
    const uint32_t g = (uint32_t)(gid % groups);
    uint32_t out[4];
    philox4x32_10(a.rk, g, (uint32_t)b + a.replica_offset, 0u, (uint32_t)kDomainInit << 28, out);
    int8_t* lat = (int8_t*)a.lattice;
    const uint32_t q = potts ? (uint32_t)a.q[b] : 2u;
#pragma unroll
    for (int e = 0; e < 4; ++e) {
        const long long p = 4ll * g + e;
        if (p >= N) break;
        const int i = (int)(p / a.L), j = (int)(p % a.L);
        int8_t v;
        if (potts) v = (int8_t)__umulhi(out[e], q);
        else v = (out[e] & 0x80000000u) ? (int8_t)1 : (int8_t)-1;
        lat[int8_index(b, a.L, i, j)] = v;
    }
}

// Bit-packed layout: one thread per 64 consecutive natural sites of a row (j = 64 x .. 64 x + 63), which are
// exactly word x of colour 0 and word x of colour 1 of that row (bit = 1 means spin -1).
__global__ void init_bits_kernel(InitArgs a) {
    const int wordsPerRow = a.L >> 6;
    const long long total = (long long)a.batch * a.L * wordsPerRow;
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= total) return;
    const int x = (int)(gid % wordsPerRow);
    const int i = (int)((gid / wordsPerRow) % a.L);
    const int b = (int)(gid / ((long long)wordsPerRow * a.L));
    uint32_t w[2] = {0u, 0u};
    const long long p0 = (long long)i * a.L + 64ll * x;  // multiple of 4
    for (int gq = 0; gq < 16; ++gq) {
        uint32_t out[4];
        philox4x32_10(a.rk, (uint32_t)((p0 >> 2) + gq), (uint32_t)b + a.replica_offset, 0u,
                      (uint32_t)kDomainInit << 28, out);
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const int jj = 4 * gq + e;          // j - 64 x
            const int c = (i + jj) & 1;         // 64 x is even
            const uint32_t down = (out[e] & 0x80000000u) ? 0u : 1u;
            w[c] |= down << (jj >> 1);
        }
    }
    uint32_t* lat = (uint32_t*)a.lattice;
    lat[(((size_t)b * 2 + 0) * a.L + i) * wordsPerRow + x] = w[0];
    lat[(((size_t)b * 2 + 1) * a.L + i) * wordsPerRow + x] = w[1];
}

__global__ void from_natural_int8_kernel(const int8_t* __restrict__ nat, int8_t* __restrict__ lat, int batch, int L) {
    const long long N = (long long)L * L;
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= N * batch) return;
    const int b = (int)(gid / N);
    const long long p = gid % N;
    const int i = (int)(p / L), j = (int)(p % L);
    lat[int8_index(b, L, i, j)] = nat[gid];
}

__global__ void to_natural_int8_kernel(const int8_t* __restrict__ lat, int8_t* __restrict__ nat, int batch, int L) {
    const long long N = (long long)L * L;
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= N * batch) return;
    const int b = (int)(gid / N);
    const long long p = gid % N;
    const int i = (int)(p / L), j = (int)(p % L);
    nat[gid] = lat[int8_index(b, L, i, j)];
}

// L % 32 == 0: one thread per 32 consecutive natural bytes of a row (two 128-bit loads) <-> one 128-bit word of each
// colour.  In row i the even columns belong to colour i & 1 and the odd columns to the other one; PRMT separates /
// interleaves them, and every global access is a coalesced 128-bit one.
__global__ void __launch_bounds__(256) from_natural_int8_vec_kernel(const uint4* __restrict__ nat, int8_t* __restrict__ lat,
                                                                    int batch, int L) {
    const int C = L >> 5;                                       // 32-byte chunks per row
    const long long total = (long long)batch * L * C;
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= total) return;
    const int x = (int)(gid % C);
    const long long bi = gid / C;                               // b * L + i
    const int i = (int)(bi % L);
    const long long b = bi / L;
    const uint4 a = __ldg(nat + 2 * gid), c = __ldg(nat + 2 * gid + 1);
    const uint4 ev = make_uint4(__byte_perm(a.x, a.y, 0x6420), __byte_perm(a.z, a.w, 0x6420),
                                __byte_perm(c.x, c.y, 0x6420), __byte_perm(c.z, c.w, 0x6420));
    const uint4 od = make_uint4(__byte_perm(a.x, a.y, 0x7531), __byte_perm(a.z, a.w, 0x7531),
                                __byte_perm(c.x, c.y, 0x7531), __byte_perm(c.z, c.w, 0x7531));
    const size_t W16 = (size_t)(L >> 5);                        // uint4 per colour-row
    uint4* l4 = (uint4*)lat;
    const int ce = i & 1;
    l4[(((size_t)b * 2 + ce) * L + i) * W16 + x] = ev;
    l4[(((size_t)b * 2 + (1 - ce)) * L + i) * W16 + x] = od;
}

__global__ void __launch_bounds__(256) to_natural_int8_vec_kernel(const int8_t* __restrict__ lat, uint4* __restrict__ nat,
                                                                  int batch, int L) {
    const int C = L >> 5;
    const long long total = (long long)batch * L * C;
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= total) return;
    const int x = (int)(gid % C);
    const long long bi = gid / C;
    const int i = (int)(bi % L);
    const long long b = bi / L;
    const size_t W16 = (size_t)(L >> 5);
    const uint4* l4 = (const uint4*)lat;
    const int ce = i & 1;
    const uint4 ev = l4[(((size_t)b * 2 + ce) * L + i) * W16 + x];
    const uint4 od = l4[(((size_t)b * 2 + (1 - ce)) * L + i) * W16 + x];
    nat[2 * gid] = make_uint4(__byte_perm(ev.x, od.x, 0x5140), __byte_perm(ev.x, od.x, 0x7362),
                              __byte_perm(ev.y, od.y, 0x5140), __byte_perm(ev.y, od.y, 0x7362));
    nat[2 * gid + 1] = make_uint4(__byte_perm(ev.z, od.z, 0x5140), __byte_perm(ev.z, od.z, 0x7362),
                                  __byte_perm(ev.w, od.w, 0x5140), __byte_perm(ev.w, od.w, 0x7362));
}

// one thread per (b, i, x): 64 natural sites <-> two words
__global__ void from_natural_bits_kernel(const int8_t* __restrict__ nat, uint32_t* __restrict__ lat, int batch, int L) {
    const int wordsPerRow = L >> 6;
    const long long total = (long long)batch * L * wordsPerRow;
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= total) return;
    const int x = (int)(gid % wordsPerRow);
    const int i = (int)((gid / wordsPerRow) % L);
    const int b = (int)(gid / ((long long)wordsPerRow * L));
    const int8_t* row = nat + ((size_t)b * L + i) * L + 64 * x;
    uint32_t w[2] = {0u, 0u};
    for (int jj = 0; jj < 64; ++jj) {
        const int c = (i + jj) & 1;
        w[c] |= (row[jj] < 0 ? 1u : 0u) << (jj >> 1);
    }
    lat[(((size_t)b * 2 + 0) * L + i) * wordsPerRow + x] = w[0];
    lat[(((size_t)b * 2 + 1) * L + i) * wordsPerRow + x] = w[1];
}

__global__ void to_natural_bits_kernel(const uint32_t* __restrict__ lat, int8_t* __restrict__ nat, int batch, int L) {
    const int wordsPerRow = L >> 6;
    const long long total = (long long)batch * L * wordsPerRow;
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= total) return;
    const int x = (int)(gid % wordsPerRow);
    const int i = (int)((gid / wordsPerRow) % L);
    const int b = (int)(gid / ((long long)wordsPerRow * L));
    uint32_t w[2];
    w[0] = lat[(((size_t)b * 2 + 0) * L + i) * wordsPerRow + x];
    w[1] = lat[(((size_t)b * 2 + 1) * L + i) * wordsPerRow + x];
    int8_t* row = nat + ((size_t)b * L + i) * L + 64 * x;
    for (int jj = 0; jj < 64; ++jj) {
        const int c = (i + jj) & 1;
        row[jj] = ((w[c] >> (jj >> 1)) & 1u) ? (int8_t)-1 : (int8_t)1;
    }
}

__global__ void validate_natural_kernel(const int8_t* __restrict__ nat, int batch, int L, int potts,
                                        const int32_t* __restrict__ q, unsigned int* bad) {
    const long long N = (long long)L * L;
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= N * batch) return;
    const int v = nat[gid];
    bool ok;
    if (potts) ok = v >= 0 && v < q[gid / N];
    else ok = (v == 1 || v == -1);
    if (!ok) atomicAdd(bad, 1u);
}

// 16 bytes per thread (N % 16 == 0): Ising bytes must be 0x01 or 0xFF, Potts bytes < q of their replica.
__global__ void __launch_bounds__(256) validate_natural_vec_kernel(const uint4* __restrict__ nat, long long n16, long long N16,
                                                                   int potts, const int32_t* __restrict__ q, unsigned int* bad) {
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= n16) return;
    const uint4 v = __ldg(nat + gid);
    const uint32_t w[4] = {v.x, v.y, v.z, v.w};
    unsigned int nbad = 0;
    if (potts) {
        const uint32_t qq = (uint32_t)q[gid / N16];            // bytes >= q (or negative): bit 7 of (byte | (byte + 0x80 - q))
        const uint32_t add = (0x80u - qq) * 0x01010101u;
#pragma unroll
        for (int k = 0; k < 4; ++k) nbad += __popc((w[k] | ((w[k] & 0x7F7F7F7Fu) + add)) & 0x80808080u);
    } else {
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            // exact zero-byte test on w ^ 0x01.. (+1 bytes) and on ~w (-1 = 0xFF bytes)
            const uint32_t a = w[k] ^ 0x01010101u, c = ~w[k];
            const uint32_t za = ~(((a & 0x7F7F7F7Fu) + 0x7F7F7F7Fu) | a | 0x7F7F7F7Fu);
            const uint32_t zc = ~(((c & 0x7F7F7F7Fu) + 0x7F7F7F7Fu) | c | 0x7F7F7F7Fu);
            nbad += 4 - __popc(za | zc);
        }
    }
    if (nbad) atomicAdd(bad, nbad);
}

inline unsigned blocks_for(long long n, int tpb) { return (unsigned)((n + tpb - 1) / tpb); }

}  // namespace

int launch_init(const InitArgs& a, int model, int layout, cudaStream_t s) {
    if (layout == 1) {
        const long long total = (long long)a.batch * a.L * (a.L >> 6);
        init_bits_kernel<<<blocks_for(total, 128), 128, 0, s>>>(a);
    } else {
        const long long N = (long long)a.L * a.L;
        const long long total = ((N + 3) >> 2) * a.batch;
        init_int8_kernel<<<blocks_for(total, 256), 256, 0, s>>>(a, model);
    }
    return 1;
}

int launch_from_natural(const int8_t* natural, void* lattice, int batch, int L, int layout, cudaStream_t s) {
    if (layout == 1) {
        const long long total = (long long)batch * L * (L >> 6);
        from_natural_bits_kernel<<<blocks_for(total, 128), 128, 0, s>>>(natural, (uint32_t*)lattice, batch, L);
    } else if (L % 32 == 0) {
        const long long total = (long long)batch * L * (L >> 5);
        from_natural_int8_vec_kernel<<<blocks_for(total, 256), 256, 0, s>>>((const uint4*)natural, (int8_t*)lattice, batch, L);
    } else {
        const long long total = (long long)batch * L * L;
        from_natural_int8_kernel<<<blocks_for(total, 256), 256, 0, s>>>(natural, (int8_t*)lattice, batch, L);
    }
    return 1;
}

int launch_to_natural(const void* lattice, int8_t* natural, int batch, int L, int layout, cudaStream_t s) {
    if (layout == 1) {
        const long long total = (long long)batch * L * (L >> 6);
        to_natural_bits_kernel<<<blocks_for(total, 128), 128, 0, s>>>((const uint32_t*)lattice, natural, batch, L);
    } else if (L % 32 == 0) {
        const long long total = (long long)batch * L * (L >> 5);
        to_natural_int8_vec_kernel<<<blocks_for(total, 256), 256, 0, s>>>((const int8_t*)lattice, (uint4*)natural, batch, L);
    } else {
        const long long total = (long long)batch * L * L;
        to_natural_int8_kernel<<<blocks_for(total, 256), 256, 0, s>>>((const int8_t*)lattice, natural, batch, L);
    }
    return 1;
}

int launch_validate_natural(const int8_t* natural, int batch, int L, int model, const int32_t* q, unsigned int* bad,
                            cudaStream_t s) {
    const long long total = (long long)batch * L * L;
    if (((long long)L * L) % 16 == 0) {
        validate_natural_vec_kernel<<<blocks_for(total >> 4, 256), 256, 0, s>>>((const uint4*)natural, total >> 4,
                                                                                ((long long)L * L) >> 4, model, q, bad);
        return 1;
    }
    validate_natural_kernel<<<blocks_for(total, 256), 256, 0, s>>>(natural, batch, L, model, q, bad);
    return 1;
}

// ---- +-J couplings: natural-layout bond signs -> per-colour bit planes (spin_set_bonds, spin.h).
// For the colour-c site (i, k), j = 2k + p, p = (i + c) & 1:
//   plane 0 (up) Jv[i-1][j], plane 1 (down) Jv[i][j], plane 2 (centre) p ? Jh[i][j-1] : Jh[i][j],
//   plane 3 (side) p ? Jh[i][j] : Jh[i][j-1];  bit = 1 iff the bond is -1.  One thread per output word quadruple.
// bad[0] counts entries that are not +-1 (each entry is read by exactly one of colour 0 / colour 1 per role, so the
// count is of reads, not of entries; only zero / non-zero matters).
namespace {
__global__ void bonds_from_natural_kernel(const int8_t* __restrict__ Jh, const int8_t* __restrict__ Jv,
                                          uint32_t* __restrict__ planes, int batch, int L, unsigned int* bad) {
    const int WW = L >> 6;
    const long long half = (long long)L * WW;
    const long long total = (long long)batch * 2 * half;
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= total) return;
    const int b = (int)(gid / (2 * half));
    const long long rem = gid - (long long)b * 2 * half;
    const int c = (int)(rem / half);
    const long long w = rem - (long long)c * half;
    const int i = (int)(w / WW), x = (int)(w - (long long)i * WW);
    const int iu = i == 0 ? L - 1 : i - 1, par = (i + c) & 1;
    const int8_t* jh = Jh + (size_t)b * L * L;
    const int8_t* jv = Jv + (size_t)b * L * L;
    uint32_t pu = 0u, pd = 0u, pc = 0u, ps = 0u;
    unsigned int nbad = 0;
    for (int t = 0; t < 32; ++t) {
        const int k = 32 * x + t, j = 2 * k + par, jl = j == 0 ? L - 1 : j - 1;
        const int up = jv[(size_t)iu * L + j], dn = jv[(size_t)i * L + j];
        const int left = jh[(size_t)i * L + jl], right = jh[(size_t)i * L + j];
        nbad += (up != 1 && up != -1) + (dn != 1 && dn != -1) + (left != 1 && left != -1) + (right != 1 && right != -1);
        const int ct = par ? left : right, sd = par ? right : left;
        pu |= (uint32_t)(up < 0) << t;
        pd |= (uint32_t)(dn < 0) << t;
        pc |= (uint32_t)(ct < 0) << t;
        ps |= (uint32_t)(sd < 0) << t;
    }
    uint32_t* base = planes + ((size_t)b * 2 + c) * 4 * half + w;
    base[0] = pu;
    base[half] = pd;
    base[2 * half] = pc;
    base[3 * half] = ps;
    if (nbad) atomicAdd(bad, nbad);
}
}  // namespace

int launch_bonds_from_natural(const int8_t* Jh, const int8_t* Jv, uint32_t* planes, int batch, int L, unsigned int* bad,
                              cudaStream_t s) {
    const long long total = (long long)batch * 2 * L * (L >> 6);
    bonds_from_natural_kernel<<<blocks_for(total, 128), 128, 0, s>>>(Jh, Jv, planes, batch, L, bad);
    return 1;
}

}  // namespace spin
