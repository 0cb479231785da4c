// stencil.cu — SURVEY.md section 8(f) #4: Algorithm 1 on the other geometries the paper names:
// the triangular lattice (Eq. 3), the 3D cubic lattice and the square lattice with
// second neighbours, which needs "more colors".  Readings S1-S6 in DESIGN.md section 13:
//   TRIANGULAR: L x L, L % 3 == 0, neighbours (i+-1, j), (i, j+-1), (i+1, j+1), (i-1, j-1), colours (i + j) mod 3;
//   CUBIC:      L^3, L even, neighbours +-1 along each axis, colours (i + j + k) & 1;
//   SQUARE_NNN: L x L, L even, 4 first (J1) + 4 diagonal second (J2) neighbours, colours 2 (i & 1) + (j & 1).
// Natural row-major int8 lattices (no colour split: with 2, 3 or 4 colours and two dimensionalities one layout serves
// all), H = -J1 sum_<1> s s' - J2 sum_<2> s s' - h sum s, dE = 2 s (J1 nn1 + J2 nn2 + h), per-replica class table
// T[d][nd1][nd2] built on the host in IEEE double (the arithmetic of spin_threshold_table).  Random word of a site:
// Philox group n >> 2, word n & 3, n = index of the site among the sites of its colour in row-major order, domain 3.
// One thread per Philox group = 4 consecutive same-colour sites of one row (a row holds a multiple of ... sites of a
// colour only when L allows; groups may straddle rows, handled per site).
#include "../../include/spin.h"
#include "spin_internal.cuh"

#include <cmath>
#include <vector>

namespace spin {
namespace {

constexpr uint32_t kDomainStencil = 3;
constexpr int kStencilRec = 64;            // uint32 per replica: T[0..49], always mask at [62] (low) and [63] (high)

struct StencilArgs {
    int8_t* lattice;
    const uint32_t* tables;                // [B][kStencilRec]
    int32_t stencil, batch, L, colour;
    uint32_t replica_offset, c2, c3;
    RoundKeys rk;
};

__device__ __forceinline__ int wrap_inc(int a, int L) { return a == L - 1 ? 0 : a + 1; }
__device__ __forceinline__ int wrap_dec(int a, int L) { return a == 0 ? L - 1 : a - 1; }

// Index arithmetic of the byte-SIMD kernels without 64-bit divisions (each costs ~100 instructions, against ~40 for the
// update of a site): the thread index splits into (replica, rest) in 32 bits whenever the launch has fewer than 2^32
// threads, and divisions by a power of two are shifts.
__device__ __forceinline__ void split_replica(long long gid, long long total, uint32_t per, int& b, uint32_t& rem) {
    if (total <= 0xFFFFFFFFll) {
        const uint32_t g = (uint32_t)gid;
        b = (int)(g / per);
        rem = g - (uint32_t)b * per;
    } else {
        b = (int)(gid / per);
        rem = (uint32_t)(gid - (long long)b * per);
    }
}
__device__ __forceinline__ void divmod_u32(uint32_t x, uint32_t d, uint32_t& quo, uint32_t& r) {
    if ((d & (d - 1u)) == 0u) { quo = x >> (__ffs((int)d) - 1); r = x & (d - 1u); }
    else { quo = x / d; r = x - quo * d; }
}

// Number of sites of one colour, and coordinates of same-colour site n (row-major order among that colour).
__device__ __host__ __forceinline__ long long colour_sites(int stencil, int L) {
    if (stencil == SPIN_STENCIL_TRIANGULAR) return (long long)L * (L / 3);
    if (stencil == SPIN_STENCIL_CUBIC) return (long long)L * L * (L / 2);
    return (long long)(L / 2) * (L / 2);
}

template <int kStencil>
__global__ void __launch_bounds__(128) stencil_pass_kernel(StencilArgs a) {
    pdl_wait();   // launched with programmatic stream serialisation: the previous pass must have completed
    const int L = a.L;
    const long long per = colour_sites(kStencil, L);
    const long long groups = (per + 3) >> 2;
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= groups * a.batch) return;
    const int b = (int)(gid / groups);
    const uint32_t g = (uint32_t)(gid % groups);
    const long long N = kStencil == SPIN_STENCIL_CUBIC ? (long long)L * L * L : (long long)L * L;
    int8_t* lat = a.lattice + (size_t)b * N;
    const uint32_t* tab = a.tables + (size_t)b * kStencilRec;
    const unsigned long long always = (unsigned long long)tab[62] | ((unsigned long long)tab[63] << 32);
    uint32_t r[4];
    philox4x32_10(a.rk, g, (uint32_t)b + a.replica_offset, a.c2, a.c3, r);
#pragma unroll
    for (int e = 0; e < 4; ++e) {
        const long long n = 4ll * g + e;
        if (n >= per) break;
        int idx;
        size_t x;
        int s;
        if (kStencil == SPIN_STENCIL_TRIANGULAR) {
            const int W = L / 3;
            const int i = (int)(n / W), m = (int)(n % W);
            const int j = 3 * m + ((a.colour - i) % 3 + 3) % 3;
            const int iu = wrap_dec(i, L), id = wrap_inc(i, L), jl = wrap_dec(j, L), jr = wrap_inc(j, L);
            x = (size_t)i * L + j;
            s = lat[x];
            const int nd = (lat[(size_t)iu * L + j] < 0) + (lat[(size_t)id * L + j] < 0) + (lat[(size_t)i * L + jl] < 0) +
                           (lat[(size_t)i * L + jr] < 0) + (lat[(size_t)id * L + jr] < 0) + (lat[(size_t)iu * L + jl] < 0);
            idx = (s < 0 ? 7 : 0) + nd;
        } else if (kStencil == SPIN_STENCIL_CUBIC) {
            const int W = L / 2;
            const long long ij = n / W;
            const int m = (int)(n % W);
            const int i = (int)(ij / L), j = (int)(ij % L);
            const int k = 2 * m + ((i + j + a.colour) & 1);
            const int iu = wrap_dec(i, L), id = wrap_inc(i, L), jl = wrap_dec(j, L), jr = wrap_inc(j, L), kl = wrap_dec(k, L), kr = wrap_inc(k, L);
            x = ((size_t)i * L + j) * L + k;
            s = lat[x];
            const int nd = (lat[((size_t)iu * L + j) * L + k] < 0) + (lat[((size_t)id * L + j) * L + k] < 0) +
                           (lat[((size_t)i * L + jl) * L + k] < 0) + (lat[((size_t)i * L + jr) * L + k] < 0) +
                           (lat[((size_t)i * L + j) * L + kl] < 0) + (lat[((size_t)i * L + j) * L + kr] < 0);
            idx = (s < 0 ? 7 : 0) + nd;
        } else {
            const int W = L / 2;
            const int ai = (int)(n / W), m = (int)(n % W);
            const int i = 2 * ai + (a.colour >> 1), j = 2 * m + (a.colour & 1);
            const int iu = wrap_dec(i, L), id = wrap_inc(i, L), jl = wrap_dec(j, L), jr = wrap_inc(j, L);
            x = (size_t)i * L + j;
            s = lat[x];
            const int nd1 = (lat[(size_t)iu * L + j] < 0) + (lat[(size_t)id * L + j] < 0) + (lat[(size_t)i * L + jl] < 0) +
                            (lat[(size_t)i * L + jr] < 0);
            const int nd2 = (lat[(size_t)iu * L + jl] < 0) + (lat[(size_t)iu * L + jr] < 0) + (lat[(size_t)id * L + jl] < 0) +
                            (lat[(size_t)id * L + jr] < 0);
            idx = (s < 0 ? 25 : 0) + nd1 * 5 + nd2;
        }
        if (((always >> idx) & 1ull) || r[e] < tab[idx]) lat[x] = (int8_t)(-s);
    }
}

// ---- cubic lattice, L % 16 == 0: byte-SIMD marching kernel.  A thread owns 16 consecutive sites along k of one (i, j)
// line (one 128-bit word of the natural layout) for kRows consecutive planes i: 8 of the 16 have the current colour = two
// Philox groups.  The neighbour lines (i+-1, j), (i, j+-1) are 128-bit words of the same k range; the k+-1 neighbours are
// the other-colour bytes of the own word (plus one edge byte on each side).  As in the int8 Ising kernel the spins are
// masked to "4 per -1 spin" per byte, the six neighbours are added per byte, and 4 nd + 32 d is the byte offset of the class
// threshold in a shared-memory table laid out [d][8].  The whole word is written back: its other-colour bytes are rewritten
// with the values they already have (no thread changes them during this pass).  The words of the planes below / of / above
// the current one stay in registers, so a plane costs three 128-bit loads (the next plane's word and the two j neighbours
// of the current one) instead of five: one word per thread was bound by its L2 traffic (80 bytes per 8 updates; 380 vs 449
// flips/ns on 8 x 128^3).  The updated sites never neighbour each other, so a plane's word stays valid as the "i - 1"
// neighbour after it was updated.
template <int kRows, bool kUniform>
__global__ void __launch_bounds__(128) cubic_march_vec_kernel(StencilArgs a) {
    pdl_wait();
    __shared__ unsigned long long stab[16];   // entry (always << 32) | T: accepted iff (64-bit) r < entry, one compare
    __shared__ uint32_t salways;
    const int L = a.L, V = L >> 4, RB = L / kRows;
    const long long per = (long long)RB * L * V;               // threads per replica: (plane block, j, v)
    const long long total = per * a.batch;
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    int b0;
    uint32_t rem0;
    split_replica((long long)blockIdx.x * blockDim.x, total, (uint32_t)per, b0, rem0);
    constexpr bool uniform = kUniform;                           // per % blockDim.x == 0 (the launcher): a block never straddles replicas
    if (uniform) {
        if (threadIdx.x < 16) {
            const uint32_t* tab = a.tables + (size_t)b0 * kStencilRec;
            const int d = threadIdx.x >> 3, nd = threadIdx.x & 7;
            const uint32_t alw = (tab[62] & 0x7Fu) | (((tab[62] >> 7) & 0x7Fu) << 8);
            stab[threadIdx.x] = nd <= 6 ? ((unsigned long long)((alw >> threadIdx.x) & 1u) << 32) | tab[d * 7 + nd] : 0ull;
            if (threadIdx.x == 0) salways = alw;
        }
        __syncthreads();
    }
    if (gid >= total) return;
    int b;
    uint32_t rem, uv, ujr, uj, urb;
    split_replica(gid, total, (uint32_t)per, b, rem);
    divmod_u32(rem, (uint32_t)V, ujr, uv);
    divmod_u32(ujr, (uint32_t)L, urb, uj);
    const int v = (int)uv, j = (int)uj, i0 = (int)urb * kRows;
    const int jl = wrap_dec(j, L), jr = wrap_inc(j, L), k0 = v << 4;
    const int kl = k0 == 0 ? L - 1 : k0 - 1, kr = k0 + 16 == L ? 0 : k0 + 16;
    int8_t* lat = a.lattice + (size_t)b * L * L * L;
    const uint32_t* gtab = a.tables + (size_t)b * kStencilRec;
    uint32_t always = salways;
    if (!uniform) always = (gtab[62] & 0x7Fu) | (((gtab[62] >> 7) & 0x7Fu) << 8);
    const uint32_t m = 0x04040404u;
    const size_t plane = (size_t)L * L;
    // words (i - 1, j), (i, j), (i + 1, j) of the k range; edge bytes of the current and the next plane
    const int iu0 = wrap_dec(i0, L), id0 = wrap_inc(i0, L);
    uint4 u = *(const uint4*)(lat + (size_t)iu0 * plane + (size_t)j * L + k0);
    uint4 c = *(const uint4*)(lat + (size_t)i0 * plane + (size_t)j * L + k0);
    uint4 d = *(const uint4*)(lat + (size_t)id0 * plane + (size_t)j * L + k0);
    uint32_t eL = (uint32_t)(uint8_t)lat[(size_t)i0 * plane + (size_t)j * L + kl];
    uint32_t eR = (uint32_t)(uint8_t)lat[(size_t)i0 * plane + (size_t)j * L + kr];
    uint32_t nL = (uint32_t)(uint8_t)lat[(size_t)id0 * plane + (size_t)j * L + kl];
    uint32_t nR = (uint32_t)(uint8_t)lat[(size_t)id0 * plane + (size_t)j * L + kr];
    uint32_t par = (uint32_t)((i0 + j + a.colour) & 1);        // k parity of the updated sites (k0 is even)
    uint32_t g0 = (uint32_t)(((long long)i0 * L + j) * (L >> 3) + 2 * v);
    const uint32_t gstep = (uint32_t)L * (uint32_t)(L >> 3);
    const uint32_t c1 = (uint32_t)b + a.replica_offset;
#pragma unroll
    for (int rr = 0; rr < kRows; ++rr) {
        const int i = i0 + rr;
        const uint4 f = *(const uint4*)(lat + (size_t)i * plane + (size_t)jl * L + k0);
        const uint4 g = *(const uint4*)(lat + (size_t)i * plane + (size_t)jr * L + k0);
        uint4 x = make_uint4(0u, 0u, 0u, 0u);
        uint32_t xL = 0u, xR = 0u;
        if (rr + 1 < kRows) {                                  // the plane after next
            int i2 = i + 2;
            i2 = i2 >= L ? i2 - L : i2;
            x = *(const uint4*)(lat + (size_t)i2 * plane + (size_t)j * L + k0);
            xL = (uint32_t)(uint8_t)lat[(size_t)i2 * plane + (size_t)j * L + kl];
            xR = (uint32_t)(uint8_t)lat[(size_t)i2 * plane + (size_t)j * L + kr];
        }
        const uint32_t cw[4] = {c.x, c.y, c.z, c.w};
        const uint32_t cm[4] = {c.x & m, c.y & m, c.z & m, c.w & m};
        const uint32_t sum4[4] = {(u.x & m) + (d.x & m) + (f.x & m) + (g.x & m), (u.y & m) + (d.y & m) + (f.y & m) + (g.y & m),
                                  (u.z & m) + (d.z & m) + (f.z & m) + (g.z & m), (u.w & m) + (d.w & m) + (f.w & m) + (g.w & m)};
        uint32_t r[8];
        philox4x32_10(a.rk, g0, c1, a.c2, a.c3, r);
        philox4x32_10(a.rk, g0 + 1u, c1, a.c2, a.c3, r + 4);
        uint32_t out[4];
#pragma unroll
        for (int w = 0; w < 4; ++w) {
            const uint32_t prevm = w == 0 ? ((eL & 4u) << 24) : (cm[w - 1] & 0xFF000000u);
            const uint32_t nextm = w == 3 ? (eR & 4u) : (cm[w + 1] & 0xFFu);
            const uint32_t left = (cm[w] << 8) | (prevm >> 24);
            const uint32_t right = (cm[w] >> 8) | (nextm << 24);
            const uint32_t t = sum4[w] + left + right + (cw[w] & 0x20202020u);                  // bytes: 4 nd + 32 d
            uint32_t flip = 0u;
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const uint32_t pos = 2u * (uint32_t)e + par;                                    // byte of the updated site
                const uint32_t idx = ((t >> (8u * pos)) & 0xFFu) >> 2;                          // d * 8 + nd
                // branch-free (a short-circuit `||` compiles to a divergent branch per site): accept -> all ones
                uint32_t acc;
                if (uniform) acc = (uint32_t)((unsigned long long)r[2 * w + e] < stab[idx]);
                else acc = ((always >> idx) & 1u) | (uint32_t)(r[2 * w + e] < gtab[(idx >> 3) * 7u + (idx & 7u)]);
                flip |= (0u - acc) & (0xFEu << (8u * pos));
            }
            out[w] = cw[w] ^ flip;
        }
        *(uint4*)(lat + (size_t)i * plane + (size_t)j * L + k0) = make_uint4(out[0], out[1], out[2], out[3]);
        u = c; c = d; d = x;                                    // (below, current, above) <- (current as it was, above, new)
        eL = nL; eR = nR; nL = xL; nR = xR;
        par ^= 1u;
        g0 += gstep;
    }
}

// ---- square lattice with second neighbours, L % 16 == 0: the same byte-SIMD scheme.  A thread owns 16 consecutive sites
// of a row of the colour's row parity; 8 of them (column parity of the colour) are updated.  With every spin masked to
// "4 per -1 spin", 5 (N + S + W + E) + (NW + NE + SW + SE) + 25 own is 4 (25 d + 5 nd1 + nd2): the byte offset of the class
// threshold in the 50-entry table.
__device__ __forceinline__ void shifted_words(const uint32_t x[4], uint32_t edgeL, uint32_t edgeR, uint32_t left[4], uint32_t right[4]) {
#pragma unroll
    for (int w = 0; w < 4; ++w) {
        const uint32_t prev = w == 0 ? edgeL : (x[w - 1] >> 24);
        const uint32_t next = w == 3 ? edgeR : (x[w + 1] & 0xFFu);
        left[w] = (x[w] << 8) | prev;          // byte e holds the site at column - 1
        right[w] = (x[w] >> 8) | (next << 24); // byte e holds the site at column + 1
    }
}

// A thread owns the word (row, v) of kRows consecutive rows of the colour's row parity (every other row).  The row below
// an updated row is the row above the next one and is not touched in this pass, so its masked and shifted words are
// reused: two rows of loads per step instead of three (one word per thread: 326 flips/ns on 16 x 1024^2, marching 4 rows:
// 355, 8 rows: 282).
template <int kRows, bool kUniform>
__global__ void __launch_bounds__(128) nnn_march_vec_kernel(StencilArgs a) {
    pdl_wait();
    __shared__ unsigned long long stab[50];   // entry (always << 32) | T: accepted iff (64-bit) r < entry, one compare
    const int L = a.L, V = L >> 4, H = L >> 1, RB = H / kRows;
    const long long per = (long long)RB * V;
    const long long total = per * a.batch;
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    int b0;
    uint32_t rem0;
    split_replica((long long)blockIdx.x * blockDim.x, total, (uint32_t)per, b0, rem0);
    constexpr bool uniform = kUniform;                           // per % blockDim.x == 0 (the launcher): a block never straddles replicas
    if (uniform) {
        const uint32_t* tab = a.tables + (size_t)b0 * kStencilRec;
        if (threadIdx.x < 50)
            stab[threadIdx.x] = ((unsigned long long)((tab[62 + (threadIdx.x >> 5)] >> (threadIdx.x & 31)) & 1u) << 32) | tab[threadIdx.x];
        __syncthreads();
    }
    if (gid >= total) return;
    int b;
    uint32_t rem, uv, urb;
    split_replica(gid, total, (uint32_t)per, b, rem);
    divmod_u32(rem, (uint32_t)V, urb, uv);
    const int v = (int)uv, ar0 = (int)urb * kRows;
    const uint32_t pj = (uint32_t)(a.colour & 1);
    const int j0 = v << 4, jl = j0 == 0 ? L - 1 : j0 - 1, jr = j0 + 16 == L ? 0 : j0 + 16;
    int8_t* lat = a.lattice + (size_t)b * L * L;
    const uint32_t m = 0x04040404u;
    const uint32_t* tab = a.tables + (size_t)b * kStencilRec;   // read by the ragged launches only (!uniform)
    unsigned long long always = 0ull;
    if (!uniform) always = (unsigned long long)tab[62] | ((unsigned long long)tab[63] << 32);
    const uint32_t c1 = (uint32_t)b + a.replica_offset;
    // the row above the first updated row: masked word and its shifted forms
    uint32_t um[4], ul[4], ur[4];
    {
        const int i0 = 2 * ar0 + (a.colour >> 1), iu = wrap_dec(i0, L);
        const uint4 u4 = *(const uint4*)(lat + (size_t)iu * L + j0);
        um[0] = u4.x & m; um[1] = u4.y & m; um[2] = u4.z & m; um[3] = u4.w & m;
        shifted_words(um, (uint32_t)(uint8_t)lat[(size_t)iu * L + jl] & 4u, (uint32_t)(uint8_t)lat[(size_t)iu * L + jr] & 4u, ul, ur);
    }
    uint32_t g0 = (uint32_t)((long long)ar0 * (L >> 3) + 2 * v);
#pragma unroll
    for (int rr = 0; rr < kRows; ++rr) {
        const int i = 2 * (ar0 + rr) + (a.colour >> 1), id = wrap_inc(i, L);
        const uint4 c4 = *(const uint4*)(lat + (size_t)i * L + j0), d4 = *(const uint4*)(lat + (size_t)id * L + j0);
        const uint32_t cw[4] = {c4.x, c4.y, c4.z, c4.w};
        const uint32_t cm[4] = {c4.x & m, c4.y & m, c4.z & m, c4.w & m};
        uint32_t dm[4] = {d4.x & m, d4.y & m, d4.z & m, d4.w & m};
        uint32_t cl[4], cr[4], dl[4], dr[4];
        shifted_words(cm, (uint32_t)(uint8_t)lat[(size_t)i * L + jl] & 4u, (uint32_t)(uint8_t)lat[(size_t)i * L + jr] & 4u, cl, cr);
        shifted_words(dm, (uint32_t)(uint8_t)lat[(size_t)id * L + jl] & 4u, (uint32_t)(uint8_t)lat[(size_t)id * L + jr] & 4u, dl, dr);
        uint32_t r[8];
        philox4x32_10(a.rk, g0, c1, a.c2, a.c3, r);
        philox4x32_10(a.rk, g0 + 1u, c1, a.c2, a.c3, r + 4);
        uint32_t out[4];
#pragma unroll
        for (int w = 0; w < 4; ++w) {
            const uint32_t first = um[w] + dm[w] + cl[w] + cr[w];             // 4 nd1 per byte
            const uint32_t second = ul[w] + ur[w] + dl[w] + dr[w];            // 4 nd2 per byte
            const uint32_t t = first * 5u + second + cm[w] * 25u;             // 4 (25 d + 5 nd1 + nd2), < 256 per byte
            uint32_t flip = 0u;
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const uint32_t pos = 2u * (uint32_t)e + pj;
                const uint32_t idx = ((t >> (8u * pos)) & 0xFFu) >> 2;
                uint32_t acc;                                                                    // branch-free
                if (uniform) acc = (uint32_t)((unsigned long long)r[2 * w + e] < stab[idx]);
                else acc = (uint32_t)((always >> idx) & 1ull) | (uint32_t)(r[2 * w + e] < tab[idx]);
                flip |= (0u - acc) & (0xFEu << (8u * pos));
            }
            out[w] = cw[w] ^ flip;
        }
        *(uint4*)(lat + (size_t)i * L + j0) = make_uint4(out[0], out[1], out[2], out[3]);
#pragma unroll
        for (int w = 0; w < 4; ++w) { um[w] = dm[w]; ul[w] = dl[w]; ur[w] = dr[w]; }   // the row below is the next row above
        g0 += (uint32_t)(L >> 3);
    }
}

// ---- triangular lattice, L % 12 == 0: byte-SIMD row-marching kernel.  A thread owns a chunk of 12 consecutive sites (three
// words) of kRows consecutive rows; the four sites of the pass's colour in a chunk, at bytes p + 3 m with
// p = (colour - i) mod 3, are one Philox group (group index i * (L / 12) + v).  Neighbours (i+-1, j), (i, j+-1),
// (i+1, j+1), (i-1, j-1): with every spin masked to "4 per -1 spin", up + down + left + right + upleft + downright +
// 32 d per byte is the byte offset of the class threshold in a shared-memory table laid out [d][8].  The masked words (and
// the two edge bytes) of the rows above / of / below the current one stay in registers, so a row costs one row of loads
// and the index arithmetic is paid once per thread.  The updated sites never neighbour each other, so the masked words of
// a row stay valid as "row above" after the row was updated (only bytes of the current colour changed, and those are
// never read as neighbours in this pass); rows of the neighbouring threads are read word-wise, their other-colour bytes
// are rewritten with the values they already have.
template <int kRows, bool kUniform, int kColour>
__global__ void __launch_bounds__(128) triangular_march_vec_kernel(StencilArgs a) {
    static_assert(kRows % 3 == 0, "the byte positions of the updated sites are compile-time only if a thread starts at a row that is a multiple of 3");
    pdl_wait();
    __shared__ unsigned long long stab[16];   // entry (always << 32) | T: accepted iff (64-bit) r < entry, one compare
    __shared__ uint32_t salways;
    const int L = a.L, V = L / 12, RB = L / kRows;             // chunks per row, row blocks per replica
    const long long per = (long long)RB * V;
    const long long total = per * a.batch;
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    int b0;
    uint32_t rem0;
    split_replica((long long)blockIdx.x * blockDim.x, total, (uint32_t)per, b0, rem0);
    constexpr bool uniform = kUniform;                           // per % blockDim.x == 0 (the launcher): a block never straddles replicas
    if (uniform) {
        if (threadIdx.x < 16) {
            const uint32_t* tab = a.tables + (size_t)b0 * kStencilRec;
            const int d = threadIdx.x >> 3, nd = threadIdx.x & 7;
            const uint32_t alw = (tab[62] & 0x7Fu) | (((tab[62] >> 7) & 0x7Fu) << 8);
            stab[threadIdx.x] = nd <= 6 ? ((unsigned long long)((alw >> threadIdx.x) & 1u) << 32) | tab[d * 7 + nd] : 0ull;
            if (threadIdx.x == 0) salways = alw;
        }
        __syncthreads();
    }
    if (gid >= total) return;
    int b;
    uint32_t rem, uv, urb;
    split_replica(gid, total, (uint32_t)per, b, rem);
    divmod_u32(rem, (uint32_t)V, urb, uv);
    const int v = (int)uv, i0 = (int)urb * kRows;
    const int j0 = 12 * v, jl = j0 == 0 ? L - 1 : j0 - 1, jr = j0 + 12 == L ? 0 : j0 + 12;
    int8_t* lat = a.lattice + (size_t)b * L * L;
    const uint32_t m = 0x04040404u;
    const uint32_t* gtab = a.tables + (size_t)b * kStencilRec;
    uint32_t always = salways;
    if (!uniform) always = (gtab[62] & 0x7Fu) | (((gtab[62] >> 7) & 0x7Fu) << 8);
    // rows i - 1, i, i + 1: masked words, edge bytes (masked), and the raw words of row i
    uint32_t um[3], cm[3], dm[3], cw[3], nw[3];
    uint32_t uL, cL, cR, dL, dR;
    {
        const int iu = wrap_dec(i0, L), id = wrap_inc(i0, L);
        const uint32_t* ru = (const uint32_t*)(lat + (size_t)iu * L + j0);
        const uint32_t* rc = (const uint32_t*)(lat + (size_t)i0 * L + j0);
        const uint32_t* rd = (const uint32_t*)(lat + (size_t)id * L + j0);
#pragma unroll
        for (int w = 0; w < 3; ++w) { um[w] = ru[w] & m; cw[w] = rc[w]; cm[w] = cw[w] & m; nw[w] = rd[w]; dm[w] = nw[w] & m; }
        uL = (uint32_t)(uint8_t)lat[(size_t)iu * L + jl] & 4u;
        cL = (uint32_t)(uint8_t)lat[(size_t)i0 * L + jl] & 4u;
        cR = (uint32_t)(uint8_t)lat[(size_t)i0 * L + jr] & 4u;
        dL = (uint32_t)(uint8_t)lat[(size_t)id * L + jl] & 4u;
        dR = (uint32_t)(uint8_t)lat[(size_t)id * L + jr] & 4u;
    }
    // byte offset of the first updated site of row i0 + rr: (colour - i) mod 3 = (kColour - rr) mod 3, as i0 % 3 == 0 - a
    // compile-time constant in the unrolled loop, so the word selects, shifts and flip masks below are immediates
    uint32_t group = (uint32_t)((long long)i0 * V + v);
    const uint32_t c1 = (uint32_t)b + a.replica_offset;
#pragma unroll
    for (int rr = 0; rr < kRows; ++rr) {
        const int i = i0 + rr;
        // the row after next (the only load of this step), issued before the arithmetic of the current row
        uint32_t xw[3] = {0u, 0u, 0u}, xL = 0u, xR = 0u;
        if (rr + 1 < kRows) {
            int i2 = i + 2;
            i2 = i2 >= L ? i2 - L : i2;
            const uint32_t* rx = (const uint32_t*)(lat + (size_t)i2 * L + j0);
            xw[0] = rx[0]; xw[1] = rx[1]; xw[2] = rx[2];
            xL = (uint32_t)(uint8_t)lat[(size_t)i2 * L + jl] & 4u;
            xR = (uint32_t)(uint8_t)lat[(size_t)i2 * L + jr] & 4u;
        }
        uint32_t r[4];
        philox4x32_10(a.rk, group, c1, a.c2, a.c3, r);
        uint32_t t[3];
#pragma unroll
        for (int w = 0; w < 3; ++w) {
            const uint32_t cprev = w == 0 ? cL : (cm[w - 1] >> 24), cnext = w == 2 ? cR : (cm[w + 1] & 0xFFu);
            const uint32_t uprev = w == 0 ? uL : (um[w - 1] >> 24), dnext = w == 2 ? dR : (dm[w + 1] & 0xFFu);
            const uint32_t left = (cm[w] << 8) | cprev, right = (cm[w] >> 8) | (cnext << 24);
            const uint32_t upleft = (um[w] << 8) | uprev, downright = (dm[w] >> 8) | (dnext << 24);
            t[w] = um[w] + dm[w] + left + right + upleft + downright + (cw[w] & 0x20202020u);   // bytes: 4 nd + 32 d
        }
        uint32_t flip[3] = {0u, 0u, 0u};
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const int pos = ((kColour - rr) % 3 + 3) % 3 + 3 * e;   // byte of the updated site within the 12
            const uint32_t word = pos < 4 ? t[0] : (pos < 8 ? t[1] : t[2]);
            const uint32_t idx = ((word >> (8 * (pos & 3))) & 0xFFu) >> 2;      // d * 8 + nd
            uint32_t acc;                                                                        // branch-free
            if (uniform) acc = (uint32_t)((unsigned long long)r[e] < stab[idx]);
            else acc = ((always >> idx) & 1u) | (uint32_t)(r[e] < gtab[(idx >> 3) * 7u + (idx & 7u)]);
            const uint32_t bit = (0u - acc) & (0xFEu << (8 * (pos & 3)));
            flip[0] |= pos < 4 ? bit : 0u;
            flip[1] |= (pos >= 4 && pos < 8) ? bit : 0u;
            flip[2] |= pos >= 8 ? bit : 0u;
        }
        uint32_t* wc = (uint32_t*)(lat + (size_t)i * L + j0);
        wc[0] = cw[0] ^ flip[0];
        wc[1] = cw[1] ^ flip[1];
        wc[2] = cw[2] ^ flip[2];
        // next row: (above, current, below) <- (current as it was, below, the row just loaded)
#pragma unroll
        for (int w = 0; w < 3; ++w) { um[w] = cm[w]; cw[w] = nw[w]; cm[w] = dm[w]; nw[w] = xw[w]; dm[w] = xw[w] & m; }
        uL = cL; cL = dL; cR = dR; dL = xL; dR = xR;
        group += (uint32_t)V;
    }
}

__global__ void stencil_init_kernel(int8_t* lattice, long long N, int batch, uint32_t replica_offset, RoundKeys rk) {
    const long long groups = (N + 3) >> 2;
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= groups * batch) return;
    const int b = (int)(gid / groups);
    const uint32_t g = (uint32_t)(gid % groups);
    uint32_t out[4];
    philox4x32_10(rk, g, (uint32_t)b + replica_offset, 0u, (uint32_t)kDomainInit << 28, out);
#pragma unroll
    for (int e = 0; e < 4; ++e) {
        const long long p = 4ll * g + e;
        if (p < N) lattice[(size_t)b * N + p] = (out[e] & 0x80000000u) ? (int8_t)1 : (int8_t)-1;
    }
}

// acc[b][0..2] += (E1, E2, M) partial sums; blocks never straddle replicas.
template <int kStencil>
__global__ void __launch_bounds__(256) stencil_observe_kernel(const int8_t* __restrict__ lattice, int L, int bpr, long long* acc) {
    __shared__ long long sh[3][8];
    const int b = blockIdx.x / bpr, blk = blockIdx.x - b * bpr;
    const long long N = kStencil == SPIN_STENCIL_CUBIC ? (long long)L * L * L : (long long)L * L;
    const int8_t* lat = lattice + (size_t)b * N;
    long long e1 = 0, e2 = 0, m = 0;
    for (long long x = (long long)blk * blockDim.x + threadIdx.x; x < N; x += (long long)bpr * blockDim.x) {
        const int s = lat[x];
        m += s;
        if (kStencil == SPIN_STENCIL_CUBIC) {
            const int k = (int)(x % L), j = (int)((x / L) % L), i = (int)(x / ((long long)L * L));
            e1 -= s * (lat[((size_t)wrap_inc(i, L) * L + j) * L + k] + lat[((size_t)i * L + wrap_inc(j, L)) * L + k] +
                       lat[((size_t)i * L + j) * L + wrap_inc(k, L)]);
        } else {
            const int i = (int)(x / L), j = (int)(x % L);
            const int id = wrap_inc(i, L), jr = wrap_inc(j, L), jl = wrap_dec(j, L);
            e1 -= s * (lat[(size_t)id * L + j] + lat[(size_t)i * L + jr]);
            if (kStencil == SPIN_STENCIL_TRIANGULAR) e1 -= s * lat[(size_t)id * L + jr];
            else e2 -= s * (lat[(size_t)id * L + jl] + lat[(size_t)id * L + jr]);
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        e1 += __shfl_xor_sync(0xFFFFFFFFu, e1, o);
        e2 += __shfl_xor_sync(0xFFFFFFFFu, e2, o);
        m += __shfl_xor_sync(0xFFFFFFFFu, m, o);
    }
    if ((threadIdx.x & 31) == 0) { sh[0][threadIdx.x >> 5] = e1; sh[1][threadIdx.x >> 5] = e2; sh[2][threadIdx.x >> 5] = m; }
    __syncthreads();
    if (threadIdx.x < 3) {
        long long t = 0;
        for (int k = 0; k < (int)(blockDim.x >> 5); ++k) t += sh[threadIdx.x][k];
        atomicAdd((unsigned long long*)acc + 3 * b + threadIdx.x, (unsigned long long)t);
    }
}

// ---- scratch of spin_stencil_observables_noalloc: the accumulators the reduction kernel adds into, in a file-scope device
// array (every GPU that loads the library holds these 96 KiB until exit) instead of a per-call allocation.  In HOST code
// the name g_noalloc_acc is a stand-in, not a device address: the launcher below asks cudaGetSymbolAddress for the
// address, once per device, with that device current.
constexpr int kNoAllocMaxBatch = 4096;
static __device__ __align__(256) long long g_noalloc_acc[3 * kNoAllocMaxBatch];

// acc[3 b + {0, 1, 2}] -> E1[b], E2[b], M[b] (device outputs, any may be NULL).
__global__ void stencil_noalloc_scatter_kernel(const long long* __restrict__ acc, int batch, long long* E1, long long* E2,
                                               long long* M) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= batch) return;
    if (E1) E1[b] = acc[3 * b];
    if (E2) E2[b] = acc[3 * b + 1];
    if (M) M[b] = acc[3 * b + 2];
}

constexpr int kNoAllocMaxDevices = 64;
long long* g_noalloc_ptr[kNoAllocMaxDevices] = {};     // device address of g_noalloc_acc on device d, once looked up

int stencil_fail(int code, const char* msg) { return set_error(code, msg); }

int check_shape(int32_t stencil, int32_t batch, int32_t L) {
    if (batch < 1) return stencil_fail(SPIN_ERR_INVALID, "spin_stencil: batch must be >= 1");
    if (stencil == SPIN_STENCIL_TRIANGULAR) {
        if (L < 3 || L % 3 != 0 || L > 65535) return stencil_fail(SPIN_ERR_INVALID, "spin_stencil: the triangular lattice needs L % 3 == 0 (three colours on a periodic lattice), 3 <= L <= 65535");
    } else if (stencil == SPIN_STENCIL_CUBIC) {
        if (L < 2 || (L & 1) || L > 1624) return stencil_fail(SPIN_ERR_INVALID, "spin_stencil: the cubic lattice needs even L, 2 <= L <= 1624");
    } else if (stencil == SPIN_STENCIL_SQUARE_NNN) {
        if (L < 2 || (L & 1) || L > 65536) return stencil_fail(SPIN_ERR_INVALID, "spin_stencil: the second-neighbour square lattice needs even L, 2 <= L <= 65536");
    } else return stencil_fail(SPIN_ERR_INVALID, "spin_stencil: unknown stencil");
    return SPIN_OK;
}

long long total_sites(int stencil, int L) { return stencil == SPIN_STENCIL_CUBIC ? (long long)L * L * L : (long long)L * L; }
int n_colours(int stencil) { return stencil == SPIN_STENCIL_TRIANGULAR ? 3 : stencil == SPIN_STENCIL_CUBIC ? 2 : 4; }

RoundKeys keys_for(uint64_t seed) {
    RoundKeys rk;
    uint32_t k0 = (uint32_t)(seed & 0xFFFFFFFFull), k1 = (uint32_t)(seed >> 32);
    for (int r = 0; r < 10; ++r) { rk.k0[r] = k0; rk.k1[r] = k1; k0 += kPhiloxW0; k1 += kPhiloxW1; }
    return rk;
}

}  // namespace
}  // namespace spin

using namespace spin;

extern "C" {

size_t spin_stencil_sites(int32_t stencil, int32_t L) {
    if (check_shape(stencil, 1, L) != SPIN_OK) return 0;
    return (size_t)total_sites(stencil, L);
}

int spin_stencil_init(int32_t stencil, int32_t batch, int32_t L, int8_t* lattice, uint64_t seed, int64_t replica_offset,
                      void* cuda_stream) {
    const int rc = check_shape(stencil, batch, L);
    if (rc != SPIN_OK) return rc;
    if (!lattice) return stencil_fail(SPIN_ERR_INVALID, "spin_stencil_init: NULL lattice");
    if (replica_offset < 0 || replica_offset + (int64_t)batch > (1ll << 32)) return stencil_fail(SPIN_ERR_INVALID, "spin_stencil: replica_offset + batch must stay within [0, 2^32]");
    const long long N = total_sites(stencil, L), total = ((N + 3) >> 2) * batch;
    stencil_init_kernel<<<(unsigned)((total + 255) / 256), 256, 0, (cudaStream_t)cuda_stream>>>(lattice, N, batch, (uint32_t)replica_offset, keys_for(seed));
    const cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? SPIN_OK : stencil_fail(SPIN_ERR_CUDA, cudaGetErrorString(e));
}

int spin_stencil_sweep(int32_t stencil, int32_t batch, int32_t L, int8_t* lattice, const double* beta, double J1, double J2,
                       double h, uint64_t seed, int64_t replica_offset, int64_t n_sweeps, int64_t sweep_offset, void* cuda_stream) {
    const int rc = check_shape(stencil, batch, L);
    if (rc != SPIN_OK) return rc;
    if (!lattice || !beta) return stencil_fail(SPIN_ERR_INVALID, "spin_stencil_sweep: NULL argument");
    if (!std::isfinite(J1) || !std::isfinite(J2) || !std::isfinite(h)) return stencil_fail(SPIN_ERR_INVALID, "spin_stencil_sweep: J1, J2 and h must be finite");
    for (int b = 0; b < batch; ++b)
        if (!std::isfinite(beta[b]) || beta[b] < 0.0) return stencil_fail(SPIN_ERR_INVALID, "spin_stencil_sweep: beta must be finite and >= 0");
    if (replica_offset < 0 || replica_offset + (int64_t)batch > (1ll << 32)) return stencil_fail(SPIN_ERR_INVALID, "spin_stencil: replica_offset + batch must stay within [0, 2^32]");
    if (n_sweeps < 0 || sweep_offset < 0 || sweep_offset > (1ll << 56) || n_sweeps > (1ll << 56) || sweep_offset + n_sweeps > (1ll << 56))
        return stencil_fail(SPIN_ERR_INVALID, "spin_stencil_sweep: sweep range must lie in [0, 2^56]");
    if (n_sweeps == 0) return SPIN_OK;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    // class table per replica: dE = 2 s (J1 nn1 + J2 nn2 + h), nn = (number of neighbours) - 2 (number of -1 neighbours)
    const int n1 = stencil == SPIN_STENCIL_SQUARE_NNN ? 4 : 6, n2 = stencil == SPIN_STENCIL_SQUARE_NNN ? 4 : 0;
    std::vector<uint32_t> rec;
    try { rec.assign((size_t)batch * kStencilRec, 0u); } catch (...) { return stencil_fail(SPIN_ERR_NOMEM, "spin_stencil_sweep: out of host memory"); }
    for (int b = 0; b < batch; ++b) {
        uint32_t* r = rec.data() + (size_t)b * kStencilRec;
        unsigned long long always = 0ull;
        for (int d = 0; d < 2; ++d)
            for (int nd1 = 0; nd1 <= n1; ++nd1)
                for (int nd2 = 0; nd2 <= n2; ++nd2) {
                    const int idx = d * (n1 + 1) * (n2 + 1) + nd1 * (n2 + 1) + nd2;
                    const double sgn = d ? -1.0 : 1.0;
                    const double dE = 2.0 * sgn * (J1 * (double)(n1 - 2 * nd1) + J2 * (double)(n2 - 2 * nd2) + h);
                    uint32_t T[1];
                    uint8_t al[1];
                    // the arithmetic of row a1 (spin_threshold_table): a one-class "Potts table" with dn = -dE, J = 1
                    const double x = beta[b] * dE;
                    if (x <= 0.0) { al[0] = 1; T[0] = 0xFFFFFFFFu; }
                    else {
                        const double v = std::floor(std::exp(-x) * 4294967296.0);
                        al[0] = 0;
                        T[0] = v >= 4294967295.0 ? 0xFFFFFFFFu : (uint32_t)v;
                    }
                    r[idx] = T[0];
                    if (al[0]) always |= 1ull << idx;
                }
        r[62] = (uint32_t)always;
        r[63] = (uint32_t)(always >> 32);
    }
    uint32_t* d_tab = nullptr;
    cudaError_t e = cudaMallocAsync(&d_tab, rec.size() * sizeof(uint32_t), s);
    if (e != cudaSuccess) return stencil_fail(SPIN_ERR_CUDA, cudaGetErrorString(e));
    e = cudaMemcpyAsync(d_tab, rec.data(), rec.size() * sizeof(uint32_t), cudaMemcpyHostToDevice, s);   // pageable: staged before return
    StencilArgs a;
    a.lattice = lattice; a.tables = d_tab; a.stencil = stencil; a.batch = batch; a.L = L;
    a.replica_offset = (uint32_t)replica_offset; a.rk = keys_for(seed);
    const long long total = ((colour_sites(stencil, L) + 3) >> 2) * batch;
    const unsigned grid = (unsigned)((total + 127) / 128);
    const int nc = n_colours(stencil);
    for (int64_t t = sweep_offset; t < sweep_offset + n_sweeps && e == cudaSuccess; ++t)
        for (int c = 0; c < nc; ++c) {
            a.colour = c;
            a.c2 = (uint32_t)((uint64_t)t & 0xFFFFFFFFull);
            a.c3 = (uint32_t)(((uint64_t)t >> 32) & 0xFFFFFFull) | ((uint32_t)c << 24) | (kDomainStencil << 28);
            if (stencil == SPIN_STENCIL_TRIANGULAR && L % 12 == 0) {
                const long long chunks = (long long)L * (L / 12) * batch;
                // 12 or 6 rows per thread (L % 12 == 0): the longer march when it still gives every SM several blocks.
                // (kUniform: the threads of one replica fill whole blocks, so a block's table comes from shared memory;
                // the colour is a template parameter: see the kernel)
                typedef void (*Kern)(StencilArgs);
                static const Kern k12[2][3] = {{triangular_march_vec_kernel<12, false, 0>, triangular_march_vec_kernel<12, false, 1>,
                                                triangular_march_vec_kernel<12, false, 2>},
                                               {triangular_march_vec_kernel<12, true, 0>, triangular_march_vec_kernel<12, true, 1>,
                                                triangular_march_vec_kernel<12, true, 2>}};
                static const Kern k6[2][3] = {{triangular_march_vec_kernel<6, false, 0>, triangular_march_vec_kernel<6, false, 1>,
                                               triangular_march_vec_kernel<6, false, 2>},
                                              {triangular_march_vec_kernel<6, true, 0>, triangular_march_vec_kernel<6, true, 1>,
                                               triangular_march_vec_kernel<6, true, 2>}};
                if (chunks / 12 >= 148ll * 8 * 128) {
                    const bool uni = ((long long)(L / 12) * (L / 12)) % 128 == 0;
                    launch_pdl(k12[uni][c], (unsigned)((chunks / 12 + 127) / 128), 128u, s, a);
                } else {
                    const bool uni = ((long long)(L / 6) * (L / 12)) % 128 == 0;
                    launch_pdl(k6[uni][c], (unsigned)((chunks / 6 + 127) / 128), 128u, s, a);
                }
            } else if (stencil == SPIN_STENCIL_TRIANGULAR) launch_pdl(stencil_pass_kernel<SPIN_STENCIL_TRIANGULAR>, grid, 128u, s, a);
            else if (stencil == SPIN_STENCIL_CUBIC && L % 16 == 0) {
                const long long words = (long long)L * L * (L >> 4) * batch;
                const bool uni = ((long long)(L / 4) * L * (L >> 4)) % 128 == 0;
                launch_pdl(uni ? cubic_march_vec_kernel<4, true> : cubic_march_vec_kernel<4, false>,
                           (unsigned)((words / 4 + 127) / 128), 128u, s, a);   // 4 planes per thread (8: 407 flips/ns)
            } else if (stencil == SPIN_STENCIL_CUBIC) launch_pdl(stencil_pass_kernel<SPIN_STENCIL_CUBIC>, grid, 128u, s, a);
            else if (L % 16 == 0) {
                const long long words = (long long)(L >> 1) * (L >> 4) * batch;
                const bool uni = ((long long)(L / 8) * (L >> 4)) % 128 == 0;
                launch_pdl(uni ? nnn_march_vec_kernel<4, true> : nnn_march_vec_kernel<4, false>,
                           (unsigned)((words / 4 + 127) / 128), 128u, s, a);
            } else launch_pdl(stencil_pass_kernel<SPIN_STENCIL_SQUARE_NNN>, grid, 128u, s, a);
        }
    if (e == cudaSuccess) e = cudaGetLastError();
    cudaFreeAsync(d_tab, s);
    return e == cudaSuccess ? SPIN_OK : stencil_fail(SPIN_ERR_CUDA, cudaGetErrorString(e));
}

int spin_stencil_observables(int32_t stencil, int32_t batch, int32_t L, const int8_t* lattice, int64_t* E1, int64_t* E2,
                             int64_t* M, void* cuda_stream) {
    const int rc = check_shape(stencil, batch, L);
    if (rc != SPIN_OK) return rc;
    if (!lattice) return stencil_fail(SPIN_ERR_INVALID, "spin_stencil_observables: NULL lattice");
    cudaStream_t s = (cudaStream_t)cuda_stream;
    long long* d_acc = nullptr;
    std::vector<long long> host;
    try { host.assign((size_t)batch * 3, 0); } catch (...) { return stencil_fail(SPIN_ERR_NOMEM, "spin_stencil_observables: out of host memory"); }
    cudaError_t e = cudaMallocAsync(&d_acc, sizeof(long long) * 3 * batch, s);
    if (e != cudaSuccess) return stencil_fail(SPIN_ERR_CUDA, cudaGetErrorString(e));
    e = cudaMemsetAsync(d_acc, 0, sizeof(long long) * 3 * batch, s);
    const long long N = total_sites(stencil, L);
    long long want = (N + 255) / 256, cap = (148ll * 16 + batch - 1) / batch;
    const int bpr = (int)(want < cap ? want : (cap < 1 ? 1 : cap));
    const unsigned grid = (unsigned)((long long)bpr * batch);
    if (stencil == SPIN_STENCIL_TRIANGULAR) stencil_observe_kernel<SPIN_STENCIL_TRIANGULAR><<<grid, 256, 0, s>>>(lattice, L, bpr, d_acc);
    else if (stencil == SPIN_STENCIL_CUBIC) stencil_observe_kernel<SPIN_STENCIL_CUBIC><<<grid, 256, 0, s>>>(lattice, L, bpr, d_acc);
    else stencil_observe_kernel<SPIN_STENCIL_SQUARE_NNN><<<grid, 256, 0, s>>>(lattice, L, bpr, d_acc);
    if (e == cudaSuccess) e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaMemcpyAsync(host.data(), d_acc, sizeof(long long) * 3 * batch, cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    cudaFreeAsync(d_acc, s);
    if (e != cudaSuccess) return stencil_fail(SPIN_ERR_CUDA, cudaGetErrorString(e));
    for (int b = 0; b < batch; ++b) {
        if (E1) E1[b] = host[3 * b];
        if (E2) E2[b] = host[3 * b + 1];
        if (M) M[b] = host[3 * b + 2];
    }
    return SPIN_OK;
}

int spin_stencil_observables_noalloc(int32_t stencil, int32_t batch, int32_t L, const int8_t* lattice, int64_t* E1_dev,
                                     int64_t* E2_dev, int64_t* M_dev, void* cuda_stream) {
    const int rc = check_shape(stencil, batch, L);
    if (rc != SPIN_OK) return rc;
    if (!lattice) return stencil_fail(SPIN_ERR_INVALID, "spin_stencil_observables_noalloc: NULL lattice");
    if (batch > kNoAllocMaxBatch)
        return stencil_fail(SPIN_ERR_INVALID, "spin_stencil_observables_noalloc: batch exceeds the fixed scratch (at most 4096 replicas "
                                              "per call); split the batch or use spin_stencil_observables");
    cudaStream_t s = (cudaStream_t)cuda_stream;
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return stencil_fail(SPIN_ERR_CUDA, cudaGetErrorString(e));
    if (dev < 0 || dev >= kNoAllocMaxDevices) return stencil_fail(SPIN_ERR_UNSUPPORTED, "spin_stencil_observables_noalloc: device ordinal >= 64");
    long long* acc = g_noalloc_ptr[dev];
    if (!acc) {
        // once per device, with that device current (two threads racing here store the same address)
        e = cudaGetSymbolAddress((void**)&acc, g_noalloc_acc);
        if (e != cudaSuccess || !acc) return stencil_fail(SPIN_ERR_CUDA, e != cudaSuccess ? cudaGetErrorString(e) : "cudaGetSymbolAddress returned NULL");
        g_noalloc_ptr[dev] = acc;
    }
    // the array keeps the previous call's sums and the kernel accumulates: clear this call's part first
    e = cudaMemsetAsync(acc, 0, sizeof(long long) * 3 * (size_t)batch, s);
    if (e != cudaSuccess) return stencil_fail(SPIN_ERR_CUDA, cudaGetErrorString(e));
    const long long N = total_sites(stencil, L);
    long long want = (N + 255) / 256, cap = (148ll * 16 + batch - 1) / batch;
    const int bpr = (int)(want < cap ? want : (cap < 1 ? 1 : cap));
    const unsigned grid = (unsigned)((long long)bpr * batch);
    if (stencil == SPIN_STENCIL_TRIANGULAR) stencil_observe_kernel<SPIN_STENCIL_TRIANGULAR><<<grid, 256, 0, s>>>(lattice, L, bpr, acc);
    else if (stencil == SPIN_STENCIL_CUBIC) stencil_observe_kernel<SPIN_STENCIL_CUBIC><<<grid, 256, 0, s>>>(lattice, L, bpr, acc);
    else stencil_observe_kernel<SPIN_STENCIL_SQUARE_NNN><<<grid, 256, 0, s>>>(lattice, L, bpr, acc);
    stencil_noalloc_scatter_kernel<<<(unsigned)((batch + 127) / 128), 128, 0, s>>>(acc, batch, (long long*)E1_dev, (long long*)E2_dev,
                                                                                 (long long*)M_dev);
    e = cudaGetLastError();
    return e == cudaSuccess ? SPIN_OK : stencil_fail(SPIN_ERR_CUDA, cudaGetErrorString(e));
}


}  // extern "C"
