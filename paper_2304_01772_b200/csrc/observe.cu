// observe.cu — rows a5-a7: exact integer per-replica reductions.
//   Ising: E_int = -sum_bonds s_i s_j, M = sum s.  Every bond of an even periodic lattice has exactly one
//          colour-0 end, so E_int = -sum_{colour-0 sites} s * (up + down + left + right)  (the
//          Hamiltonian is the neighbour-sum map times the lattice; each bond once, P2).
//   Potts: E_int = -sum_{colour-0 sites} #(neighbours equal), M = max_k N_k (P8).
//   Moments: n, sum E, sum E^2 (128 bit), sum M, sum |M|, sum M^2, sum E*M.
// Warp-shuffle + shared-memory block reduction, one 64-bit atomic per block and quantity.
#include "spin_internal.cuh"

namespace spin {

namespace {

__device__ __forceinline__ int warp_sum(int v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, o);
    return v;
}

// Block-reduce two ints and add them to 64-bit accumulators.  All threads of the block must call.
__device__ __forceinline__ void block_add2(int e, int m, long long* E_acc, long long* M_acc) {
    __shared__ int se[32], sm[32];
    e = warp_sum(e);
    m = warp_sum(m);
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    if (lane == 0) { se[w] = e; sm[w] = m; }
    __syncthreads();
    if (w == 0) {
        const int nw = (blockDim.x + 31) >> 5;
        e = lane < nw ? se[lane] : 0;
        m = lane < nw ? sm[lane] : 0;
        e = warp_sum(e);
        m = warp_sum(m);
        if (lane == 0) {
            if (E_acc && e) atomicAdd((unsigned long long*)E_acc, (unsigned long long)(long long)e);
            if (M_acc && m) atomicAdd((unsigned long long*)M_acc, (unsigned long long)(long long)m);
        }
    }
}

// Ising int8, any even L: one thread per row-pair position; grid = (blocks per replica) * batch.
// Thread handles column index k of row i for both colours.
__global__ void ising_int8_observe_kernel(const int8_t* __restrict__ lat, int L, int bpr, long long* E_acc,
                                          long long* M_acc) {
    const int W = L >> 1;
    const int b = blockIdx.x / bpr, blk = blockIdx.x - b * bpr;
    const size_t half = (size_t)L * W;
    const int8_t* c0 = lat + (size_t)b * 2 * half;
    const int8_t* c1 = c0 + half;
    int e = 0, m = 0;
    for (long long n = (long long)blk * blockDim.x + threadIdx.x; n < (long long)half; n += (long long)bpr * blockDim.x) {
        const int i = (int)(n / W), k = (int)(n % W);
        const int p = i & 1;                                  // colour 0: column parity = row parity
        const int iu = i == 0 ? L - 1 : i - 1, id = i == L - 1 ? 0 : i + 1;
        const int ks = p ? (k == W - 1 ? 0 : k + 1) : (k == 0 ? W - 1 : k - 1);
        const int s = c0[n];
        const int nn = c1[(size_t)iu * W + k] + c1[(size_t)id * W + k] + c1[(size_t)i * W + k] + c1[(size_t)i * W + ks];
        e -= s * nn;
        m += s + c1[n];
    }
    block_add2(e, m, E_acc ? E_acc + b : nullptr, M_acc ? M_acc + b : nullptr);
}

// Ising int8, L % 32 == 0: one thread per 16-site strip of a colour-0 row, 128-bit loads, byte-SIMD.
// For +-1 bytes own ^ nbr is 0x00 (equal) or 0xFE (different): s * nbr summed over a strip and its 4 neighbours is
// 64 - 2 * #different; the number of -1 spins of a word is popc(word & 0x80808080).
__global__ void __launch_bounds__(256) ising_int8_observe_vec_kernel(const int8_t* __restrict__ lat, int L, int bpr,
                                                                     long long* E_acc, long long* M_acc) {
    const int W = L >> 1, W16 = W >> 4, W4 = W >> 2;
    const int b = blockIdx.x / bpr, blk = blockIdx.x - b * bpr;
    const size_t half = (size_t)L * W;
    const uint4* c0 = (const uint4*)(lat + (size_t)b * 2 * half);
    const uint4* c1 = (const uint4*)(lat + (size_t)b * 2 * half + half);
    const uint32_t* c1w = (const uint32_t*)c1;
    const int strips = L * W16;
    int diff = 0, neg = 0, cnt = 0;
    for (int n = blk * blockDim.x + threadIdx.x; n < strips; n += bpr * blockDim.x) {
        const int i = n / W16, x = n - i * W16;
        const int iu = i == 0 ? L - 1 : i - 1, id = i == L - 1 ? 0 : i + 1;
        const uint4 own = __ldg(c0 + n), ct = __ldg(c1 + n);
        const uint4 up = __ldg(c1 + (size_t)iu * W16 + x), dn = __ldg(c1 + (size_t)id * W16 + x);
        uint32_t s0, s1, s2, s3;
        if (i & 1) {                                           // colour 0: side neighbour is other[i][k+1] on odd rows
            const uint32_t e = __ldg(c1w + (size_t)i * W4 + (x == W16 - 1 ? 0 : 4 * x + 4));
            s0 = __byte_perm(ct.x, ct.y, 0x4321); s1 = __byte_perm(ct.y, ct.z, 0x4321);
            s2 = __byte_perm(ct.z, ct.w, 0x4321); s3 = __byte_perm(ct.w, e, 0x4321);
        } else {
            const uint32_t e = __ldg(c1w + (size_t)i * W4 + (x == 0 ? W4 - 1 : 4 * x - 1));
            s0 = __byte_perm(e, ct.x, 0x6543); s1 = __byte_perm(ct.x, ct.y, 0x6543);
            s2 = __byte_perm(ct.y, ct.z, 0x6543); s3 = __byte_perm(ct.z, ct.w, 0x6543);
        }
        const uint32_t m2 = 0x02020202u, m8 = 0x80808080u;
        diff += __popc((own.x ^ up.x) & m2) + __popc((own.x ^ dn.x) & m2) + __popc((own.x ^ ct.x) & m2) + __popc((own.x ^ s0) & m2);
        diff += __popc((own.y ^ up.y) & m2) + __popc((own.y ^ dn.y) & m2) + __popc((own.y ^ ct.y) & m2) + __popc((own.y ^ s1) & m2);
        diff += __popc((own.z ^ up.z) & m2) + __popc((own.z ^ dn.z) & m2) + __popc((own.z ^ ct.z) & m2) + __popc((own.z ^ s2) & m2);
        diff += __popc((own.w ^ up.w) & m2) + __popc((own.w ^ dn.w) & m2) + __popc((own.w ^ ct.w) & m2) + __popc((own.w ^ s3) & m2);
        neg += __popc(own.x & m8) + __popc(own.y & m8) + __popc(own.z & m8) + __popc(own.w & m8);
        neg += __popc(ct.x & m8) + __popc(ct.y & m8) + __popc(ct.z & m8) + __popc(ct.w & m8);
        ++cnt;
    }
    // per strip: 16 sites x 4 bonds, and 32 spins (both colours)
    block_add2(-(64 * cnt - 2 * diff), 32 * cnt - 2 * neg, E_acc ? E_acc + b : nullptr, M_acc ? M_acc + b : nullptr);
}

// bonds (or nullptr): sign planes of the +-J couplings, [B][2][4][L][L/64]; only the colour-0 planes are read.
__global__ void ising_bits_observe_kernel(const uint32_t* __restrict__ lat, const uint32_t* __restrict__ bonds, int L,
                                          int bpr, long long* E_acc, long long* M_acc) {
    const int WW = L >> 6;
    const int b = blockIdx.x / bpr, blk = blockIdx.x - b * bpr;
    const size_t half = (size_t)L * WW;
    const uint32_t* c0 = lat + (size_t)b * 2 * half;
    const uint32_t* c1 = c0 + half;
    int e = 0, m = 0;
    for (long long n = (long long)blk * blockDim.x + threadIdx.x; n < (long long)half; n += (long long)bpr * blockDim.x) {
        const int i = (int)(n / WW), x = (int)(n % WW);
        const int iu = i == 0 ? L - 1 : i - 1, id = i == L - 1 ? 0 : i + 1;
        const uint32_t own = c0[n], ct = c1[(size_t)i * WW + x];
        uint32_t sd;
        if (i & 1) sd = (ct >> 1) | (c1[(size_t)i * WW + (x == WW - 1 ? 0 : x + 1)] << 31);
        else sd = (ct << 1) | (c1[(size_t)i * WW + (x == 0 ? WW - 1 : x - 1)] >> 31);
        // s * nbr = +1 if equal, -1 if different: sum over 32 sites and 4 neighbours = 128 - 2 * (#different);
        // with bond signs J s s' = -1 iff (s differs from s') xor (bond is -1)
        uint32_t bu = 0u, bd = 0u, bc = 0u, bs = 0u;
        if (bonds) {
            const uint32_t* pb = bonds + (size_t)b * 2 * 4 * half + n;
            bu = pb[0]; bd = pb[half]; bc = pb[2 * half]; bs = pb[3 * half];
        }
        const int diff = __popc(own ^ c1[(size_t)iu * WW + x] ^ bu) + __popc(own ^ c1[(size_t)id * WW + x] ^ bd) +
                         __popc(own ^ ct ^ bc) + __popc(own ^ sd ^ bs);
        e -= 128 - 2 * diff;
        m += 64 - 2 * (__popc(own) + __popc(c1[n]));
    }
    block_add2(e, m, E_acc ? E_acc + b : nullptr, M_acc ? M_acc + b : nullptr);
}

__global__ void potts_int8_observe_kernel(const uint8_t* __restrict__ lat, int L, int bpr, long long* E_acc,
                                          unsigned int* hist) {
    __shared__ unsigned int sh[128];
    const int W = L >> 1;
    const int b = blockIdx.x / bpr, blk = blockIdx.x - b * bpr;
    const size_t half = (size_t)L * W;
    const uint8_t* c0 = lat + (size_t)b * 2 * half;
    const uint8_t* c1 = c0 + half;
    for (int t = threadIdx.x; t < 128; t += blockDim.x) sh[t] = 0u;
    __syncthreads();
    int e = 0;
    for (long long n = (long long)blk * blockDim.x + threadIdx.x; n < (long long)half; n += (long long)bpr * blockDim.x) {
        const int i = (int)(n / W), k = (int)(n % W);
        const int p = i & 1;
        const int iu = i == 0 ? L - 1 : i - 1, id = i == L - 1 ? 0 : i + 1;
        const int ks = p ? (k == W - 1 ? 0 : k + 1) : (k == 0 ? W - 1 : k - 1);
        const unsigned s = c0[n];
        e -= (c1[(size_t)iu * W + k] == s) + (c1[(size_t)id * W + k] == s) + (c1[(size_t)i * W + k] == s) +
             (c1[(size_t)i * W + ks] == s);
        if (hist) {
            atomicAdd(&sh[s & 127u], 1u);
            atomicAdd(&sh[c1[n] & 127u], 1u);
        }
    }
    __syncthreads();
    if (hist)
        for (int t = threadIdx.x; t < 128; t += blockDim.x)
            if (sh[t]) atomicAdd(&hist[(size_t)b * 128 + t], sh[t]);
    block_add2(e, 0, E_acc ? E_acc + b : nullptr, nullptr);
}

// Potts uint8, L % 32 == 0: one thread per 16-site strip of a colour-0 row (128-bit loads, byte-SIMD).  States are
// < 128, so bit 7 of (a ^ b) + 0x7F is "a != b" per byte.  The histogram is counted in registers by comparing whole
// words with each state when q <= 8 (no shared-memory atomics on a handful of hot bins), else with shared atomics.
__device__ __forceinline__ int neq_count(uint32_t a, uint32_t b) {
    return __popc(((a ^ b) + 0x7F7F7F7Fu) & 0x80808080u);
}

__global__ void __launch_bounds__(256) potts_int8_observe_vec_kernel(const uint8_t* __restrict__ lat, int L, int bpr,
                                                                     const int32_t* __restrict__ qv, long long* E_acc,
                                                                     unsigned int* hist) {
    __shared__ unsigned int sh[128];
    const int W = L >> 1, W16 = W >> 4, W4 = W >> 2;
    const int b = blockIdx.x / bpr, blk = blockIdx.x - b * bpr;
    const size_t half = (size_t)L * W;
    const uint4* c0 = (const uint4*)(lat + (size_t)b * 2 * half);
    const uint4* c1 = (const uint4*)(lat + (size_t)b * 2 * half + half);
    const uint32_t* c1w = (const uint32_t*)c1;
    const int q = qv[b];
    const bool small = q <= 8;
    for (int t = threadIdx.x; t < 128; t += blockDim.x) sh[t] = 0u;
    __syncthreads();
    const int strips = L * W16;
    int diff = 0, cnt = 0;
    int hk[8] = {0, 0, 0, 0, 0, 0, 0, 0};                    // sites NOT in state k (q <= 8)
    for (int n = blk * blockDim.x + threadIdx.x; n < strips; n += bpr * blockDim.x) {
        const int i = n / W16, x = n - i * W16;
        const int iu = i == 0 ? L - 1 : i - 1, id = i == L - 1 ? 0 : i + 1;
        const uint4 own = __ldg(c0 + n), ct = __ldg(c1 + n);
        const uint4 up = __ldg(c1 + (size_t)iu * W16 + x), dn = __ldg(c1 + (size_t)id * W16 + x);
        uint32_t s0, s1, s2, s3;
        if (i & 1) {
            const uint32_t e = __ldg(c1w + (size_t)i * W4 + (x == W16 - 1 ? 0 : 4 * x + 4));
            s0 = __byte_perm(ct.x, ct.y, 0x4321); s1 = __byte_perm(ct.y, ct.z, 0x4321);
            s2 = __byte_perm(ct.z, ct.w, 0x4321); s3 = __byte_perm(ct.w, e, 0x4321);
        } else {
            const uint32_t e = __ldg(c1w + (size_t)i * W4 + (x == 0 ? W4 - 1 : 4 * x - 1));
            s0 = __byte_perm(e, ct.x, 0x6543); s1 = __byte_perm(ct.x, ct.y, 0x6543);
            s2 = __byte_perm(ct.y, ct.z, 0x6543); s3 = __byte_perm(ct.z, ct.w, 0x6543);
        }
        diff += neq_count(own.x, up.x) + neq_count(own.x, dn.x) + neq_count(own.x, ct.x) + neq_count(own.x, s0);
        diff += neq_count(own.y, up.y) + neq_count(own.y, dn.y) + neq_count(own.y, ct.y) + neq_count(own.y, s1);
        diff += neq_count(own.z, up.z) + neq_count(own.z, dn.z) + neq_count(own.z, ct.z) + neq_count(own.z, s2);
        diff += neq_count(own.w, up.w) + neq_count(own.w, dn.w) + neq_count(own.w, ct.w) + neq_count(own.w, s3);
        ++cnt;
        if (hist) {
            const uint32_t w[8] = {own.x, own.y, own.z, own.w, ct.x, ct.y, ct.z, ct.w};
            if (small) {
#pragma unroll
                for (int k = 0; k < 8; ++k) {
                    if (k >= q) break;                        // block-uniform
                    const uint32_t kk = 0x01010101u * (uint32_t)k;
#pragma unroll
                    for (int j = 0; j < 8; ++j) hk[k] += neq_count(w[j], kk);
                }
            } else {
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    atomicAdd(&sh[w[j] & 127u], 1u);
                    atomicAdd(&sh[(w[j] >> 8) & 127u], 1u);
                    atomicAdd(&sh[(w[j] >> 16) & 127u], 1u);
                    atomicAdd(&sh[(w[j] >> 24) & 127u], 1u);
                }
            }
        }
    }
    if (hist && small) {
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            int v = k < q ? 32 * cnt - hk[k] : 0;             // sites in state k
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, o);
            if ((threadIdx.x & 31) == 0 && v) atomicAdd(&sh[k], (unsigned int)v);
        }
    }
    __syncthreads();
    if (hist)
        for (int t = threadIdx.x; t < 128; t += blockDim.x)
            if (sh[t]) atomicAdd(&hist[(size_t)b * 128 + t], sh[t]);
    // per strip: 16 sites x 4 bonds; E_int = -(#equal bonds)
    block_add2(-(64 * cnt - diff), 0, E_acc ? E_acc + b : nullptr, nullptr);
}

__global__ void potts_finalize_kernel(unsigned int* hist, const int32_t* __restrict__ q, int batch, long long* M_out) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= batch) return;
    unsigned int best = 0u;
    for (int k = 0; k < 128; ++k) {
        const unsigned int v = hist[(size_t)b * 128 + k];
        if (k < q[b] && v > best) best = v;
        hist[(size_t)b * 128 + k] = 0u;
    }
    if (M_out) M_out[b] = (long long)best;
}

__global__ void accumulate_moments_kernel(long long* moments, const long long* __restrict__ E,
                                          const long long* __restrict__ M, int batch) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= batch) return;
    long long* m = moments + 8 * (size_t)b;
    const long long e = E[b], mag = M[b];
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

inline int blocks_per_replica(long long items, int tpb, int batch) {
    // enough blocks to fill the GPU a few times over, but never more than the work
    long long want = (items + tpb - 1) / tpb;
    long long cap = (148ll * 16 + batch - 1) / batch;
    if (cap < 1) cap = 1;
    return (int)(want < cap ? want : cap);
}

}  // namespace

int launch_ising_int8_observe(const void* lattice, int batch, int L, long long* E_acc, long long* M_acc, cudaStream_t s) {
    if (L % 32 == 0) {
        const long long strips = (long long)L * (L >> 5);
        const int tpb = 256, bpr = blocks_per_replica(strips, tpb, batch);
        ising_int8_observe_vec_kernel<<<(unsigned)((long long)bpr * batch), tpb, 0, s>>>((const int8_t*)lattice, L, bpr, E_acc, M_acc);
        return 1;
    }
    const long long half = (long long)L * (L >> 1);
    const int tpb = 256, bpr = blocks_per_replica(half, tpb, batch);
    ising_int8_observe_kernel<<<(unsigned)((long long)bpr * batch), tpb, 0, s>>>((const int8_t*)lattice, L, bpr, E_acc, M_acc);
    return 1;
}

int launch_ising_bits_observe(const void* lattice, const uint32_t* bonds, int batch, int L, long long* E_acc,
                              long long* M_acc, cudaStream_t s) {
    const long long half = (long long)L * (L >> 6);
    const int tpb = 256, bpr = blocks_per_replica(half, tpb, batch);
    ising_bits_observe_kernel<<<(unsigned)((long long)bpr * batch), tpb, 0, s>>>((const uint32_t*)lattice, bonds, L, bpr, E_acc, M_acc);
    return 1;
}

int launch_potts_int8_observe(const void* lattice, int batch, int L, const int32_t* q, long long* E_acc,
                              unsigned int* hist, cudaStream_t s) {
    if (L % 32 == 0) {
        const long long strips = (long long)L * (L >> 5);
        const int tpb = 256, bpr = blocks_per_replica(strips, tpb, batch);
        potts_int8_observe_vec_kernel<<<(unsigned)((long long)bpr * batch), tpb, 0, s>>>((const uint8_t*)lattice, L, bpr, q, E_acc, hist);
        return 1;
    }
    const long long half = (long long)L * (L >> 1);
    const int tpb = 256, bpr = blocks_per_replica(half, tpb, batch);
    potts_int8_observe_kernel<<<(unsigned)((long long)bpr * batch), tpb, 0, s>>>((const uint8_t*)lattice, L, bpr, E_acc, hist);
    return 1;
}

int launch_potts_finalize(unsigned int* hist, const int32_t* q, int batch, long long* M_out, cudaStream_t s) {
    potts_finalize_kernel<<<(batch + 127) / 128, 128, 0, s>>>(hist, q, batch, M_out);
    return 1;
}

int launch_accumulate_moments(long long* moments, const long long* E, const long long* M, int batch, cudaStream_t s) {
    accumulate_moments_kernel<<<(batch + 127) / 128, 128, 0, s>>>(moments, E, M, batch);
    return 1;
}

}  // namespace spin
