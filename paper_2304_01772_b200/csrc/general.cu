// general.cu — SURVEY.md section 8(f) #2: the Hamiltonians as the paper writes them, with a coupling per bond and a
// field per site (Eq. 1; Eq. 5 with its field term), on the int8 checkerboard layout.
// These are the general-purpose kernels (one thread per Philox group, byte loads): every shape, every coupling; the
// tuned row-marching kernels stay responsible for the uniform model and the bit-packed +-J glass.
//   * Ising with +-1 bond signs: the bond-weighted neighbour sum is still in {-4..4}, so the 10-class table applies.
//   * Ising with real J_ij and B_i: dE takes 32 values per site (own spin x 16 neighbour configurations); the host
//     evaluates Alg. 1's acceptance for each of them in IEEE double exactly as for the class table (O4) and
//     the kernel looks up thr[site][16 d + cfg]: bit-exact against the oracle by construction, 132 bytes of table per
//     site and replica, HBM-bound.
//   * Potts with a field h on the state label and optional +-1 bond signs: class (dn, new - old), host-built table
//     [9][255] per replica.
#include "spin_internal.cuh"

namespace spin {
namespace {

__device__ __forceinline__ size_t split_index(int b, int L, int i, int j) {
    return (((size_t)b * 2 + ((i + j) & 1)) * L + i) * (size_t)(L >> 1) + (size_t)(j >> 1);
}

// Decodes the thread's Philox group into (replica, first same-colour site); shared by the three kernels.
struct GroupPos {
    int b;
    uint32_t g;
    bool valid;
};
__device__ __forceinline__ GroupPos group_pos(const SweepArgs& a, int sites_per_group) {
    const long long half = (long long)a.L * (a.L >> 1);
    const long long groups = (half + sites_per_group - 1) / sites_per_group;
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    GroupPos p;
    const long long total = groups * a.batch;
    p.valid = gid < total;
    p.b = 0;
    p.g = 0u;
    if (p.valid) {
        if (total <= 0xFFFFFFFFll) {                               // 32-bit division (the 64-bit one costs ~100 instructions)
            const uint32_t ug = (uint32_t)gid, gr = (uint32_t)groups;
            p.b = (int)(ug / gr);
            p.g = ug - (uint32_t)p.b * gr;
        } else {
            p.b = (int)(gid / groups);
            p.g = (uint32_t)(gid % groups);
        }
    }
    return p;
}

// Natural coordinates of same-colour site n of colour c.
__device__ __forceinline__ void site_coords(int L, int colour, long long n, int& i, int& j) {
    const uint32_t W = (uint32_t)L >> 1, un = (uint32_t)n;      // n < L * L / 2 <= 2^31: 32-bit arithmetic, no division for L = 2^k
    const uint32_t row = (W & (W - 1u)) == 0u ? un >> (__ffs((int)W) - 1) : un / W;
    const int k = (int)(un - row * W);
    i = (int)row;
    j = 2 * k + ((i + colour) & 1);
}

__global__ void ising_int8_bonds_kernel(SweepArgs a, const int8_t* __restrict__ Jh, const int8_t* __restrict__ Jv) {
    pdl_wait();   // launched with programmatic stream serialisation: the previous half-sweep must have completed
    const GroupPos p = group_pos(a, 4);
    if (!p.valid) return;
    const int L = a.L;
    const long long half = (long long)L * (L >> 1);
    const uint32_t* tab = a.tables + (size_t)p.b * kTableStride;
    int8_t* lat = (int8_t*)a.lattice;
    const size_t nb = (size_t)p.b * L * L;
    uint32_t r[4];
    philox4x32_10(a.rk, p.g, (uint32_t)p.b + a.replica_offset, a.c2, a.c3, r);
#pragma unroll
    for (int e = 0; e < 4; ++e) {
        const long long n = 4ll * p.g + e;
        if (n >= half) break;
        int i, j;
        site_coords(L, a.colour, n, i, j);
        const int iu = i == 0 ? L - 1 : i - 1, id = i == L - 1 ? 0 : i + 1, jl = j == 0 ? L - 1 : j - 1, jr = j == L - 1 ? 0 : j + 1;
        const size_t own = split_index(p.b, L, i, j);
        const int s = lat[own];
        const int nn = Jv[nb + (size_t)iu * L + j] * lat[split_index(p.b, L, iu, j)] + Jv[nb + (size_t)i * L + j] * lat[split_index(p.b, L, id, j)] +
                       Jh[nb + (size_t)i * L + jl] * lat[split_index(p.b, L, i, jl)] + Jh[nb + (size_t)i * L + j] * lat[split_index(p.b, L, i, jr)];
        const int idx = (s < 0 ? 8 : 0) + ((4 - nn) >> 1);          // d * 8 + (number of -1 bond-weighted neighbours)
        if ((r[e] <= tab[idx]) && !((tab[kTabNever] >> idx) & 1u)) lat[own] = (int8_t)(-s);
    }
}

// thr: [B][L*L][32] uint32 T (accept iff r < T), alw: [B][L*L] bit k = class k always accepts; k = 16 d + cfg,
// cfg bit 0 / 1 / 2 / 3 = the up / down / left / right neighbour is -1.
__global__ void ising_int8_general_kernel(SweepArgs a, const uint32_t* __restrict__ thr, const uint32_t* __restrict__ alw) {
    pdl_wait();   // launched with programmatic stream serialisation: the previous half-sweep must have completed
    const GroupPos p = group_pos(a, 4);
    if (!p.valid) return;
    const int L = a.L;
    const long long half = (long long)L * (L >> 1);
    int8_t* lat = (int8_t*)a.lattice;
    const size_t nb = (size_t)p.b * L * L;
    uint32_t r[4];
    philox4x32_10(a.rk, p.g, (uint32_t)p.b + a.replica_offset, a.c2, a.c3, r);
#pragma unroll
    for (int e = 0; e < 4; ++e) {
        const long long n = 4ll * p.g + e;
        if (n >= half) break;
        int i, j;
        site_coords(L, a.colour, n, i, j);
        const int iu = i == 0 ? L - 1 : i - 1, id = i == L - 1 ? 0 : i + 1, jl = j == 0 ? L - 1 : j - 1, jr = j == L - 1 ? 0 : j + 1;
        const size_t own = split_index(p.b, L, i, j);
        const int s = lat[own];
        const int cfg = (lat[split_index(p.b, L, iu, j)] < 0 ? 1 : 0) | (lat[split_index(p.b, L, id, j)] < 0 ? 2 : 0) |
                        (lat[split_index(p.b, L, i, jl)] < 0 ? 4 : 0) | (lat[split_index(p.b, L, i, jr)] < 0 ? 8 : 0);
        const int k = (s < 0 ? 16 : 0) + cfg;
        const size_t site = nb + (size_t)i * L + j;
        const bool acc = ((alw[site] >> k) & 1u) || r[e] < thr[site * 32 + k];
        if (acc) lat[own] = (int8_t)(-s);
    }
}

// tab2: [B][9][255] entries (always << 32) | T, index (dn + 4) * 255 + (new - old + 127).  Jh / Jv: natural int8 bond
// signs or nullptr.
__global__ void potts_int8_general_kernel(SweepArgs a, const unsigned long long* __restrict__ tab2,
                                          const int8_t* __restrict__ Jh, const int8_t* __restrict__ Jv) {
    pdl_wait();
    const GroupPos p = group_pos(a, 2);
    if (!p.valid) return;
    const int L = a.L;
    const long long half = (long long)L * (L >> 1);
    const uint32_t q = a.tables[(size_t)p.b * kTableStride + kTabQ];
    const unsigned long long* tab = tab2 + (size_t)p.b * 9 * 255;
    uint8_t* lat = (uint8_t*)a.lattice;
    const size_t nb = (size_t)p.b * L * L;
    uint32_t r[4];
    philox4x32_10(a.rk, p.g, (uint32_t)p.b + a.replica_offset, a.c2, a.c3, r);
#pragma unroll
    for (int e = 0; e < 2; ++e) {
        const long long n = 2ll * p.g + e;
        if (n >= half) break;
        int i, j;
        site_coords(L, a.colour, n, i, j);
        const int iu = i == 0 ? L - 1 : i - 1, id = i == L - 1 ? 0 : i + 1, jl = j == 0 ? L - 1 : j - 1, jr = j == L - 1 ? 0 : j + 1;
        const size_t own = split_index(p.b, L, i, j);
        const int old = lat[own];
        int nw = old + 1 + (int)__umulhi(r[2 * e], q - 1u);
        if (nw >= (int)q) nw -= (int)q;
        const int v[4] = {lat[split_index(p.b, L, iu, j)], lat[split_index(p.b, L, id, j)], lat[split_index(p.b, L, i, jl)],
                          lat[split_index(p.b, L, i, jr)]};
        int sg[4] = {1, 1, 1, 1};
        if (Jh) {
            sg[0] = Jv[nb + (size_t)iu * L + j]; sg[1] = Jv[nb + (size_t)i * L + j];
            sg[2] = Jh[nb + (size_t)i * L + jl]; sg[3] = Jh[nb + (size_t)i * L + j];
        }
        int dn = 0;
#pragma unroll
        for (int t = 0; t < 4; ++t) dn += sg[t] * ((int)(v[t] == nw) - (int)(v[t] == old));
        const unsigned long long ent = tab[(dn + 4) * 255 + (nw - old + 127)];
        if ((ent >> 32) || r[2 * e + 1] < (uint32_t)ent) lat[own] = (uint8_t)nw;
    }
}

__device__ __forceinline__ double block_sum_double(double v, double* sh) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, o);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
    __syncthreads();
    double t = 0.0;
    if (threadIdx.x == 0) for (int k = 0; k < (int)(blockDim.x >> 5); ++k) t += sh[k];
    __syncthreads();
    return t;
}

// E[b] += -sum_bonds J_ij s_i s_j - sum_i B_i s_i over the block's sites (double; blocks never straddle replicas).
__global__ void __launch_bounds__(256) ising_general_energy_kernel(const int8_t* __restrict__ lat, const double* __restrict__ Jh,
                                                                   const double* __restrict__ Jv, const double* __restrict__ B,
                                                                   int L, int bpr, double* E) {
    __shared__ double sh[8];
    const int b = blockIdx.x / bpr, blk = blockIdx.x - b * bpr;
    const long long N = (long long)L * L;
    double e = 0.0;
    for (long long x = (long long)blk * blockDim.x + threadIdx.x; x < N; x += (long long)bpr * blockDim.x) {
        const int i = (int)(x / L), j = (int)(x % L);
        const int id = i == L - 1 ? 0 : i + 1, jr = j == L - 1 ? 0 : j + 1;
        const double s = (double)lat[split_index(b, L, i, j)];
        e -= Jh[b * N + x] * s * (double)lat[split_index(b, L, i, jr)];
        e -= Jv[b * N + x] * s * (double)lat[split_index(b, L, id, j)];
        e -= B[b * N + x] * s;
    }
    const double t = block_sum_double(e, sh);
    if (threadIdx.x == 0) atomicAdd(E + b, t);
}

// Potts, natural bond signs (or nullptr): E_acc[b] += -sum_bonds J_ij delta, S_acc[b] += sum of labels.
__global__ void __launch_bounds__(256) potts_general_observe_kernel(const uint8_t* __restrict__ lat, const int8_t* __restrict__ Jh,
                                                                    const int8_t* __restrict__ Jv, int L, int bpr,
                                                                    long long* E_acc, long long* S_acc) {
    __shared__ long long se[8], ss[8];
    const int b = blockIdx.x / bpr, blk = blockIdx.x - b * bpr;
    const long long N = (long long)L * L;
    long long e = 0, sl = 0;
    for (long long x = (long long)blk * blockDim.x + threadIdx.x; x < N; x += (long long)bpr * blockDim.x) {
        const int i = (int)(x / L), j = (int)(x % L);
        const int id = i == L - 1 ? 0 : i + 1, jr = j == L - 1 ? 0 : j + 1;
        const int s = lat[split_index(b, L, i, j)];
        const int jh = Jh ? Jh[b * N + x] : 1, jv = Jv ? Jv[b * N + x] : 1;
        e -= jh * (int)(lat[split_index(b, L, i, jr)] == s) + jv * (int)(lat[split_index(b, L, id, j)] == s);
        sl += s;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        e += __shfl_xor_sync(0xFFFFFFFFu, e, o);
        sl += __shfl_xor_sync(0xFFFFFFFFu, sl, o);
    }
    if ((threadIdx.x & 31) == 0) { se[threadIdx.x >> 5] = e; ss[threadIdx.x >> 5] = sl; }
    __syncthreads();
    if (threadIdx.x == 0) {
        long long te = 0, ts = 0;
        for (int k = 0; k < (int)(blockDim.x >> 5); ++k) { te += se[k]; ts += ss[k]; }
        if (E_acc) atomicAdd((unsigned long long*)E_acc + b, (unsigned long long)te);
        if (S_acc) atomicAdd((unsigned long long*)S_acc + b, (unsigned long long)ts);
    }
}

// Ising int8 with natural +-1 bond signs: E_acc[b] += -sum_bonds J_ij s_i s_j, M_acc[b] += sum s.
__global__ void __launch_bounds__(256) ising_int8_bonds_observe_kernel(const int8_t* __restrict__ lat, const int8_t* __restrict__ Jh,
                                                                       const int8_t* __restrict__ Jv, int L, int bpr,
                                                                       long long* E_acc, long long* M_acc) {
    __shared__ long long se[8], ss[8];
    const int b = blockIdx.x / bpr, blk = blockIdx.x - b * bpr;
    const long long N = (long long)L * L;
    long long e = 0, m = 0;
    for (long long x = (long long)blk * blockDim.x + threadIdx.x; x < N; x += (long long)bpr * blockDim.x) {
        const int i = (int)(x / L), j = (int)(x % L);
        const int id = i == L - 1 ? 0 : i + 1, jr = j == L - 1 ? 0 : j + 1;
        const int s = lat[split_index(b, L, i, j)];
        e -= s * (Jh[b * N + x] * lat[split_index(b, L, i, jr)] + Jv[b * N + x] * lat[split_index(b, L, id, j)]);
        m += s;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        e += __shfl_xor_sync(0xFFFFFFFFu, e, o);
        m += __shfl_xor_sync(0xFFFFFFFFu, m, o);
    }
    if ((threadIdx.x & 31) == 0) { se[threadIdx.x >> 5] = e; ss[threadIdx.x >> 5] = m; }
    __syncthreads();
    if (threadIdx.x == 0) {
        long long te = 0, ts = 0;
        for (int k = 0; k < (int)(blockDim.x >> 5); ++k) { te += se[k]; ts += ss[k]; }
        if (E_acc) atomicAdd((unsigned long long*)E_acc + b, (unsigned long long)te);
        if (M_acc) atomicAdd((unsigned long long*)M_acc + b, (unsigned long long)ts);
    }
}

inline int bpr_for(long long items, int batch) {
    long long want = (items + 255) / 256, cap = (148ll * 16 + batch - 1) / batch;
    if (cap < 1) cap = 1;
    return (int)(want < cap ? want : cap);
}

}  // namespace

int launch_ising_int8_bonds_half_sweep(const SweepArgs& a, const int8_t* Jh, const int8_t* Jv, cudaStream_t s) {
    const long long total = (((long long)a.L * (a.L >> 1) + 3) >> 2) * a.batch;
    launch_pdl(ising_int8_bonds_kernel, (unsigned)((total + 127) / 128), 128u, s, a, Jh, Jv);
    return 1;
}

int launch_ising_int8_general_half_sweep(const SweepArgs& a, const uint32_t* thr, const uint32_t* alw, cudaStream_t s) {
    const long long total = (((long long)a.L * (a.L >> 1) + 3) >> 2) * a.batch;
    launch_pdl(ising_int8_general_kernel, (unsigned)((total + 127) / 128), 128u, s, a, thr, alw);
    return 1;
}

int launch_potts_int8_general_half_sweep(const SweepArgs& a, const unsigned long long* tab2, const int8_t* Jh, const int8_t* Jv,
                                         cudaStream_t s) {
    const long long total = (((long long)a.L * (a.L >> 1) + 1) >> 1) * a.batch;
    launch_pdl(potts_int8_general_kernel, (unsigned)((total + 127) / 128), 128u, s, a, tab2, Jh, Jv);
    return 1;
}

int launch_ising_general_energy(const void* lattice, const double* Jh, const double* Jv, const double* B, int batch, int L,
                                double* E, cudaStream_t s) {
    const int bpr = bpr_for((long long)L * L, batch);
    ising_general_energy_kernel<<<(unsigned)((long long)bpr * batch), 256, 0, s>>>((const int8_t*)lattice, Jh, Jv, B, L, bpr, E);
    return 1;
}

int launch_potts_general_observe(const void* lattice, const int8_t* Jh, const int8_t* Jv, int batch, int L, long long* E_acc,
                                 long long* S_acc, cudaStream_t s) {
    const int bpr = bpr_for((long long)L * L, batch);
    potts_general_observe_kernel<<<(unsigned)((long long)bpr * batch), 256, 0, s>>>((const uint8_t*)lattice, Jh, Jv, L, bpr, E_acc, S_acc);
    return 1;
}

int launch_ising_int8_bonds_observe(const void* lattice, const int8_t* Jh, const int8_t* Jv, int batch, int L, long long* E_acc,
                                    long long* M_acc, cudaStream_t s) {
    const int bpr = bpr_for((long long)L * L, batch);
    ising_int8_bonds_observe_kernel<<<(unsigned)((long long)bpr * batch), 256, 0, s>>>((const int8_t*)lattice, Jh, Jv, L, bpr, E_acc, M_acc);
    return 1;
}

}  // namespace spin
