// cpm.cu — SURVEY.md section 8(f) #3: the Cellular Potts Model of the paper (Eq. 7, Table II) with the
// checkerboard Metropolis rule (Algorithm 1).  Readings C1-C9: a site of the current colour
// (four colours 2 (i & 1) + (j & 1): no two Moore neighbours share one) copies the identifier of one of its eight Moore
// neighbours chosen by r_prop >> 29; dH = adhesion change over the eight neighbours with the type-dependent J of Table
// II + the area term lambda [(new != 0)(2 (a_new - A_new) + 1) + (old != 0)(-2 (a_old - A_old) + 1)] with the areas
// counted at the start of the colour pass; J, lambda, A integers, so dH is an exact integer and the acceptance of
// Alg. 1 is a host-built table T[dH] = floor(exp(-beta dH) 2^32) per replica (the arithmetic of spin_threshold_table).
// Natural row-major int8 lattice of identifiers 0..q-1 (0 = medium).  Per colour pass: zero + count the areas (shared-
// memory histogram), then one thread per Philox group (two sites).
#include "../../include/spin.h"
#include "spin_internal.cuh"

#include <cmath>
#include <cstring>
#include <vector>

namespace spin {
namespace {

constexpr uint32_t kDomainCpm = 4;
constexpr int kMaxTypes = 4;

struct CpmParams {
    int8_t tau[128];
    int32_t A[128];
    int32_t J[kMaxTypes * kMaxTypes];
    long long lambda;
    int32_t q, ntypes;
};

struct CpmArgs {
    int8_t* lattice;
    const int32_t* areas;          // [B][128], counted before the pass
    const uint32_t* T;             // [B][dmax + 1]
    const uint8_t* beta_zero;      // [B]
    int32_t batch, L, colour, dmax;
    uint32_t replica_offset, c2, c3;
    RoundKeys rk;
};

__global__ void __launch_bounds__(256) cpm_area_kernel(const int8_t* __restrict__ lattice, int L, int bpr, int32_t* areas) {
    __shared__ int sh[128];
    const int b = blockIdx.x / bpr, blk = blockIdx.x - b * bpr;
    const long long N = (long long)L * L;
    for (int k = threadIdx.x; k < 128; k += blockDim.x) sh[k] = 0;
    __syncthreads();
    for (long long x = (long long)blk * blockDim.x + threadIdx.x; x < N; x += (long long)bpr * blockDim.x)
        atomicAdd(&sh[lattice[(size_t)b * N + x] & 127], 1);
    __syncthreads();
    for (int k = threadIdx.x; k < 128; k += blockDim.x)
        if (sh[k]) atomicAdd(&areas[b * 128 + k], sh[k]);
}

// One proposal (readings C1, C3-C6): returns the new identifier of site (i, j), or -1 if it keeps its value.
// The resident kernel reads tau / A / J from SHARED-memory copies of the parameters: indexing the kernel-parameter
// (constant) bank with per-thread cell identifiers serialises a warp up to 32-fold.  The short-lived blocks of the
// general pass kernel keep the parameter bank (filling shared tables per block costs more than it saves there).
struct CpmTables {
    const int8_t* tau;
    const int32_t* A;
    const int32_t* J;
    long long lambda;
    int ntypes;
};

// kPair: D[a * qs + b] = (a != b) ? J[tau a][tau b] : 0 for all pairs of identifiers (shared memory, resident kernel): the
// adhesion change is then two reads and two adds per neighbour.
template <typename P, bool kPair = false>   // CpmParams (kernel parameters) or CpmTables (shared-memory copies): same member names
__device__ __forceinline__ int cpm_site(const int8_t* lat, int L, int i, int j, uint32_t r_prop, uint32_t r_acc,
                                        const int32_t* areas, const P& p, const uint32_t* T, int dmax, bool beta_zero,
                                        const int32_t* D = nullptr, int qs = 0) {
    const int iu = i == 0 ? L - 1 : i - 1, id = i == L - 1 ? 0 : i + 1, jl = j == 0 ? L - 1 : j - 1, jr = j == L - 1 ? 0 : j + 1;
    const int old = lat[(size_t)i * L + j];
    // the proposed value first: most sites sit inside a cell or the medium, where it equals the old one and nothing else
    // is needed.  Direction k of the Moore order (-1,-1) (-1,0) (-1,1) (0,-1) (0,1) (1,-1) (1,0) (1,1): cell k + (k >= 4)
    // of the 3 x 3 block around the site.
    const uint32_t dir = r_prop >> 29;
    const int cell = (int)dir + (dir >= 4u ? 1 : 0);
    const int cr = cell / 3, cc = cell - 3 * cr;
    const int pi = cr == 0 ? iu : (cr == 1 ? i : id), pj = cc == 0 ? jl : (cc == 1 ? j : jr);
    const int nw = lat[(size_t)pi * L + pj];
    if (nw == old) return -1;
    const int nb[8] = {lat[(size_t)iu * L + jl], lat[(size_t)iu * L + j], lat[(size_t)iu * L + jr], lat[(size_t)i * L + jl],
                       lat[(size_t)i * L + jr], lat[(size_t)id * L + jl], lat[(size_t)id * L + j], lat[(size_t)id * L + jr]};
    int dJ = 0;
    if (kPair) {
        const int32_t* Dn = D + nw * qs;
        const int32_t* Do = D + old * qs;
#pragma unroll
        for (int k = 0; k < 8; ++k) dJ += Dn[nb[k]] - Do[nb[k]];
    } else {
    const int tn = p.tau[nw], to = p.tau[old];
    // Branch-free: both J entries are read for every neighbour and selected (conditional adds compile to a divergent branch
    // each).  |J| <= 2^20 and 16 terms: the adhesion part is exact in 32 bits.
    const int32_t* Jn = p.J + tn * p.ntypes;
    const int32_t* Jo = p.J + to * p.ntypes;
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        const int ty = p.tau[nb[k]];
        const int jn = Jn[ty], jo = Jo[ty];
        dJ += (nw != nb[k] ? jn : 0) - (old != nb[k] ? jo : 0);
    }
    }
    const long long an = p.lambda * (2ll * ((long long)areas[nw] - p.A[nw]) + 1);
    const long long ao = p.lambda * (-2ll * ((long long)areas[old] - p.A[old]) + 1);
    const long long dH = (long long)dJ + (nw != 0 ? an : 0ll) + (old != 0 ? ao : 0ll);
    bool acc = dH <= 0 || beta_zero;
    if (!acc && dH <= (long long)dmax) acc = r_acc < T[dH];
    return acc ? nw : -1;
}

__device__ __forceinline__ CpmTables load_tables(const CpmParams& p, int8_t* stau, int32_t* sA, int32_t* sJ) {
    for (int k = threadIdx.x; k < 128; k += blockDim.x) { stau[k] = p.tau[k]; sA[k] = p.A[k]; }
    if (threadIdx.x < kMaxTypes * kMaxTypes) sJ[threadIdx.x] = p.J[threadIdx.x];
    CpmTables t;
    t.tau = stau; t.A = sA; t.J = sJ; t.lambda = p.lambda; t.ntypes = p.ntypes;
    return t;
}

__global__ void __launch_bounds__(128) cpm_pass_kernel(CpmArgs a, CpmParams p) {
    const int L = a.L, W = L >> 1;
    const long long per = (long long)W * W, groups = (per + 1) >> 1;
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= groups * a.batch) return;
    const int b = (int)(gid / groups);
    const uint32_t g = (uint32_t)(gid % groups);
    int8_t* lat = a.lattice + (size_t)b * L * L;
    uint32_t r[4];
    philox4x32_10(a.rk, g, (uint32_t)b + a.replica_offset, a.c2, a.c3, r);
#pragma unroll
    for (int e = 0; e < 2; ++e) {
        const long long n = 2ll * g + e;
        if (n >= per) break;
        const int i = 2 * (int)(n / W) + (a.colour >> 1), j = 2 * (int)(n % W) + (a.colour & 1);
        const int nw = cpm_site(lat, L, i, j, r[2 * e], r[2 * e + 1], a.areas + b * 128, p, a.T + (size_t)b * (a.dmax + 1), a.dmax,
                                a.beta_zero[b] != 0);
        if (nw >= 0) lat[(size_t)i * L + j] = (int8_t)nw;
    }
}

// Resident variant for small lattices (the paper's set-up is 36 cells of 25 sites: a few thousand sites): one CTA per
// replica keeps the lattice and the area counters in shared memory and runs every sweep of the call in one launch.  The
// areas are counted once; during a colour pass accepted copies add to a separate delta array, which is folded into the
// areas after the pass - so every proposal of a pass still sees the counts of the start of that pass (reading C3).
template <bool kPair>
__global__ void __launch_bounds__(512) cpm_resident_kernel(CpmArgs a, CpmParams pp, unsigned long long t0, long long n_sweeps) {
    extern __shared__ __align__(16) int8_t slat[];
    __shared__ int32_t sarea[128], sdelta[128];
    __shared__ int8_t stau[128];
    __shared__ int32_t sA[128], sJ[kMaxTypes * kMaxTypes];
    const CpmTables p = load_tables(pp, stau, sA, sJ);
    const int L = a.L, W = L >> 1, b = blockIdx.x;
    const int N = L * L;
    int8_t* glat = a.lattice + (size_t)b * N;
    for (int k = threadIdx.x; k < 128; k += blockDim.x) { sarea[k] = 0; sdelta[k] = 0; }
    for (int k = threadIdx.x; k < (N >> 2); k += blockDim.x) ((uint32_t*)slat)[k] = ((const uint32_t*)glat)[k];
    __syncthreads();
    int32_t* D = (int32_t*)(slat + ((N + 15) & ~15));          // kPair: [q][q] behind the lattice
    const int qs = pp.q;
    if (kPair)
        for (int k = threadIdx.x; k < qs * qs; k += blockDim.x) {
            const int ia = k / qs, ib = k - ia * qs;
            D[k] = ia != ib ? sJ[stau[ia] * p.ntypes + stau[ib]] : 0;
        }
    {   // initial count: the medium (0) usually dominates, so it is counted in a register and reduced per warp
        int zeros = 0;
        for (int x = threadIdx.x; x < N; x += blockDim.x) {
            const int s = slat[x];
            if (s == 0) ++zeros; else atomicAdd(&sarea[s], 1);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) zeros += __shfl_xor_sync(0xFFFFFFFFu, zeros, o);
        if ((threadIdx.x & 31) == 0 && zeros) atomicAdd(&sarea[0], zeros);
    }
    __syncthreads();
    const int per = W * W, groups = (per + 1) >> 1;
    const int wshift = (W & (W - 1)) == 0 ? __ffs(W) - 1 : -1;
    const uint32_t* T = a.T + (size_t)b * (a.dmax + 1);
    const bool bz = a.beta_zero[b] != 0;
    for (long long s = 0; s < n_sweeps; ++s) {
        const unsigned long long t = t0 + (unsigned long long)s;
        const uint32_t c2 = (uint32_t)(t & 0xFFFFFFFFull);
        for (int colour = 0; colour < 4; ++colour) {
            const uint32_t c3 = (uint32_t)((t >> 32) & 0xFFFFFFull) | ((uint32_t)colour << 24) | (kDomainCpm << 28);
            for (int g = threadIdx.x; g < groups; g += blockDim.x) {
                uint32_t r[4];
                philox4x32_10(a.rk, (uint32_t)g, (uint32_t)b + a.replica_offset, c2, c3, r);
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const int n = 2 * g + e;
                    if (n >= per) break;
                    const int row = wshift >= 0 ? n >> wshift : n / W, col = n - row * W;   // no division for L = 2^k
                    const int i = 2 * row + (colour >> 1), j = 2 * col + (colour & 1);
                    const int nw = cpm_site<CpmTables, kPair>(slat, L, i, j, r[2 * e], r[2 * e + 1], sarea, p, T, a.dmax, bz, D, qs);
                    if (nw >= 0) {
                        const int old = slat[i * L + j];
                        slat[i * L + j] = (int8_t)nw;         // only this thread touches a site of the current colour
                        atomicAdd(&sdelta[nw], 1);
                        atomicAdd(&sdelta[old], -1);
                    }
                }
            }
            __syncthreads();
            if (threadIdx.x < 128) { sarea[threadIdx.x] += sdelta[threadIdx.x]; sdelta[threadIdx.x] = 0; }
            __syncthreads();
        }
    }
    for (int k = threadIdx.x; k < (N >> 2); k += blockDim.x) ((uint32_t*)glat)[k] = ((const uint32_t*)slat)[k];
}

// acc[b][0] += adhesion energy, acc[b][1 + lo * ntypes + hi] += boundary pairs, per forward Moore pair.
__global__ void __launch_bounds__(256) cpm_observe_kernel(const int8_t* __restrict__ lattice, int L, int bpr, CpmParams p,
                                                          long long* acc) {
    __shared__ long long sh[1 + kMaxTypes * kMaxTypes];
    const int b = blockIdx.x / bpr, blk = blockIdx.x - b * bpr;
    const long long N = (long long)L * L;
    const int8_t* lat = lattice + (size_t)b * N;
    if (threadIdx.x < 1 + kMaxTypes * kMaxTypes) sh[threadIdx.x] = 0;
    __syncthreads();
    for (long long x = (long long)blk * blockDim.x + threadIdx.x; x < N; x += (long long)bpr * blockDim.x) {
        const int i = (int)(x / L), j = (int)(x % L);
        const int id = i == L - 1 ? 0 : i + 1, jl = j == 0 ? L - 1 : j - 1, jr = j == L - 1 ? 0 : j + 1;
        const int s = lat[x];
        const int ys[4] = {lat[(size_t)i * L + jr], lat[(size_t)id * L + jl], lat[(size_t)id * L + j], lat[(size_t)id * L + jr]};
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            if (ys[k] == s) continue;
            const int t0 = p.tau[s], t1 = p.tau[ys[k]];
            atomicAdd((unsigned long long*)&sh[0], (unsigned long long)(long long)p.J[t0 * p.ntypes + t1]);
            atomicAdd((unsigned long long*)&sh[1 + min(t0, t1) * p.ntypes + max(t0, t1)], 1ull);
        }
    }
    __syncthreads();
    if (threadIdx.x < 1 + kMaxTypes * kMaxTypes && sh[threadIdx.x])
        atomicAdd((unsigned long long*)acc + (size_t)b * (1 + kMaxTypes * kMaxTypes) + threadIdx.x, (unsigned long long)sh[threadIdx.x]);
}

int cpm_fail(int code, const char* msg) { return set_error(code, msg); }

int make_params(int32_t batch, int32_t L, int32_t q, const int32_t* tau, const int32_t* Jtab, int32_t ntypes, int64_t lambda,
                const int32_t* A, CpmParams& p) {
    if (batch < 1 || L < 2 || (L & 1) || L > 32768) return cpm_fail(SPIN_ERR_INVALID, "spin_cpm: batch >= 1 and even L in 2..32768 required");
    if (q < 1 || q > 127 || ntypes < 1 || ntypes > kMaxTypes) return cpm_fail(SPIN_ERR_INVALID, "spin_cpm: 1 <= q <= 127 identifiers and 1 <= ntypes <= 4 types required");
    if (!tau || !Jtab || !A) return cpm_fail(SPIN_ERR_INVALID, "spin_cpm: NULL parameter array");
    if (lambda < 0 || lambda > (1ll << 20)) return cpm_fail(SPIN_ERR_INVALID, "spin_cpm: lambda must be in 0..2^20");
    std::memset(&p, 0, sizeof p);
    for (int k = 0; k < q; ++k) {
        if (tau[k] < 0 || tau[k] >= ntypes) return cpm_fail(SPIN_ERR_INVALID, "spin_cpm: tau[k] must be a type index in 0..ntypes-1");
        if (A[k] < 0) return cpm_fail(SPIN_ERR_INVALID, "spin_cpm: target areas must be >= 0");
        p.tau[k] = (int8_t)tau[k];
        p.A[k] = A[k];
    }
    for (int a = 0; a < ntypes; ++a)
        for (int c = 0; c < ntypes; ++c) {
            if (Jtab[a * ntypes + c] != Jtab[c * ntypes + a]) return cpm_fail(SPIN_ERR_INVALID, "spin_cpm: the J table must be symmetric (PAPER.md:222)");
            if (Jtab[a * ntypes + c] < -(1 << 20) || Jtab[a * ntypes + c] > (1 << 20)) return cpm_fail(SPIN_ERR_INVALID, "spin_cpm: |J| must be <= 2^20");
            p.J[a * ntypes + c] = Jtab[a * ntypes + c];
        }
    p.lambda = lambda; p.q = q; p.ntypes = ntypes;
    return SPIN_OK;
}

}  // namespace
}  // namespace spin

using namespace spin;

extern "C" {

int spin_cpm_sweep(int32_t batch, int32_t L, int32_t q, int8_t* lattice, const int32_t* tau, const int32_t* Jtab, int32_t ntypes,
                   int64_t lambda, const int32_t* A, const double* beta, uint64_t seed, int64_t replica_offset, int64_t n_sweeps,
                   int64_t sweep_offset, void* cuda_stream) {
    CpmParams p;
    int rc = make_params(batch, L, q, tau, Jtab, ntypes, lambda, A, p);
    if (rc != SPIN_OK) return rc;
    if (!lattice || !beta) return cpm_fail(SPIN_ERR_INVALID, "spin_cpm_sweep: NULL argument");
    if (replica_offset < 0 || replica_offset + (int64_t)batch > (1ll << 32)) return cpm_fail(SPIN_ERR_INVALID, "spin_cpm: replica_offset + batch must stay within [0, 2^32]");
    if (n_sweeps < 0 || sweep_offset < 0 || sweep_offset > (1ll << 56) || n_sweeps > (1ll << 56) || sweep_offset + n_sweeps > (1ll << 56))
        return cpm_fail(SPIN_ERR_INVALID, "spin_cpm_sweep: sweep range must lie in [0, 2^56]");
    // acceptance table T[b][d], d = 1 .. dmax: the smallest d at which every replica's threshold has reached 0
    const int kCap = 65536;
    int dmax = 1;
    for (int b = 0; b < batch; ++b) {
        if (!std::isfinite(beta[b]) || beta[b] < 0.0) return cpm_fail(SPIN_ERR_INVALID, "spin_cpm_sweep: beta must be finite and >= 0");
        if (beta[b] == 0.0) continue;
        if (b > 0 && beta[b] == beta[b - 1]) continue;      // same table as the previous replica
        int d = 1;
        while (d <= kCap && std::floor(std::exp(-(beta[b] * (double)d)) * 4294967296.0) >= 1.0) ++d;
        if (d > kCap) return cpm_fail(SPIN_ERR_UNSUPPORTED, "spin_cpm_sweep: beta is so small that exp(-beta dH) 2^32 >= 1 beyond dH = 65536; use beta = 0 or a larger beta");
        if (d > dmax) dmax = d;
    }
    if (n_sweeps == 0) return SPIN_OK;
    std::vector<uint32_t> T;
    std::vector<uint8_t> bz;
    try { T.assign((size_t)batch * (dmax + 1), 0u); bz.assign(batch, 0); } catch (...) { return cpm_fail(SPIN_ERR_NOMEM, "spin_cpm_sweep: out of host memory"); }
    for (int b = 0; b < batch; ++b) {
        bz[b] = beta[b] == 0.0 ? 1 : 0;
        if (b > 0 && beta[b] == beta[b - 1]) {                // replicas at one temperature share the (identical) table
            std::memcpy(&T[(size_t)b * (dmax + 1)], &T[(size_t)(b - 1) * (dmax + 1)], sizeof(uint32_t) * (dmax + 1));
            continue;
        }
        for (int d = 1; d <= dmax; ++d) {
            const double x = beta[b] * (double)d;              // O4 with dE = d > 0
            if (x <= 0.0) { T[(size_t)b * (dmax + 1) + d] = 0xFFFFFFFFu; continue; }
            const double v = std::floor(std::exp(-x) * 4294967296.0);
            T[(size_t)b * (dmax + 1) + d] = v >= 4294967295.0 ? 0xFFFFFFFFu : (uint32_t)v;
        }
    }
    cudaStream_t s = (cudaStream_t)cuda_stream;
    uint32_t* d_T = nullptr;
    uint8_t* d_bz = nullptr;
    int32_t* d_areas = nullptr;
    cudaError_t e = cudaMallocAsync(&d_T, T.size() * sizeof(uint32_t), s);
    if (e == cudaSuccess) e = cudaMallocAsync(&d_bz, batch, s);
    if (e == cudaSuccess) e = cudaMallocAsync(&d_areas, sizeof(int32_t) * 128 * batch, s);
    if (e == cudaSuccess) e = cudaMemcpyAsync(d_T, T.data(), T.size() * sizeof(uint32_t), cudaMemcpyHostToDevice, s);
    if (e == cudaSuccess) e = cudaMemcpyAsync(d_bz, bz.data(), batch, cudaMemcpyHostToDevice, s);
    if (e == cudaSuccess) {
        CpmArgs a;
        a.lattice = lattice; a.areas = d_areas; a.T = d_T; a.beta_zero = d_bz; a.batch = batch; a.L = L; a.dmax = dmax;
        a.replica_offset = (uint32_t)replica_offset;
        uint32_t k0 = (uint32_t)(seed & 0xFFFFFFFFull), k1 = (uint32_t)(seed >> 32);
        for (int r = 0; r < 10; ++r) { a.rk.k0[r] = k0; a.rk.k1[r] = k1; k0 += kPhiloxW0; k1 += kPhiloxW1; }
        const long long N = (long long)L * L;
        long long want = (N + 255) / 256, cap = (148ll * 8 + batch - 1) / batch;
        const int bpr = (int)(want < cap ? want : (cap < 1 ? 1 : cap));
        const long long groups = (((long long)(L / 2) * (L / 2) + 1) >> 1) * batch;
        // small lattices: one CTA per replica, everything in shared memory, all sweeps in one launch
        const bool resident = N <= 65536 && (N & 3) == 0 && (L <= 128 || batch >= 148);
        if (resident) {
            a.colour = 0; a.c2 = 0; a.c3 = 0;
            // one Philox group (two sites) per thread and colour pass where the lattice has that many (the passes are latency
            // chains: 60 -> measured below with 512 threads for L = 64)
            const unsigned res_threads = (L / 2) * (L / 2) / 2 >= 512 ? 512u : 256u;
            // the pair table of the adhesion energies ([q][q] int32 behind the lattice) while it stays small (q <= 64: 16 KiB)
            const bool pair = q <= 64;
            const size_t smem = pair ? (size_t)((N + 15) & ~15ll) + sizeof(int32_t) * q * q : (size_t)N;
            if (smem > 49152) e = cudaFuncSetAttribute(pair ? cpm_resident_kernel<true> : cpm_resident_kernel<false>,
                                                       cudaFuncAttributeMaxDynamicSharedMemorySize, 65536 + 16384);
            if (e == cudaSuccess) {
                if (pair) cpm_resident_kernel<true><<<(unsigned)batch, res_threads, smem, s>>>(a, p, (unsigned long long)sweep_offset, (long long)n_sweeps);
                else cpm_resident_kernel<false><<<(unsigned)batch, res_threads, smem, s>>>(a, p, (unsigned long long)sweep_offset, (long long)n_sweeps);
            }
        }
        for (int64_t t = sweep_offset; !resident && t < sweep_offset + n_sweeps && e == cudaSuccess; ++t)
            for (int c = 0; c < 4; ++c) {
                e = cudaMemsetAsync(d_areas, 0, sizeof(int32_t) * 128 * batch, s);
                cpm_area_kernel<<<(unsigned)((long long)bpr * batch), 256, 0, s>>>(lattice, L, bpr, d_areas);
                a.colour = c;
                a.c2 = (uint32_t)((uint64_t)t & 0xFFFFFFFFull);
                a.c3 = (uint32_t)(((uint64_t)t >> 32) & 0xFFFFFFull) | ((uint32_t)c << 24) | (kDomainCpm << 28);
                cpm_pass_kernel<<<(unsigned)((groups + 127) / 128), 128, 0, s>>>(a, p);
            }
        if (e == cudaSuccess) e = cudaGetLastError();
    }
    if (d_T) cudaFreeAsync(d_T, s);
    if (d_bz) cudaFreeAsync(d_bz, s);
    if (d_areas) cudaFreeAsync(d_areas, s);
    return e == cudaSuccess ? SPIN_OK : cpm_fail(SPIN_ERR_CUDA, cudaGetErrorString(e));
}

int spin_cpm_observables(int32_t batch, int32_t L, int32_t q, const int8_t* lattice, const int32_t* tau, const int32_t* Jtab,
                         int32_t ntypes, int64_t lambda, const int32_t* A, int64_t* H_adh, int64_t* H_area, int64_t* areas,
                         int64_t* boundary, void* cuda_stream) {
    CpmParams p;
    const int rc = make_params(batch, L, q, tau, Jtab, ntypes, lambda, A, p);
    if (rc != SPIN_OK) return rc;
    if (!lattice) return cpm_fail(SPIN_ERR_INVALID, "spin_cpm_observables: NULL lattice");
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const int kAcc = 1 + kMaxTypes * kMaxTypes;
    std::vector<long long> hacc;
    std::vector<int32_t> har;
    try { hacc.assign((size_t)batch * kAcc, 0); har.assign((size_t)batch * 128, 0); } catch (...) { return cpm_fail(SPIN_ERR_NOMEM, "spin_cpm_observables: out of host memory"); }
    long long* d_acc = nullptr;
    int32_t* d_areas = nullptr;
    cudaError_t e = cudaMallocAsync(&d_acc, sizeof(long long) * kAcc * batch, s);
    if (e == cudaSuccess) e = cudaMallocAsync(&d_areas, sizeof(int32_t) * 128 * batch, s);
    if (e == cudaSuccess) e = cudaMemsetAsync(d_acc, 0, sizeof(long long) * kAcc * batch, s);
    if (e == cudaSuccess) e = cudaMemsetAsync(d_areas, 0, sizeof(int32_t) * 128 * batch, s);
    if (e == cudaSuccess) {
        const long long N = (long long)L * L;
        long long want = (N + 255) / 256, cap = (148ll * 8 + batch - 1) / batch;
        const int bpr = (int)(want < cap ? want : (cap < 1 ? 1 : cap));
        cpm_area_kernel<<<(unsigned)((long long)bpr * batch), 256, 0, s>>>(lattice, L, bpr, d_areas);
        cpm_observe_kernel<<<(unsigned)((long long)bpr * batch), 256, 0, s>>>(lattice, L, bpr, p, d_acc);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaMemcpyAsync(hacc.data(), d_acc, sizeof(long long) * kAcc * batch, cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaMemcpyAsync(har.data(), d_areas, sizeof(int32_t) * 128 * batch, cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (d_acc) cudaFreeAsync(d_acc, s);
    if (d_areas) cudaFreeAsync(d_areas, s);
    if (e != cudaSuccess) return cpm_fail(SPIN_ERR_CUDA, cudaGetErrorString(e));
    for (int b = 0; b < batch; ++b) {
        if (H_adh) H_adh[b] = hacc[(size_t)b * kAcc];
        long long ha = 0;
        for (int k = 0; k < q; ++k) {
            const long long ar = har[(size_t)b * 128 + k];
            if (areas) areas[(size_t)b * q + k] = ar;
            if (k >= 1) ha += lambda * (ar - A[k]) * (ar - A[k]);     // O(q) host arithmetic on the exact device counts
        }
        if (H_area) H_area[b] = ha;
        if (boundary)
            for (int a = 0; a < ntypes; ++a)
                for (int c = 0; c < ntypes; ++c)
                    boundary[((size_t)b * ntypes + a) * ntypes + c] = a <= c ? hacc[(size_t)b * kAcc + 1 + a * ntypes + c] : 0;
    }
    return SPIN_OK;
}

}  // extern "C"
