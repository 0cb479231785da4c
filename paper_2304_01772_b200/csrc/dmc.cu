// dmc.cu — SURVEY.md section 8(f) #1: the paper's Differentiable Monte Carlo step (Algorithm 2 and Eq. 4,
// PAPER.md:125, 140-158) for the 2D Ising model with per-bond couplings (Eq. 1), forward and
// hand-written backward (dLoss/dJ_ij, dLoss/dbeta, dLoss/dh, dLoss/ds_0; the training use is PAPER.md:308-332).
//
// Per site x of the current colour (readings D1-D8):
//   F = sum_n J_xn s_n + h,  dE = 2 s F,  p = exp(-beta dE),  r = (w >> 8) 2^-24 (w: the Ising sweep's Philox word),
//   q = 1 / (1 + exp(-alpha (p - r))),  s <- q (-s) + (1 - q) s.
// Float lattices in the NATURAL layout [B][L][L] (fp32, or fp64 for tight parity), couplings Jh / Jv [B][L][L] as in
// spin_set_bonds.  The path is HBM-bound (a few dozen flops and two exponentials per 16-32 bytes), so the kernels are
// plain streaming kernels: one thread per V consecutive sites of a row (one 16-byte vector of the lattice and of every
// operand row), coalesced vector loads / stores, the three lattice rows and the two coupling arrays read once per
// half-sweep, grids of whole rows.  A half-sweep is out of place (state k -> state k+1), which is what the backward
// pass needs anyway (it re-reads the state every half-sweep started from).
//
// Backward of one half-sweep, with A = alpha q (1-q) p at the updated sites (0 elsewhere):
//   pass 1 (updated sites):  G_x = g_x 4 beta A s^2  (= dLoss/dF_x),  D_x = g_x ((1-2q) + 4 beta A s F);  D_y = g_y elsewhere;
//                            dLoss/dbeta += g_x 4 A s^2 F,  dLoss/dh += G_x          (block reduction + one atomic)
//   pass 2 (all sites):      g_prev_x = D_x + sum_n G_n J_xn;  dJh[i][j] += G[i][j] s[i][j+1] + G[i][j+1] s[i][j],
//                            dJv[i][j] += G[i][j] s[i+1][j] + G[i+1][j] s[i][j]      (every bond has one updated end)
// No atomics on the lattice-sized arrays, no scattered accesses.
#include "../../include/spin.h"
#include "spin_internal.cuh"

#include <cmath>
#include <cstdio>

namespace spin {
namespace {

template <typename T, int V>
struct alignas(sizeof(T) * V) Vec {
    T v[V];
};

template <typename T> __device__ __forceinline__ T exp_t(T x);
template <> __device__ __forceinline__ float exp_t<float>(float x) { return expf(x); }
template <> __device__ __forceinline__ double exp_t<double>(double x) { return exp(x); }

struct DmcArgs {
    int32_t batch, L;
    uint32_t replica_offset;
    uint32_t c2, c3;          // Philox counter words of (t, colour), domain ISING (reading D4)
    int32_t colour;
    double h, alpha;
    const double* beta;       // device [B]
    RoundKeys rk;
};

// Everything Algorithm 2 computes for the V sites a thread owns.  upd[e]: the site has the current colour.
template <typename T, int V>
struct Sites {
    T s[V], F[V], p[V], q[V];
    bool upd[V];
};

// Loads the thread's neighbourhood from the state `src` and evaluates lines 2-8 of Algorithm 2 for its updated sites.
template <typename T, int V>
__device__ __forceinline__ void eval_sites(const DmcArgs& a, const T* __restrict__ src, const T* __restrict__ Jh,
                                           const T* __restrict__ Jv, int b, int i, int j0, Sites<T, V>& o) {
    const int L = a.L;
    const size_t base = (size_t)b * L * L;
    const int iu = i == 0 ? L - 1 : i - 1, id = i == L - 1 ? 0 : i + 1;
    const int jl = j0 == 0 ? L - 1 : j0 - 1, jr = j0 + V == L ? 0 : j0 + V;
    const Vec<T, V> sc = *(const Vec<T, V>*)(src + base + (size_t)i * L + j0);
    const Vec<T, V> su = *(const Vec<T, V>*)(src + base + (size_t)iu * L + j0);
    const Vec<T, V> sd = *(const Vec<T, V>*)(src + base + (size_t)id * L + j0);
    const Vec<T, V> jh = *(const Vec<T, V>*)(Jh + base + (size_t)i * L + j0);
    const Vec<T, V> jvu = *(const Vec<T, V>*)(Jv + base + (size_t)iu * L + j0);
    const Vec<T, V> jvc = *(const Vec<T, V>*)(Jv + base + (size_t)i * L + j0);
    const T sl = src[base + (size_t)i * L + jl], sr = src[base + (size_t)i * L + jr];
    const T jhl = Jh[base + (size_t)i * L + jl];
    // one Philox call covers the thread's updated sites when V == 4 (L % 4 == 0: n and n+1 share a group); with V == 2
    // there is one updated site
    const T beta = (T)a.beta[b];
    uint32_t r[4];
    uint32_t have = 0xFFFFFFFFu;
#pragma unroll
    for (int e = 0; e < V; ++e) {
        const int j = j0 + e;
        o.s[e] = sc.v[e];
        o.upd[e] = ((i + j) & 1) == a.colour;
        o.F[e] = o.p[e] = o.q[e] = (T)0;
        if (!o.upd[e]) continue;
        const uint32_t n = (uint32_t)i * (uint32_t)(L >> 1) + (uint32_t)(j >> 1);
        if ((n >> 2) != have) {
            have = n >> 2;
            philox4x32_10(a.rk, have, (uint32_t)b + a.replica_offset, a.c2, a.c3, r);
        }
        const uint32_t w = (n & 3u) == 0u ? r[0] : (n & 3u) == 1u ? r[1] : (n & 3u) == 2u ? r[2] : r[3];
        const T rr = (T)(w >> 8) * (T)(1.0 / 16777216.0);
        const T left = e == 0 ? sl : sc.v[e > 0 ? e - 1 : 0];
        const T right = e == V - 1 ? sr : sc.v[e < V - 1 ? e + 1 : V - 1];
        const T jleft = e == 0 ? jhl : jh.v[e > 0 ? e - 1 : 0];
        // same association order as the oracle: up, down, left, right, then h
        const T F = jvu.v[e] * su.v[e] + jvc.v[e] * sd.v[e] + jleft * left + jh.v[e] * right + (T)a.h;
        const T dE = (T)2 * o.s[e] * F;
        const T p = exp_t<T>(-beta * dE);
        o.F[e] = F;
        o.p[e] = p;
        o.q[e] = (T)1 / ((T)1 + exp_t<T>(-(T)a.alpha * (p - rr)));
    }
}

template <typename T, int V>
__global__ void __launch_bounds__(256) dmc_forward_kernel(DmcArgs a, const T* __restrict__ src, T* __restrict__ dst,
                                                          const T* __restrict__ Jh, const T* __restrict__ Jv) {
    const int vpr = a.L / V;                                   // vectors per row
    const long long total = (long long)a.batch * a.L * vpr;
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= total) return;
    const int x = (int)(gid % vpr);
    const long long bi = gid / vpr;
    const int i = (int)(bi % a.L), b = (int)(bi / a.L);
    Sites<T, V> st;
    eval_sites<T, V>(a, src, Jh, Jv, b, i, x * V, st);
    Vec<T, V> out;
#pragma unroll
    for (int e = 0; e < V; ++e)
        out.v[e] = st.upd[e] ? st.q[e] * (-st.s[e]) + ((T)1 - st.q[e]) * st.s[e] : st.s[e];      // line 9
    *(Vec<T, V>*)(dst + (size_t)b * a.L * a.L + (size_t)i * a.L + x * V) = out;
}

// ---- fused forward sweep (fp32, L % 8 == 0, L <= 2048): both colours of a sweep in ONE pass.  A block owns a tile of R
// whole rows.  Phase A applies the colour-0 half-sweep to rows i0-1 .. i0+R (one halo row on each side, recomputed by the
// neighbouring tile as well: the counter-based random numbers make the redundant updates identical) and keeps the result
// in shared memory; phase B applies the colour-1 half-sweep to rows i0 .. i0+R-1 from shared memory and writes the final
// rows.  The lattice and the couplings are read from HBM once per SWEEP instead of once per half-sweep (the second
// read of the couplings hits L1/L2): about (R+4)/R * 4 + 4 + (R+2)/R * 8 = 18 B/site/sweep at R = 14 instead of 32.
// A thread's unit of work is 8 consecutive sites of a row = the 4 sites of one colour = one Philox call (all 4 words).
// The arithmetic per site is the two-pass kernels' up to the last bits (fast reciprocal, FMA contraction): both are held
// to the fp32 tolerance against the oracle, not to each other.
__device__ __forceinline__ float dmc_site(float s, float su, float sd, float sl, float sr, float jvu, float jvc, float jl,
                                          float jr, float h, float beta, float alpha, uint32_t w) {
    const float rr = (float)(w >> 8) * (float)(1.0 / 16777216.0);
    const float F = jvu * su + jvc * sd + jl * sl + jr * sr + h;
    const float dE = 2.0f * s * F;
    const float p = expf(-beta * dE);
    const float q = __fdividef(1.0f, 1.0f + expf(-alpha * (p - rr)));       // MUFU.RCP + FMUL, 2 ulp
    return q * (-s) + (1.0f - q) * s;
}

// Updates the 4 sites of parity kPar (columns j0 + kPar + 2m) among 8 consecutive sites c[0..7] of row i.
template <int kPar>
__device__ __forceinline__ void dmc_chunk_par(const DmcArgs& a, const uint32_t r[4], const float c[8], const float u[8],
                                              const float d[8], float left, float right, const float jh[8], float jhl,
                                              const float jvu[8], const float jvc[8], float beta, float out[8]) {
#pragma unroll
    for (int e = 0; e < 8; ++e) out[e] = c[e];
#pragma unroll
    for (int m = 0; m < 4; ++m) {
        const int e = 2 * m + kPar;
        const float sl = e == 0 ? left : c[e > 0 ? e - 1 : 0];
        const float sr = e == 7 ? right : c[e < 7 ? e + 1 : 7];
        const float jl = e == 0 ? jhl : jh[e > 0 ? e - 1 : 0];
        out[e] = dmc_site(c[e], u[e], d[e], sl, sr, jvu[e], jvc[e], jl, jh[e], (float)a.h, beta, (float)a.alpha, r[m]);
    }
}

__device__ __forceinline__ void dmc_chunk(const DmcArgs& a, int b, int i, int cidx, int par, uint32_t c3, const float c[8],
                                          const float u[8], const float d[8], float left, float right, const float jh[8],
                                          float jhl, const float jvu[8], const float jvc[8], float beta, float out[8]) {
    uint32_t r[4];
    philox4x32_10(a.rk, (uint32_t)i * (uint32_t)(a.L >> 3) + (uint32_t)cidx, (uint32_t)b + a.replica_offset, a.c2, c3, r);
    if (par == 0) dmc_chunk_par<0>(a, r, c, u, d, left, right, jh, jhl, jvu, jvc, beta, out);
    else dmc_chunk_par<1>(a, r, c, u, d, left, right, jh, jhl, jvu, jvc, beta, out);
}

__device__ __forceinline__ void load8(const float* p, float v[8]) {
    const float4 x = *(const float4*)p, y = *(const float4*)(p + 4);
    v[0] = x.x; v[1] = x.y; v[2] = x.z; v[3] = x.w; v[4] = y.x; v[5] = y.y; v[6] = y.z; v[7] = y.w;
}
__device__ __forceinline__ void store8(float* p, const float v[8]) {
    *(float4*)p = make_float4(v[0], v[1], v[2], v[3]);
    *(float4*)(p + 4) = make_float4(v[4], v[5], v[6], v[7]);
}

__global__ void __launch_bounds__(256) dmc_fused_sweep_kernel(DmcArgs a, const float* __restrict__ src, float* __restrict__ mid,
                                                              float* __restrict__ dst, const float* __restrict__ Jh,
                                                              const float* __restrict__ Jv, int R, int tiles) {
    extern __shared__ __align__(16) float sA[];               // (R + 2) rows of L floats: the state after colour 0
    const int L = a.L, cpr = L >> 3;
    const int b = blockIdx.x / tiles, tile = blockIdx.x - b * tiles;
    const int i0 = tile * R, rows = min(R, L - i0);
    const size_t base = (size_t)b * L * L;
    const float beta = (float)a.beta[b];
    const uint32_t c3lo = a.c3 & ~(0xFu << 24);               // colour field cleared
    // phase A: colour 0 on rows i0 - 1 .. i0 + rows
    for (int task = threadIdx.x; task < (rows + 2) * cpr; task += blockDim.x) {
        const int ra = task / cpr, cidx = task - ra * cpr;
        int i = i0 - 1 + ra;
        i = i < 0 ? L - 1 : (i >= L ? i - L : i);
        const int iu = i == 0 ? L - 1 : i - 1, id = i == L - 1 ? 0 : i + 1, j0 = cidx << 3;
        const int jl = j0 == 0 ? L - 1 : j0 - 1, jr = j0 + 8 == L ? 0 : j0 + 8;
        float c[8], u[8], d[8], jh[8], jvu[8], jvc[8], out[8];
        load8(src + base + (size_t)i * L + j0, c);
        load8(src + base + (size_t)iu * L + j0, u);
        load8(src + base + (size_t)id * L + j0, d);
        load8(Jh + base + (size_t)i * L + j0, jh);
        load8(Jv + base + (size_t)iu * L + j0, jvu);
        load8(Jv + base + (size_t)i * L + j0, jvc);
        dmc_chunk(a, b, i, cidx, i & 1, c3lo, c, u, d, src[base + (size_t)i * L + jl], src[base + (size_t)i * L + jr], jh,
                  Jh[base + (size_t)i * L + jl], jvu, jvc, beta, out);
        store8(sA + (size_t)ra * L + j0, out);
        if (mid && ra >= 1 && ra <= rows) store8(mid + base + (size_t)i * L + j0, out);
    }
    __syncthreads();
    // phase B: colour 1 on rows i0 .. i0 + rows - 1, neighbours from shared memory
    for (int task = threadIdx.x; task < rows * cpr; task += blockDim.x) {
        const int rb = task / cpr, cidx = task - rb * cpr;
        const int ra = rb + 1, i = i0 + rb, j0 = cidx << 3;
        const int iu = i == 0 ? L - 1 : i - 1;
        const int jl = j0 == 0 ? L - 1 : j0 - 1, jr = j0 + 8 == L ? 0 : j0 + 8;
        float c[8], u[8], d[8], jh[8], jvu[8], jvc[8], out[8];
        load8(sA + (size_t)ra * L + j0, c);
        load8(sA + (size_t)(ra - 1) * L + j0, u);
        load8(sA + (size_t)(ra + 1) * L + j0, d);
        load8(Jh + base + (size_t)i * L + j0, jh);
        load8(Jv + base + (size_t)iu * L + j0, jvu);
        load8(Jv + base + (size_t)i * L + j0, jvc);
        dmc_chunk(a, b, i, cidx, 1 - (i & 1), c3lo | (1u << 24), c, u, d, sA[(size_t)ra * L + jl], sA[(size_t)ra * L + jr], jh,
                  Jh[base + (size_t)i * L + jl], jvu, jvc, beta, out);
        store8(dst + base + (size_t)i * L + j0, out);
    }
}

// ---- row-marching forward sweep (fp32, 256 <= L <= 2048, L % 8 == 0): the fused sweep above re-reads the couplings from
// L2 for the second colour and pays a full memory latency per task; here a thread owns one 8-site chunk COLUMN and
// marches down the R rows of its tile with everything it needs twice kept in registers: three source rows, three
// colour-0 rows, the couplings of the current and the previous row.  Per row step: prefetch the next source row and the
// next row's couplings, compute the colour-0 update A_i of row i, publish the two edge values of A_i to shared memory (the
// neighbouring chunks need them for the colour-1 update), barrier, compute the colour-1 update of row i-1 from A_{i-2},
// A_{i-1}, A_i and store it.  A block is one full row of chunks (L/8 threads), so the periodic wrap in the row stays in the
// block; tiles overlap by one halo row at each end (recomputed, identical by construction).  Every source element and
// every coupling is loaded from HBM exactly once per sweep (+ 4/R for the halo rows).
__global__ void __launch_bounds__(256) dmc_march_sweep_kernel(DmcArgs a, const float* __restrict__ src, float* __restrict__ mid,
                                                              float* __restrict__ dst, const float* __restrict__ Jh,
                                                              const float* __restrict__ Jv, int R, int tiles) {
    __shared__ float sEdge[3][256][2];                       // [row slot][chunk][first, last] of the colour-0 row
    const int L = a.L, cpr = L >> 3, cidx = threadIdx.x;
    const int b = blockIdx.x / tiles, tile = blockIdx.x - b * tiles;
    const int i0 = tile * R, rows = min(R, L - i0);
    const size_t base = (size_t)b * L * L;
    const float beta = (float)a.beta[b];
    const uint32_t c3lo = a.c3 & ~(0xFu << 24);
    const int j0 = cidx << 3;
    const int jl = j0 == 0 ? L - 1 : j0 - 1, jr = j0 + 8 == L ? 0 : j0 + 8;
    const int cl = cidx == 0 ? cpr - 1 : cidx - 1, cr = cidx == cpr - 1 ? 0 : cidx + 1;
    auto wrapi = [L](int i) { return i < 0 ? i + L : (i >= L ? i - L : i); };
    // source rows i-1, i, i+1 of the first step (i = i0 - 1), couplings of row i and Jv of row i-1
    float Sm[8], Sc[8], Sp[8], Sn[8];                         // rows i-1, i, i+1 and the prefetched i+2
    float Am[8], Ac[8], An[8];                                // colour-0 rows i-2, i-1, i (An = newest)
    float JhC[8], JhP[8], JhN[8], JvM[8], JvC[8], JvP2[8], JvN[8];
    float jhlC, jhlP = 0.f, jhlN, slC, srC, slN, srN;
    int i = wrapi(i0 - 1);
    load8(src + base + (size_t)wrapi(i - 1) * L + j0, Sm);
    load8(src + base + (size_t)i * L + j0, Sc);
    load8(src + base + (size_t)wrapi(i + 1) * L + j0, Sp);
    load8(Jh + base + (size_t)i * L + j0, JhC);
    load8(Jv + base + (size_t)wrapi(i - 1) * L + j0, JvM);
    load8(Jv + base + (size_t)i * L + j0, JvC);
    jhlC = Jh[base + (size_t)i * L + jl];
    slC = src[base + (size_t)i * L + jl];
    srC = src[base + (size_t)i * L + jr];
#pragma unroll
    for (int e = 0; e < 8; ++e) { Am[e] = 0.f; Ac[e] = 0.f; JhP[e] = 0.f; JvP2[e] = 0.f; }
    for (int step = 0; step < rows + 2; ++step) {
        // rows of this step: i (colour 0), i - 1 (colour 1, once step >= 2)
        const int inext = i == L - 1 ? 0 : i + 1;             // row i + 1
        const int inn = inext == L - 1 ? 0 : inext + 1;       // row i + 2
        const bool more = step + 1 < rows + 2;
        if (more) {                                           // prefetch what the next step needs
            load8(src + base + (size_t)inn * L + j0, Sn);
            load8(Jh + base + (size_t)inext * L + j0, JhN);
            load8(Jv + base + (size_t)inext * L + j0, JvN);
            jhlN = Jh[base + (size_t)inext * L + jl];
            slN = src[base + (size_t)inext * L + jl];
            srN = src[base + (size_t)inext * L + jr];
        }
        // colour 0 on row i
        dmc_chunk(a, b, i, cidx, i & 1, c3lo, Sc, Sm, Sp, slC, srC, JhC, jhlC, JvM, JvC, beta, An);
        const int slot = step % 3;
        sEdge[slot][cidx][0] = An[0];
        sEdge[slot][cidx][1] = An[7];
        if (mid && step >= 1 && step <= rows) store8(mid + base + (size_t)i * L + j0, An);
        __syncthreads();
        if (step >= 2) {
            // colour 1 on row i - 1: neighbours A_{i-2} (Am), A_i (An), own A_{i-1} (Ac); couplings of row i - 1
            const int ip = i == 0 ? L - 1 : i - 1;
            const int ps = (step + 2) % 3;                    // slot of step - 1
            float out[8];
            dmc_chunk(a, b, ip, cidx, 1 - (ip & 1), c3lo | (1u << 24), Ac, Am, An, sEdge[ps][cl][1], sEdge[ps][cr][0], JhP, jhlP,
                      JvP2, JvM, beta, out);
            store8(dst + base + (size_t)ip * L + j0, out);
        }
        // rotate the windows: rows move up by one
#pragma unroll
        for (int e = 0; e < 8; ++e) {
            Am[e] = Ac[e]; Ac[e] = An[e];
            JhP[e] = JhC[e]; JvP2[e] = JvM[e]; JvM[e] = JvC[e];
            Sm[e] = Sc[e]; Sc[e] = Sp[e];
            if (more) { Sp[e] = Sn[e]; JhC[e] = JhN[e]; JvC[e] = JvN[e]; }
        }
        jhlP = jhlC;
        if (more) { jhlC = jhlN; slC = slN; srC = srN; }
        i = inext;
    }
}

// ---- row-marching backward half-sweep (fp32, 256 <= L <= 2048, L % 8 == 0): passes 1 and 2 below fused, so that G and D
// never travel through HBM.  Same skeleton as dmc_march_sweep_kernel: a thread owns one 8-site chunk column; per step it
// computes G_{i+1}, D_{i+1} of the next row (recomputing p, q from the stored state), publishes the edge values of G_{i+1},
// and finishes row i, which needs G_{i-1}, G_i, G_{i+1}:
//   g_prev_i[j] = D_i[j] + G_{i-1}[j] Jv_{i-1}[j] + G_{i+1}[j] Jv_i[j] + G_i[j-1] Jh_i[j-1] + G_i[j+1] Jh_i[j]
//   dJh_i[j] += G_i[j] s_i[j+1] + G_i[j+1] s_i[j],   dJv_i[j] += G_i[j] s_{i+1}[j] + G_{i+1}[j] s_i[j]
// Per site and half-sweep: read s, Jh, Jv, g (16 B), write g_prev (4), read-modify-write dJh, dJv (16) = 36 B instead of 64.
template <int kPar>
__device__ __forceinline__ void dmc_chunk_bwd_par(const DmcArgs& a, const uint32_t r[4], const float c[8], const float u[8],
                                                  const float d[8], float left, float right, const float jh[8], float jhl,
                                                  const float jvu[8], const float jvc[8], float beta, const float g[8],
                                                  float G[8], float D[8], double& sb, double& sh) {
#pragma unroll
    for (int e = 0; e < 8; ++e) { G[e] = 0.f; D[e] = g[e]; }
#pragma unroll
    for (int m = 0; m < 4; ++m) {
        const int e = 2 * m + kPar;
        const float sl = e == 0 ? left : c[e > 0 ? e - 1 : 0];
        const float sr = e == 7 ? right : c[e < 7 ? e + 1 : 7];
        const float jl = e == 0 ? jhl : jh[e > 0 ? e - 1 : 0];
        const float sx = c[e];
        const float rr = (float)(r[m] >> 8) * (float)(1.0 / 16777216.0);
        const float F = jvu[e] * u[e] + jvc[e] * d[e] + jl * sl + jh[e] * sr + (float)a.h;
        const float p = expf(-beta * (2.0f * sx * F));
        const float q = __fdividef(1.0f, 1.0f + expf(-(float)a.alpha * (p - rr)));
        const float A = (float)a.alpha * q * (1.0f - q) * p;
        D[e] = g[e] * ((1.0f - 2.0f * q) + 4.0f * beta * A * sx * F);
        G[e] = g[e] * (4.0f * beta * A * sx * sx);
        sb += (double)(g[e] * (4.0f * A * sx * sx * F));
        sh += (double)G[e];
    }
}

__global__ void __launch_bounds__(256) dmc_march_backward_kernel(DmcArgs a, const float* __restrict__ src, const float* __restrict__ Jh,
                                                                 const float* __restrict__ Jv, const float* __restrict__ gnew,
                                                                 float* __restrict__ gprev, float* __restrict__ gJh,
                                                                 float* __restrict__ gJv, double* gbeta, double* gh, int R, int tiles) {
    __shared__ float sEdge[3][256][2];                       // [row slot][chunk][first, last] of G
    __shared__ double red[2][8];
    const int L = a.L, cpr = L >> 3, cidx = threadIdx.x;
    const int b = blockIdx.x / tiles, tile = blockIdx.x - b * tiles;
    const int i0 = tile * R, rows = min(R, L - i0);
    const size_t base = (size_t)b * L * L;
    const float beta = (float)a.beta[b];
    const int j0 = cidx << 3;
    const int jl = j0 == 0 ? L - 1 : j0 - 1, jr = j0 + 8 == L ? 0 : j0 + 8;
    const int cl = cidx == 0 ? cpr - 1 : cidx - 1, cr = cidx == cpr - 1 ? 0 : cidx + 1;
    auto wrapi = [L](int i) { return i < 0 ? i + L : (i >= L ? i - L : i); };
    double sb = 0.0, sh = 0.0;
    // the step for row i computes G_i, D_i (rows i0 - 1 .. i0 + rows) and finishes row i - 1 (rows i0 .. i0 + rows - 1)
    float Sm[8], Sc[8], Sp[8], Sn[8];                         // state rows i-1, i, i+1, prefetched i+2
    float Gm[8], Gc[8], Gn[8], Dc[8], Dn[8];                  // G rows i-2, i-1, i; D rows i-1, i
    float JhC[8], JhP[8], JhN[8], JvM[8], JvC[8], JvP2[8], JvN[8], gC[8], gN[8];
    float jhlC, jhlP = 0.f, jhlN, slC, srC, slN, srN, srP = 0.f;
    int i = wrapi(i0 - 1);
    load8(src + base + (size_t)wrapi(i - 1) * L + j0, Sm);
    load8(src + base + (size_t)i * L + j0, Sc);
    load8(src + base + (size_t)wrapi(i + 1) * L + j0, Sp);
    load8(Jh + base + (size_t)i * L + j0, JhC);
    load8(Jv + base + (size_t)wrapi(i - 1) * L + j0, JvM);
    load8(Jv + base + (size_t)i * L + j0, JvC);
    load8(gnew + base + (size_t)i * L + j0, gC);
    jhlC = Jh[base + (size_t)i * L + jl];
    slC = src[base + (size_t)i * L + jl];
    srC = src[base + (size_t)i * L + jr];
#pragma unroll
    for (int e = 0; e < 8; ++e) { Gm[e] = 0.f; Gc[e] = 0.f; Dc[e] = 0.f; JhP[e] = 0.f; JvP2[e] = 0.f; }
    for (int step = 0; step < rows + 2; ++step) {
        const int inext = i == L - 1 ? 0 : i + 1;
        const int inn = inext == L - 1 ? 0 : inext + 1;
        const bool more = step + 1 < rows + 2;
        if (more) {
            load8(src + base + (size_t)inn * L + j0, Sn);
            load8(Jh + base + (size_t)inext * L + j0, JhN);
            load8(Jv + base + (size_t)inext * L + j0, JvN);
            load8(gnew + base + (size_t)inext * L + j0, gN);
            jhlN = Jh[base + (size_t)inext * L + jl];
            slN = src[base + (size_t)inext * L + jl];
            srN = src[base + (size_t)inext * L + jr];
        }
        // the gradient rows this step will update (row i - 1): issue their loads now, use them after the barrier
        const int ipre = i == 0 ? L - 1 : i - 1;
        const size_t offpre = base + (size_t)ipre * L + j0;
        float ah[8], av[8];
        if (step >= 2) { load8(gJh + offpre, ah); load8(gJv + offpre, av); }
        {   // G_i, D_i; the beta / h sums count interior rows only (the halo rows belong to the neighbouring tiles)
            uint32_t r[4];
            philox4x32_10(a.rk, (uint32_t)i * (uint32_t)(L >> 3) + (uint32_t)cidx, (uint32_t)b + a.replica_offset, a.c2, a.c3, r);
            double tb = 0.0, th = 0.0;
            if (((i + a.colour) & 1) == 0) dmc_chunk_bwd_par<0>(a, r, Sc, Sm, Sp, slC, srC, JhC, jhlC, JvM, JvC, beta, gC, Gn, Dn, tb, th);
            else dmc_chunk_bwd_par<1>(a, r, Sc, Sm, Sp, slC, srC, JhC, jhlC, JvM, JvC, beta, gC, Gn, Dn, tb, th);
            if (step >= 1 && step <= rows) { sb += tb; sh += th; }
        }
        const int slot = step % 3;
        sEdge[slot][cidx][0] = Gn[0];
        sEdge[slot][cidx][1] = Gn[7];
        __syncthreads();
        if (step >= 2) {
            // finish row ip = i - 1: G_{i-2} = Gm, G_{i-1} = Gc, G_i = Gn; state rows: s_{i-1} = Sm, s_i = Sc;
            // couplings: Jh_{i-1} = JhP (left edge jhlP), Jv_{i-2} = JvP2, Jv_{i-1} = JvM
            const int ip = i == 0 ? L - 1 : i - 1;
            const int ps = (step + 2) % 3;
            const float gl = sEdge[ps][cl][1], gr = sEdge[ps][cr][0];
            const size_t off = offpre;
            float out[8];
#pragma unroll
            for (int e = 0; e < 8; ++e) {
                const float gleft = e == 0 ? gl : Gc[e > 0 ? e - 1 : 0];
                const float gright = e == 7 ? gr : Gc[e < 7 ? e + 1 : 7];
                const float jleft = e == 0 ? jhlP : JhP[e > 0 ? e - 1 : 0];
                const float sright = e == 7 ? srP : Sm[e < 7 ? e + 1 : 7];
                out[e] = Dc[e] + (Gm[e] * JvP2[e] + Gn[e] * JvM[e] + gleft * jleft + gright * JhP[e]);
                ah[e] += Gc[e] * sright + gright * Sm[e];
                av[e] += Gc[e] * Sc[e] + Gn[e] * Sm[e];
            }
            store8(gprev + off, out);
            store8(gJh + off, ah);
            store8(gJv + off, av);
        }
#pragma unroll
        for (int e = 0; e < 8; ++e) {
            Gm[e] = Gc[e]; Gc[e] = Gn[e]; Dc[e] = Dn[e];
            JhP[e] = JhC[e]; JvP2[e] = JvM[e]; JvM[e] = JvC[e];
            Sm[e] = Sc[e]; Sc[e] = Sp[e];
            if (more) { Sp[e] = Sn[e]; JhC[e] = JhN[e]; JvC[e] = JvN[e]; gC[e] = gN[e]; }
        }
        jhlP = jhlC; srP = srC;
        if (more) { jhlC = jhlN; slC = slN; srC = srN; }
        i = inext;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        sb += __shfl_xor_sync(0xFFFFFFFFu, sb, o);
        sh += __shfl_xor_sync(0xFFFFFFFFu, sh, o);
    }
    if ((threadIdx.x & 31) == 0) { red[0][threadIdx.x >> 5] = sb; red[1][threadIdx.x >> 5] = sh; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double tb = 0.0, th = 0.0;
        for (int k = 0; k < (int)((blockDim.x + 31) >> 5); ++k) { tb += red[0][k]; th += red[1][k]; }
        atomicAdd(gbeta + b, tb);
        atomicAdd(gh + b, th);
    }
}

// Backward pass 1: blocks never straddle replicas (grid = blocks per replica x batch), so the beta / h sums reduce per block.
template <typename T, int V>
__global__ void __launch_bounds__(256) dmc_backward1_kernel(DmcArgs a, const T* __restrict__ src, const T* __restrict__ Jh,
                                                            const T* __restrict__ Jv, const T* __restrict__ gnew,
                                                            T* __restrict__ D, T* __restrict__ G, double* gbeta, double* gh,
                                                            int bpr) {
    __shared__ double red[2][8];
    const int vpr = a.L / V;
    const int per = a.L * vpr;
    const int b = blockIdx.x / bpr, blk = blockIdx.x - b * bpr;
    const int u = blk * blockDim.x + threadIdx.x;
    double sb = 0.0, sh = 0.0;
    if (u < per) {
        const int i = u / vpr, x = u - i * vpr;
        Sites<T, V> st;
        eval_sites<T, V>(a, src, Jh, Jv, b, i, x * V, st);
        const size_t off = (size_t)b * a.L * a.L + (size_t)i * a.L + x * V;
        const Vec<T, V> g = *(const Vec<T, V>*)(gnew + off);
        const T beta = (T)a.beta[b];
        Vec<T, V> d, gg;
#pragma unroll
        for (int e = 0; e < V; ++e) {
            if (!st.upd[e]) { d.v[e] = g.v[e]; gg.v[e] = (T)0; continue; }
            const T A = (T)a.alpha * st.q[e] * ((T)1 - st.q[e]) * st.p[e];
            const T s = st.s[e];
            d.v[e] = g.v[e] * (((T)1 - (T)2 * st.q[e]) + (T)4 * beta * A * s * st.F[e]);
            gg.v[e] = g.v[e] * ((T)4 * beta * A * s * s);
            sb += (double)(g.v[e] * ((T)4 * A * s * s * st.F[e]));
            sh += (double)gg.v[e];
        }
        *(Vec<T, V>*)(D + off) = d;
        *(Vec<T, V>*)(G + off) = gg;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        sb += __shfl_xor_sync(0xFFFFFFFFu, sb, o);
        sh += __shfl_xor_sync(0xFFFFFFFFu, sh, o);
    }
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    if (lane == 0) { red[0][w] = sb; red[1][w] = sh; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double tb = 0.0, th = 0.0;
        for (int k = 0; k < (int)(blockDim.x >> 5); ++k) { tb += red[0][k]; th += red[1][k]; }
        atomicAdd(gbeta + b, tb);
        atomicAdd(gh + b, th);
    }
}

// Backward pass 2, all sites: g_prev = D + sum_n G_n J_xn (in place in D), and the coupling gradients.
template <typename T, int V>
__global__ void __launch_bounds__(256) dmc_backward2_kernel(int batch, int L, const T* __restrict__ src,
                                                            const T* __restrict__ Jh, const T* __restrict__ Jv,
                                                            const T* __restrict__ G, T* __restrict__ D, T* __restrict__ gJh,
                                                            T* __restrict__ gJv) {
    const int vpr = L / V;
    const long long total = (long long)batch * L * vpr;
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gid >= total) return;
    const int x = (int)(gid % vpr);
    const long long bi = gid / vpr;
    const int i = (int)(bi % L), b = (int)(bi / L);
    const int j0 = x * V;
    const size_t base = (size_t)b * L * L;
    const int iu = i == 0 ? L - 1 : i - 1, id = i == L - 1 ? 0 : i + 1;
    const int jl = j0 == 0 ? L - 1 : j0 - 1, jr = j0 + V == L ? 0 : j0 + V;
    const size_t off = base + (size_t)i * L + j0, offu = base + (size_t)iu * L + j0, offd = base + (size_t)id * L + j0;
    const Vec<T, V> gc = *(const Vec<T, V>*)(G + off), gu = *(const Vec<T, V>*)(G + offu), gd = *(const Vec<T, V>*)(G + offd);
    const Vec<T, V> sc = *(const Vec<T, V>*)(src + off), sd = *(const Vec<T, V>*)(src + offd);
    const Vec<T, V> jh = *(const Vec<T, V>*)(Jh + off), jvu = *(const Vec<T, V>*)(Jv + offu), jvc = *(const Vec<T, V>*)(Jv + off);
    const T gl = G[base + (size_t)i * L + jl], gr = G[base + (size_t)i * L + jr];
    const T jhl = Jh[base + (size_t)i * L + jl], sr = src[base + (size_t)i * L + jr];
    Vec<T, V> d = *(const Vec<T, V>*)(D + off);
    Vec<T, V> ah = *(const Vec<T, V>*)(gJh + off), av = *(const Vec<T, V>*)(gJv + off);
#pragma unroll
    for (int e = 0; e < V; ++e) {
        const T gleft = e == 0 ? gl : gc.v[e > 0 ? e - 1 : 0];
        const T gright = e == V - 1 ? gr : gc.v[e < V - 1 ? e + 1 : V - 1];
        const T jleft = e == 0 ? jhl : jh.v[e > 0 ? e - 1 : 0];
        const T sright = e == V - 1 ? sr : sc.v[e < V - 1 ? e + 1 : V - 1];
        d.v[e] += gu.v[e] * jvu.v[e] + gd.v[e] * jvc.v[e] + gleft * jleft + gright * jh.v[e];
        ah.v[e] += gc.v[e] * sright + gright * sc.v[e];
        av.v[e] += gc.v[e] * sd.v[e] + gd.v[e] * sc.v[e];
    }
    *(Vec<T, V>*)(D + off) = d;
    *(Vec<T, V>*)(gJh + off) = ah;
    *(Vec<T, V>*)(gJv + off) = av;
}

template <typename T>
__global__ void dmc_discretise_kernel(T* s, long long n) {
    const long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (k < n) s[k] = s[k] < (T)0 ? (T)-1 : (T)1;             // Eq. 4
}

}  // namespace
}  // namespace spin

// ---- host side ---------------------------------------------------------------------------------------------------
namespace {

using namespace spin;

int dmc_fail(int code, const char* msg) { return spin::set_error(code, msg); }   // thread-local spin_last_error (spin_api.cu)

struct DmcShape {
    int32_t batch, L, dtype;
    size_t elems() const { return (size_t)batch * L * L; }
    size_t bytes() const { return elems() * (dtype == SPIN_DTYPE_F64 ? 8 : 4); }
};

int check_common(int32_t batch, int32_t L, int32_t dtype, const double* beta, double h, double alpha, int64_t replica_offset,
                 int64_t n_sweeps, int64_t sweep_offset) {
    if (batch < 1 || L < 2 || (L & 1) || L > 65536) return dmc_fail(SPIN_ERR_INVALID, "spin_dmc: batch >= 1 and even L in 2..65536 required");
    if (dtype != SPIN_DTYPE_F32 && dtype != SPIN_DTYPE_F64) return dmc_fail(SPIN_ERR_INVALID, "spin_dmc: dtype must be SPIN_DTYPE_F32 or SPIN_DTYPE_F64");
    if (!beta) return dmc_fail(SPIN_ERR_INVALID, "spin_dmc: beta is NULL");
    for (int b = 0; b < batch; ++b)
        if (!std::isfinite(beta[b]) || beta[b] < 0.0) return dmc_fail(SPIN_ERR_INVALID, "spin_dmc: beta must be finite and >= 0");
    if (!std::isfinite(h) || !std::isfinite(alpha) || alpha < 0.0) return dmc_fail(SPIN_ERR_INVALID, "spin_dmc: h finite and alpha finite, >= 0 required");
    if (replica_offset < 0 || replica_offset + (int64_t)batch > (1ll << 32)) return dmc_fail(SPIN_ERR_INVALID, "spin_dmc: replica_offset + batch must stay within [0, 2^32]");
    if (n_sweeps < 0 || sweep_offset < 0 || sweep_offset > (1ll << 56) || n_sweeps > (1ll << 56) || sweep_offset + n_sweeps > (1ll << 56))
        return dmc_fail(SPIN_ERR_INVALID, "spin_dmc: sweep range must lie in [0, 2^56]");
    return SPIN_OK;
}

// The temporaries come from the device's default stream-ordered pool; keep freed blocks cached in the pool (the default
// release threshold of 0 returns them to the driver at every synchronisation, which costs milliseconds per call).
void keep_pool_memory() {
    int dev = 0;
    cudaMemPool_t pool;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetDefaultMemPool(&pool, dev) != cudaSuccess) { cudaGetLastError(); return; }
    unsigned long long keep = ~0ull;
    cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
    cudaGetLastError();
}

DmcArgs make_args(int32_t batch, int32_t L, double h, double alpha, const double* d_beta, uint64_t seed,
                  int64_t replica_offset, int64_t t, int colour) {
    DmcArgs a;
    a.batch = batch; a.L = L; a.replica_offset = (uint32_t)replica_offset;
    a.c2 = (uint32_t)((uint64_t)t & 0xFFFFFFFFull);
    a.c3 = (uint32_t)(((uint64_t)t >> 32) & 0xFFFFFFull) | ((uint32_t)colour << 24) | ((uint32_t)kDomainIsing << 28);
    a.colour = colour; a.h = h; a.alpha = alpha; a.beta = d_beta;
    uint32_t k0 = (uint32_t)(seed & 0xFFFFFFFFull), k1 = (uint32_t)(seed >> 32);
    for (int r = 0; r < 10; ++r) { a.rk.k0[r] = k0; a.rk.k1[r] = k1; k0 += kPhiloxW0; k1 += kPhiloxW1; }
    return a;
}

template <typename T, int V>
void launch_forward(const DmcArgs& a, const void* src, void* dst, const void* Jh, const void* Jv, cudaStream_t s) {
    const long long total = (long long)a.batch * a.L * (a.L / V);
    dmc_forward_kernel<T, V><<<(unsigned)((total + 255) / 256), 256, 0, s>>>(a, (const T*)src, (T*)dst, (const T*)Jh, (const T*)Jv);
}

// Rows per tile of the fused sweep: (R + 2) rows of L floats in at most 64 KiB (96 KiB for L > 1024) of shared memory.
int fused_tile_rows(int L) {
    const int budget = L > 1024 ? 96 * 1024 : 64 * 1024;
    int R = budget / (4 * L) - 2;
    if (R > 64) R = 64;
    if (R > L) R = L;
    return R;
}
bool fused_ok(int dtype, int L) { return dtype == SPIN_DTYPE_F32 && L % 8 == 0 && L <= 2048 && fused_tile_rows(L) >= 4; }

cudaError_t forward_sweep_fused(const DmcArgs& a, const void* src, void* mid, void* dst, const void* Jh, const void* Jv,
                                cudaStream_t s) {
    if (a.L >= 256) {                                         // row-marching kernel: one block = one row of chunks, R rows per tile
        const int R = 32, tiles = (a.L + R - 1) / R;
        dmc_march_sweep_kernel<<<(unsigned)((long long)tiles * a.batch), a.L >> 3, 0, s>>>(a, (const float*)src, (float*)mid, (float*)dst,
                                                                                         (const float*)Jh, (const float*)Jv, R, tiles);
        return cudaGetLastError();
    }
    const int R = fused_tile_rows(a.L), tiles = (a.L + R - 1) / R;
    const size_t smem = (size_t)(R + 2) * a.L * sizeof(float);
    cudaError_t e = cudaFuncSetAttribute(dmc_fused_sweep_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024);
    if (e != cudaSuccess) return e;
    dmc_fused_sweep_kernel<<<(unsigned)((long long)tiles * a.batch), 256, smem, s>>>(a, (const float*)src, (float*)mid, (float*)dst,
                                                                                   (const float*)Jh, (const float*)Jv, R, tiles);
    return cudaGetLastError();
}

void forward_half(int dtype, const DmcArgs& a, const void* src, void* dst, const void* Jh, const void* Jv, cudaStream_t s) {
    if (dtype == SPIN_DTYPE_F64) launch_forward<double, 2>(a, src, dst, Jh, Jv, s);
    else if (a.L % 4 == 0) launch_forward<float, 4>(a, src, dst, Jh, Jv, s);
    else launch_forward<float, 2>(a, src, dst, Jh, Jv, s);
}

template <typename T, int V>
void launch_backward(const DmcArgs& a, const void* src, const void* Jh, const void* Jv, const void* gnew, void* D, void* G,
                     double* gbeta, double* gh, void* gJh, void* gJv, cudaStream_t s) {
    const int per = a.L * (a.L / V);
    const int bpr = (per + 255) / 256;
    dmc_backward1_kernel<T, V><<<(unsigned)((long long)bpr * a.batch), 256, 0, s>>>(a, (const T*)src, (const T*)Jh, (const T*)Jv,
                                                                                  (const T*)gnew, (T*)D, (T*)G, gbeta, gh, bpr);
    const long long total = (long long)a.batch * per;
    dmc_backward2_kernel<T, V><<<(unsigned)((total + 255) / 256), 256, 0, s>>>(a.batch, a.L, (const T*)src, (const T*)Jh,
                                                                              (const T*)Jv, (const T*)G, (T*)D, (T*)gJh, (T*)gJv);
}

void backward_half(int dtype, const DmcArgs& a, const void* src, const void* Jh, const void* Jv, const void* gnew, void* D,
                   void* G, double* gbeta, double* gh, void* gJh, void* gJv, cudaStream_t s) {
    if (dtype == SPIN_DTYPE_F32 && a.L % 8 == 0 && a.L >= 256 && a.L <= 2048) {
        const int R = 32, tiles = (a.L + R - 1) / R;          // fused row-marching kernel: g_prev lands in D, G is unused
        dmc_march_backward_kernel<<<(unsigned)((long long)tiles * a.batch), a.L >> 3, 0, s>>>(
            a, (const float*)src, (const float*)Jh, (const float*)Jv, (const float*)gnew, (float*)D, (float*)gJh, (float*)gJv, gbeta, gh,
            R, tiles);
        return;
    }
    if (dtype == SPIN_DTYPE_F64) launch_backward<double, 2>(a, src, Jh, Jv, gnew, D, G, gbeta, gh, gJh, gJv, s);
    else if (a.L % 4 == 0) launch_backward<float, 4>(a, src, Jh, Jv, gnew, D, G, gbeta, gh, gJh, gJv, s);
    else launch_backward<float, 2>(a, src, Jh, Jv, gnew, D, G, gbeta, gh, gJh, gJv, s);
}

#define DMC_TRY(expr)                                                                             \
    do {                                                                                          \
        cudaError_t e_ = (expr);                                                                  \
        if (e_ != cudaSuccess) { rc = dmc_fail(SPIN_ERR_CUDA, cudaGetErrorString(e_)); goto done; } \
    } while (0)

}  // namespace

extern "C" {

int spin_dmc_forward(int32_t batch, int32_t L, int32_t dtype, const void* s0, const void* Jh, const void* Jv, double h,
                     const double* beta, double alpha, uint64_t seed, int64_t replica_offset, int64_t n_sweeps,
                     int64_t sweep_offset, void* s_out, void* traj, void* cuda_stream) {
    int rc = check_common(batch, L, dtype, beta, h, alpha, replica_offset, n_sweeps, sweep_offset);
    if (rc != SPIN_OK) return rc;
    if (!s0 || !Jh || !Jv || !s_out) return dmc_fail(SPIN_ERR_INVALID, "spin_dmc_forward: NULL device pointer");
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const DmcShape sh{batch, L, dtype};
    const size_t bytes = sh.bytes();
    double* d_beta = nullptr;
    void* tmp = nullptr;
    keep_pool_memory();
    DMC_TRY(cudaMallocAsync(&d_beta, sizeof(double) * batch, s));
    DMC_TRY(cudaMemcpyAsync(d_beta, beta, sizeof(double) * batch, cudaMemcpyHostToDevice, s));
    if (traj) DMC_TRY(cudaMemcpyAsync(traj, s0, bytes, cudaMemcpyDeviceToDevice, s));
    else if (n_sweeps > 0) DMC_TRY(cudaMallocAsync(&tmp, bytes, s));
    if (fused_ok(dtype, L)) {
        // one kernel per sweep: state 2k -> (state 2k+1 into the trajectory, if any) -> state 2k+2.  Out of place, so
        // without a trajectory the sweeps ping-pong between tmp and s_out, ending in s_out.
        const void* cur = s0;
        for (int64_t k = 0; k < n_sweeps; ++k) {
            void* mid = traj ? (void*)((char*)traj + (size_t)(2 * k + 1) * bytes) : nullptr;
            void* dst = traj ? (void*)((char*)traj + (size_t)(2 * k + 2) * bytes) : (((n_sweeps - k) & 1) ? s_out : tmp);
            if (!traj && dst == cur) dst = (dst == s_out) ? tmp : s_out;      // s0 == s_out on the first sweep
            const DmcArgs a = make_args(batch, L, h, alpha, d_beta, seed, replica_offset, sweep_offset + k, 0);
            DMC_TRY(forward_sweep_fused(a, cur, mid, dst, Jh, Jv, s));
            cur = dst;
        }
        if (cur != s_out) DMC_TRY(cudaMemcpyAsync(s_out, cur, bytes, cudaMemcpyDeviceToDevice, s));
    } else {
        const void* cur = s0;
        for (int64_t k = 0; k < n_sweeps; ++k)
            for (int c = 0; c < 2; ++c) {
                // with a trajectory: state 2k+c -> state 2k+c+1; without: ping-pong so that the last state lands in s_out
                void* dst = traj ? (void*)((char*)traj + (size_t)(2 * k + c + 1) * bytes) : (c == 0 ? tmp : s_out);
                const DmcArgs a = make_args(batch, L, h, alpha, d_beta, seed, replica_offset, sweep_offset + k, c);
                forward_half(dtype, a, cur, dst, Jh, Jv, s);
                cur = dst;
            }
        if (cur != s_out) DMC_TRY(cudaMemcpyAsync(s_out, cur, bytes, cudaMemcpyDeviceToDevice, s));
    }
    DMC_TRY(cudaGetLastError());
done:
    if (tmp) cudaFreeAsync(tmp, s);
    if (d_beta) cudaFreeAsync(d_beta, s);
    return rc;
}

int spin_dmc_backward(int32_t batch, int32_t L, int32_t dtype, const void* traj, const void* Jh, const void* Jv, double h,
                      const double* beta, double alpha, uint64_t seed, int64_t replica_offset, int64_t n_sweeps,
                      int64_t sweep_offset, const void* grad_out, void* grad_s0, void* grad_Jh, void* grad_Jv,
                      double* grad_beta, double* grad_h, void* cuda_stream) {
    int rc = check_common(batch, L, dtype, beta, h, alpha, replica_offset, n_sweeps, sweep_offset);
    if (rc != SPIN_OK) return rc;
    if (!traj || !Jh || !Jv || !grad_out || !grad_s0 || !grad_Jh || !grad_Jv)
        return dmc_fail(SPIN_ERR_INVALID, "spin_dmc_backward: NULL device pointer");
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const DmcShape sh{batch, L, dtype};
    const size_t bytes = sh.bytes();
    double* d_small = nullptr;     // [beta | grad_beta | grad_h]
    void* ws = nullptr;            // [g ping | g pong | G]
    keep_pool_memory();
    DMC_TRY(cudaMallocAsync(&d_small, sizeof(double) * 3 * batch, s));
    DMC_TRY(cudaMemcpyAsync(d_small, beta, sizeof(double) * batch, cudaMemcpyHostToDevice, s));
    DMC_TRY(cudaMemsetAsync(d_small + batch, 0, sizeof(double) * 2 * batch, s));
    DMC_TRY(cudaMallocAsync(&ws, 3 * bytes, s));
    DMC_TRY(cudaMemsetAsync(grad_Jh, 0, bytes, s));
    DMC_TRY(cudaMemsetAsync(grad_Jv, 0, bytes, s));
    {
        char* g0 = (char*)ws;
        char* g1 = g0 + bytes;
        void* G = g1 + bytes;
        const void* gnew = grad_out;
        int flip = 0;
        for (int64_t k = n_sweeps - 1; k >= 0; --k)
            for (int c = 1; c >= 0; --c) {
                const void* before = (const char*)traj + (size_t)(2 * k + c) * bytes;
                void* D = flip ? g1 : g0;
                const DmcArgs a = make_args(batch, L, h, alpha, d_small, seed, replica_offset, sweep_offset + k, c);
                backward_half(dtype, a, before, Jh, Jv, gnew, D, G, d_small + batch, d_small + 2 * batch, grad_Jh, grad_Jv, s);
                gnew = D;
                flip ^= 1;
            }
        DMC_TRY(cudaMemcpyAsync(grad_s0, gnew, bytes, cudaMemcpyDeviceToDevice, s));
    }
    DMC_TRY(cudaGetLastError());
    if (grad_beta) DMC_TRY(cudaMemcpyAsync(grad_beta, d_small + batch, sizeof(double) * batch, cudaMemcpyDeviceToHost, s));
    if (grad_h) DMC_TRY(cudaMemcpyAsync(grad_h, d_small + 2 * batch, sizeof(double) * batch, cudaMemcpyDeviceToHost, s));
    if (grad_beta || grad_h) DMC_TRY(cudaStreamSynchronize(s));
done:
    if (ws) cudaFreeAsync(ws, s);
    if (d_small) cudaFreeAsync(d_small, s);
    return rc;
}

int spin_dmc_discretise(int32_t dtype, void* s, int64_t n, void* cuda_stream) {
    if (!s || n < 0) return dmc_fail(SPIN_ERR_INVALID, "spin_dmc_discretise: NULL pointer or negative count");
    if (dtype != SPIN_DTYPE_F32 && dtype != SPIN_DTYPE_F64) return dmc_fail(SPIN_ERR_INVALID, "spin_dmc_discretise: unknown dtype");
    if (n == 0) return SPIN_OK;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const unsigned grid = (unsigned)((n + 255) / 256);
    if (dtype == SPIN_DTYPE_F64) spin::dmc_discretise_kernel<double><<<grid, 256, 0, st>>>((double*)s, n);
    else spin::dmc_discretise_kernel<float><<<grid, 256, 0, st>>>((float*)s, n);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return dmc_fail(SPIN_ERR_CUDA, cudaGetErrorString(e));
    return SPIN_OK;
}

}  // extern "C"
