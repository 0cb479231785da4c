// ORACLE — TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, slow, single-threaded CPU implementation of the hot path of
// arXiv 2304.01772 ("A differentiable programming framework for spin models"):
// the checkerboard Metropolis sweep over a batch of 2D periodic lattices (Ising and
// q-state Potts) and the per-replica energy / magnetisation reductions.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
// legs may build, load or call this file.  It shares no code, header, table or constant
// generator with the CUDA library under paper_2304_01772_b200/csrc/, and neither
// includes the other.
//
// What it follows (line numbers are /root/reference/PAPER.md):
//   * Algorithm 1 "Standard Metropolis-Hastings algorithm with parallelization"
//     (PAPER.md:127-138): propose, local energy of both states, checkerboard colour,
//     dE per site of one colour, accept if dE <= 0 else with probability exp(-beta dH).
//   * Checkerboard method (Fig. 1): black squares first, then white.
//   * Ising Hamiltonian Eq. 1 with the 4-neighbour kernel Eq. 2
//     (PAPER.md:105-115): local energy = spin x (sum of up/down/left/right).
//   * Potts Hamiltonian Eq. 5, four one-neighbour kernels Eq. 6
//     with a Kronecker delta, proposal uniform over the q-1 other
//     states.
//   * Batch dimension = independent lattices / temperatures.
// Where the paper is silent the readings of DESIGN.md section 3 (= SURVEY.md section 8(c),
// O1-O8 and P1-P17) are taken; each is marked "reading Pn" below.
//
// Sign convention (reading P1): H = -J sum_<ij> s_i s_j - h sum_i s_i (Ising),
// H = -J sum_<ij> delta(s_i,s_j) (Potts).  The paper writes H = +sum J s s with the
// ferromagnet at J<0, so J_here = -J_paper, h_here = -B_paper.
//
// Data layout: natural, row-major int8 lattices [batch][L][L]; Ising spins are -1/+1,
// Potts states are 0..q-1.  No tiling, no vectorisation, no colour-split storage: one site
// at a time, in the order "for colour, for replica, for row, for column".
//
// Pins (tests/test_oracle_*.py, all `-m "not gpu"`): Philox known-answer vectors; threshold
// tables against closed-form values; beta=0 all-flip; Z2 mirror; chunking and replica
// independence; parity/bound invariants of E and M; exact enumeration of the 4x4 Ising torus
// and of 2x2 / 4x4 Potts tori; Onsager's energy at beta=0.30 and 0.60 on L=128; half-sweep
// detailed balance and sweep stationarity on 2x2 from the transition matrix; Potts self-dual
// point bracket; T->0 monotone energy and ground-state fixed points.  Every exported function
// below is covered by at least one of these; none is "parity unpinned".

#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>

namespace {

// ---- O2: Philox-4x32, 10 rounds (Salmon et al., "Parallel random numbers: as easy as
// 1, 2, 3", SC'11).  Multipliers and Weyl key increments are the published constants.
const uint32_t PHILOX_M0 = 0xD2511F53u;  // multiplies counter word 0
const uint32_t PHILOX_M1 = 0xCD9E8D57u;  // multiplies counter word 2
const uint32_t PHILOX_W0 = 0x9E3779B9u;  // key[0] increment per round
const uint32_t PHILOX_W1 = 0xBB67AE85u;  // key[1] increment per round

void philox4x32_10(const uint32_t ctr_in[4], const uint32_t key_in[2], uint32_t out[4]) {
    uint32_t c0 = ctr_in[0], c1 = ctr_in[1], c2 = ctr_in[2], c3 = ctr_in[3];
    uint32_t k0 = key_in[0], k1 = key_in[1];
    for (int round = 0; round < 10; ++round) {
        if (round > 0) { k0 += PHILOX_W0; k1 += PHILOX_W1; }
        uint64_t p0 = (uint64_t)PHILOX_M0 * (uint64_t)c0;
        uint64_t p1 = (uint64_t)PHILOX_M1 * (uint64_t)c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

enum { DOMAIN_INIT = 0, DOMAIN_ISING = 1, DOMAIN_POTTS = 2 };

// O2 counter assembly: c0 = group, c1 = replica, c2 = low 32 bits of the sweep index t,
// c3 = bits 32..55 of t | colour << 24 | domain << 28.  Key = (seed low, seed high).
void draw(uint64_t seed, uint32_t group, uint32_t replica, uint64_t t, uint32_t colour,
          uint32_t domain, uint32_t out[4]) {
    uint32_t ctr[4];
    ctr[0] = group;
    ctr[1] = replica;
    ctr[2] = (uint32_t)(t & 0xFFFFFFFFull);
    ctr[3] = (uint32_t)((t >> 32) & 0xFFFFFFull) | (colour << 24) | (domain << 28);
    uint32_t key[2] = {(uint32_t)(seed & 0xFFFFFFFFull), (uint32_t)(seed >> 32)};
    philox4x32_10(ctr, key, out);
}

inline int wrap(int a, int L) { return a < 0 ? a + L : (a >= L ? a - L : a); }

// O4: acceptance of one class.  x = beta*dE; x <= 0 -> always (Alg. 1 line 6, "dE <= 0
// accept", reading P5); else threshold floor(exp(-x) 2^32) clipped to 2^32-1
// (Alg. 1 line 9, p = exp(-beta dH); reading P6).
void threshold(double beta, double dE, uint32_t* T, uint8_t* always) {
    double x = beta * dE;
    if (x <= 0.0) { *always = 1; *T = 0xFFFFFFFFu; return; }
    double v = std::floor(std::exp(-x) * 4294967296.0);
    *always = 0;
    *T = (v >= 4294967295.0) ? 0xFFFFFFFFu : (uint32_t)v;
}

inline bool accept(uint32_t r, uint32_t T, uint8_t always) { return always || r < T; }

}  // namespace

extern "C" {

// O2.  Exposed for the known-answer pin Q1.
void oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    philox4x32_10(ctr, key, out);
}

// O2 counter assembly and O4 acceptance of one class, exported unchanged for the other oracle files (general_oracle.cpp).
void oracle_draw(uint64_t seed, uint32_t group, uint32_t replica, uint64_t t, uint32_t colour, uint32_t domain,
                 uint32_t out[4]) {
    draw(seed, group, replica, t, colour, domain, out);
}
void oracle_threshold(double beta, double dE, uint32_t* T, uint8_t* always) { threshold(beta, dE, T, always); }

// O4, Ising.  Class index = 5*(s+1)/2 + (nn+4)/2; dE of flipping s with neighbour sum nn is
// H(-s) - H(s) = 2 s (J nn + h) (Eq. 1 with reading P1; local energy = spin x neighbour sum,
// PAPER.md:123).
void oracle_ising_table(double beta, double J, double h, uint32_t T[10], uint8_t always[10]) {
    for (int si = 0; si < 2; ++si) {
        for (int ni = 0; ni < 5; ++ni) {
            double s = si == 0 ? -1.0 : 1.0;
            double nn = (double)(2 * ni - 4);
            double dE = 2.0 * s * (J * nn + h);
            threshold(beta, dE, &T[5 * si + ni], &always[5 * si + ni]);
        }
    }
}

// O4, Potts.  Class index = dn+4, dn = n_new - n_old in -4..4; dE = -J dn (Eq. 5, P1).
void oracle_potts_table(double beta, double J, uint32_t T[9], uint8_t always[9]) {
    for (int di = 0; di < 9; ++di) {
        double dn = (double)(di - 4);
        double dE = -(J * dn);
        threshold(beta, dE, &T[di], &always[di]);
    }
}

// O3 / a0: initial lattice from Philox(seed), domain INIT, t = 0, colour 0, group = p>>2,
// word = out[p&3] with p = i*L + j.  Ising: +1 iff bit 31 set.  Potts: (word*q) >> 32.
// q[b] == 2 with model Ising; q[b] in 2..127 with model Potts.
void oracle_init(int8_t* spins, int32_t batch, int32_t L, int32_t model_potts, const int32_t* q,
                 uint64_t seed, int64_t replica_offset) {
    const int64_t N = (int64_t)L * L;
    for (int32_t b = 0; b < batch; ++b) {
        int8_t* lat = spins + (int64_t)b * N;
        uint32_t replica = (uint32_t)(b + replica_offset);
        for (int64_t p = 0; p < N; ++p) {
            uint32_t out[4];
            draw(seed, (uint32_t)(p >> 2), replica, 0, 0, DOMAIN_INIT, out);
            uint32_t word = out[p & 3];
            if (!model_potts) {
                lat[p] = (word & 0x80000000u) ? (int8_t)1 : (int8_t)-1;
            } else {
                lat[p] = (int8_t)(((uint64_t)word * (uint64_t)q[b]) >> 32);
            }
        }
    }
}

// O5 + O7 (rows a2/a3): one Ising half-sweep of colour `colour` at sweep index t.
// For every site (i,j) with (i+j)&1 == colour: s = sigma(i,j), nn = up+down+left+right with
// periodic wrap and multiplicity (O1), class (s,nn), r = word n&3 of Philox group n>>2 where
// n = i*(L/2) + (j>>1); flip iff accepted.  Sites of one colour see only the other colour, so
// the in-place update equals the synchronous one.
void oracle_ising_half_sweep(int8_t* spins, int32_t batch, int32_t L, const double* beta, double J,
                             double h, uint64_t seed, int64_t replica_offset, int64_t t,
                             int32_t colour) {
    const int64_t N = (int64_t)L * L;
    const int half = L / 2;
    for (int32_t b = 0; b < batch; ++b) {
        uint32_t T[10];
        uint8_t always[10];
        oracle_ising_table(beta[b], J, h, T, always);
        int8_t* lat = spins + (int64_t)b * N;
        uint32_t replica = (uint32_t)(b + replica_offset);
        for (int i = 0; i < L; ++i) {
            for (int j = 0; j < L; ++j) {
                if (((i + j) & 1) != colour) continue;
                int s = lat[(int64_t)i * L + j];
                int nn = lat[(int64_t)wrap(i - 1, L) * L + j] + lat[(int64_t)wrap(i + 1, L) * L + j] +
                         lat[(int64_t)i * L + wrap(j - 1, L)] + lat[(int64_t)i * L + wrap(j + 1, L)];
                int64_t n = (int64_t)i * half + (j >> 1);
                uint32_t out[4];
                draw(seed, (uint32_t)(n >> 2), replica, (uint64_t)t, (uint32_t)colour, DOMAIN_ISING, out);
                uint32_t r = out[n & 3];
                int cls = 5 * ((s + 1) / 2) + (nn + 4) / 2;
                if (accept(r, T[cls], always[cls])) lat[(int64_t)i * L + j] = (int8_t)(-s);
            }
        }
    }
}

// O6 + O7: one Potts half-sweep.  r_prop = out[2(n&1)], r_acc = out[2(n&1)+1] of group n>>1.
// new = old + 1 + floor(r_prop (q-1) / 2^32) mod q (reading P9);
// dn = n_new - n_old counted over the 4 neighbours with multiplicity (Eq. 6).
void oracle_potts_half_sweep(int8_t* spins, int32_t batch, int32_t L, const int32_t* q,
                             const double* beta, double J, uint64_t seed, int64_t replica_offset,
                             int64_t t, int32_t colour) {
    const int64_t N = (int64_t)L * L;
    const int half = L / 2;
    for (int32_t b = 0; b < batch; ++b) {
        uint32_t T[9];
        uint8_t always[9];
        oracle_potts_table(beta[b], J, T, always);
        int8_t* lat = spins + (int64_t)b * N;
        uint32_t replica = (uint32_t)(b + replica_offset);
        const int qb = q[b];
        for (int i = 0; i < L; ++i) {
            for (int j = 0; j < L; ++j) {
                if (((i + j) & 1) != colour) continue;
                int old = lat[(int64_t)i * L + j];
                int nb[4] = {lat[(int64_t)wrap(i - 1, L) * L + j], lat[(int64_t)wrap(i + 1, L) * L + j],
                             lat[(int64_t)i * L + wrap(j - 1, L)], lat[(int64_t)i * L + wrap(j + 1, L)]};
                int64_t n = (int64_t)i * half + (j >> 1);
                uint32_t out[4];
                draw(seed, (uint32_t)(n >> 1), replica, (uint64_t)t, (uint32_t)colour, DOMAIN_POTTS, out);
                uint32_t r_prop = out[2 * (n & 1)];
                uint32_t r_acc = out[2 * (n & 1) + 1];
                int d = (int)(((uint64_t)r_prop * (uint64_t)(qb - 1)) >> 32);
                int nw = old + 1 + d;
                if (nw >= qb) nw -= qb;
                int n_old = 0, n_new = 0;
                for (int a = 0; a < 4; ++a) {
                    n_old += (nb[a] == old);
                    n_new += (nb[a] == nw);
                }
                int cls = (n_new - n_old) + 4;
                if (accept(r_acc, T[cls], always[cls])) lat[(int64_t)i * L + j] = (int8_t)nw;
            }
        }
    }
}

// O8 (rows a5/a6), Ising: S = 1/2 sum_sites s*nn (each bond once, with multiplicity; reading P2),
// E_int = -S, M = sum s.
void oracle_ising_observables(const int8_t* spins, int32_t batch, int32_t L, int64_t* E, int64_t* M) {
    const int64_t N = (int64_t)L * L;
    for (int32_t b = 0; b < batch; ++b) {
        const int8_t* lat = spins + (int64_t)b * N;
        int64_t twoS = 0, m = 0;
        for (int i = 0; i < L; ++i) {
            for (int j = 0; j < L; ++j) {
                int s = lat[(int64_t)i * L + j];
                int nn = lat[(int64_t)wrap(i - 1, L) * L + j] + lat[(int64_t)wrap(i + 1, L) * L + j] +
                         lat[(int64_t)i * L + wrap(j - 1, L)] + lat[(int64_t)i * L + wrap(j + 1, L)];
                twoS += s * nn;
                m += s;
            }
        }
        E[b] = -(twoS / 2);
        M[b] = m;
    }
}

// O8, Potts: D = 1/2 sum_sites n_same, E_int = -D, M = max_k N_k (reading P8).
void oracle_potts_observables(const int8_t* spins, int32_t batch, int32_t L, const int32_t* q,
                              int64_t* E, int64_t* M) {
    const int64_t N = (int64_t)L * L;
    for (int32_t b = 0; b < batch; ++b) {
        const int8_t* lat = spins + (int64_t)b * N;
        int64_t twoD = 0;
        int64_t count[128];
        for (int k = 0; k < 128; ++k) count[k] = 0;
        for (int i = 0; i < L; ++i) {
            for (int j = 0; j < L; ++j) {
                int s = lat[(int64_t)i * L + j];
                twoD += (lat[(int64_t)wrap(i - 1, L) * L + j] == s) + (lat[(int64_t)wrap(i + 1, L) * L + j] == s) +
                        (lat[(int64_t)i * L + wrap(j - 1, L)] == s) + (lat[(int64_t)i * L + wrap(j + 1, L)] == s);
                count[s] += 1;
            }
        }
        int64_t best = 0;
        for (int k = 0; k < q[b]; ++k) best = count[k] > best ? count[k] : best;
        E[b] = -(twoD / 2);
        M[b] = best;
    }
}

// Row a7: fold one (E_int, M) sample per replica into moments[b][8] =
// {n, sum E, sum E^2 low 64 bits, sum E^2 high 64 bits, sum M, sum |M|, sum M^2, sum E*M}
// (reading P15: sum E^2 is a 128-bit integer in two limbs; the rest are int64).
void oracle_accumulate_moments(int64_t* moments, int32_t batch, const int64_t* E, const int64_t* M) {
    for (int32_t b = 0; b < batch; ++b) {
        int64_t* m = moments + 8 * (int64_t)b;
        unsigned __int128 e2 = ((unsigned __int128)(uint64_t)m[3] << 64) | (unsigned __int128)(uint64_t)m[2];
        __int128 e = (__int128)E[b];
        e2 += (unsigned __int128)(e * e);
        m[0] += 1;
        m[1] += E[b];
        m[2] = (int64_t)(uint64_t)e2;
        m[3] = (int64_t)(uint64_t)(e2 >> 64);
        m[4] += M[b];
        m[5] += M[b] < 0 ? -M[b] : M[b];
        m[6] += M[b] * M[b];
        m[7] += E[b] * M[b];
    }
}

// Rows a2-a7 (O7): sweeps t = sweep_offset .. sweep_offset+n_sweeps-1, colour 0 then colour 1
// (reading P3: colour 0 = (i+j) even goes first).  After every full sweep, if E_trace/M_trace
// are non-NULL the pair (E_int, M) of every replica is stored at [local sweep][b]; if moments
// is non-NULL the pair is folded into it.  model_potts == 0: Ising (q ignored, may be NULL).
void oracle_sweep(int8_t* spins, int32_t batch, int32_t L, int32_t model_potts, const int32_t* q,
                  const double* beta, double J, double h, uint64_t seed, int64_t replica_offset,
                  int64_t n_sweeps, int64_t sweep_offset, int64_t* E_trace, int64_t* M_trace,
                  int64_t* moments) {
    int64_t* E = (int64_t*)std::malloc(sizeof(int64_t) * (size_t)batch);
    int64_t* M = (int64_t*)std::malloc(sizeof(int64_t) * (size_t)batch);
    for (int64_t local = 0; local < n_sweeps; ++local) {
        int64_t t = sweep_offset + local;
        for (int colour = 0; colour < 2; ++colour) {
            if (model_potts)
                oracle_potts_half_sweep(spins, batch, L, q, beta, J, seed, replica_offset, t, colour);
            else
                oracle_ising_half_sweep(spins, batch, L, beta, J, h, seed, replica_offset, t, colour);
        }
        if (E_trace || M_trace || moments) {
            if (model_potts) oracle_potts_observables(spins, batch, L, q, E, M);
            else oracle_ising_observables(spins, batch, L, E, M);
            if (E_trace) std::memcpy(E_trace + local * batch, E, sizeof(int64_t) * (size_t)batch);
            if (M_trace) std::memcpy(M_trace + local * batch, M, sizeof(int64_t) * (size_t)batch);
            if (moments) oracle_accumulate_moments(moments, batch, E, M);
        }
    }
    std::free(E);
    std::free(M);
}

// ---- +-J couplings (Eq. 1 is written with per-bond J_ij, and the
// paper's Fig. 9 minimises a +-J spin glass).  Reading: every bond carries a sign
// Jh[b][i][j] (between (i,j) and (i,j+1 mod L)) or Jv[b][i][j] (between (i,j) and (i+1 mod L,j)), values +-1, and
// H = -J sum_bonds J_ij s_i s_j - h sum_i s_i.  The local field of a site is the bond-weighted neighbour sum
// nn = Jv[i-1][j] s(i-1,j) + Jv[i][j] s(i+1,j) + Jh[i][j-1] s(i,j-1) + Jh[i][j] s(i,j+1), still in {-4..4}, so
// the class table, the random words and the accept rule are those of the uniform model (O2, O4, O5).
void oracle_ising_bonds_half_sweep(int8_t* spins, const int8_t* Jh, const int8_t* Jv, int32_t batch, int32_t L,
                                   const double* beta, double J, double h, uint64_t seed,
                                   int64_t replica_offset, int64_t t, int32_t colour) {
    const int64_t N = (int64_t)L * L;
    const int half = L / 2;
    for (int32_t b = 0; b < batch; ++b) {
        uint32_t T[10];
        uint8_t always[10];
        oracle_ising_table(beta[b], J, h, T, always);
        int8_t* lat = spins + (int64_t)b * N;
        const int8_t* jh = Jh + (int64_t)b * N;
        const int8_t* jv = Jv + (int64_t)b * N;
        uint32_t replica = (uint32_t)(b + replica_offset);
        for (int i = 0; i < L; ++i) {
            for (int j = 0; j < L; ++j) {
                if (((i + j) & 1) != colour) continue;
                int s = lat[(int64_t)i * L + j];
                int nn = jv[(int64_t)wrap(i - 1, L) * L + j] * lat[(int64_t)wrap(i - 1, L) * L + j] +
                         jv[(int64_t)i * L + j] * lat[(int64_t)wrap(i + 1, L) * L + j] +
                         jh[(int64_t)i * L + wrap(j - 1, L)] * lat[(int64_t)i * L + wrap(j - 1, L)] +
                         jh[(int64_t)i * L + j] * lat[(int64_t)i * L + wrap(j + 1, L)];
                int64_t n = (int64_t)i * half + (j >> 1);
                uint32_t out[4];
                draw(seed, (uint32_t)(n >> 2), replica, (uint64_t)t, (uint32_t)colour, DOMAIN_ISING, out);
                uint32_t r = out[n & 3];
                int cls = 5 * ((s + 1) / 2) + (nn + 4) / 2;
                if (accept(r, T[cls], always[cls])) lat[(int64_t)i * L + j] = (int8_t)(-s);
            }
        }
    }
}

// E_int = -sum_bonds J_ij s_i s_j (each bond once: the right and the down bond of every site), M = sum s.
void oracle_ising_bonds_observables(const int8_t* spins, const int8_t* Jh, const int8_t* Jv, int32_t batch,
                                    int32_t L, int64_t* E, int64_t* M) {
    const int64_t N = (int64_t)L * L;
    for (int32_t b = 0; b < batch; ++b) {
        const int8_t* lat = spins + (int64_t)b * N;
        const int8_t* jh = Jh + (int64_t)b * N;
        const int8_t* jv = Jv + (int64_t)b * N;
        int64_t S = 0, m = 0;
        for (int i = 0; i < L; ++i) {
            for (int j = 0; j < L; ++j) {
                int s = lat[(int64_t)i * L + j];
                S += s * (jh[(int64_t)i * L + j] * lat[(int64_t)i * L + wrap(j + 1, L)] +
                          jv[(int64_t)i * L + j] * lat[(int64_t)wrap(i + 1, L) * L + j]);
                m += s;
            }
        }
        E[b] = -S;
        M[b] = m;
    }
}

void oracle_sweep_bonds(int8_t* spins, const int8_t* Jh, const int8_t* Jv, int32_t batch, int32_t L,
                        const double* beta, double J, double h, uint64_t seed, int64_t replica_offset,
                        int64_t n_sweeps, int64_t sweep_offset, int64_t* E_trace, int64_t* M_trace) {
    int64_t* E = (int64_t*)std::malloc(sizeof(int64_t) * (size_t)batch);
    int64_t* M = (int64_t*)std::malloc(sizeof(int64_t) * (size_t)batch);
    for (int64_t local = 0; local < n_sweeps; ++local) {
        int64_t t = sweep_offset + local;
        for (int colour = 0; colour < 2; ++colour)
            oracle_ising_bonds_half_sweep(spins, Jh, Jv, batch, L, beta, J, h, seed, replica_offset, t, colour);
        if (E_trace || M_trace) {
            oracle_ising_bonds_observables(spins, Jh, Jv, batch, L, E, M);
            if (E_trace) std::memcpy(E_trace + local * batch, E, sizeof(int64_t) * (size_t)batch);
            if (M_trace) std::memcpy(M_trace + local * batch, M, sizeof(int64_t) * (size_t)batch);
        }
    }
    std::free(E);
    std::free(M);
}

}  // extern "C"
