// ORACLE — TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Extensions of the plain CPU oracle (spin_oracle.cpp) for SURVEY.md section 8(f) #2: the Hamiltonians as the paper
// writes them, with a coupling per bond and a field per site (Eq. 1: H = sum J_ij s_i s_j + sum B_i s_i;
// Eq. 5, the same with a Kronecker delta and the field on the state label), sampled by the same
// checkerboard Metropolis rule (Algorithm 1) with the same random words (O2) and the same
// acceptance arithmetic (O4: x = beta dE; x <= 0 always, else r < floor(exp(-x) 2^32)).  Library sign convention (P1):
//   Ising:  H = -sum_bonds J_ij s_i s_j - sum_i B_i s_i                 (J_ij, B_i real)
//   Potts:  H = -J sum_bonds J_ij delta(s_i, s_j) - h sum_i s_i         (J_ij = +-1 bond signs, s_i in 0..q-1: the field
//                                                                        term of Eq. 5 is linear in the state label, P7)
// Natural row-major layouts; Jh[b][i][j] couples (i,j)-(i,j+1 mod L), Jv[b][i][j] couples (i,j)-(i+1 mod L,j).
// One site at a time, every dE evaluated in IEEE double in the order written below, no table.
//
// Pins (tests/test_oracle_general.py): uniform / +-1 couplings reproduce spin_oracle.cpp bit for bit; gauge
// transformation J'_ij = x_i J_ij x_j, B'_i = x_i B_i maps trajectories exactly; long-run averages against brute-force
// Boltzmann sums (4x4 Ising with random real couplings and fields; 2x2 and 2x4... Potts with field); large-field and
// T -> 0 limits; observables against explicit bond lists.
#include <cmath>
#include <cstdint>
#include <cstdlib>

extern "C" void oracle_draw(uint64_t seed, uint32_t group, uint32_t replica, uint64_t t, uint32_t colour, uint32_t domain,
                            uint32_t out[4]);
extern "C" void oracle_threshold(double beta, double dE, uint32_t* T, uint8_t* always);

namespace {
inline int wrap(int a, int L) { return a < 0 ? a + L : (a >= L ? a - L : a); }
enum { DOMAIN_ISING = 1, DOMAIN_POTTS = 2 };
}  // namespace

extern "C" {

// Ising, real couplings and per-site fields.  dE of flipping s at (i,j): 2 s F with the local field
//   F = Jv[i-1][j] s(i-1,j) + Jv[i][j] s(i+1,j) + Jh[i][j-1] s(i,j-1) + Jh[i][j] s(i,j+1) + B[i][j]
// (sum in this order).  Random word: as in the uniform model (group n>>2, word n&3, domain ISING).
void oracle_ising_general_half_sweep(int8_t* spins, const double* Jh, const double* Jv, const double* B, int32_t batch,
                                     int32_t L, const double* beta, uint64_t seed, int64_t replica_offset, int64_t t,
                                     int32_t colour) {
    const int64_t N = (int64_t)L * L;
    const int half = L / 2;
    for (int32_t b = 0; b < batch; ++b) {
        int8_t* lat = spins + b * N;
        const double* jh = Jh + b * N;
        const double* jv = Jv + b * N;
        const double* fb = B + b * N;
        for (int i = 0; i < L; ++i)
            for (int j = 0; j < L; ++j) {
                if (((i + j) & 1) != colour) continue;
                const int iu = wrap(i - 1, L), id = wrap(i + 1, L), jl = wrap(j - 1, L), jr = wrap(j + 1, L);
                const double s = (double)lat[(int64_t)i * L + j];
                const double F = jv[(int64_t)iu * L + j] * (double)lat[(int64_t)iu * L + j] +
                                 jv[(int64_t)i * L + j] * (double)lat[(int64_t)id * L + j] +
                                 jh[(int64_t)i * L + jl] * (double)lat[(int64_t)i * L + jl] +
                                 jh[(int64_t)i * L + j] * (double)lat[(int64_t)i * L + jr] + fb[(int64_t)i * L + j];
                const double dE = 2.0 * s * F;
                uint32_t T;
                uint8_t always;
                oracle_threshold(beta[b], dE, &T, &always);
                const int64_t n = (int64_t)i * half + (j >> 1);
                uint32_t out[4];
                oracle_draw(seed, (uint32_t)(n >> 2), (uint32_t)(b + replica_offset), (uint64_t)t, (uint32_t)colour, DOMAIN_ISING, out);
                if (always || out[n & 3] < T) lat[(int64_t)i * L + j] = (int8_t)(-lat[(int64_t)i * L + j]);
            }
    }
}

// Energy of the general Ising model in double: E[b] = -sum_bonds J_ij s_i s_j - sum_i B_i s_i (row-major site order,
// right bond then down bond then field per site); M[b] = sum s (exact integer).
void oracle_ising_general_observables(const int8_t* spins, const double* Jh, const double* Jv, const double* B,
                                      int32_t batch, int32_t L, double* E, int64_t* M) {
    const int64_t N = (int64_t)L * L;
    for (int32_t b = 0; b < batch; ++b) {
        const int8_t* lat = spins + b * N;
        double e = 0.0;
        int64_t m = 0;
        for (int i = 0; i < L; ++i)
            for (int j = 0; j < L; ++j) {
                const int64_t x = (int64_t)i * L + j;
                const double s = (double)lat[x];
                e -= Jh[b * N + x] * s * (double)lat[(int64_t)i * L + wrap(j + 1, L)];
                e -= Jv[b * N + x] * s * (double)lat[(int64_t)wrap(i + 1, L) * L + j];
                e -= B[b * N + x] * s;
                m += lat[x];
            }
        E[b] = e;
        M[b] = m;
    }
}

// Potts with +-1 bond signs (NULL: all +1) and a field on the state label.  Proposal as in O6.  With
// n_old / n_new = bond-weighted numbers of neighbours equal to the old / the proposed state (each bond contributes its
// sign), dE = -(J (n_new - n_old)) - (h (new - old)), evaluated as dE = -(J*dn) - h*dl in double.
void oracle_potts_general_half_sweep(int8_t* spins, const int8_t* Jh, const int8_t* Jv, int32_t batch, int32_t L,
                                     const int32_t* q, const double* beta, double J, double h, uint64_t seed,
                                     int64_t replica_offset, int64_t t, int32_t colour) {
    const int64_t N = (int64_t)L * L;
    const int half = L / 2;
    for (int32_t b = 0; b < batch; ++b) {
        int8_t* lat = spins + b * N;
        const int qb = q[b];
        for (int i = 0; i < L; ++i)
            for (int j = 0; j < L; ++j) {
                if (((i + j) & 1) != colour) continue;
                const int iu = wrap(i - 1, L), id = wrap(i + 1, L), jl = wrap(j - 1, L), jr = wrap(j + 1, L);
                const int old = lat[(int64_t)i * L + j];
                const int nb[4] = {lat[(int64_t)iu * L + j], lat[(int64_t)id * L + j], lat[(int64_t)i * L + jl], lat[(int64_t)i * L + jr]};
                int sg[4] = {1, 1, 1, 1};
                if (Jh) {
                    sg[0] = Jv[b * N + (int64_t)iu * L + j];
                    sg[1] = Jv[b * N + (int64_t)i * L + j];
                    sg[2] = Jh[b * N + (int64_t)i * L + jl];
                    sg[3] = Jh[b * N + (int64_t)i * L + j];
                }
                const int64_t n = (int64_t)i * half + (j >> 1);
                uint32_t out[4];
                oracle_draw(seed, (uint32_t)(n >> 1), (uint32_t)(b + replica_offset), (uint64_t)t, (uint32_t)colour, DOMAIN_POTTS, out);
                const uint32_t r_prop = out[2 * (n & 1)], r_acc = out[2 * (n & 1) + 1];
                const int d = (int)(((uint64_t)r_prop * (uint64_t)(qb - 1)) >> 32);
                int nw = old + 1 + d;
                if (nw >= qb) nw -= qb;
                int dn = 0;
                for (int a = 0; a < 4; ++a) dn += sg[a] * ((nb[a] == nw) - (nb[a] == old));
                const double dE = -(J * (double)dn) - h * (double)(nw - old);
                uint32_t T;
                uint8_t always;
                oracle_threshold(beta[b], dE, &T, &always);
                if (always || r_acc < T) lat[(int64_t)i * L + j] = (int8_t)nw;
            }
    }
}

// E_int[b] = -sum_bonds J_ij delta(s_i, s_j) (exact integer), S[b] = sum of the state labels (the field couples to it),
// M[b] = max_k N_k.  Energy = J E_int - h S.
void oracle_potts_general_observables(const int8_t* spins, const int8_t* Jh, const int8_t* Jv, int32_t batch, int32_t L,
                                      const int32_t* q, int64_t* E, int64_t* S, int64_t* M) {
    const int64_t N = (int64_t)L * L;
    for (int32_t b = 0; b < batch; ++b) {
        const int8_t* lat = spins + b * N;
        int64_t e = 0, sl = 0, cnt[128] = {0};
        for (int i = 0; i < L; ++i)
            for (int j = 0; j < L; ++j) {
                const int64_t x = (int64_t)i * L + j;
                const int s = lat[x];
                const int jh = Jh ? Jh[b * N + x] : 1, jv = Jv ? Jv[b * N + x] : 1;
                e -= jh * (lat[(int64_t)i * L + wrap(j + 1, L)] == s);
                e -= jv * (lat[(int64_t)wrap(i + 1, L) * L + j] == s);
                sl += s;
                cnt[s] += 1;
            }
        int64_t best = 0;
        for (int k = 0; k < q[b]; ++k) if (cnt[k] > best) best = cnt[k];
        E[b] = e; S[b] = sl; M[b] = best;
    }
}

}  // extern "C"
