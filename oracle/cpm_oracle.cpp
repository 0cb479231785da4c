// ORACLE — TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// the Cellular Potts Model of the paper (Eq. 7, Table II) sampled with
// Algorithm 1 on a colouring that makes the parallel update well defined.  Plain loops, natural
// row-major int8 lattice of cell identifiers ("spins") sigma in 0..q-1, 0 = the medium.  Shares no code with
// paper_2304_01772_b200/csrc/.
//
//   H = 1/2 sum_x sum_{y in Moore(x)} J[tau(s_x)][tau(s_y)] (1 - delta(s_x, s_y)) + lambda sum_{s >= 1} (a_s - A_s)^2  (Eq. 7)
// with tau(s) the type of cell s (medium, light, dark, ...), a_s its area, A_s its target area; the medium's area is
// unconstrained.  "The interaction uses the Moore neighborhood with second neighbors".
//
// Readings (C1-C9):
//   C1 proposal: "change the value in a given lattice position for another in its vicinity": the
//      target site copies the identifier of ONE of its 8 Moore neighbours, chosen uniformly by r_prop >> 29 in the order
//      (-1,-1), (-1,0), (-1,1), (0,-1), (0,1), (1,-1), (1,0), (1,1); a copy of an equal identifier changes nothing.
//   C2 parallel update: four colours c = 2 (i & 1) + (j & 1) (no two Moore neighbours share one); a sweep is
//      the four colour passes in order.
//   C3 areas are counted once at the START of every colour pass and held fixed during it (a tensor implementation
//      evaluates all sites of a pass from one snapshot); the area term of a proposal old -> new is
//      lambda [(new != 0)(2 (a_new - A_new) + 1) + (old != 0)(-2 (a_old - A_old) + 1)].
//   C4 adhesion term: sum over the 8 Moore neighbours y of (new != s_y) J[tau(new)][tau(s_y)] - (old != s_y) J[tau(old)][tau(s_y)].
//   C5 J, lambda and A are integers (Table II and the paper's lambda = 1, A = 25 are), so dH is an exact integer.
//   C6 acceptance: O4 on x = beta dH (dH <= 0 always; else r_acc < floor(exp(-x) 2^32)), beta = 1 / (k_B T).
//   C7 random words: Philox group n >> 1, r_prop = word 2 (n & 1), r_acc = word 2 (n & 1) + 1, n = (i >> 1) (L/2) + (j >> 1)
//      (the index of the site among the sites of its colour), counter as O2 with domain 4 = CPM.
//   C8 periodic boundaries, L even.    C9 types and target areas are per cell identifier, shared by the replicas.
//
// Pins (tests/test_oracle_cpm.py): the exported dH of a proposal equals H(after) - H(before) of an explicit Eq.-7
// Hamiltonian written in the test (exact integers, random lattices and proposals); one site by hand through the
// exported Philox (direction, words, acceptance); beta = 0 accepts every copy: the pass equals a numpy gather; areas sum
// to L^2, no identifier is created, an all-medium lattice and a lambda = 0 single-colour lattice are fixed points;
// observables against explicit double loops.
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <vector>

extern "C" void oracle_draw(uint64_t seed, uint32_t group, uint32_t replica, uint64_t t, uint32_t colour, uint32_t domain,
                            uint32_t out[4]);
extern "C" void oracle_threshold(double beta, double dE, uint32_t* T, uint8_t* always);

namespace {
enum { DOMAIN_CPM = 4 };
const int MOORE[8][2] = {{-1, -1}, {-1, 0}, {-1, 1}, {0, -1}, {0, 1}, {1, -1}, {1, 0}, {1, 1}};
inline int wrap(int a, int L) { return a < 0 ? a + L : (a >= L ? a - L : a); }

// C3 + C4 for the proposal old -> nw at (i, j); areas = the snapshot counts.
int64_t delta_H(const int8_t* lat, int L, const int32_t* tau, const int32_t* Jtab, int ntypes, int64_t lambda,
                const int32_t* A, const int64_t* areas, int i, int j, int nw) {
    const int old = lat[(int64_t)i * L + j];
    if (nw == old) return 0;
    int64_t d = 0;
    for (int a = 0; a < 8; ++a) {
        const int sy = lat[(int64_t)wrap(i + MOORE[a][0], L) * L + wrap(j + MOORE[a][1], L)];
        if (nw != sy) d += Jtab[tau[nw] * ntypes + tau[sy]];
        if (old != sy) d -= Jtab[tau[old] * ntypes + tau[sy]];
    }
    if (nw != 0) d += lambda * (2 * (areas[nw] - A[nw]) + 1);
    if (old != 0) d += lambda * (-2 * (areas[old] - A[old]) + 1);
    return d;
}
}  // namespace

extern "C" {

int64_t oracle_cpm_delta(const int8_t* lat, int32_t L, int32_t q, const int32_t* tau, const int32_t* Jtab, int32_t ntypes,
                         int64_t lambda, const int32_t* A, int32_t i, int32_t j, int32_t nw) {
    std::vector<int64_t> areas(q, 0);
    for (int64_t x = 0; x < (int64_t)L * L; ++x) areas[lat[x]] += 1;
    return delta_H(lat, L, tau, Jtab, ntypes, lambda, A, areas.data(), i, j, nw);
}

void oracle_cpm_colour_pass(int8_t* spins, int32_t batch, int32_t L, int32_t q, const int32_t* tau, const int32_t* Jtab,
                            int32_t ntypes, int64_t lambda, const int32_t* A, const double* beta, uint64_t seed,
                            int64_t replica_offset, int64_t t, int32_t colour) {
    const int64_t N = (int64_t)L * L;
    const int half = L / 2;
    for (int32_t b = 0; b < batch; ++b) {
        int8_t* lat = spins + b * N;
        std::vector<int64_t> areas(q, 0);
        for (int64_t x = 0; x < N; ++x) areas[lat[x]] += 1;                      // C3: snapshot
        for (int i = colour >> 1; i < L; i += 2)
            for (int j = colour & 1; j < L; j += 2) {
                const int64_t n = (int64_t)(i >> 1) * half + (j >> 1);
                uint32_t out[4];
                oracle_draw(seed, (uint32_t)(n >> 1), (uint32_t)(b + replica_offset), (uint64_t)t, (uint32_t)colour, DOMAIN_CPM, out);
                const uint32_t r_prop = out[2 * (n & 1)], r_acc = out[2 * (n & 1) + 1];
                const int dir = (int)(r_prop >> 29);
                const int nw = lat[(int64_t)wrap(i + MOORE[dir][0], L) * L + wrap(j + MOORE[dir][1], L)];
                if (nw == lat[(int64_t)i * L + j]) continue;
                const int64_t dH = delta_H(lat, L, tau, Jtab, ntypes, lambda, A, areas.data(), i, j, nw);
                uint32_t T;
                uint8_t always;
                oracle_threshold(beta[b], (double)dH, &T, &always);
                if (always || r_acc < T) lat[(int64_t)i * L + j] = (int8_t)nw;
            }
    }
}

void oracle_cpm_sweep(int8_t* spins, int32_t batch, int32_t L, int32_t q, const int32_t* tau, const int32_t* Jtab,
                      int32_t ntypes, int64_t lambda, const int32_t* A, const double* beta, uint64_t seed,
                      int64_t replica_offset, int64_t n_sweeps, int64_t sweep_offset) {
    for (int64_t t = sweep_offset; t < sweep_offset + n_sweeps; ++t)
        for (int c = 0; c < 4; ++c)
            oracle_cpm_colour_pass(spins, batch, L, q, tau, Jtab, ntypes, lambda, A, beta, seed, replica_offset, t, c);
}

// H_adh[b] (first term of Eq. 7: every unordered Moore pair once), H_area[b] (second term), areas [batch][q],
// boundary [batch][ntypes][ntypes]: number of unordered Moore pairs with different identifiers and types (tau <= tau')
// stored at [min][max] (Fig. 6's boundary lengths).
void oracle_cpm_observables(const int8_t* spins, int32_t batch, int32_t L, int32_t q, const int32_t* tau, const int32_t* Jtab,
                            int32_t ntypes, int64_t lambda, const int32_t* A, int64_t* H_adh, int64_t* H_area,
                            int64_t* areas, int64_t* boundary) {
    const int64_t N = (int64_t)L * L;
    const int FWD[4][2] = {{0, 1}, {1, -1}, {1, 0}, {1, 1}};
    for (int32_t b = 0; b < batch; ++b) {
        const int8_t* lat = spins + b * N;
        int64_t* ar = areas + (int64_t)b * q;
        int64_t* bl = boundary + (int64_t)b * ntypes * ntypes;
        for (int k = 0; k < q; ++k) ar[k] = 0;
        for (int k = 0; k < ntypes * ntypes; ++k) bl[k] = 0;
        int64_t h = 0;
        for (int i = 0; i < L; ++i)
            for (int j = 0; j < L; ++j) {
                const int s = lat[(int64_t)i * L + j];
                ar[s] += 1;
                for (int a = 0; a < 4; ++a) {
                    const int sy = lat[(int64_t)wrap(i + FWD[a][0], L) * L + wrap(j + FWD[a][1], L)];
                    if (sy == s) continue;
                    h += Jtab[tau[s] * ntypes + tau[sy]];
                    const int lo = tau[s] < tau[sy] ? tau[s] : tau[sy], hi = tau[s] < tau[sy] ? tau[sy] : tau[s];
                    bl[lo * ntypes + hi] += 1;
                }
            }
        int64_t ha = 0;
        for (int k = 1; k < q; ++k) ha += lambda * (ar[k] - A[k]) * (ar[k] - A[k]);
        H_adh[b] = h;
        H_area[b] = ha;
    }
}

}  // extern "C"
