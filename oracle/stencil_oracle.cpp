// ORACLE — TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// the checkerboard Metropolis rule of Algorithm 1 on the other lattice
// geometries the paper names — "2D convolution for square or triangular networks, and 3D convolution for cubic networks"
// (PAPER.md:105), the triangular-lattice kernels of Eq. 3, and second-neighbour interactions
// ("using more colors to obtain interactions beyond first neighbors").  Plain loops, one site at a time,
// natural row-major int8 lattices, Ising spins +-1.  Shares no code with paper_2304_01772_b200/csrc/.
//
// Geometries (readings S1-S6):
//   TRIANGULAR (0): L x L sites, L % 3 == 0, six neighbours (i+-1, j), (i, j+-1), (i+1, j+1), (i-1, j-1) — the triangular
//       lattice sheared onto the square grid (the paper's Eq. 3 pads with null spins instead; the connectivity is the
//       same).  Three colours c = (i + j) mod 3: no two neighbours share one.
//   CUBIC (1): L x L x L sites, L even, six neighbours +-1 along each axis, two colours c = (i + j + k) & 1.
//   SQUARE_NNN (2): L x L sites, L even, four first neighbours (coupling J1) and four diagonal second neighbours
//       (coupling J2), four colours c = 2 (i & 1) + (j & 1).
// H = -J1 sum_<first> s s' - J2 sum_<second> s s' - h sum s; neighbours with multiplicity (periodic wrap, small L).
// dE of flipping s: 2 s (J1 nn1 + J2 nn2 + h), evaluated as written; acceptance O4 (oracle_threshold).
// Sweep t: colours 0, 1, .. in order.  Random word of a site: Philox group n >> 2, word n & 3, where n is the index of
// the site among the sites of its colour in row-major order; counter (group, replica, t low, t high | colour << 24 |
// domain << 28) with domain 3 = STENCIL.  Initial lattice: as O3 over the natural site index (domain INIT).
//
// Pins (tests/test_oracle_stencil.py): brute-force Boltzmann sums (3x3 and 3x6 triangular incl. the frustrated
// antiferromagnet, 2x2x2 and 2x2x4... cubic, 4x4 J1-J2), J2 = 0 long-run averages against the exact 4x4 square-lattice
// values of SURVEY Q7, beta = 0 flips everything, T -> 0 monotone energy, colour classes are independent sets,
// one site by hand through the exported Philox, observables against explicit bond lists.
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <vector>

extern "C" void oracle_draw(uint64_t seed, uint32_t group, uint32_t replica, uint64_t t, uint32_t colour, uint32_t domain,
                            uint32_t out[4]);
extern "C" void oracle_threshold(double beta, double dE, uint32_t* T, uint8_t* always);

namespace {

enum { TRIANGULAR = 0, CUBIC = 1, SQUARE_NNN = 2 };
enum { DOMAIN_INIT = 0, DOMAIN_STENCIL = 3 };

struct Geometry {
    int stencil, L, dims;          // dims: 2 or 3
    int n_colours;
    int n1, n2;                    // numbers of first / second neighbours
    int off1[6][3], off2[4][3];    // offsets (di, dj, dk)
};

Geometry make_geometry(int stencil, int L) {
    Geometry g;
    std::memset(&g, 0, sizeof g);
    g.stencil = stencil;
    g.L = L;
    if (stencil == TRIANGULAR) {
        g.dims = 2; g.n_colours = 3; g.n1 = 6; g.n2 = 0;
        const int o[6][3] = {{-1, 0, 0}, {1, 0, 0}, {0, -1, 0}, {0, 1, 0}, {1, 1, 0}, {-1, -1, 0}};
        std::memcpy(g.off1, o, sizeof o);
    } else if (stencil == CUBIC) {
        g.dims = 3; g.n_colours = 2; g.n1 = 6; g.n2 = 0;
        const int o[6][3] = {{-1, 0, 0}, {1, 0, 0}, {0, -1, 0}, {0, 1, 0}, {0, 0, -1}, {0, 0, 1}};
        std::memcpy(g.off1, o, sizeof o);
    } else {
        g.dims = 2; g.n_colours = 4; g.n1 = 4; g.n2 = 4;
        const int o1[4][3] = {{-1, 0, 0}, {1, 0, 0}, {0, -1, 0}, {0, 1, 0}};
        const int o2[4][3] = {{-1, -1, 0}, {-1, 1, 0}, {1, -1, 0}, {1, 1, 0}};
        std::memcpy(g.off1, o1, sizeof o1);
        std::memcpy(g.off2, o2, sizeof o2);
    }
    return g;
}

inline int64_t n_sites(const Geometry& g) { return g.dims == 3 ? (int64_t)g.L * g.L * g.L : (int64_t)g.L * g.L; }
inline int wrapL(int a, int L) { a %= L; return a < 0 ? a + L : a; }

inline int colour_of(const Geometry& g, int i, int j, int k) {
    if (g.stencil == TRIANGULAR) return (i + j) % 3;
    if (g.stencil == CUBIC) return (i + j + k) & 1;
    return 2 * (i & 1) + (j & 1);
}

inline int64_t site_index(const Geometry& g, int i, int j, int k) {
    return g.dims == 3 ? ((int64_t)i * g.L + j) * g.L + k : (int64_t)i * g.L + j;
}

}  // namespace

extern "C" {

int64_t oracle_stencil_sites(int32_t stencil, int32_t L) { return n_sites(make_geometry(stencil, L)); }

// O3 over the natural index p: group p >> 2, word p & 3, +1 iff bit 31.
void oracle_stencil_init(int8_t* spins, int32_t stencil, int32_t batch, int32_t L, uint64_t seed, int64_t replica_offset) {
    const Geometry g = make_geometry(stencil, L);
    const int64_t N = n_sites(g);
    for (int32_t b = 0; b < batch; ++b)
        for (int64_t p = 0; p < N; ++p) {
            uint32_t out[4];
            oracle_draw(seed, (uint32_t)(p >> 2), (uint32_t)(b + replica_offset), 0, 0, DOMAIN_INIT, out);
            spins[b * N + p] = (out[p & 3] & 0x80000000u) ? (int8_t)1 : (int8_t)-1;
        }
}

// One pass over the sites of colour `colour` (row-major), sweep index t.
void oracle_stencil_colour_pass(int8_t* spins, int32_t stencil, int32_t batch, int32_t L, const double* beta, double J1,
                                double J2, double h, uint64_t seed, int64_t replica_offset, int64_t t, int32_t colour) {
    const Geometry g = make_geometry(stencil, L);
    const int64_t N = n_sites(g);
    const int K = g.dims == 3 ? L : 1;
    for (int32_t b = 0; b < batch; ++b) {
        int8_t* lat = spins + b * N;
        int64_t n = 0;                                        // running index among the sites of this colour
        for (int i = 0; i < L; ++i)
            for (int j = 0; j < L; ++j)
                for (int k = 0; k < K; ++k) {
                    if (colour_of(g, i, j, k) != colour) continue;
                    const int64_t x = site_index(g, i, j, k);
                    const int s = lat[x];
                    int nn1 = 0, nn2 = 0;
                    for (int a = 0; a < g.n1; ++a)
                        nn1 += lat[site_index(g, wrapL(i + g.off1[a][0], L), wrapL(j + g.off1[a][1], L), g.dims == 3 ? wrapL(k + g.off1[a][2], L) : 0)];
                    for (int a = 0; a < g.n2; ++a)
                        nn2 += lat[site_index(g, wrapL(i + g.off2[a][0], L), wrapL(j + g.off2[a][1], L), 0)];
                    const double dE = 2.0 * (double)s * (J1 * (double)nn1 + J2 * (double)nn2 + h);
                    uint32_t T;
                    uint8_t always;
                    oracle_threshold(beta[b], dE, &T, &always);
                    uint32_t out[4];
                    oracle_draw(seed, (uint32_t)(n >> 2), (uint32_t)(b + replica_offset), (uint64_t)t, (uint32_t)colour, DOMAIN_STENCIL, out);
                    if (always || out[n & 3] < T) lat[x] = (int8_t)(-s);
                    ++n;
                }
    }
}

void oracle_stencil_sweep(int8_t* spins, int32_t stencil, int32_t batch, int32_t L, const double* beta, double J1, double J2,
                          double h, uint64_t seed, int64_t replica_offset, int64_t n_sweeps, int64_t sweep_offset) {
    const Geometry g = make_geometry(stencil, L);
    for (int64_t t = sweep_offset; t < sweep_offset + n_sweeps; ++t)
        for (int c = 0; c < g.n_colours; ++c)
            oracle_stencil_colour_pass(spins, stencil, batch, L, beta, J1, J2, h, seed, replica_offset, t, c);
}

// E1 = -sum over first-neighbour bonds of s s', E2 = -sum over second-neighbour bonds (each bond once: the "forward"
// half of the offsets, with multiplicity), M = sum s.  Energy = J1 E1 + J2 E2 - h M.
void oracle_stencil_observables(const int8_t* spins, int32_t stencil, int32_t batch, int32_t L, int64_t* E1, int64_t* E2,
                                int64_t* M) {
    const Geometry g = make_geometry(stencil, L);
    const int64_t N = n_sites(g);
    const int K = g.dims == 3 ? L : 1;
    for (int32_t b = 0; b < batch; ++b) {
        const int8_t* lat = spins + b * N;
        int64_t e1 = 0, e2 = 0, m = 0;
        for (int i = 0; i < L; ++i)
            for (int j = 0; j < L; ++j)
                for (int k = 0; k < K; ++k) {
                    const int s = lat[site_index(g, i, j, k)];
                    for (int a = 0; a < g.n1; ++a) {
                        const int* o = g.off1[a];
                        const bool forward = o[0] > 0 || (o[0] == 0 && (o[1] > 0 || (o[1] == 0 && o[2] > 0)));
                        if (!forward) continue;
                        e1 -= s * lat[site_index(g, wrapL(i + o[0], L), wrapL(j + o[1], L), g.dims == 3 ? wrapL(k + o[2], L) : 0)];
                    }
                    for (int a = 0; a < g.n2; ++a) {
                        const int* o = g.off2[a];
                        if (o[0] <= 0) continue;               // (1,-1) and (1,1)
                        e2 -= s * lat[site_index(g, wrapL(i + o[0], L), wrapL(j + o[1], L), 0)];
                    }
                    m += s;
                }
        E1[b] = e1; E2[b] = e2; M[b] = m;
    }
}

}  // extern "C"
