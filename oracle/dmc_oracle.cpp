// ORACLE — TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain fp64 CPU implementation of the paper's Differentiable Monte Carlo step (Algorithm 2 and Eq. 4,
// /root/reference/PAPER.md:125, 140-158) for the 2D Ising model with per-bond couplings (Eq. 1 with J_ij,
// PAPER.md:99-103), and of its analytic gradient (the derivative of a scalar loss with respect to the
// per-bond couplings, the inverse temperatures, the field and the initial lattice: PAPER.md:308-320,
// "the derivative of the loss with respect to the parameters J_ij").
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may build, load or call this file.
// It shares no code with paper_2304_01772_b200/csrc/.  The random words come from the oracle's own Philox
// (spin_oracle.cpp, oracle_philox4x32_10), with the counter layout of DESIGN.md O2 written out below.
//
// Algorithm 2, line by line, with the readings of DESIGN.md section 12 (D1-D8):
//   1  propose s' for the lattice                      D1: the Ising proposal is the flip, s' = -s (reading P4)
//   2-3 convolution with the stencil, times the state  local energy e(s) = -s F, F = sum_n J_xn s_n + h
//                                                      (Eq. 1-2 with per-bond J_ij, library sign convention P1)
//   4  checkerboard                                    D6: colour 0 = (i+j) even first, then colour 1; only the
//                                                      sites of the current colour change in a half-sweep
//   5  dE = e(s') - e(s)                               D2: dE = 2 s F
//   6  p = exp(-beta dE)                               D3: not clamped to 1 (p > 1 when dE < 0)
//   7  random numbers r                                D4: r = (w >> 8) / 2^24, w = the Philox word of the Ising
//                                                      sweep at the same (seed, replica, site, t, colour)
//   8  q = 1 / (1 + exp(-alpha (p - r)))               D5: minus signs restored from PAPER.md:154
//   9  s <- q s' + (1 - q) s                           = s (1 - 2 q)
//   11 discretise, Eq. 4: s <- -1 if s < 0 else +1     D7
// Layout: natural row-major double arrays [batch][L][L]; Jh[b][i][j] couples (i,j)-(i,j+1 mod L),
// Jv[b][i][j] couples (i,j)-(i+1 mod L,j), as in spin_set_bonds.  One site at a time.
//
// Pins (tests/test_oracle_dmc.py, `-m "not gpu"`): central finite differences of the forward pass for every
// gradient (J per bond, beta, h, initial lattice) on 4x4 and 6x6; alpha -> infinity followed by Eq. 4
// reproduces the discrete Algorithm-1 lattice of spin_oracle.cpp (oracle_sweep_bonds) bit for bit; 0 < q < 1 and
// |s| <= 1 preserved; one site recomputed by hand from the Philox word; alpha = 0 gives q = 1/2, s -> 0;
// uniform couplings equal the bond-free formula.
#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <vector>

extern "C" void oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);

namespace {

inline int wrap(int a, int L) { return a < 0 ? a + L : (a >= L ? a - L : a); }

// D4.  The word the Ising sweep of spin_oracle.cpp would use for site (i, j) of colour c at sweep t
// (O2: group = n >> 2, word n & 3, n = i (L/2) + (j >> 1), domain ISING = 1), reduced to its top 24 bits.
double uniform_r(uint64_t seed, uint32_t replica, uint64_t t, int colour, int L, int i, int j) {
    const int64_t n = (int64_t)i * (L / 2) + (j >> 1);
    uint32_t ctr[4], key[2], out[4];
    ctr[0] = (uint32_t)(n >> 2);
    ctr[1] = replica;
    ctr[2] = (uint32_t)(t & 0xFFFFFFFFull);
    ctr[3] = (uint32_t)((t >> 32) & 0xFFFFFFull) | ((uint32_t)colour << 24) | (1u << 28);
    key[0] = (uint32_t)(seed & 0xFFFFFFFFull);
    key[1] = (uint32_t)(seed >> 32);
    oracle_philox4x32_10(ctr, key, out);
    return (double)(out[n & 3] >> 8) / 16777216.0;
}

struct Site {           // everything Algorithm 2 computes for one site, kept for the backward pass
    double F, dE, p, r, q;
};

// Lines 2-8 of Algorithm 2 for site (i, j) of replica lattice `lat`.
Site site_forward(const double* lat, const double* Jh, const double* Jv, int L, int i, int j, double h, double beta,
                  double alpha, double r) {
    const int iu = wrap(i - 1, L), id = wrap(i + 1, L), jl = wrap(j - 1, L), jr = wrap(j + 1, L);
    Site x;
    x.F = Jv[(int64_t)iu * L + j] * lat[(int64_t)iu * L + j] + Jv[(int64_t)i * L + j] * lat[(int64_t)id * L + j] +
          Jh[(int64_t)i * L + jl] * lat[(int64_t)i * L + jl] + Jh[(int64_t)i * L + j] * lat[(int64_t)i * L + jr] + h;
    const double s = lat[(int64_t)i * L + j];
    x.dE = 2.0 * s * x.F;                                    // line 5 (D2)
    x.p = std::exp(-beta * x.dE);                            // line 6 (D3)
    x.r = r;                                                 // line 7 (D4)
    x.q = 1.0 / (1.0 + std::exp(-alpha * (x.p - x.r)));      // line 8 (D5)
    return x;
}

}  // namespace

extern "C" {

// One DMC half-sweep of colour `colour` at sweep index t, in place (sites of one colour only see the other colour).
// q_out (may be NULL): [batch][L][L], receives q at the updated sites (untouched elsewhere) for the 0 < q < 1 pin.
void oracle_dmc_half_sweep(double* s, const double* Jh, const double* Jv, int32_t batch, int32_t L, double h,
                           const double* beta, double alpha, uint64_t seed, int64_t replica_offset, int64_t t,
                           int32_t colour, double* q_out) {
    const int64_t N = (int64_t)L * L;
    for (int32_t b = 0; b < batch; ++b) {
        double* lat = s + b * N;
        const double* jh = Jh + b * N;
        const double* jv = Jv + b * N;
        for (int i = 0; i < L; ++i)
            for (int j = 0; j < L; ++j) {
                if (((i + j) & 1) != colour) continue;
                const double r = uniform_r(seed, (uint32_t)(b + replica_offset), (uint64_t)t, colour, L, i, j);
                const Site x = site_forward(lat, jh, jv, L, i, j, h, beta[b], alpha, r);
                const double sx = lat[(int64_t)i * L + j];
                lat[(int64_t)i * L + j] = x.q * (-sx) + (1.0 - x.q) * sx;      // line 9, s' = -s (D1)
                if (q_out) q_out[b * N + (int64_t)i * L + j] = x.q;
            }
    }
}

// n_sweeps full sweeps (colour 0 then colour 1), t = sweep_offset ...  traj (may be NULL):
// [2 n_sweeps + 1][batch][L][L]; traj[0] = the initial lattice, traj[2k + 1 + c] = the lattice after half-sweep c of
// sweep k.  s is updated in place to the final lattice.
void oracle_dmc_forward(double* s, const double* Jh, const double* Jv, int32_t batch, int32_t L, double h,
                        const double* beta, double alpha, uint64_t seed, int64_t replica_offset, int64_t n_sweeps,
                        int64_t sweep_offset, double* traj) {
    const int64_t tot = (int64_t)batch * L * L;
    if (traj) for (int64_t k = 0; k < tot; ++k) traj[k] = s[k];
    for (int64_t k = 0; k < n_sweeps; ++k)
        for (int c = 0; c < 2; ++c) {
            oracle_dmc_half_sweep(s, Jh, Jv, batch, L, h, beta, alpha, seed, replica_offset, sweep_offset + k, c, nullptr);
            if (traj) for (int64_t m = 0; m < tot; ++m) traj[(2 * k + 1 + c) * tot + m] = s[m];
        }
}

// Eq. 4 (line 11).
void oracle_dmc_discretise(double* s, int64_t n) {
    for (int64_t k = 0; k < n; ++k) s[k] = s[k] < 0.0 ? -1.0 : 1.0;
}

// Reverse-mode derivative of a scalar loss through oracle_dmc_forward.  grad_out = dLoss/d(final lattice).  Outputs
// (all overwritten): grad_s0 [batch][L][L], grad_Jh, grad_Jv [batch][L][L], grad_beta [batch], grad_h [batch].
// Per updated site x of a half-sweep (s = value before, s_new = s (1 - 2q)), with A = alpha q (1-q) p:
//   d s_new / d s    = (1 - 2q) + 4 beta A s F          (through q: dq/dp = alpha q (1-q), dp/ds = -2 beta F p)
//   d s_new / d F    = 4 beta A s^2                     (dp/dF = -2 beta s p)
//   d s_new / d beta = 4 A s^2 F                        (dp/dbeta = -dE p)
//   dF/ds_n = J_xn, dF/dJ_xn = s_n, dF/dh = 1;  sites of the other colour pass through unchanged.
void oracle_dmc_backward(const double* traj, const double* Jh, const double* Jv, int32_t batch, int32_t L, double h,
                         const double* beta, double alpha, uint64_t seed, int64_t replica_offset, int64_t n_sweeps,
                         int64_t sweep_offset, const double* grad_out, double* grad_s0, double* grad_Jh, double* grad_Jv,
                         double* grad_beta, double* grad_h) {
    const int64_t N = (int64_t)L * L, tot = (int64_t)batch * N;
    std::vector<double> g(grad_out, grad_out + tot), gprev(tot);
    for (int64_t k = 0; k < tot; ++k) { grad_Jh[k] = 0.0; grad_Jv[k] = 0.0; }
    for (int32_t b = 0; b < batch; ++b) { grad_beta[b] = 0.0; grad_h[b] = 0.0; }
    for (int64_t k = n_sweeps - 1; k >= 0; --k)
        for (int c = 1; c >= 0; --c) {
            const double* before = traj + (2 * k + c) * tot;      // lattice this half-sweep started from
            for (int64_t m = 0; m < tot; ++m) gprev[m] = 0.0;
            for (int32_t b = 0; b < batch; ++b) {
                const double* lat = before + b * N;
                const double* jh = Jh + b * N;
                const double* jv = Jv + b * N;
                double* gp = gprev.data() + b * N;
                const double* gn = g.data() + b * N;
                for (int i = 0; i < L; ++i)
                    for (int j = 0; j < L; ++j) {
                        const int64_t x = (int64_t)i * L + j;
                        if (((i + j) & 1) != c) { gp[x] += gn[x]; continue; }       // untouched site
                        const double r = uniform_r(seed, (uint32_t)(b + replica_offset), (uint64_t)(sweep_offset + k), c, L, i, j);
                        const Site st = site_forward(lat, jh, jv, L, i, j, h, beta[b], alpha, r);
                        const double sx = lat[x];
                        const double A = alpha * st.q * (1.0 - st.q) * st.p;
                        const double dnew_ds = (1.0 - 2.0 * st.q) + 4.0 * beta[b] * A * sx * st.F;
                        const double dnew_dF = 4.0 * beta[b] * A * sx * sx;
                        const double dnew_dbeta = 4.0 * A * sx * sx * st.F;
                        const double G = gn[x] * dnew_dF;
                        gp[x] += gn[x] * dnew_ds;
                        grad_beta[b] += gn[x] * dnew_dbeta;
                        grad_h[b] += G;
                        const int iu = wrap(i - 1, L), id = wrap(i + 1, L), jl = wrap(j - 1, L), jr = wrap(j + 1, L);
                        // the four bonds of x and the neighbours they lead to
                        gp[(int64_t)iu * L + j] += G * jv[(int64_t)iu * L + j];
                        gp[(int64_t)id * L + j] += G * jv[x];
                        gp[(int64_t)i * L + jl] += G * jh[(int64_t)i * L + jl];
                        gp[(int64_t)i * L + jr] += G * jh[x];
                        grad_Jv[b * N + (int64_t)iu * L + j] += G * lat[(int64_t)iu * L + j];
                        grad_Jv[b * N + x] += G * lat[(int64_t)id * L + j];
                        grad_Jh[b * N + (int64_t)i * L + jl] += G * lat[(int64_t)i * L + jl];
                        grad_Jh[b * N + x] += G * lat[(int64_t)i * L + jr];
                    }
            }
            g.swap(gprev);
        }
    for (int64_t k = 0; k < tot; ++k) grad_s0[k] = g[k];
}

}  // extern "C"
