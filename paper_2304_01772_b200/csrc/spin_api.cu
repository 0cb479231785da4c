// spin_api.cu — host control and the C ABI of include/spin.h: handle state, argument validation, acceptance
// tables (row a1), Philox round keys, kernel selection, the sweep loop (row a4) and the measurement loop.
// No step of the method runs on the CPU except the O(batch) table build, which the paper's acceptance rule
// defines in floating point (Alg. 1 line 9) and which is evaluated in IEEE double here.
#include "../../include/spin.h"
#include "spin_internal.cuh"

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

using namespace spin;

namespace {

thread_local std::string g_last_error;

int fail(int code, const char* fmt, ...) __attribute__((format(printf, 2, 3)));
int fail(int code, const char* fmt, ...) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    try { g_last_error = buf; } catch (...) {}   // no exception may cross the C boundary
    return code;
}

int cuda_fail(cudaError_t e, const char* what) {
    return fail(SPIN_ERR_CUDA, "%s: %s", what, cudaGetErrorString(e));
}

#define CUDA_TRY(expr)                                      \
    do {                                                    \
        cudaError_t e_ = (expr);                            \
        if (e_ != cudaSuccess) return cuda_fail(e_, #expr); \
    } while (0)

// ---- row a1: acceptance of one class (O4; Alg. 1 lines 6-9) -----------------
struct ClassAccept {
    uint32_t T;      // floor(exp(-x) 2^32), clipped
    bool always;     // x <= 0
};

ClassAccept class_accept(double beta, double dE) {
    ClassAccept c;
    const double x = beta * dE;
    if (x <= 0.0) {
        c.always = true;
        c.T = 0xFFFFFFFFu;
        return c;
    }
    const double v = std::floor(std::exp(-x) * 4294967296.0);
    c.always = false;
    c.T = v >= 4294967295.0 ? 0xFFFFFFFFu : (uint32_t)v;
    return c;
}

// Ising class (s, nn): dE = 2 s (J nn + h)
ClassAccept ising_class(double beta, double J, double h, int s, int nn) {
    const double dE = 2.0 * (double)s * (J * (double)nn + h);
    return class_accept(beta, dE);
}

// Potts class dn: dE = -J dn
ClassAccept potts_class(double beta, double J, int dn) {
    const double dE = -(J * (double)dn);
    return class_accept(beta, dE);
}

// Device record: accept iff r <= U, except classes in the never mask.
void encode(const ClassAccept& c, int idx, uint32_t* rec) {
    if (c.always) rec[idx] = 0xFFFFFFFFu;
    else if (c.T == 0u) { rec[idx] = 0u; rec[kTabNever] |= 1u << idx; }
    else rec[idx] = c.T - 1u;
}

}  // namespace

namespace spin {
int set_error(int code, const char* msg) { return fail(code, "%s", msg); }
}  // namespace spin

struct spin_sim {
    int32_t batch = 0, L = 0, model = 0, layout = 0;
    uint64_t seed = 0;
    uint32_t replica_offset = 0;
    std::vector<int32_t> q;          // per replica (Ising: 2)
    void* lattice = nullptr;
    bool owns_lattice = false;
    size_t lattice_bytes = 0;
    cudaStream_t stream = nullptr;
    int device = 0;
    // scratch (device)
    uint32_t* d_tables = nullptr;    // [B][kTableStride]
    int32_t* d_q = nullptr;          // [B]
    long long* d_EM = nullptr;       // [2][B] accumulators
    unsigned int* d_hist = nullptr;  // [B][128] (Potts)
    unsigned int* d_bad = nullptr;   // validation counter
    uint32_t* d_bonds = nullptr;     // +-J sign planes [B][2][4][L][L/64] (bit-packed layout) or nullptr
    int8_t* d_bond_nat = nullptr;    // +-J signs in the natural layout [2][B][L][L] (Jh then Jv): int8 Ising and Potts
    // real couplings and per-site fields (Ising, int8 layout): host copies for the threshold build, device copies for
    // the energy, the per-site thresholds [B][N][32] + always masks [B][N], and the beta they were built for
    std::vector<double> g_Jh, g_Jv, g_B, g_beta;
    double* d_gen = nullptr;         // [3][B][N] doubles: Jh, Jv, B
    uint32_t* d_thr = nullptr;
    uint32_t* d_alw = nullptr;
    bool general = false;
    unsigned long long* d_tab2 = nullptr;   // Potts with a field / bond signs: [B][9][255] (always << 32) | T
    bool potts_general = false;             // the current tables were built for the general Potts kernel
    uint32_t* d_sched = nullptr;            // tables of spin_sweep_schedule [n_steps][B][kTableStride] (grow-only)
    size_t sched_bytes = 0;
    uint32_t* h_sched = nullptr;            // pinned staging of the same size, guarded by sched_ev (recorded after its upload)
    cudaEvent_t sched_ev = nullptr;
    void* d_shadow = nullptr;               // second lattice of the tiled kernel (allocated on first use)
    unsigned int* d_counter = nullptr;      // grid-barrier word of the persistent kernel
    bool any_never = false;                 // some replica's current table has a never-accepted class
    uint8_t* d_aux = nullptr;        // bit-packed kernel's constant 2 KiB lookup table, on this handle's device
    int8_t* d_stage = nullptr;       // natural-layout staging for spin_get_spins / spin_set_spins / spin_set_bonds (grow-only)
    size_t stage_bytes = 0;
    long long* d_mom = nullptr;      // [B][8] moments of spin_sweep_measure
    long long* d_macc = nullptr;     // [B][3] sums of the fused E / M reduction (streaming spin_sweep_measure), lazily allocated
    long long* d_trace = nullptr;    // trace buffer of spin_sweep_measure (grow-only)
    size_t trace_bytes = 0;
    // scratch (host, pinned): two table buffers used alternately, each guarded by the event recorded after its upload,
    // so that spin_sweep never waits for earlier sweeps, only (rarely) for the copy issued two calls ago
    uint32_t* h_tables[2] = {nullptr, nullptr};
    cudaEvent_t table_ev[2] = {nullptr, nullptr};
    int table_slot = 0;
    long long* h_EM = nullptr;       // [2][B] pinned, spin_observables
    RoundKeys rk;
    int64_t launches = 0;
    // second stream for the replica groups of a streaming sweep (streaming_begin / streaming_end), created on first use
    cudaStream_t aux_stream = nullptr;
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
    // CUDA graph of kGraphSweeps streaming sweeps whose nodes read the sweep index from d_graph_t (sweep_graph below)
    cudaGraphExec_t graph_exec = nullptr;
    unsigned long long* d_graph_t = nullptr;
    const unsigned long long* capture_t = nullptr;   // non-NULL only while the graph is being captured
    int graph_launches = 0;                          // kernels per replay
    const uint32_t* graph_bonds = nullptr;           // SweepArgs::bonds the graph was captured with
    bool graph_failed = false;
    int32_t policy = SPIN_POLICY_AUTO;
};

namespace {

RoundKeys make_round_keys(uint64_t seed) {
    RoundKeys rk;
    uint32_t k0 = (uint32_t)(seed & 0xFFFFFFFFull), k1 = (uint32_t)(seed >> 32);
    for (int r = 0; r < 10; ++r) {
        rk.k0[r] = k0;
        rk.k1[r] = k1;
        k0 += kPhiloxW0;
        k1 += kPhiloxW1;
    }
    return rk;
}

bool shape_ok(int32_t batch, int32_t L) { return batch >= 1 && L >= 2 && (L & 1) == 0 && L <= 65536; }

int check_sweep_args(const spin_sim* sim, const double* beta, double J, double h, int64_t n_sweeps, int64_t off) {
    if (!sim) return fail(SPIN_ERR_INVALID, "spin_sweep: NULL handle");
    if (!beta) return fail(SPIN_ERR_INVALID, "spin_sweep: beta is NULL");
    if (!std::isfinite(J) || !std::isfinite(h)) return fail(SPIN_ERR_INVALID, "spin_sweep: J and h must be finite");
    if (n_sweeps < 0 || off < 0) return fail(SPIN_ERR_INVALID, "spin_sweep: n_sweeps and sweep_offset must be >= 0");
    if (off > (1ll << 56) || n_sweeps > (1ll << 56) || off + n_sweeps > (1ll << 56))
        return fail(SPIN_ERR_INVALID, "spin_sweep: sweep_offset + n_sweeps exceeds 2^56");
    for (int b = 0; b < sim->batch; ++b)
        if (!std::isfinite(beta[b]) || beta[b] < 0.0)
            return fail(SPIN_ERR_INVALID, "spin_sweep: beta[%d] must be finite and >= 0", b);
    return SPIN_OK;
}

// One replica's device record for (beta, J, h).
void build_record(const spin_sim* sim, int b, double beta, double J, double h, uint32_t* rec) {
    std::memset(rec, 0, sizeof(uint32_t) * kTableStride);
    if (sim->model == SPIN_MODEL_ISING) {
        for (int d = 0; d < 2; ++d)
            for (int nd = 0; nd <= 4; ++nd) {
                const int s = d ? -1 : 1, nn = 4 - 2 * nd;
                encode(ising_class(beta, J, h, s, nn), d * 8 + nd, rec);
            }
    } else {
        for (int dn = -4; dn <= 4; ++dn) encode(potts_class(beta, J, dn), dn + 4, rec);
    }
    rec[kTabQ] = (uint32_t)sim->q[b];
}

// Real couplings and per-site fields: Alg. 1's acceptance for each of the 32 (own spin, neighbour configuration) classes
// of every site, evaluated on the host in IEEE double in the order the oracle uses (general_oracle.cpp): local field
// F = Jv[i-1][j] s_up + Jv[i][j] s_down + Jh[i][j-1] s_left + Jh[i][j] s_right + B[i][j], dE = 2 s F, then O4.
int upload_general_thresholds(spin_sim* sim, const double* beta) {
    const int L = sim->L;
    const size_t N = (size_t)L * L, B = (size_t)sim->batch;
    bool same = sim->g_beta.size() == B;
    for (size_t b = 0; same && b < B; ++b) same = sim->g_beta[b] == beta[b];
    if (same) return SPIN_OK;                               // thresholds on the device are current
    std::vector<uint32_t> thr, alw;
    try { thr.resize(B * N * 32); alw.resize(B * N); }
    catch (...) { return fail(SPIN_ERR_NOMEM, "spin_sweep: out of host memory for %zu per-site thresholds", B * N * 32); }
    for (size_t b = 0; b < B; ++b)
        for (int i = 0; i < L; ++i)
            for (int j = 0; j < L; ++j) {
                const int iu = i == 0 ? L - 1 : i - 1, jl = j == 0 ? L - 1 : j - 1;
                const size_t x = b * N + (size_t)i * L + j;
                const double ju = sim->g_Jv[b * N + (size_t)iu * L + j], jd = sim->g_Jv[x];
                const double jlft = sim->g_Jh[b * N + (size_t)i * L + jl], jrgt = sim->g_Jh[x], fb = sim->g_B[x];
                uint32_t mask = 0u;
                for (int k = 0; k < 32; ++k) {
                    const double s = (k & 16) ? -1.0 : 1.0;
                    const double su = (k & 1) ? -1.0 : 1.0, sd = (k & 2) ? -1.0 : 1.0, sl = (k & 4) ? -1.0 : 1.0, sr = (k & 8) ? -1.0 : 1.0;
                    const double F = ju * su + jd * sd + jlft * sl + jrgt * sr + fb;
                    const ClassAccept c = class_accept(beta[b], 2.0 * s * F);
                    thr[x * 32 + k] = c.T;
                    if (c.always) mask |= 1u << k;
                }
                alw[x] = mask;
            }
    CUDA_TRY(cudaMemcpyAsync(sim->d_thr, thr.data(), thr.size() * sizeof(uint32_t), cudaMemcpyHostToDevice, sim->stream));
    CUDA_TRY(cudaMemcpyAsync(sim->d_alw, alw.data(), alw.size() * sizeof(uint32_t), cudaMemcpyHostToDevice, sim->stream));
    CUDA_TRY(cudaStreamSynchronize(sim->stream));           // the host vectors go out of scope
    try { sim->g_beta.assign(beta, beta + B); } catch (...) { sim->g_beta.clear(); }   // no cache: rebuilt next call
    return SPIN_OK;
}

// Potts with a field on the state label and / or bond signs: class (dn, dl = new - old), dE = -(J dn) - h dl.
int upload_potts_general(spin_sim* sim, const double* beta, double J, double h) {
    const size_t B = (size_t)sim->batch;
    if (!sim->d_tab2) CUDA_TRY(cudaMalloc(&sim->d_tab2, sizeof(unsigned long long) * 9 * 255 * B));
    std::vector<unsigned long long> tab;
    try { tab.assign(B * 9 * 255, 0ull); }
    catch (...) { return fail(SPIN_ERR_NOMEM, "spin_sweep: out of host memory for the Potts class tables"); }
    for (size_t b = 0; b < B; ++b) {
        const int q = sim->q[b];
        for (int dn = -4; dn <= 4; ++dn)
            for (int dl = -(q - 1); dl <= q - 1; ++dl) {
                const double dE = -(J * (double)dn) - h * (double)dl;
                const ClassAccept c = class_accept(beta[b], dE);
                tab[(b * 9 + (size_t)(dn + 4)) * 255 + (size_t)(dl + 127)] = ((unsigned long long)(c.always ? 1 : 0) << 32) | c.T;
            }
    }
    CUDA_TRY(cudaMemcpyAsync(sim->d_tab2, tab.data(), tab.size() * sizeof(unsigned long long), cudaMemcpyHostToDevice, sim->stream));
    CUDA_TRY(cudaStreamSynchronize(sim->stream));
    return SPIN_OK;
}

// Build the per-replica records on the host and enqueue their copy.
int upload_tables(spin_sim* sim, const double* beta, double J, double h) {
    // the upload issued two calls ago may still be reading this pinned buffer; nothing else is waited for
    const int slot = sim->table_slot;
    sim->table_slot ^= 1;
    uint32_t* h_tab = sim->h_tables[slot];
    CUDA_TRY(cudaEventSynchronize(sim->table_ev[slot]));
    sim->any_never = false;
    for (int b = 0; b < sim->batch; ++b) {
        build_record(sim, b, beta[b], J, h, h_tab + (size_t)b * kTableStride);
        if (h_tab[(size_t)b * kTableStride + kTabNever]) sim->any_never = true;
    }
    CUDA_TRY(cudaMemcpyAsync(sim->d_tables, h_tab, sizeof(uint32_t) * kTableStride * (size_t)sim->batch,
                             cudaMemcpyHostToDevice, sim->stream));
    CUDA_TRY(cudaEventRecord(sim->table_ev[slot], sim->stream));
    if (sim->general) {
        const int rg = upload_general_thresholds(sim, beta);
        if (rg != SPIN_OK) return rg;
    }
    sim->potts_general = sim->model == SPIN_MODEL_POTTS && (h != 0.0 || sim->d_bond_nat != nullptr);
    if (sim->potts_general) {
        const int rp = upload_potts_general(sim, beta, J, h);
        if (rp != SPIN_OK) return rp;
    }
    return SPIN_OK;
}

SweepArgs sweep_args(const spin_sim* sim, int64_t t, int colour) {
    SweepArgs a;
    a.lattice = sim->lattice;
    a.tables = sim->d_tables;
    a.batch = sim->batch;
    a.L = sim->L;
    a.replica_offset = sim->replica_offset;
    a.c2 = (uint32_t)((uint64_t)t & 0xFFFFFFFFull);
    const uint32_t domain = sim->model == SPIN_MODEL_ISING ? kDomainIsing : kDomainPotts;
    a.c3 = (uint32_t)(((uint64_t)t >> 32) & 0xFFFFFFull) | ((uint32_t)colour << 24) | (domain << 28);
    a.colour = colour;
    a.aux = sim->d_aux;
    a.bonds = sim->d_bonds;
    a.rk = sim->rk;
    a.pdl_trigger = kPdlAtExit;
    a.plan_scale = 1;
    a.potts_tab2 = nullptr;
    a.measure_acc = nullptr;
    a.fin_E = nullptr; a.fin_M = nullptr; a.fin_mom = nullptr; a.fin_pending = 0;
    a.t_dev = sim->capture_t;
    a.t_rel = sim->capture_t ? (uint32_t)t : 0u;
    return a;
}

// Shapes AUTO sends to the temporally blocked tile kernel (ising_int8.cu) for plain sweeps: up to 16 replicas and 2^21
// sites in all, i.e. launches that leave the streaming kernels latency-bound and give one CTA per replica too few CTAs.
// Measured (profiles/r2_policy_grid.md): 1 x 640^2 271 vs 87 flips/ns streaming, 16 x 128^2 201 vs 73 resident,
// 16 x 256^2 265 vs 235, 1 x 1024^2 265 vs 219, 4 x 640^2 351 vs 325; beyond that it loses (16 x 416^2 412 vs 407 is a
// tie, 4 x 1024^2 470 vs 576, 64 x 128^2 269 vs 291 resident).
bool prefer_tiled(const spin_sim* sim) {
    if (sim->model != SPIN_MODEL_ISING || sim->layout != SPIN_LAYOUT_INT8 || sim->general || sim->d_bond_nat) return false;
    if (sim->policy != SPIN_POLICY_AUTO) return false;
    return sim->L >= 64 && sim->batch <= 16 && (long long)sim->batch * sim->L * sim->L <= (1ll << 21) &&
           ising_int8_tiled_fits(sim->batch, sim->L);
}

// Shared-memory-resident path (ising_int8.cu): Ising, int8 layout, replica fits one CTA.  AUTO uses it when the
// batch gives every SM work (or when the lattice is so small that the streaming kernels are launch-bound anyway).
bool use_resident(const spin_sim* sim, bool measure) {
    if (sim->model != SPIN_MODEL_ISING || sim->layout != SPIN_LAYOUT_INT8 || !ising_int8_resident_fits(sim->L)) return false;
    if (sim->general || sim->d_bond_nat) return false;            // per-bond couplings run on the general kernels
    if (sim->policy == SPIN_POLICY_STREAMING || sim->policy == SPIN_POLICY_PERSISTENT || sim->policy == SPIN_POLICY_TILED ||
        sim->policy == SPIN_POLICY_GRAPH) return false;
    if (sim->policy == SPIN_POLICY_RESIDENT) return true;
    // Measured on B200 (profiles/r2_policy_grid.md): one CTA per replica wins while a half-sweep of a replica is a handful
    // of warps and there are many replicas (L <= 128: 503 vs 229 flips/ns at 256 x 64^2, 767 vs 579 at 256 x 128^2).
    if (!measure && prefer_tiled(sim)) return false;               // few small replicas: the tiled kernel spreads them over the SMs
    // larger replicas stream: with the batch swept as two replica groups even the ragged L = 160 / 224 shapes are faster
    // there (256 x 224^2: 930 vs 763 flips/ns), and measured runs have the reduction fused into the colour-1 launch
    // (1024 x 256^2 with moments: 1171 vs 1047)
    return sim->L <= 128;
}

// Bit-packed resident kernel (ising_bits.cu): uniform couplings, replica fits one CTA.  On request only
// (SPIN_POLICY_RESIDENT): one CTA per replica idles SMs or loses to the two-group streaming path on every measured shape
// (64 x 1024^2 406 vs 1266 flips/ns, 148 x 1024^2 939 vs 1339, 1024 x 256^2 1220 vs 1330).
bool use_bits_resident(const spin_sim* sim) {
    if (sim->model != SPIN_MODEL_ISING || sim->layout != SPIN_LAYOUT_BITPACKED || sim->d_bonds) return false;
    if (!ising_bits_resident_fits(sim->L)) return false;
    return sim->policy == SPIN_POLICY_RESIDENT;
}

bool enqueue_bits_resident(spin_sim* sim, int64_t t0, int64_t n_sweeps, const uint32_t* tables = nullptr) {
    ResidentArgs a;
    a.lattice = sim->lattice;
    a.tables = tables ? tables : sim->d_tables;
    a.batch = sim->batch; a.L = sim->L; a.replica_offset = sim->replica_offset; a.measure = 0u;
    a.t0 = (unsigned long long)t0; a.n_sweeps = n_sweeps;
    a.E_trace = nullptr; a.M_trace = nullptr; a.moments = nullptr;
    a.rk = sim->rk;
    const int n = launch_ising_bits_resident(a, sim->d_aux, sim->stream);
    sim->launches += n;
    return n > 0;
}

// Persistent cooperative kernel (ising_int8.cu): uniform Ising model, int8 layout, L % 32 == 0, no never-classes in the
// current tables.  On request only (SPIN_POLICY_PERSISTENT): a grid barrier costs ~2.3 us here, and since the streaming
// kernels release the next launch where its blocks get a balanced placement (spin_internal.cuh, PdlTrigger) they are
// faster on every shape of the measured grid (profiles/r2_policy_grid.md: 1 x 1024^2 224 vs 213 flips/ns, 4 x 640^2
// 327 vs 279, 16 x 256^2 236 vs 214).
bool use_persistent(const spin_sim* sim) {
    if (sim->model != SPIN_MODEL_ISING || sim->layout != SPIN_LAYOUT_INT8 || sim->L % 32 != 0) return false;
    if (sim->general || sim->d_bond_nat || sim->any_never) return false;
    return sim->policy == SPIN_POLICY_PERSISTENT;
}

SweepArgs sweep_args(const spin_sim* sim, int64_t t, int colour);

// Temporally blocked tile kernel (ising_int8.cu): uniform Ising model, int8 layout, L % 8 == 0; four sweeps per launch on
// tiles with halos, at most one tile per SM, one thread per 4-site word for the whole launch.  AUTO: prefer_tiled().
bool use_tiled(const spin_sim* sim) {
    if (sim->model != SPIN_MODEL_ISING || sim->layout != SPIN_LAYOUT_INT8) return false;
    if (sim->general || sim->d_bond_nat) return false;
    if (!ising_int8_tiled_fits(sim->batch, sim->L)) return false;
    if (sim->policy == SPIN_POLICY_TILED) return true;
    return prefer_tiled(sim);
}

bool enqueue_tiled(spin_sim* sim, int64_t t0, int64_t n_sweeps, const uint32_t* tables = nullptr) {
    if (!sim->d_shadow && cudaMalloc(&sim->d_shadow, sim->lattice_bytes) != cudaSuccess) {
        cudaGetLastError();
        sim->d_shadow = nullptr;
        return false;
    }
    SweepArgs a = sweep_args(sim, t0, 0);
    if (tables) a.tables = tables;
    const int n = launch_ising_int8_tiled(a, sim->d_shadow, (unsigned long long)t0, n_sweeps, sim->stream);
    sim->launches += n;
    return n > 0;
}

// Returns false when the cooperative launch was not possible (the caller streams instead).
bool enqueue_persistent(spin_sim* sim, int64_t t0, int64_t n_sweeps, const uint32_t* tables = nullptr) {
    SweepArgs a = sweep_args(sim, t0, 0);
    if (tables) a.tables = tables;
    for (int64_t done = 0; done < n_sweeps;) {
        const int64_t chunk = n_sweeps - done < (1ll << 20) ? n_sweeps - done : (1ll << 20);   // barrier counter stays below 2^31
        const int n = launch_ising_int8_persistent(a, (unsigned long long)(t0 + done), chunk, sim->d_counter, sim->stream);
        if (n == 0) {
            if (done == 0) return false;
            for (int64_t t = t0 + done; t < t0 + n_sweeps; ++t) {      // finish on the streaming path
                SweepArgs h0 = sweep_args(sim, t, 0), h1 = sweep_args(sim, t, 1);
                if (tables) { h0.tables = tables; h1.tables = tables; }
                sim->launches += launch_ising_int8_half_sweep(h0, sim->stream);
                sim->launches += launch_ising_int8_half_sweep(h1, sim->stream);
            }
            return true;
        }
        sim->launches += n;
        done += chunk;
    }
    return true;
}

void enqueue_resident(spin_sim* sim, int64_t t0, int64_t n_sweeps, bool measure, long long* E_trace, long long* M_trace,
                      long long* moments, const uint32_t* tables = nullptr) {
    ResidentArgs a;
    a.lattice = sim->lattice;
    a.tables = tables ? tables : sim->d_tables;
    a.batch = sim->batch;
    a.L = sim->L;
    a.replica_offset = sim->replica_offset;
    a.measure = measure ? 1u : 0u;
    a.t0 = (unsigned long long)t0;
    a.n_sweeps = n_sweeps;
    a.E_trace = E_trace;
    a.M_trace = M_trace;
    a.moments = moments;
    a.rk = sim->rk;
    sim->launches += launch_ising_int8_resident(a, sim->stream);
}

void enqueue_half_sweep(spin_sim* sim, int64_t t, int colour, const uint32_t* tables = nullptr) {
    SweepArgs a = sweep_args(sim, t, colour);
    if (tables) a.tables = tables;                          // a step of spin_sweep_schedule
    const size_t nat = (size_t)sim->batch * sim->L * sim->L;
    if (sim->model == SPIN_MODEL_POTTS) {
        if (sim->potts_general && (sim->d_bond_nat || sim->L % 32 != 0))
            sim->launches += launch_potts_int8_general_half_sweep(a, sim->d_tab2, sim->d_bond_nat,
                                                                  sim->d_bond_nat ? sim->d_bond_nat + nat : nullptr, sim->stream);
        else {
            if (sim->potts_general) a.potts_tab2 = sim->d_tab2;   // a field, uniform couplings: the row-marching kernel's field variant
            sim->launches += launch_potts_int8_half_sweep(a, sim->stream);
        }
    } else if (sim->layout == SPIN_LAYOUT_BITPACKED) sim->launches += launch_ising_bits_half_sweep(a, sim->stream);
    else if (sim->general) sim->launches += launch_ising_int8_general_half_sweep(a, sim->d_thr, sim->d_alw, sim->stream);
    else if (sim->d_bond_nat) sim->launches += launch_ising_int8_bonds_half_sweep(a, sim->d_bond_nat, sim->d_bond_nat + nat, sim->stream);
    else sim->launches += launch_ising_int8_half_sweep(a, sim->stream);
}

// ---- streaming sweeps on two replica groups ---------------------------------------------------------------------------
// A chain of dependent half-sweep launches leaves the GPU idle between them (the drain of one launch, the release and
// ramp-up of the next).  Replicas are independent, so the batch is split in two halves whose chains run on two streams: the
// gaps of one are covered by the kernels of the other.  Measured (profiles/r2_pdl_placement.md): 64 x 1024^2 int8 1178 ->
// 1278 flips/ns, bit-packed 1269 -> 1351; 16 x 2560^2 1089 -> 1226 / 1287 -> 1383; 16 x 1024^2 956 -> 1153; it loses when a
// half is too small to fill the GPU on its own turn (16 x 640^2 724 -> 695, 4 x 1024^2 598 -> 525), so it is used from 0.15
// (bit-packed), 0.2 (Potts), 0.3 (int8) waves of 8-row blocks upwards.  Class-table models only (the general kernels index natural-order coupling arrays).
int streaming_groups(const spin_sim* sim) {
    if (sim->batch < 2 || sim->general || sim->d_bond_nat) return 1;   // (Potts with a field and uniform couplings: groups as usual)
    if (sim->policy != SPIN_POLICY_AUTO && sim->policy != SPIN_POLICY_STREAMING && sim->policy != SPIN_POLICY_GRAPH) return 1;
    const bool bits = sim->layout == SPIN_LAYOUT_BITPACKED;
    if (sim->L % (bits ? 64 : 32) != 0) return 1;                // the generic kernels are not planned
    const int perSm = sim->model == SPIN_MODEL_POTTS ? kPottsBlocksPerSm : bits ? kIsingBitsBlocksPerSm : kIsingInt8BlocksPerSm;
    const double threads8 = (double)(sim->L / 8) * (sim->L >> (bits ? 6 : 5)) * sim->batch;
    const double from = sim->model == SPIN_MODEL_POTTS ? 0.2 : bits ? 0.15 : 0.3;   // measured crossovers, in waves of 8-row blocks
    return threads8 >= from * 128.0 * 148.0 * perSm ? 2 : 1;
}

// Fork: the second stream waits for everything enqueued so far on the handle's stream.  Returns the number of groups
// actually available (1 if the stream / events cannot be created).
int streaming_begin(spin_sim* sim) {
    int G = streaming_groups(sim);
    if (G < 2) return 1;
    if (!sim->aux_stream) {
        if (cudaStreamCreateWithFlags(&sim->aux_stream, cudaStreamNonBlocking) != cudaSuccess ||
            cudaEventCreateWithFlags(&sim->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&sim->ev_join, cudaEventDisableTiming) != cudaSuccess) {
            cudaGetLastError();
            if (sim->aux_stream) cudaStreamDestroy(sim->aux_stream);
            if (sim->graph_exec) cudaGraphExecDestroy(sim->graph_exec);
    if (sim->d_graph_t) cudaFree(sim->d_graph_t);
    if (sim->ev_fork) cudaEventDestroy(sim->ev_fork);
            sim->aux_stream = nullptr; sim->ev_fork = nullptr; sim->ev_join = nullptr;
            return 1;
        }
    }
    if (cudaEventRecord(sim->ev_fork, sim->stream) != cudaSuccess || cudaStreamWaitEvent(sim->aux_stream, sim->ev_fork, 0) != cudaSuccess) {
        cudaGetLastError();
        return 1;
    }
    return G;
}

// Join: the handle's stream waits for the second one (every later operation of the handle sees all replicas done).
void streaming_end(spin_sim* sim, int G) {
    if (G < 2) return;
    cudaEventRecord(sim->ev_join, sim->aux_stream);
    cudaStreamWaitEvent(sim->stream, sim->ev_join, 0);
}

// n_sweeps sweeps from t0 for all replicas: the half-sweeps of the groups interleaved in issue order.
void enqueue_streaming(spin_sim* sim, int G, int64_t t0, int64_t n_sweeps, const uint32_t* tables = nullptr) {
    if (G < 2) {
        for (int64_t t = t0; t < t0 + n_sweeps; ++t) {
            enqueue_half_sweep(sim, t, 0, tables);
            enqueue_half_sweep(sim, t, 1, tables);
        }
        return;
    }
    const size_t perReplica = sim->lattice_bytes / (size_t)sim->batch;
    const size_t bondWords = (size_t)2 * 4 * sim->L * (sim->L >> 6);       // sign planes of one replica (bit-packed +-J)
    for (int64_t t = t0; t < t0 + n_sweeps; ++t)
        for (int colour = 0; colour < 2; ++colour)
            for (int g = 0; g < G; ++g) {
                const int b0 = (int)((long long)sim->batch * g / G), b1 = (int)((long long)sim->batch * (g + 1) / G);
                SweepArgs a = sweep_args(sim, t, colour);
                a.lattice = (char*)sim->lattice + perReplica * (size_t)b0;
                a.tables = (tables ? tables : sim->d_tables) + (size_t)b0 * kTableStride;
                a.batch = b1 - b0;
                a.replica_offset = sim->replica_offset + (uint32_t)b0;
                if (a.bonds) a.bonds += bondWords * (size_t)b0;
                a.plan_scale = G;
                if (sim->potts_general) a.potts_tab2 = sim->d_tab2 + (size_t)9 * 255 * b0;
                cudaStream_t st = g == 0 ? sim->stream : sim->aux_stream;
                if (sim->model == SPIN_MODEL_POTTS) sim->launches += launch_potts_int8_half_sweep(a, st);
                else if (sim->layout == SPIN_LAYOUT_BITPACKED) sim->launches += launch_ising_bits_half_sweep(a, st);
                else sim->launches += launch_ising_int8_half_sweep(a, st);
            }
}

// ---- streaming sweeps with the E / M reduction fused into the colour-1 launch (spin_sweep_measure) ----------------------
// Uniform Ising model, int8 layout, L % 32 == 0: the colour-1 kernel variant adds three sums per replica into d_macc and a
// thread per replica of the NEXT sweep's colour-0 launch (a finalisation kernel after the last sweep) turns them into E
// and M, writes the trace sample and / or accumulates the moments, and clears the sums.  Two launches per sweep, as for
// spin_sweep, instead of two launches, a memset, a reduction over the whole lattice and the moment kernel; the same replica
// groups as spin_sweep.  (A finalisation kernel per sweep in the chain cost 10 us per sweep: it keeps the next colour-0
// launch from being staged behind the colour-1 launch.)
bool fused_measure_eligible(const spin_sim* sim) {
    return sim->model == SPIN_MODEL_ISING && sim->layout == SPIN_LAYOUT_INT8 && sim->L % 32 == 0 && !sim->general && !sim->d_bond_nat;
}

// E_trace / M_trace: device [n_sweeps][B] or nullptr; d_mom: device [B][8] or nullptr.
int enqueue_streaming_measure(spin_sim* sim, int64_t t0, int64_t n_sweeps, long long* E_trace, long long* M_trace, long long* d_mom) {
    const size_t B = (size_t)sim->batch;
    if (!sim->d_macc) {
        const cudaError_t e = cudaMalloc(&sim->d_macc, sizeof(long long) * 3 * B);
        if (e != cudaSuccess) { sim->d_macc = nullptr; return fail(SPIN_ERR_NOMEM, "cudaMalloc for the measurement sums: %s", cudaGetErrorString(e)); }
    }
    CUDA_TRY(cudaMemsetAsync(sim->d_macc, 0, sizeof(long long) * 3 * B, sim->stream));
    const int G = streaming_begin(sim);
    const size_t perReplica = sim->lattice_bytes / B;
    const long long sites = (long long)sim->L * sim->L;
    for (int64_t local = 0; local <= n_sweeps; ++local) {
        // sweep `local` (none after the last); its colour-0 launch first finalises sweep local - 1
        for (int colour = 0; colour < (local < n_sweeps ? 2 : 0); ++colour)
            for (int g = 0; g < G; ++g) {
                const int b0 = (int)((long long)sim->batch * g / G), b1 = (int)((long long)sim->batch * (g + 1) / G);
                SweepArgs a = sweep_args(sim, t0 + local, colour);
                a.lattice = (char*)sim->lattice + perReplica * (size_t)b0;
                a.tables = sim->d_tables + (size_t)b0 * kTableStride;
                a.batch = b1 - b0;
                a.replica_offset = sim->replica_offset + (uint32_t)b0;
                a.plan_scale = G;
                a.measure_acc = sim->d_macc + 3 * (size_t)b0;
                if (colour == 0 && local > 0) {
                    a.fin_pending = 1;
                    a.fin_E = E_trace ? E_trace + (size_t)(local - 1) * B + b0 : nullptr;
                    a.fin_M = M_trace ? M_trace + (size_t)(local - 1) * B + b0 : nullptr;
                    a.fin_mom = d_mom ? d_mom + 8 * (size_t)b0 : nullptr;
                }
                sim->launches += launch_ising_int8_half_sweep(a, g == 0 ? sim->stream : sim->aux_stream);
            }
        if (local == n_sweeps)
            for (int g = 0; g < G; ++g) {
                const int b0 = (int)((long long)sim->batch * g / G), b1 = (int)((long long)sim->batch * (g + 1) / G);
                sim->launches += launch_ising_measure_finalize(sim->d_macc + 3 * (size_t)b0, b1 - b0, sites,
                                                               E_trace ? E_trace + (size_t)(local - 1) * B + b0 : nullptr,
                                                               M_trace ? M_trace + (size_t)(local - 1) * B + b0 : nullptr,
                                                               d_mom ? d_mom + 8 * (size_t)b0 : nullptr, g == 0 ? sim->stream : sim->aux_stream);
            }
    }
    streaming_end(sim, G);
    return SPIN_OK;
}

// ---- streaming sweeps replayed from a CUDA graph (SPIN_POLICY_GRAPH) ----------------------------------------------------
// A chain of half-sweep launches costs the host 2-4 us per launch (about half of what the GPU needs per launch on the
// paper's mid-size shapes), so a busy or jittery host thread shows up in the sweep rate.  Under this policy a graph of
// kGraphSweeps sweeps is captured once per handle from the very launchers of the streaming path (same kernels, same launch
// plan, same replica groups; the capture keeps the programmatic edges); its kernels take the sweep index from device memory
// (SweepArgs::t_dev + t_rel, the kDevT instantiations) and a last node advances it, so a replay needs no parameter update:
// one cudaGraphLaunch per 64 sweeps.  Measured (profiles/r2_pdl_placement.md): host time per 240 sweeps 1.2-3.2 ms ->
// 0.03 ms; GPU rate 1-5 % below the stream launches (1 x 2560^2 695 vs 720 flips/ns, 64 x 1024^2 1282 vs 1284): replaying
// is not faster on the GPU than programmatic dependent launches, it only takes the host out of the loop.
constexpr int kGraphSweeps = 64;

__global__ void graph_set_t_kernel(unsigned long long* t, unsigned long long v) { *t = v; }
__global__ void graph_advance_t_kernel(unsigned long long* t, unsigned long long k) { *t += k; }

// Class-table models on the row-marching kernels (the only ones with kDevT instantiations).
bool use_graph(const spin_sim* sim) {
    if (sim->policy != SPIN_POLICY_GRAPH || sim->graph_failed) return false;
    if (sim->stream == nullptr || sim->stream == cudaStreamLegacy) return false;   // the legacy default stream cannot be captured
    if (sim->general || sim->d_bond_nat || sim->potts_general) return false;
    return sim->L % (sim->layout == SPIN_LAYOUT_BITPACKED ? 64 : 32) == 0;
}

// Returns 1 if all n_sweeps sweeps were enqueued, 0 if the caller should use the stream path (nothing enqueued), -1 on a
// CUDA error after part of the work was enqueued.
int enqueue_graph_sweeps(spin_sim* sim, int64_t t0, int64_t n_sweeps) {
    if (!use_graph(sim) || n_sweeps < kGraphSweeps) return 0;
    if (sim->graph_exec && sim->graph_bonds != sim->d_bonds) {      // spin_set_bonds since the capture
        cudaGraphExecDestroy(sim->graph_exec);
        sim->graph_exec = nullptr;
    }
    if (!sim->graph_exec) {
        if (!sim->d_graph_t && cudaMalloc(&sim->d_graph_t, sizeof(unsigned long long)) != cudaSuccess) {
            cudaGetLastError();
            sim->d_graph_t = nullptr;
            sim->graph_failed = true;
            return 0;
        }
        const int probe = streaming_begin(sim);                     // creates the second stream and the events outside the capture
        streaming_end(sim, probe);
        const int64_t l0 = sim->launches;
        cudaGraph_t graph = nullptr;
        if (cudaStreamBeginCapture(sim->stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) {
            cudaGetLastError();
            sim->graph_failed = true;
            return 0;
        }
        sim->capture_t = sim->d_graph_t;
        const int G = streaming_begin(sim);
        enqueue_streaming(sim, G, 0, kGraphSweeps);
        streaming_end(sim, G);
        sim->capture_t = nullptr;
        graph_advance_t_kernel<<<1, 1, 0, sim->stream>>>(sim->d_graph_t, (unsigned long long)kGraphSweeps);
        const cudaError_t e1 = cudaStreamEndCapture(sim->stream, &graph);
        sim->graph_launches = (int)(sim->launches - l0) + 1;
        sim->launches = l0;                                          // nothing ran yet: replays are counted below
        cudaError_t e2 = cudaErrorUnknown;
        if (e1 == cudaSuccess && graph) e2 = cudaGraphInstantiate(&sim->graph_exec, graph, 0);
        if (graph) cudaGraphDestroy(graph);
        if (e1 != cudaSuccess || e2 != cudaSuccess) {
            cudaGetLastError();
            sim->graph_exec = nullptr;
            sim->graph_failed = true;                                // this handle streams from now on
            return 0;
        }
        sim->graph_bonds = sim->d_bonds;
    }
    graph_set_t_kernel<<<1, 1, 0, sim->stream>>>(sim->d_graph_t, (unsigned long long)t0);
    sim->launches += 1;
    int64_t done = 0;
    for (; done + kGraphSweeps <= n_sweeps; done += kGraphSweeps) {
        if (cudaGraphLaunch(sim->graph_exec, sim->stream) != cudaSuccess) return -1;
        sim->launches += sim->graph_launches;
    }
    if (done < n_sweeps) {                                           // the ragged rest as plain launches
        const int G = streaming_begin(sim);
        enqueue_streaming(sim, G, t0 + done, n_sweeps - done);
        streaming_end(sim, G);
    }
    return 1;
}

// Enqueue the reductions of the current lattice into E_out[b], M_out[b] (device int64, either may be NULL).
// The targets are zeroed first (the kernels accumulate).
int enqueue_observe(spin_sim* sim, long long* E_out, long long* M_out) {
    const size_t nb = sizeof(long long) * (size_t)sim->batch;
    if (E_out) CUDA_TRY(cudaMemsetAsync(E_out, 0, nb, sim->stream));
    const size_t nat = (size_t)sim->batch * sim->L * sim->L;
    if (sim->model == SPIN_MODEL_POTTS) {
        // with bond signs the energy comes from the general reduction; the histogram (M) from the regular one
        const bool signs = sim->d_bond_nat != nullptr;
        if (signs && E_out) sim->launches += launch_potts_general_observe(sim->lattice, sim->d_bond_nat, sim->d_bond_nat + nat, sim->batch,
                                                                          sim->L, E_out, nullptr, sim->stream);
        if (!signs || M_out)
            sim->launches += launch_potts_int8_observe(sim->lattice, sim->batch, sim->L, sim->d_q, signs ? nullptr : E_out,
                                                       M_out ? sim->d_hist : nullptr, sim->stream);
        if (M_out) sim->launches += launch_potts_finalize(sim->d_hist, sim->d_q, sim->batch, M_out, sim->stream);
    } else {
        if (M_out) CUDA_TRY(cudaMemsetAsync(M_out, 0, nb, sim->stream));
        if (sim->layout == SPIN_LAYOUT_INT8 && sim->d_bond_nat)
            sim->launches += launch_ising_int8_bonds_observe(sim->lattice, sim->d_bond_nat, sim->d_bond_nat + nat, sim->batch, sim->L,
                                                             E_out, M_out, sim->stream);
        else if (sim->layout == SPIN_LAYOUT_BITPACKED)
            sim->launches += launch_ising_bits_observe(sim->lattice, sim->d_bonds, sim->batch, sim->L, E_out, M_out, sim->stream);
        else
            sim->launches += launch_ising_int8_observe(sim->lattice, sim->batch, sim->L, E_out, M_out, sim->stream);
    }
    CUDA_TRY(cudaGetLastError());
    return SPIN_OK;
}

// Grow-only device staging buffers kept in the handle (no cudaMalloc / cudaFree on the per-call paths).
int ensure_stage(spin_sim* sim, size_t bytes) {
    if (sim->stage_bytes >= bytes) return SPIN_OK;
    CUDA_TRY(cudaStreamSynchronize(sim->stream));
    if (sim->d_stage) cudaFree(sim->d_stage);
    sim->d_stage = nullptr;
    sim->stage_bytes = 0;
    cudaError_t e = cudaMalloc(&sim->d_stage, bytes);
    if (e != cudaSuccess) { sim->d_stage = nullptr; return fail(SPIN_ERR_NOMEM, "cudaMalloc(%zu) for staging: %s", bytes, cudaGetErrorString(e)); }
    sim->stage_bytes = bytes;
    return SPIN_OK;
}

int ensure_trace(spin_sim* sim, size_t bytes) {
    if (sim->trace_bytes >= bytes) return SPIN_OK;
    CUDA_TRY(cudaStreamSynchronize(sim->stream));
    if (sim->d_trace) cudaFree(sim->d_trace);
    sim->d_trace = nullptr;
    sim->trace_bytes = 0;
    cudaError_t e = cudaMalloc(&sim->d_trace, bytes);
    if (e != cudaSuccess) { sim->d_trace = nullptr; return fail(SPIN_ERR_NOMEM, "cudaMalloc(%zu) for the trace: %s", bytes, cudaGetErrorString(e)); }
    sim->trace_bytes = bytes;
    return SPIN_OK;
}

}  // namespace

// =====================================================================================================
extern "C" {

const char* spin_last_error(void) { return g_last_error.c_str(); }

size_t spin_buffer_bytes(int32_t batch, int32_t L, int32_t model, int32_t layout) {
    if (!shape_ok(batch, L)) return 0;
    if (layout == SPIN_LAYOUT_BITPACKED) {
        if (model != SPIN_MODEL_ISING || L % 64 != 0) return 0;
        return (size_t)batch * L * L / 8;
    }
    if (layout != SPIN_LAYOUT_INT8) return 0;
    return (size_t)batch * L * L;
}

int spin_threshold_table(int32_t model, double beta, double J, double h, uint32_t* T, uint8_t* always) {
    if (!T || !always) return fail(SPIN_ERR_INVALID, "spin_threshold_table: NULL output");
    if (!std::isfinite(beta) || beta < 0.0 || !std::isfinite(J) || !std::isfinite(h))
        return fail(SPIN_ERR_INVALID, "spin_threshold_table: beta must be finite and >= 0, J and h finite");
    if (model == SPIN_MODEL_ISING) {
        for (int si = 0; si < 2; ++si)
            for (int ni = 0; ni < 5; ++ni) {
                const ClassAccept c = ising_class(beta, J, h, si ? 1 : -1, 2 * ni - 4);
                T[5 * si + ni] = c.T;
                always[5 * si + ni] = c.always ? 1 : 0;
            }
        return 10;
    }
    if (model == SPIN_MODEL_POTTS) {
        for (int dn = -4; dn <= 4; ++dn) {
            const ClassAccept c = potts_class(beta, J, dn);
            T[dn + 4] = c.T;
            always[dn + 4] = c.always ? 1 : 0;
        }
        return 9;
    }
    return fail(SPIN_ERR_INVALID, "spin_threshold_table: unknown model %d", model);
}

void spin_destroy(spin_sim* sim) {
    if (!sim) return;
    cudaSetDevice(sim->device);
    if (sim->stream || sim->lattice) cudaStreamSynchronize(sim->stream);
    if (sim->aux_stream) {
        cudaStreamSynchronize(sim->aux_stream);
        cudaStreamDestroy(sim->aux_stream);
    }
    if (sim->ev_fork) cudaEventDestroy(sim->ev_fork);
    if (sim->ev_join) cudaEventDestroy(sim->ev_join);
    if (sim->owns_lattice && sim->lattice) cudaFree(sim->lattice);
    if (sim->d_tables) cudaFree(sim->d_tables);
    if (sim->d_bonds) cudaFree(sim->d_bonds);
    if (sim->d_q) cudaFree(sim->d_q);
    if (sim->d_EM) cudaFree(sim->d_EM);
    if (sim->d_hist) cudaFree(sim->d_hist);
    if (sim->d_bad) cudaFree(sim->d_bad);
    if (sim->d_bond_nat) cudaFree(sim->d_bond_nat);
    if (sim->d_gen) cudaFree(sim->d_gen);
    if (sim->d_thr) cudaFree(sim->d_thr);
    if (sim->d_alw) cudaFree(sim->d_alw);
    if (sim->d_tab2) cudaFree(sim->d_tab2);
    if (sim->d_sched) cudaFree(sim->d_sched);
    if (sim->h_sched) cudaFreeHost(sim->h_sched);
    if (sim->sched_ev) cudaEventDestroy(sim->sched_ev);
    if (sim->d_shadow) cudaFree(sim->d_shadow);
    if (sim->d_counter) cudaFree(sim->d_counter);
    if (sim->d_aux) cudaFree(sim->d_aux);
    if (sim->d_stage) cudaFree(sim->d_stage);
    if (sim->d_mom) cudaFree(sim->d_mom);
    if (sim->d_macc) cudaFree(sim->d_macc);
    if (sim->d_trace) cudaFree(sim->d_trace);
    for (int k = 0; k < 2; ++k) {
        if (sim->h_tables[k]) cudaFreeHost(sim->h_tables[k]);
        if (sim->table_ev[k]) cudaEventDestroy(sim->table_ev[k]);
    }
    if (sim->h_EM) cudaFreeHost(sim->h_EM);
    delete sim;
}

static int create_impl(spin_sim* sim, void* device_buffer, size_t buffer_bytes) {
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev < 1)
        return fail(SPIN_ERR_CUDA, "no CUDA device available (%s); this library has no CPU fallback",
                    e != cudaSuccess ? cudaGetErrorString(e) : "device count is 0");
    CUDA_TRY(cudaGetDevice(&sim->device));
    sim->lattice_bytes = spin_buffer_bytes(sim->batch, sim->L, sim->model, sim->layout);
    if (device_buffer) {
        if (buffer_bytes < sim->lattice_bytes)
            return fail(SPIN_ERR_INVALID, "device_buffer holds %zu bytes, %zu needed", buffer_bytes, sim->lattice_bytes);
        if (((uintptr_t)device_buffer & 15u) != 0) return fail(SPIN_ERR_INVALID, "device_buffer must be 16-byte aligned");
        sim->lattice = device_buffer;
        sim->owns_lattice = false;
    } else {
        e = cudaMalloc(&sim->lattice, sim->lattice_bytes);
        if (e != cudaSuccess) {
            sim->lattice = nullptr;
            return fail(e == cudaErrorMemoryAllocation ? SPIN_ERR_NOMEM : SPIN_ERR_CUDA, "cudaMalloc(%zu): %s",
                        sim->lattice_bytes, cudaGetErrorString(e));
        }
        sim->owns_lattice = true;
    }
    const size_t B = (size_t)sim->batch;
    CUDA_TRY(cudaMalloc(&sim->d_tables, sizeof(uint32_t) * kTableStride * B));
    CUDA_TRY(cudaMalloc(&sim->d_q, sizeof(int32_t) * B));
    CUDA_TRY(cudaMalloc(&sim->d_EM, sizeof(long long) * 2 * B));
    CUDA_TRY(cudaMalloc(&sim->d_bad, sizeof(unsigned int)));
    CUDA_TRY(cudaMalloc(&sim->d_counter, sizeof(unsigned int)));
    if (sim->model == SPIN_MODEL_POTTS) {
        CUDA_TRY(cudaMalloc(&sim->d_hist, sizeof(unsigned int) * 128 * B));
        CUDA_TRY(cudaMemsetAsync(sim->d_hist, 0, sizeof(unsigned int) * 128 * B, sim->stream));
    }
    for (int k = 0; k < 2; ++k) {
        CUDA_TRY(cudaMallocHost(&sim->h_tables[k], sizeof(uint32_t) * kTableStride * B));
        CUDA_TRY(cudaEventCreateWithFlags(&sim->table_ev[k], cudaEventDisableTiming));
    }
    CUDA_TRY(cudaMallocHost(&sim->h_EM, sizeof(long long) * 2 * B));
    CUDA_TRY(cudaMalloc(&sim->d_mom, sizeof(long long) * 8 * B));
    // per-device kernel state lives in the handle (a handle belongs to the device current at creation)
    if (sim->layout == SPIN_LAYOUT_BITPACKED) {
        sim->d_aux = ising_bits_make_aux_table();
        if (!sim->d_aux) return fail(SPIN_ERR_CUDA, "could not allocate the bit-packed kernel's lookup table");
    }
    if (sim->model == SPIN_MODEL_ISING && sim->layout == SPIN_LAYOUT_INT8 && ising_int8_resident_fits(sim->L))
        CUDA_TRY(ising_int8_resident_configure());
    CUDA_TRY(cudaMemcpyAsync(sim->d_q, sim->q.data(), sizeof(int32_t) * B, cudaMemcpyHostToDevice, sim->stream));
    // row a0: initial lattice
    InitArgs ia;
    ia.lattice = sim->lattice;
    ia.q = sim->d_q;
    ia.batch = sim->batch;
    ia.L = sim->L;
    ia.replica_offset = sim->replica_offset;
    ia.rk = sim->rk;
    sim->launches += launch_init(ia, sim->model, sim->layout, sim->stream);
    CUDA_TRY(cudaGetLastError());
    CUDA_TRY(cudaStreamSynchronize(sim->stream));   // q vector / args no longer referenced after this
    return SPIN_OK;
}

spin_sim* spin_create_ex(int32_t batch, int32_t L, int32_t model, const int32_t* q_per_replica, int32_t q_uniform,
                         uint64_t seed, int32_t layout, int64_t replica_offset, void* device_buffer,
                         size_t buffer_bytes, void* cuda_stream) {
    if (batch < 1) { fail(SPIN_ERR_INVALID, "spin_create: batch must be >= 1"); return nullptr; }
    if (L < 2 || (L & 1)) { fail(SPIN_ERR_INVALID, "spin_create: L must be even and >= 2 (checkerboard on a periodic lattice)"); return nullptr; }
    if (L > 65536) { fail(SPIN_ERR_INVALID, "spin_create: L must be <= 65536"); return nullptr; }
    if (model != SPIN_MODEL_ISING && model != SPIN_MODEL_POTTS) { fail(SPIN_ERR_INVALID, "spin_create: unknown model %d", model); return nullptr; }
    if (layout != SPIN_LAYOUT_INT8 && layout != SPIN_LAYOUT_BITPACKED) { fail(SPIN_ERR_INVALID, "spin_create: unknown layout %d", layout); return nullptr; }
    if (replica_offset < 0 || replica_offset + (int64_t)batch > (1ll << 32)) { fail(SPIN_ERR_INVALID, "spin_create: replica_offset + batch must stay within [0, 2^32]"); return nullptr; }
    if (layout == SPIN_LAYOUT_BITPACKED && model != SPIN_MODEL_ISING) { fail(SPIN_ERR_UNSUPPORTED, "spin_create: the bit-packed layout is Ising only"); return nullptr; }
    if (layout == SPIN_LAYOUT_BITPACKED && L % 64 != 0) { fail(SPIN_ERR_UNSUPPORTED, "spin_create: the bit-packed layout needs L %% 64 == 0"); return nullptr; }
    spin_sim* sim = new (std::nothrow) spin_sim;
    if (!sim) { fail(SPIN_ERR_NOMEM, "spin_create: out of host memory"); return nullptr; }
    try {
    sim->batch = batch; sim->L = L; sim->model = model; sim->layout = layout; sim->seed = seed;
    sim->replica_offset = (uint32_t)replica_offset;
    sim->stream = (cudaStream_t)cuda_stream;
    sim->rk = make_round_keys(seed);
    sim->q.resize(batch);
    for (int b = 0; b < batch; ++b) {
        const int32_t qb = model == SPIN_MODEL_ISING ? 2 : (q_per_replica ? q_per_replica[b] : q_uniform);
        if (qb < 2 || qb > 127) {
            fail(SPIN_ERR_INVALID, "spin_create: q[%d] = %d outside 2..127", b, qb);
            delete sim;
            sim = nullptr;
            return nullptr;
        }
        sim->q[b] = qb;
    }
    const int rc = create_impl(sim, device_buffer, buffer_bytes);
    if (rc != SPIN_OK) {
        char keep[512];
        snprintf(keep, sizeof keep, "%s", g_last_error.c_str());
        spin_destroy(sim);
        sim = nullptr;
        cudaGetLastError();
        fail(rc, "%s", keep);
        return nullptr;
    }
    } catch (...) {   // std::bad_alloc from the host-side containers
        if (sim) spin_destroy(sim);
        fail(SPIN_ERR_NOMEM, "spin_create: out of host memory");
        return nullptr;
    }
    return sim;
}

spin_sim* spin_create(int32_t batch, int32_t L, int32_t q, uint64_t seed) {
    if (q < 2 || q > 127) { fail(SPIN_ERR_INVALID, "spin_create: q = %d outside 2..127", q); return nullptr; }
    return spin_create_ex(batch, L, q == 2 ? SPIN_MODEL_ISING : SPIN_MODEL_POTTS, nullptr, q, seed, SPIN_LAYOUT_INT8, 0,
                          nullptr, 0, nullptr);
}

int spin_set_stream(spin_sim* sim, void* cuda_stream) {
    if (!sim) return fail(SPIN_ERR_INVALID, "spin_set_stream: NULL handle");
    CUDA_TRY(cudaStreamSynchronize(sim->stream));
    sim->stream = (cudaStream_t)cuda_stream;
    return SPIN_OK;
}

int spin_synchronize(spin_sim* sim) {
    if (!sim) return fail(SPIN_ERR_INVALID, "spin_synchronize: NULL handle");
    CUDA_TRY(cudaStreamSynchronize(sim->stream));
    return SPIN_OK;
}

int64_t spin_kernel_launches(const spin_sim* sim) { return sim ? sim->launches : 0; }

const char* spin_kernel_variant(const spin_sim* sim) {
    if (!sim) return "";
    if (sim->model == SPIN_MODEL_POTTS) return potts_int8_variant(sim->L);
    if (use_bits_resident(sim)) return "ising_bits_resident";
    if (sim->layout == SPIN_LAYOUT_BITPACKED) return "ising_bits_rows32";
    if (use_resident(sim, false)) return "ising_int8_resident";
    if (use_tiled(sim)) return "ising_int8_tiled";
    if (use_persistent(sim)) return "ising_int8_persistent";
    return ising_int8_variant(sim->L);
}

// +-J couplings (Eq. 1 with per-bond J_ij).  The natural-layout signs are
// turned into per-colour bit planes (init_layout.cu): for the colour-c site (i, k), j = 2k + p, p = (i + c) & 1,
//   plane 0 (up)     Jv[i-1][j]          plane 1 (down)  Jv[i][j]
//   plane 2 (centre, the other-colour site with the same k)   p ? Jh[i][j-1] : Jh[i][j]
//   plane 3 (side,   the other-colour site k+1 if p else k-1) p ? Jh[i][j]   : Jh[i][j-1]
// bit = 1 iff the bond is -1.
int spin_set_bonds(spin_sim* sim, const int8_t* Jh, const int8_t* Jv) {
    if (!sim) return fail(SPIN_ERR_INVALID, "spin_set_bonds: NULL handle");
    if ((Jh == nullptr) != (Jv == nullptr)) return fail(SPIN_ERR_INVALID, "spin_set_bonds: Jh and Jv must both be given or both be NULL");
    CUDA_TRY(cudaSetDevice(sim->device));
    if (!Jh) {   // back to uniform couplings
        CUDA_TRY(cudaStreamSynchronize(sim->stream));
        if (sim->d_bonds) cudaFree(sim->d_bonds);
        sim->d_bonds = nullptr;
        if (sim->d_bond_nat) cudaFree(sim->d_bond_nat);
        sim->d_bond_nat = nullptr;
        return SPIN_OK;
    }
    if (sim->general) return fail(SPIN_ERR_INVALID, "spin_set_bonds: the handle has real couplings (spin_set_couplings); remove them first");
    if (sim->layout == SPIN_LAYOUT_INT8) {
        // int8 layout (Ising and Potts): the signs stay in the natural layout on the device, read by the general kernels
        const size_t n = (size_t)sim->batch * sim->L * sim->L;
        int8_t* d_new = nullptr;
        cudaError_t e = cudaMalloc(&d_new, 2 * n);
        if (e != cudaSuccess) return fail(SPIN_ERR_NOMEM, "spin_set_bonds: cudaMalloc: %s", cudaGetErrorString(e));
        unsigned int bad = 0;
        e = cudaMemcpyAsync(d_new, Jh, n, cudaMemcpyHostToDevice, sim->stream);
        if (e == cudaSuccess) e = cudaMemcpyAsync(d_new + n, Jv, n, cudaMemcpyHostToDevice, sim->stream);
        if (e == cudaSuccess) e = cudaMemsetAsync(sim->d_bad, 0, sizeof(unsigned int), sim->stream);
        if (e == cudaSuccess) {
            // +-1 validation = the Ising-spin validation over the two arrays
            sim->launches += launch_validate_natural(d_new, 2 * sim->batch, sim->L, SPIN_MODEL_ISING, nullptr, sim->d_bad, sim->stream);
            e = cudaMemcpyAsync(&bad, sim->d_bad, sizeof bad, cudaMemcpyDeviceToHost, sim->stream);
        }
        if (e == cudaSuccess) e = cudaStreamSynchronize(sim->stream);
        if (e != cudaSuccess) { cudaFree(d_new); return cuda_fail(e, "spin_set_bonds"); }
        if (bad) { cudaFree(d_new); return fail(SPIN_ERR_INVALID, "spin_set_bonds: bond signs must be +1 or -1"); }
        if (sim->d_bond_nat) cudaFree(sim->d_bond_nat);
        sim->d_bond_nat = d_new;
        return SPIN_OK;
    }
    // natural-layout signs -> device staging -> per-colour bit planes (validated on the device; a rejected call leaves
    // the handle's couplings as they were)
    const int L = sim->L;
    const size_t nat = (size_t)sim->batch * L * L;
    const size_t words = (size_t)sim->batch * 2 * 4 * L * (size_t)(L >> 6);
    const int rs = ensure_stage(sim, 2 * nat);
    if (rs != SPIN_OK) return rs;
    int8_t* d_nat = sim->d_stage;
    uint32_t* d_new = nullptr;
    cudaError_t e = cudaMalloc(&d_new, words * sizeof(uint32_t));
    if (e != cudaSuccess) return fail(SPIN_ERR_NOMEM, "spin_set_bonds: cudaMalloc: %s", cudaGetErrorString(e));
    unsigned int bad = 0;
    e = cudaMemcpyAsync(d_nat, Jh, nat, cudaMemcpyHostToDevice, sim->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(d_nat + nat, Jv, nat, cudaMemcpyHostToDevice, sim->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(sim->d_bad, 0, sizeof(unsigned int), sim->stream);
    if (e == cudaSuccess) {
        sim->launches += launch_bonds_from_natural(d_nat, d_nat + nat, d_new, sim->batch, L, sim->d_bad, sim->stream);
        e = cudaMemcpyAsync(&bad, sim->d_bad, sizeof bad, cudaMemcpyDeviceToHost, sim->stream);
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(sim->stream);
    if (e != cudaSuccess) { cudaFree(d_new); return cuda_fail(e, "spin_set_bonds"); }
    if (bad) { cudaFree(d_new); return fail(SPIN_ERR_INVALID, "spin_set_bonds: bond signs must be +1 or -1"); }
    if (sim->d_bonds) cudaFree(sim->d_bonds);
    sim->d_bonds = d_new;
    return SPIN_OK;
}

int spin_set_couplings(spin_sim* sim, const double* Jh, const double* Jv, const double* Bf) {
    if (!sim) return fail(SPIN_ERR_INVALID, "spin_set_couplings: NULL handle");
    const bool none = !Jh && !Jv && !Bf;
    if (!none && (!Jh || !Jv || !Bf)) return fail(SPIN_ERR_INVALID, "spin_set_couplings: Jh, Jv and B must all be given or all be NULL");
    CUDA_TRY(cudaSetDevice(sim->device));
    if (none) {
        CUDA_TRY(cudaStreamSynchronize(sim->stream));
        if (sim->d_gen) cudaFree(sim->d_gen);
        if (sim->d_thr) cudaFree(sim->d_thr);
        if (sim->d_alw) cudaFree(sim->d_alw);
        sim->d_gen = nullptr; sim->d_thr = nullptr; sim->d_alw = nullptr;
        sim->general = false;
        try { sim->g_Jh.clear(); sim->g_Jv.clear(); sim->g_B.clear(); sim->g_beta.clear(); } catch (...) {}
        return SPIN_OK;
    }
    if (sim->model != SPIN_MODEL_ISING || sim->layout != SPIN_LAYOUT_INT8)
        return fail(SPIN_ERR_UNSUPPORTED, "spin_set_couplings: real couplings are implemented for the Ising model in the int8 layout");
    if (sim->d_bond_nat) return fail(SPIN_ERR_INVALID, "spin_set_couplings: the handle has +-J bond signs (spin_set_bonds); remove them first");
    const size_t n = (size_t)sim->batch * sim->L * sim->L;
    for (size_t k = 0; k < n; ++k)
        if (!std::isfinite(Jh[k]) || !std::isfinite(Jv[k]) || !std::isfinite(Bf[k]))
            return fail(SPIN_ERR_INVALID, "spin_set_couplings: couplings and fields must be finite");
    try {
        sim->g_Jh.assign(Jh, Jh + n); sim->g_Jv.assign(Jv, Jv + n); sim->g_B.assign(Bf, Bf + n);
        sim->g_beta.clear();
    } catch (...) { sim->general = false; return fail(SPIN_ERR_NOMEM, "spin_set_couplings: out of host memory"); }
    CUDA_TRY(cudaStreamSynchronize(sim->stream));
    if (!sim->d_gen) {
        cudaError_t e = cudaMalloc(&sim->d_gen, 3 * n * sizeof(double));
        if (e == cudaSuccess) e = cudaMalloc(&sim->d_thr, n * 32 * sizeof(uint32_t));
        if (e == cudaSuccess) e = cudaMalloc(&sim->d_alw, n * sizeof(uint32_t));
        if (e != cudaSuccess) {
            if (sim->d_gen) cudaFree(sim->d_gen);
            if (sim->d_thr) cudaFree(sim->d_thr);
            sim->d_gen = nullptr; sim->d_thr = nullptr; sim->d_alw = nullptr; sim->general = false;
            return fail(SPIN_ERR_NOMEM, "spin_set_couplings: cudaMalloc (132 bytes of thresholds per site): %s", cudaGetErrorString(e));
        }
    }
    CUDA_TRY(cudaMemcpyAsync(sim->d_gen, Jh, n * sizeof(double), cudaMemcpyHostToDevice, sim->stream));
    CUDA_TRY(cudaMemcpyAsync(sim->d_gen + n, Jv, n * sizeof(double), cudaMemcpyHostToDevice, sim->stream));
    CUDA_TRY(cudaMemcpyAsync(sim->d_gen + 2 * n, Bf, n * sizeof(double), cudaMemcpyHostToDevice, sim->stream));
    CUDA_TRY(cudaStreamSynchronize(sim->stream));
    sim->general = true;
    return SPIN_OK;
}

int spin_energy_general(spin_sim* sim, double* E) {
    if (!sim || !E) return fail(SPIN_ERR_INVALID, "spin_energy_general: NULL argument");
    if (!sim->general) return fail(SPIN_ERR_INVALID, "spin_energy_general: the handle has no real couplings (spin_set_couplings)");
    CUDA_TRY(cudaSetDevice(sim->device));
    const size_t B = (size_t)sim->batch, n = B * sim->L * sim->L;
    double* d_E = (double*)sim->d_EM;                       // [2][B] int64 scratch, reused as B doubles
    CUDA_TRY(cudaMemsetAsync(d_E, 0, sizeof(double) * B, sim->stream));
    sim->launches += launch_ising_general_energy(sim->lattice, sim->d_gen, sim->d_gen + n, sim->d_gen + 2 * n, sim->batch, sim->L, d_E, sim->stream);
    CUDA_TRY(cudaGetLastError());
    CUDA_TRY(cudaMemcpyAsync(sim->h_EM, d_E, sizeof(double) * B, cudaMemcpyDeviceToHost, sim->stream));
    CUDA_TRY(cudaStreamSynchronize(sim->stream));
    std::memcpy(E, sim->h_EM, sizeof(double) * B);
    return SPIN_OK;
}

int spin_potts_label_sum(spin_sim* sim, int64_t* S) {
    if (!sim || !S) return fail(SPIN_ERR_INVALID, "spin_potts_label_sum: NULL argument");
    if (sim->model != SPIN_MODEL_POTTS) return fail(SPIN_ERR_INVALID, "spin_potts_label_sum: Potts handles only");
    CUDA_TRY(cudaSetDevice(sim->device));
    const size_t B = (size_t)sim->batch;
    CUDA_TRY(cudaMemsetAsync(sim->d_EM, 0, sizeof(long long) * B, sim->stream));
    sim->launches += launch_potts_general_observe(sim->lattice, nullptr, nullptr, sim->batch, sim->L, nullptr, sim->d_EM, sim->stream);
    CUDA_TRY(cudaGetLastError());
    CUDA_TRY(cudaMemcpyAsync(sim->h_EM, sim->d_EM, sizeof(long long) * B, cudaMemcpyDeviceToHost, sim->stream));
    CUDA_TRY(cudaStreamSynchronize(sim->stream));
    std::memcpy(S, sim->h_EM, sizeof(long long) * B);
    return SPIN_OK;
}

int spin_sweep_schedule(spin_sim* sim, const double* beta_steps, int64_t n_steps, double J, double h, int64_t sweeps_per_step,
                        int64_t sweep_offset) {
    if (!sim || !beta_steps) return fail(SPIN_ERR_INVALID, "spin_sweep_schedule: NULL argument");
    if (n_steps < 0 || sweeps_per_step < 0 || n_steps > (1ll << 24)) return fail(SPIN_ERR_INVALID, "spin_sweep_schedule: n_steps in 0..2^24 and sweeps_per_step >= 0 required");
    if (sweeps_per_step > 0 && n_steps > (1ll << 56) / sweeps_per_step) return fail(SPIN_ERR_INVALID, "spin_sweep_schedule: sweep range exceeds 2^56");
    const size_t B = (size_t)sim->batch;
    for (int64_t k = 0; k < n_steps; ++k) {
        const int rc = check_sweep_args(sim, beta_steps + (size_t)k * B, J, h, sweeps_per_step, sweep_offset + k * sweeps_per_step);
        if (rc != SPIN_OK) return rc;
    }
    if (n_steps == 0 || sweeps_per_step == 0) return SPIN_OK;
    if (sim->general || (sim->model == SPIN_MODEL_POTTS && (h != 0.0 || sim->d_bond_nat)))
        return fail(SPIN_ERR_UNSUPPORTED, "spin_sweep_schedule: class-table models only (uniform or +-J couplings, Potts without field); "
                    "call spin_sweep per step for real couplings");
    CUDA_TRY(cudaSetDevice(sim->device));
    // every step's records are built now and uploaded in ONE copy; the kernels of step k read their own slice, so the
    // whole schedule is enqueued without a host synchronisation between steps
    const size_t bytes = sizeof(uint32_t) * kTableStride * B * (size_t)n_steps;
    if (!sim->sched_ev) CUDA_TRY(cudaEventCreateWithFlags(&sim->sched_ev, cudaEventDisableTiming));
    if (sim->sched_bytes < bytes) {
        CUDA_TRY(cudaStreamSynchronize(sim->stream));
        if (sim->d_sched) cudaFree(sim->d_sched);
        if (sim->h_sched) cudaFreeHost(sim->h_sched);
        sim->d_sched = nullptr; sim->h_sched = nullptr; sim->sched_bytes = 0;
        cudaError_t e = cudaMalloc(&sim->d_sched, bytes);
        if (e == cudaSuccess) e = cudaMallocHost(&sim->h_sched, bytes);
        if (e != cudaSuccess) {
            if (sim->d_sched) cudaFree(sim->d_sched);
            sim->d_sched = nullptr; sim->h_sched = nullptr;
            return fail(SPIN_ERR_NOMEM, "spin_sweep_schedule: allocating %zu bytes of tables: %s", bytes, cudaGetErrorString(e));
        }
        sim->sched_bytes = bytes;
    }
    CUDA_TRY(cudaEventSynchronize(sim->sched_ev));          // the previous schedule's upload has left the pinned buffer
    for (int64_t k = 0; k < n_steps; ++k)
        for (size_t b = 0; b < B; ++b)
            build_record(sim, (int)b, beta_steps[(size_t)k * B + b], J, h, sim->h_sched + ((size_t)k * B + b) * kTableStride);
    // NOTE: earlier sweeps of this stream that still read d_sched (a previous schedule) are ordered before this copy
    CUDA_TRY(cudaMemcpyAsync(sim->d_sched, sim->h_sched, bytes, cudaMemcpyHostToDevice, sim->stream));
    CUDA_TRY(cudaEventRecord(sim->sched_ev, sim->stream));
    sim->potts_general = false;
    const bool resident = use_resident(sim, false);
    bool sched_never = false;
    for (size_t k = 0; k < (size_t)n_steps * B; ++k) sched_never = sched_never || sim->h_sched[k * kTableStride + kTabNever] != 0u;
    sim->any_never = sched_never;
    const bool tiled = !resident && use_tiled(sim);
    const bool persistent = !resident && !tiled && use_persistent(sim);
    const bool streams = !resident && !tiled && !persistent && !use_bits_resident(sim);
    const int G = streams ? streaming_begin(sim) : 1;
    for (int64_t k = 0; k < n_steps; ++k) {
        const uint32_t* tab = sim->d_sched + (size_t)k * B * kTableStride;
        const int64_t t0 = sweep_offset + k * sweeps_per_step;
        if (resident) {
            enqueue_resident(sim, t0, sweeps_per_step, false, nullptr, nullptr, nullptr, tab);
        } else if (use_bits_resident(sim) && enqueue_bits_resident(sim, t0, sweeps_per_step, tab)) {
        } else if (tiled && enqueue_tiled(sim, t0, sweeps_per_step, tab)) {
        } else if (persistent && enqueue_persistent(sim, t0, sweeps_per_step, tab)) {
        } else enqueue_streaming(sim, G, t0, sweeps_per_step, tab);
    }
    streaming_end(sim, G);
    CUDA_TRY(cudaGetLastError());
    return SPIN_OK;
}

int spin_set_policy(spin_sim* sim, int32_t policy) {
    if (!sim) return fail(SPIN_ERR_INVALID, "spin_set_policy: NULL handle");
    if (policy != SPIN_POLICY_AUTO && policy != SPIN_POLICY_STREAMING && policy != SPIN_POLICY_RESIDENT &&
        policy != SPIN_POLICY_PERSISTENT && policy != SPIN_POLICY_TILED && policy != SPIN_POLICY_GRAPH)
        return fail(SPIN_ERR_INVALID, "spin_set_policy: unknown policy %d", (int)policy);
    sim->policy = policy;
    return SPIN_OK;
}

int spin_sweep(spin_sim* sim, const double* beta, double J, double h, int64_t n_sweeps, int64_t sweep_offset) {
    const int rc = check_sweep_args(sim, beta, J, h, n_sweeps, sweep_offset);
    if (rc != SPIN_OK) return rc;
    if (n_sweeps == 0) return SPIN_OK;
    CUDA_TRY(cudaSetDevice(sim->device));
    const int rt = upload_tables(sim, beta, J, h);
    if (rt != SPIN_OK) return rt;
    if (use_resident(sim, false)) {
        enqueue_resident(sim, sweep_offset, n_sweeps, false, nullptr, nullptr, nullptr);
    } else if (use_bits_resident(sim) && enqueue_bits_resident(sim, sweep_offset, n_sweeps)) {
    } else if (use_tiled(sim) && enqueue_tiled(sim, sweep_offset, n_sweeps)) {
    } else if (!(use_persistent(sim) && enqueue_persistent(sim, sweep_offset, n_sweeps))) {
        const int rg = enqueue_graph_sweeps(sim, sweep_offset, n_sweeps);
        if (rg < 0) return fail(SPIN_ERR_CUDA, "spin_sweep: cudaGraphLaunch failed: %s", cudaGetErrorString(cudaGetLastError()));
        if (rg == 0) {
            const int G = streaming_begin(sim);
            enqueue_streaming(sim, G, sweep_offset, n_sweeps);
            streaming_end(sim, G);
        }
    }
    CUDA_TRY(cudaGetLastError());
    return SPIN_OK;
}

int spin_observables_dev(spin_sim* sim, int64_t* E_dev, int64_t* M_dev) {
    if (!sim) return fail(SPIN_ERR_INVALID, "spin_observables_dev: NULL handle");
    CUDA_TRY(cudaSetDevice(sim->device));
    return enqueue_observe(sim, (long long*)E_dev, (long long*)M_dev);
}

int spin_observables(spin_sim* sim, int64_t* E, int64_t* M) {
    if (!sim) return fail(SPIN_ERR_INVALID, "spin_observables: NULL handle");
    CUDA_TRY(cudaSetDevice(sim->device));
    const size_t B = (size_t)sim->batch;
    const int rc = enqueue_observe(sim, sim->d_EM, sim->d_EM + B);
    if (rc != SPIN_OK) return rc;
    CUDA_TRY(cudaMemcpyAsync(sim->h_EM, sim->d_EM, sizeof(long long) * 2 * B, cudaMemcpyDeviceToHost, sim->stream));
    CUDA_TRY(cudaStreamSynchronize(sim->stream));
    if (E) std::memcpy(E, sim->h_EM, sizeof(long long) * B);
    if (M) std::memcpy(M, sim->h_EM + B, sizeof(long long) * B);
    return SPIN_OK;
}

int spin_get_spins(spin_sim* sim, int8_t* out) {
    if (!sim || !out) return fail(SPIN_ERR_INVALID, "spin_get_spins: NULL argument");
    CUDA_TRY(cudaSetDevice(sim->device));
    const size_t n = (size_t)sim->batch * sim->L * sim->L;
    const int rs = ensure_stage(sim, n);
    if (rs != SPIN_OK) return rs;
    sim->launches += launch_to_natural(sim->lattice, sim->d_stage, sim->batch, sim->L, sim->layout, sim->stream);
    CUDA_TRY(cudaMemcpyAsync(out, sim->d_stage, n, cudaMemcpyDeviceToHost, sim->stream));
    CUDA_TRY(cudaStreamSynchronize(sim->stream));
    return SPIN_OK;
}

int spin_set_spins(spin_sim* sim, const int8_t* in) {
    if (!sim || !in) return fail(SPIN_ERR_INVALID, "spin_set_spins: NULL argument");
    CUDA_TRY(cudaSetDevice(sim->device));
    const size_t n = (size_t)sim->batch * sim->L * sim->L;
    const int rs = ensure_stage(sim, n);
    if (rs != SPIN_OK) return rs;
    unsigned int bad = 0;
    CUDA_TRY(cudaMemcpyAsync(sim->d_stage, in, n, cudaMemcpyHostToDevice, sim->stream));
    CUDA_TRY(cudaMemsetAsync(sim->d_bad, 0, sizeof(unsigned int), sim->stream));
    sim->launches += launch_validate_natural(sim->d_stage, sim->batch, sim->L, sim->model, sim->d_q, sim->d_bad, sim->stream);
    CUDA_TRY(cudaMemcpyAsync(&bad, sim->d_bad, sizeof bad, cudaMemcpyDeviceToHost, sim->stream));
    CUDA_TRY(cudaStreamSynchronize(sim->stream));
    if (bad) return fail(SPIN_ERR_INVALID, "spin_set_spins: %u values are not valid states", bad);
    sim->launches += launch_from_natural(sim->d_stage, sim->lattice, sim->batch, sim->L, sim->layout, sim->stream);
    CUDA_TRY(cudaGetLastError());
    CUDA_TRY(cudaStreamSynchronize(sim->stream));   // the caller may reuse `in`; the staging buffer may be reused
    return SPIN_OK;
}

int spin_sweep_measure(spin_sim* sim, const double* beta, double J, double h, int64_t n_sweeps, int64_t sweep_offset,
                       int64_t* E_trace, int64_t* M_trace, int64_t* moments) {
    const int rc = check_sweep_args(sim, beta, J, h, n_sweeps, sweep_offset);
    if (rc != SPIN_OK) return rc;
    if (n_sweeps == 0) return SPIN_OK;
    CUDA_TRY(cudaSetDevice(sim->device));
    const size_t B = (size_t)sim->batch;
    const bool want_trace = E_trace || M_trace;
    if (want_trace && n_sweeps > (int64_t)((size_t)1 << 40) / (int64_t)(B * 16))
        return fail(SPIN_ERR_INVALID, "spin_sweep_measure: n_sweeps * batch too large for one traced call; chunk it");
    if (moments) {
        // sum M^2 and sum E*M are plain int64: |M| <= N, |E_int| <= 2N, so n samples stay below 2^63 iff n * 2 N^2 < 2^63
        // (sum E^2 has two limbs).  Reject rather than wrap (documented in spin.h).
        const long double N = (long double)sim->L * (long double)sim->L;
        long double nmax = 0;
        for (size_t b = 0; b < B; ++b) {
            if (moments[8 * b] < 0) return fail(SPIN_ERR_INVALID, "spin_sweep_measure: moments[%zu][0] (sample count) is negative", b);
            if ((long double)moments[8 * b] > nmax) nmax = (long double)moments[8 * b];
        }
        if ((nmax + (long double)n_sweeps) * 2.0L * N * N >= 9223372036854775807.0L)
            return fail(SPIN_ERR_INVALID, "spin_sweep_measure: %lld more samples on L = %d could overflow the 64-bit "
                        "sums of M^2 and E*M (limit: samples * 2 L^4 < 2^63); accumulate in shorter runs",
                        (long long)n_sweeps, sim->L);
    }
    const bool resident = use_resident(sim, true);
    // traces wanted: device trace [2][n_sweeps][B].  Otherwise the streaming path reuses one [2][B] sample slot every
    // sweep, and the resident kernel keeps its sums in registers and takes null trace pointers.
    const size_t trace_elems = want_trace ? (size_t)n_sweeps * B : (resident ? 0 : B);
    if (trace_elems) {
        const int rs = ensure_trace(sim, sizeof(long long) * 2 * trace_elems);
        if (rs != SPIN_OK) return rs;
    }
    long long* d_trace = trace_elems ? sim->d_trace : nullptr;
    long long* d_mom = moments ? sim->d_mom : nullptr;
    const int rt = upload_tables(sim, beta, J, h);
    if (rt != SPIN_OK) return rt;
    if (moments) CUDA_TRY(cudaMemcpyAsync(d_mom, moments, sizeof(long long) * 8 * B, cudaMemcpyHostToDevice, sim->stream));
    if (resident) {
        enqueue_resident(sim, sweep_offset, n_sweeps, true, want_trace ? d_trace : nullptr,
                         want_trace ? d_trace + trace_elems : nullptr, d_mom);
    } else if (fused_measure_eligible(sim)) {
        const int rf = enqueue_streaming_measure(sim, sweep_offset, n_sweeps, want_trace ? d_trace : nullptr,
                                                 want_trace ? d_trace + trace_elems : nullptr, d_mom);
        if (rf != SPIN_OK) { cudaStreamSynchronize(sim->stream); return rf; }
    } else {
        for (int64_t local = 0; local < n_sweeps; ++local) {
            const int64_t t = sweep_offset + local;
            enqueue_half_sweep(sim, t, 0);
            enqueue_half_sweep(sim, t, 1);
            long long* Et = d_trace + (want_trace ? (size_t)local * B : 0);
            long long* Mt = d_trace + trace_elems + (want_trace ? (size_t)local * B : 0);
            const int ro = enqueue_observe(sim, Et, Mt);
            if (ro != SPIN_OK) { cudaStreamSynchronize(sim->stream); return ro; }
            if (moments) sim->launches += launch_accumulate_moments(d_mom, Et, Mt, sim->batch, sim->stream);
        }
    }
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess && E_trace) e = cudaMemcpyAsync(E_trace, d_trace, sizeof(long long) * trace_elems, cudaMemcpyDeviceToHost, sim->stream);
    if (e == cudaSuccess && M_trace) e = cudaMemcpyAsync(M_trace, d_trace + trace_elems, sizeof(long long) * trace_elems, cudaMemcpyDeviceToHost, sim->stream);
    if (e == cudaSuccess && moments) e = cudaMemcpyAsync(moments, d_mom, sizeof(long long) * 8 * B, cudaMemcpyDeviceToHost, sim->stream);
    const cudaError_t es = cudaStreamSynchronize(sim->stream);
    if (e == cudaSuccess) e = es;
    if (e != cudaSuccess) return cuda_fail(e, "spin_sweep_measure");
    return SPIN_OK;
}

}  // extern "C"
