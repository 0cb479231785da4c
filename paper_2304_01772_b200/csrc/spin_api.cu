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
    uint8_t* d_aux = nullptr;        // bit-packed kernel's constant 2 KiB lookup table, on this handle's device
    int8_t* d_stage = nullptr;       // natural-layout staging for spin_get_spins / spin_set_spins / spin_set_bonds (grow-only)
    size_t stage_bytes = 0;
    long long* d_mom = nullptr;      // [B][8] moments of spin_sweep_measure
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
    if (sim->model == SPIN_MODEL_POTTS && h != 0.0)
        return fail(SPIN_ERR_UNSUPPORTED, "spin_sweep: a field term is not supported for the Potts model (h must be 0)");
    return SPIN_OK;
}

// Build the per-replica records on the host and enqueue their copy.
int upload_tables(spin_sim* sim, const double* beta, double J, double h) {
    // the upload issued two calls ago may still be reading this pinned buffer; nothing else is waited for
    const int slot = sim->table_slot;
    sim->table_slot ^= 1;
    uint32_t* h_tab = sim->h_tables[slot];
    CUDA_TRY(cudaEventSynchronize(sim->table_ev[slot]));
    std::memset(h_tab, 0, sizeof(uint32_t) * kTableStride * (size_t)sim->batch);
    for (int b = 0; b < sim->batch; ++b) {
        uint32_t* rec = h_tab + (size_t)b * kTableStride;
        if (sim->model == SPIN_MODEL_ISING) {
            for (int d = 0; d < 2; ++d)
                for (int nd = 0; nd <= 4; ++nd) {
                    const int s = d ? -1 : 1, nn = 4 - 2 * nd;
                    encode(ising_class(beta[b], J, h, s, nn), d * 8 + nd, rec);
                }
        } else {
            for (int dn = -4; dn <= 4; ++dn) encode(potts_class(beta[b], J, dn), dn + 4, rec);
        }
        rec[kTabQ] = (uint32_t)sim->q[b];
    }
    CUDA_TRY(cudaMemcpyAsync(sim->d_tables, h_tab, sizeof(uint32_t) * kTableStride * (size_t)sim->batch,
                             cudaMemcpyHostToDevice, sim->stream));
    CUDA_TRY(cudaEventRecord(sim->table_ev[slot], sim->stream));
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
    return a;
}

// Shared-memory-resident path (ising_int8.cu): Ising, int8 layout, replica fits one CTA.  AUTO uses it when the
// batch gives every SM work (or when the lattice is so small that the streaming kernels are launch-bound anyway).
bool use_resident(const spin_sim* sim, bool measure) {
    if (sim->model != SPIN_MODEL_ISING || sim->layout != SPIN_LAYOUT_INT8 || !ising_int8_resident_fits(sim->L)) return false;
    if (sim->policy == SPIN_POLICY_STREAMING) return false;
    if (sim->policy == SPIN_POLICY_RESIDENT) return true;
    const long long sites = (long long)sim->batch * sim->L * sim->L;
    if (sites <= (1ll << 20)) return true;                         // launch-latency-bound shapes
    // the streaming kernel's blocks cover (L/8) x (L/32) thread strips of ONE replica: below 64 of them (L = 64, 96,
    // 160, ...) its blocks are a fraction of a warp and the resident kernel is faster (L = 64: 922 vs 576 flips/ns)
    int tpb = 128;
    const int perReplica = (sim->L / 8) * (sim->L / 32);
    while (perReplica % tpb) tpb >>= 1;
    if (tpb < 64 && sim->batch >= 148) return true;
    return measure && sim->batch >= 296;                           // fused per-sweep reductions, >= 2 CTAs per SM
}

void enqueue_resident(spin_sim* sim, int64_t t0, int64_t n_sweeps, bool measure, long long* E_trace, long long* M_trace,
                      long long* moments) {
    ResidentArgs a;
    a.lattice = sim->lattice;
    a.tables = sim->d_tables;
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

void enqueue_half_sweep(spin_sim* sim, int64_t t, int colour) {
    const SweepArgs a = sweep_args(sim, t, colour);
    if (sim->model == SPIN_MODEL_POTTS) sim->launches += launch_potts_int8_half_sweep(a, sim->stream);
    else if (sim->layout == SPIN_LAYOUT_BITPACKED) sim->launches += launch_ising_bits_half_sweep(a, sim->stream);
    else sim->launches += launch_ising_int8_half_sweep(a, sim->stream);
}

// Enqueue the reductions of the current lattice into E_out[b], M_out[b] (device int64, either may be NULL).
// The targets are zeroed first (the kernels accumulate).
int enqueue_observe(spin_sim* sim, long long* E_out, long long* M_out) {
    const size_t nb = sizeof(long long) * (size_t)sim->batch;
    if (E_out) CUDA_TRY(cudaMemsetAsync(E_out, 0, nb, sim->stream));
    if (sim->model == SPIN_MODEL_POTTS) {
        sim->launches += launch_potts_int8_observe(sim->lattice, sim->batch, sim->L, sim->d_q, E_out, M_out ? sim->d_hist : nullptr, sim->stream);
        if (M_out) sim->launches += launch_potts_finalize(sim->d_hist, sim->d_q, sim->batch, M_out, sim->stream);
    } else {
        if (M_out) CUDA_TRY(cudaMemsetAsync(M_out, 0, nb, sim->stream));
        if (sim->layout == SPIN_LAYOUT_BITPACKED)
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
    if (sim->owns_lattice && sim->lattice) cudaFree(sim->lattice);
    if (sim->d_tables) cudaFree(sim->d_tables);
    if (sim->d_bonds) cudaFree(sim->d_bonds);
    if (sim->d_q) cudaFree(sim->d_q);
    if (sim->d_EM) cudaFree(sim->d_EM);
    if (sim->d_hist) cudaFree(sim->d_hist);
    if (sim->d_bad) cudaFree(sim->d_bad);
    if (sim->d_aux) cudaFree(sim->d_aux);
    if (sim->d_stage) cudaFree(sim->d_stage);
    if (sim->d_mom) cudaFree(sim->d_mom);
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
    if (sim->layout == SPIN_LAYOUT_BITPACKED) return "ising_bits_rows32";
    if (use_resident(sim, false)) return "ising_int8_resident";
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
        return SPIN_OK;
    }
    if (sim->model != SPIN_MODEL_ISING || sim->layout != SPIN_LAYOUT_BITPACKED)
        return fail(SPIN_ERR_UNSUPPORTED, "spin_set_bonds: +-J couplings are implemented for the bit-packed Ising layout only");
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

int spin_set_policy(spin_sim* sim, int32_t policy) {
    if (!sim) return fail(SPIN_ERR_INVALID, "spin_set_policy: NULL handle");
    if (policy != SPIN_POLICY_AUTO && policy != SPIN_POLICY_STREAMING && policy != SPIN_POLICY_RESIDENT)
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
    } else {
        for (int64_t t = sweep_offset; t < sweep_offset + n_sweeps; ++t) {
            enqueue_half_sweep(sim, t, 0);
            enqueue_half_sweep(sim, t, 1);
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
