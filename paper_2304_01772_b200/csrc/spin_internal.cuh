// spin_internal.cuh — declarations shared by the translation units of libspin.so (CUDA side only).
// Nothing here is shared with oracle/: the oracle has its own generator, tables and loops.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

namespace spin {

// ---- Philox-4x32-10 (O2).  Round keys are precomputed on the host. -------------
constexpr uint32_t kPhiloxM0 = 0xD2511F53u;
constexpr uint32_t kPhiloxM1 = 0xCD9E8D57u;
constexpr uint32_t kPhiloxW0 = 0x9E3779B9u;
constexpr uint32_t kPhiloxW1 = 0xBB67AE85u;

enum : uint32_t { kDomainInit = 0, kDomainIsing = 1, kDomainPotts = 2 };

struct RoundKeys {
    uint32_t k0[10];
    uint32_t k1[10];
};

// One Philox call.  c1..c3 are uniform over a launch in every kernel of this library, so the compiler
// keeps them (and the round keys, which come from the constant bank) in uniform registers.
__device__ __forceinline__ void philox4x32_10(const RoundKeys& rk, uint32_t c0, uint32_t c1, uint32_t c2,
                                              uint32_t c3, uint32_t out[4]) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)kPhiloxM0 * c0;
        const uint64_t p1 = (uint64_t)kPhiloxM1 * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ rk.k0[r];
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ rk.k1[r];
        c1 = (uint32_t)p1;
        c3 = (uint32_t)p0;
        c0 = n0;
        c2 = n2;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// ---- device-side acceptance tables -------------------------------------------------------------------
// One record of kTableStride uint32 per replica.
//   Ising: U[d*8 + nd] at [0..15], d = 1 iff the site's spin is -1, nd = number of -1 neighbours (0..4);
//          a flip of that class is accepted iff r <= U (U = T-1, or 0xFFFFFFFF for "always").
//   Potts: U[dn + 4] at [0..8].
//   [16] = bit mask of classes that can never be accepted (T == 0: r <= U cannot express it);
//   [17] = q of the replica (Potts).
constexpr int kTableStride = 32;
constexpr int kTabNever = 16;
constexpr int kTabQ = 17;

struct SweepArgs {
    void* lattice;            // int8: [B][2][L][L/2] bytes; bit-packed: [B][2][L][L/64] uint32
    const uint32_t* tables;   // [B][kTableStride]
    int32_t batch;
    int32_t L;
    uint32_t replica_offset;
    uint32_t c2;              // low 32 bits of the sweep index t
    uint32_t c3;              // (t >> 32) & 0xFFFFFF | colour << 24 | domain << 28
    int32_t colour;
    const uint8_t* aux;       // bit-packed kernel: nibble-pair -> 4 * class byte table (spin_sim::d_aux), else nullptr
    const uint32_t* bonds;    // bit-packed +-J couplings: [B][2][4][L][L/64] words (bit = bond is -1; planes up, down,
                              // centre, side of the colour's sites), or nullptr for uniform couplings
    RoundKeys rk;
    int32_t pdl_trigger;      // PdlTrigger: where the row-marching kernels release the next launch (set by the launchers)
    long long* measure_acc;   // non-NULL (int8 Ising rows kernel, colour 1): [batch][3] sums the launch adds into for the fused
                              // E / M reduction (ising_int8.cu, kMeasure); indexed by the launch's own replica index
    // colour-0 launches of a measured run (fin_pending != 0): before its own work, one thread per replica turns the sums the
    // previous sweep's colour-1 launch left in measure_acc into E / M (fin_E / fin_M: that sweep's trace sample, device
    // [batch] or NULL; fin_mom: device [batch][8] or NULL) and clears them - no separate launch in the chain
    long long* fin_E;
    long long* fin_M;
    long long* fin_mom;
    int32_t fin_pending;
    const unsigned long long* potts_tab2;   // non-NULL (Potts rows kernel): field on the state label - entries
                                            // (always << 32) | T indexed [replica][dn + 4][new - old + 127] (spin_api.cu)
    const unsigned long long* t_dev;   // non-NULL: the launch is a node of a CUDA graph (spin_api.cu, sweep_graph) and its sweep
    uint32_t t_rel;                    // index is *t_dev + t_rel, read after pdl_wait(); c2 / c3 then hold colour and domain only
    int32_t plan_scale;       // the launch is one of plan_scale concurrent ones (replica groups on their own streams,
                              // spin_api.cu): the launch plan is made for the whole batch
};

// Shared-memory-resident multi-sweep kernel (small lattices: one CTA holds a whole replica and runs all sweeps of a
// call in one launch, with the per-sweep E / M reductions and the moment accumulation fused in).
struct ResidentArgs {
    void* lattice;            // int8: [B][2][L][L/2]
    const uint32_t* tables;   // [B][kTableStride]
    int32_t batch;
    int32_t L;
    uint32_t replica_offset;
    uint32_t measure;         // 1: reduce E, M after every sweep
    unsigned long long t0;    // first sweep index
    long long n_sweeps;
    long long* E_trace;       // device [n_sweeps][B] or nullptr
    long long* M_trace;       // device [n_sweeps][B] or nullptr
    long long* moments;       // device [B][8] in/out or nullptr
    RoundKeys rk;
};

// Temporally blocked tile kernel (launch-bound shapes): a CTA owns TR rows x TK same-colour columns of one replica plus a
// halo of HR rows / HK columns on every side and advances `sweeps` full sweeps per launch in shared memory.
struct TiledArgs {
    const void* src;          // int8: [B][2][L][L/2], read by every tile (interior + halo)
    void* dst;                // same shape, a DIFFERENT buffer: tiles of one launch read each other's interiors as halos,
                              // so the advanced interiors go to a second lattice and the two swap roles per launch
    const uint32_t* tables;   // [B][kTableStride]
    int32_t batch, L;
    uint32_t replica_offset;
    unsigned long long t0;    // first sweep index of this launch
    int32_t sweeps;           // sweeps in this launch (2 * sweeps <= HR rows, sweeps <= HK same-colour columns)
    int32_t TR, TK, HR, HK;   // TK, HK multiples of 4 (k = same-colour column index)
    int32_t tilesR, tilesK;
    RoundKeys rk;
};

struct InitArgs {
    void* lattice;
    const int32_t* q;         // [B] (Potts) or nullptr
    int32_t batch;
    int32_t L;
    uint32_t replica_offset;
    RoundKeys rk;
};

// ---- programmatic dependent launch -------------------------------------------------------------------
// The sweep is a chain of short dependent kernels (two per sweep).  Launching them with the programmatic
// stream-serialisation attribute lets launch n+1 be staged while launch n runs; pdl_wait() then blocks until launch n
// has completed and its writes are visible, and comes before the first access to the lattice.
// WHERE launch n releases launch n+1 decides where the blocks of n+1 are placed (measured, profiles/r2_pdl_placement.md):
// released at the start of n, the blocks of n+1 (and n+2, ..) become resident beside those of n, on whatever SMs have
// room, and when a grid is around one wave or less that placement is lopsided for the whole launch (16 x 1024^2
// bit-packed: 297 flips/ns, against 930-1030 with the same kernel released later).  Released when the blocks of n exit
// (no explicit trigger), n+1 is placed on an empty GPU and is balanced.  With several waves the early release wins a
// few percent (the next launch's blocks take the slots the last wave frees).  plan_rows() below picks the release
// point together with the rows per thread.
enum PdlTrigger : int32_t {
    kPdlAtExit = 0,      // no explicit trigger: the dependent launch is released as this launch's blocks exit
    kPdlAtStart = 1,     // first instruction of every block
    kPdlLastRows = 2,    // when a thread starts its last two rows
};
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// What the inner update functions need for a Philox call besides the group and the replica.
struct PhiloxCtx {
    const RoundKeys& rk;
    uint32_t c2, c3;
};

// Counter words 2 and 3 of a launch: from the arguments, or (kDevT, graph nodes) from the sweep index in device memory.
template <bool kDevT>
__device__ __forceinline__ void sweep_counter_words(const SweepArgs& a, uint32_t& c2, uint32_t& c3) {
    c2 = a.c2;
    c3 = a.c3;
    if (kDevT) {
        const unsigned long long t = *(const volatile unsigned long long*)a.t_dev + a.t_rel;
        c2 = (uint32_t)(t & 0xFFFFFFFFull);
        c3 = (a.c3 & 0xFF000000u) | (uint32_t)((t >> 32) & 0xFFFFFFull);
    }
}

template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kernel)(KArgs...), unsigned grid, unsigned block, cudaStream_t s, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid, 1, 1);
    cfg.blockDim = dim3(block, 1, 1);
    cfg.dynamicSmemBytes = 0;
    cfg.stream = s;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

// Threads per block for `units` thread-units of one replica: the multiple of 32 (at most 128) that wastes the fewest
// lanes in the ragged last block; ties go to the larger block.
inline int pick_block(int units) {
    int best = 128;
    long long bestPad = -1;
    for (int t = 128; t >= 32; t -= 32) {
        const long long pad = (long long)((units + t - 1) / t) * t;
        if (bestPad < 0 || pad < bestPad) { best = t; bestPad = pad; }
    }
    return best;
}

// Rows per thread (2, 4 or 8) and release point of a row-marching half-sweep launch.  w8 = waves the 8-row grid would
// make (threads of 8 rows / (slots x 128), slots = 148 x resident blocks per SM of that kernel).  Long threads amortise
// the per-thread set-up and the two halo rows; short threads fill the GPU when the launch is small.  The thresholds are
// the crossovers of a measured (batch, L) grid per kernel (profiles/r2_pdl_placement.md); min8 = fewest 8-row threads
// per replica for which 8 or 4 rows keep a block reasonably full.
// Resident blocks per SM of the three row-marching kernels (their __launch_bounds__), i.e. 148 x this = block slots.
constexpr int kIsingInt8BlocksPerSm = 5;   // 96 registers
constexpr int kIsingBitsBlocksPerSm = 8;   // 64 registers
constexpr int kPottsBlocksPerSm = 4;

struct RowsPlan {
    int rows;
    int32_t trigger;
};
inline RowsPlan plan_rows(long long threads8, int perReplica8, int slots, double w_r2, double w_r8, bool early_r8) {
    const double w8 = (double)threads8 / (128.0 * slots);
    RowsPlan p;
    if (perReplica8 < 64 || w8 < w_r2) p.rows = 2;
    else if (w8 < w_r8) p.rows = 4;
    else p.rows = 8;
    p.trigger = (p.rows == 8 && early_r8) ? kPdlAtStart : kPdlAtExit;
    return p;
}

// Records the thread-local spin_last_error() text and returns `code` (spin_api.cu).
int set_error(int code, const char* msg);

// ---- launchers (each returns the number of kernels it launched; errors via cudaGetLastError) --------
int launch_init(const InitArgs& a, int model, int layout, cudaStream_t s);

int launch_ising_int8_half_sweep(const SweepArgs& a, cudaStream_t s);      // picks generic / vectorised
int launch_potts_int8_half_sweep(const SweepArgs& a, cudaStream_t s);
int launch_ising_bits_half_sweep(const SweepArgs& a, cudaStream_t s);
bool ising_bits_resident_fits(int L);                                       // bit-packed replica fits one CTA's shared memory
int launch_ising_bits_resident(const ResidentArgs& a, const uint8_t* aux, cudaStream_t s);   // 0: not launched
uint8_t* ising_bits_make_aux_table();      // allocates + fills the constant 2 KiB lookup table on the current device (owned by the caller)
const char* ising_int8_variant(int L);
bool ising_int8_resident_fits(int L);                                       // a replica fits one CTA's shared memory
int launch_ising_int8_persistent(const SweepArgs& a, unsigned long long t0, long long n_sweeps, unsigned int* counter,
                                 cudaStream_t s);                           // 0: not launched, use the streaming path
// Enqueues n_sweeps sweeps from t0 with the tiled kernel (ceil(n_sweeps / sweeps-per-launch) launches); returns the
// number of kernels launched, 0 if the shape does not qualify.
int launch_ising_int8_tiled(const SweepArgs& a, void* shadow, unsigned long long t0, long long n_sweeps, cudaStream_t s);
bool ising_int8_tiled_fits(int batch, int L);
cudaError_t ising_int8_resident_configure();                                // per device: allow > 48 KiB dynamic shared memory
int launch_ising_int8_resident(const ResidentArgs& a, cudaStream_t s);      // all n_sweeps in one launch
const char* potts_int8_variant(int L);

// General couplings (general.cu): natural-layout device arrays.
int launch_ising_int8_bonds_half_sweep(const SweepArgs& a, const int8_t* Jh, const int8_t* Jv, cudaStream_t s);
int launch_ising_int8_general_half_sweep(const SweepArgs& a, const uint32_t* thr, const uint32_t* alw, cudaStream_t s);
int launch_potts_int8_general_half_sweep(const SweepArgs& a, const unsigned long long* tab2, const int8_t* Jh, const int8_t* Jv,
                                         cudaStream_t s);
int launch_ising_general_energy(const void* lattice, const double* Jh, const double* Jv, const double* B, int batch, int L,
                                double* E, cudaStream_t s);                  // E[b] += ..., zero on entry
int launch_potts_general_observe(const void* lattice, const int8_t* Jh, const int8_t* Jv, int batch, int L, long long* E_acc,
                                 long long* S_acc, cudaStream_t s);
int launch_ising_int8_bonds_observe(const void* lattice, const int8_t* Jh, const int8_t* Jv, int batch, int L, long long* E_acc,
                                    long long* M_acc, cudaStream_t s);

// Observables: accumulate into E_acc[b], M_acc[b] (int64, must be zero on entry; Potts uses hist).
int launch_ising_int8_observe(const void* lattice, int batch, int L, long long* E_acc, long long* M_acc, cudaStream_t s);
int launch_ising_bits_observe(const void* lattice, const uint32_t* bonds, int batch, int L, long long* E_acc, long long* M_acc, cudaStream_t s);
// Potts: E_acc as above; hist: [B][128] uint32, zero on entry; M is produced by launch_potts_finalize.
int launch_potts_int8_observe(const void* lattice, int batch, int L, const int32_t* q, long long* E_acc, unsigned int* hist, cudaStream_t s);
// M_out[b] = max_k hist[b][k], then hist is cleared for the next use.
int launch_potts_finalize(unsigned int* hist, const int32_t* q, int batch, long long* M_out, cudaStream_t s);
// moments[b][8] += sample (E[b], M[b])
// Fused E / M of the int8 Ising streaming path: turns the sums the colour-1 launch left in acc[batch][3] into E, M (written
// to E_out / M_out if non-NULL), accumulates the moments (if non-NULL) and clears acc.  sites = L * L.
int launch_ising_measure_finalize(long long* acc, int batch, long long sites, long long* E_out, long long* M_out,
                                  long long* moments, cudaStream_t s);
int launch_accumulate_moments(long long* moments, const long long* E, const long long* M, int batch, cudaStream_t s);

// Natural <-> internal layout.  natural: [B][L][L] int8 on the device.
int launch_from_natural(const int8_t* natural, void* lattice, int batch, int L, int layout, cudaStream_t s);
int launch_to_natural(const void* lattice, int8_t* natural, int batch, int L, int layout, cudaStream_t s);
// bad[0] = number of invalid values (Ising: not +-1; Potts: outside 0..q[b]-1).  bad must be zero on entry.
// +-J bond signs, natural [B][L][L] int8 on the device -> sign planes [B][2][4][L][L/64]; bad[0] (zero on entry) gets the
// number of reads that were not +-1.
int launch_bonds_from_natural(const int8_t* Jh, const int8_t* Jv, uint32_t* planes, int batch, int L, unsigned int* bad,
                              cudaStream_t s);
int launch_validate_natural(const int8_t* natural, int batch, int L, int model, const int32_t* q, unsigned int* bad, cudaStream_t s);

}  // namespace spin
