/* spin.h — C ABI of libspin.so: batched checkerboard Metropolis sweeps for the 2D Ising and q-state
 * Potts models on one NVIDIA B200 (sm_100a).
 *
 * What the library computes is the hot path of arXiv 2304.01772, "A differentiable programming
 * framework for spin models" (citations are line numbers of /root/reference/PAPER.md):
 *   - Algorithm 1, "Standard Metropolis-Hastings algorithm with parallelization":
 *     propose a new state per site, evaluate the local energy change dE from the 4 nearest
 *     neighbours, accept if dE <= 0, else with probability exp(-beta dH);
 *   - the checkerboard method (Fig. 1): all sites of one colour are updated in
 *     parallel, black squares first, then white squares;
 *   - the Ising Hamiltonian Eq. 1 with the 4-neighbour stencil Eq. 2 and the
 *     Potts Hamiltonian Eq. 5 with the four one-neighbour stencils Eq. 6 and the "one of the other
 *     q-1 states" proposal;
 *   - the batch dimension = independent lattices, each with its own temperature;
 *   - energy / magnetisation bookkeeping.
 * The readings taken where the paper is silent (sign of J, colour order, RNG, dE == 0, ...) are
 * listed in DESIGN.md section 3.  Library sign convention: H = -J sum_<ij> s_i s_j - h sum_i s_i
 * (Ising, s = +-1) and H = -J sum_<ij> delta(s_i, s_j) (Potts, s in 0..q-1); J > 0 is the
 * ferromagnet (the paper's J = -1).  k_B = 1, beta = 1/T.
 *
 * Random numbers: Philox-4x32-10 keyed by (seed; group, replica, sweep t, colour, domain); see
 * DESIGN.md section 3 (O2).  Results are a pure function of (seed, replica index, t): running
 * n sweeps from offset 0 equals running them in chunks, and replica b of a batch equals replica 0
 * of a handle created with replica_offset = b.
 *
 * General conventions
 *   - Every function is extern "C"; no exception crosses the boundary; no global state other than a
 *     thread-local last-error string.
 *   - "host" pointers are ordinary CPU memory (pinned or pageable); "device" pointers are CUDA device
 *     memory on the handle's device.  Unless stated otherwise pointers are host pointers.
 *   - The caller owns every array it passes; the library keeps no caller pointer after a call returns,
 *     except device_buffer of spin_create_ex (owned by the caller, must outlive the handle).
 *   - int functions return SPIN_OK or a negative code; on SPIN_ERR_INVALID / SPIN_ERR_UNSUPPORTED no
 *     caller array and no lattice has been modified.  spin_create* return NULL on failure.  The reason
 *     is available from spin_last_error().
 *   - One handle is used from one host thread at a time.  All work of a handle is enqueued on the
 *     handle's CUDA stream; calls that return results in host memory synchronise that stream.
 *   - There is no CPU fallback: without a CUDA device spin_create* fail with SPIN_ERR_CUDA text.
 */
#ifndef SPIN_H_
#define SPIN_H_

#include <stddef.h>
#include <stdint.h>

#if defined(__GNUC__)
#define SPIN_API __attribute__((visibility("default")))
#else
#define SPIN_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

typedef struct spin_sim spin_sim; /* opaque handle, owned by the library */

enum { SPIN_OK = 0, SPIN_ERR_INVALID = -1, SPIN_ERR_NOMEM = -2, SPIN_ERR_CUDA = -3, SPIN_ERR_UNSUPPORTED = -4 };
enum { SPIN_MODEL_ISING = 0, SPIN_MODEL_POTTS = 1 };
enum { SPIN_LAYOUT_INT8 = 0, SPIN_LAYOUT_BITPACKED = 1 }; /* bit-packed: Ising only, L % 64 == 0 */

/* ---------------------------------------------------------------------------------------------
 * Core calls (BASELINE.json north star; problem statement PAPER.md:93-95, 127-138)
 * ------------------------------------------------------------------------------------------- */

/* Create `batch` periodic L x L lattices on the current CUDA device and initialise them uniformly at
 * random from Philox(seed) ("a random initial state"; O3).
 * q == 2: Ising, int8 spins -1/+1.  q >= 3: Potts, uint8 states 0..q-1, the same q in every replica.
 * Layout int8, replica_offset 0, library-owned memory, the default (NULL) stream.
 * Invalid: batch < 1, L < 2 or odd, q < 2 or q > 127.  Returns NULL on failure. */
SPIN_API spin_sim* spin_create(int32_t batch, int32_t L, int32_t q, uint64_t seed);

/* Run Metropolis sweeps t = sweep_offset .. sweep_offset + n_sweeps - 1; each sweep updates colour 0
 * ((i+j) even) and then colour 1 (Alg. 1 + checkerboard).
 * beta: host, [batch], inverse temperature of each replica (finite, >= 0); copied before return.
 * J, h: coupling and field (finite).  Potts: the field acts on the state label, H = -J sum delta - h sum_i s_i (Eq. 5,
 * PAPER.md:166; reading P7); h != 0 (or bond signs) selects the general Potts kernel.
 * n_sweeps >= 0, sweep_offset >= 0, sweep_offset + n_sweeps <= 2^56.
 * Asynchronous on the handle's stream: the call builds the acceptance tables (O(batch) host work), enqueues their
 * upload and the sweep kernels, and returns without waiting for earlier work of the stream (the two pinned table
 * buffers alternate; only the upload issued two calls earlier is waited for). */
SPIN_API int spin_sweep(spin_sim* sim, const double* beta, double J, double h, int64_t n_sweeps, int64_t sweep_offset);

/* Exact integer observables of the current lattices (O8).
 * E: host, [batch]: E_int = -(sum over bonds of s_i s_j) (Ising) or -(number of equal bonds) (Potts),
 *    every bond once, double bonds of L == 2 counted twice.  Energy = J E_int - h M (Ising), J E_int (Potts).
 * M: host, [batch]: sum of spins (Ising) or the population of the most common state (Potts).
 * Either pointer may be NULL.  Synchronises the stream. */
SPIN_API int spin_observables(spin_sim* sim, int64_t* E, int64_t* M);

/* Destroy a handle (frees library-owned device memory).  NULL is a no-op. */
SPIN_API void spin_destroy(spin_sim* sim);

/* Thread-local description of the last failure in this thread; valid until the next failing call. */
SPIN_API const char* spin_last_error(void);

/* ---------------------------------------------------------------------------------------------
 * Calls needed by the five BASELINE.json configurations and the parity tests
 * ------------------------------------------------------------------------------------------- */

/* Bytes of device memory a lattice buffer of this shape needs (0 if the shape is invalid).
 * int8 layout: batch * L * L bytes, stored [batch][colour][L][L/2] (colour = (i+j)&1, column index
 * k = j >> 1), Ising bytes are -1/+1, Potts bytes 0..q-1.
 * bit-packed layout: batch * L * L / 8 bytes, stored [batch][colour][L][L/64] uint32 words, bit b of
 * word w = site k = 32 w + b, bit set = spin -1. */
SPIN_API size_t spin_buffer_bytes(int32_t batch, int32_t L, int32_t model, int32_t layout);

/* Full constructor.
 * model: SPIN_MODEL_*.  q_per_replica: host, [batch], or NULL to use q_uniform for every replica
 * (Ising: q is ignored and taken as 2).  layout: SPIN_LAYOUT_*.  replica_offset >= 0: replica b is
 * keyed in the generator as b + replica_offset (must stay below 2^32).
 * device_buffer: NULL (library allocates and owns spin_buffer_bytes(...) bytes) or a 16-byte-aligned
 * device pointer to at least that many bytes, owned by the caller, which must outlive the handle;
 * buffer_bytes is its size (ignored when NULL).  cuda_stream: a cudaStream_t, NULL = default stream.
 * The lattice is initialised from Philox(seed) as in spin_create.
 * SPIN_ERR_UNSUPPORTED (NULL return): bit-packed with Potts or with L % 64 != 0. */
SPIN_API spin_sim* spin_create_ex(int32_t batch, int32_t L, int32_t model, const int32_t* q_per_replica, int32_t q_uniform,
                         uint64_t seed, int32_t layout, int64_t replica_offset, void* device_buffer,
                         size_t buffer_bytes, void* cuda_stream);

/* Use another CUDA stream for subsequent work (the previous stream is synchronised first). */
SPIN_API int spin_set_stream(spin_sim* sim, void* cuda_stream);

/* Copy the lattices out / in, in the natural layout [batch][L][L] int8 (Ising -1/+1, Potts 0..q-1).
 * Host pointers; both synchronise the stream.  spin_set_spins validates every value
 * (SPIN_ERR_INVALID, lattice unchanged). */
SPIN_API int spin_get_spins(spin_sim* sim, int8_t* out);
SPIN_API int spin_set_spins(spin_sim* sim, const int8_t* in);

/* spin_sweep with measurements after every full sweep (rows a5-a7 of DESIGN.md section 1).
 * E_trace, M_trace: host, [n_sweeps][batch] or NULL: (E_int, M) after each sweep.
 * moments: host, [batch][8], in/out, or NULL: every sweep adds one sample to
 *   {n, sum E, sum E^2 (low 64 bits), sum E^2 (high 64 bits), sum M, sum |M|, sum M^2, sum E*M}
 *   with E = E_int; all int64, sum E^2 is one 128-bit integer in two limbs.  sum M^2 and sum E*M are plain int64
 *   (|M| <= L^2, |E_int| <= 2 L^2): a call is rejected with SPIN_ERR_INVALID, nothing run, when
 *   (max_b moments[b][0] + n_sweeps) * 2 L^4 >= 2^63, i.e. when they could wrap (L = 8192: 1024 samples; L <= 1024:
 *   more than 4e6 samples); accumulate longer runs in several moment arrays.
 * With both traces NULL no per-sweep trace is stored (a moments-only run of any length needs O(batch) memory).
 * Synchronises the stream. */
SPIN_API int spin_sweep_measure(spin_sim* sim, const double* beta, double J, double h, int64_t n_sweeps, int64_t sweep_offset,
                       int64_t* E_trace, int64_t* M_trace, int64_t* moments);

/* spin_observables into device memory (E_dev, M_dev: device, [batch], either may be NULL); enqueued on
 * the stream, no synchronisation. */
SPIN_API int spin_observables_dev(spin_sim* sim, int64_t* E_dev, int64_t* M_dev);

/* Wait for all work enqueued on the handle's stream. */
SPIN_API int spin_synchronize(spin_sim* sim);

/* The acceptance table of one replica, computed on the host in IEEE double exactly as the sweeps use it
 * (Alg. 1 lines 6-9; O4).  Needs no GPU.
 * Ising: 10 classes, index 5*(s+1)/2 + (nn+4)/2 (s = -1 first, neighbour sum nn ascending), dE = 2 s (J nn + h).
 * Potts: 9 classes, index dn + 4, dn = n_new - n_old, dE = -J dn (h ignored).
 * T[c] = floor(exp(-beta dE) 2^32) clipped to 2^32-1; always[c] = 1 iff beta*dE <= 0 (accept regardless of
 * the random word).  A move of class c is accepted iff always[c] or r < T[c] (r: 32-bit Philox word).
 * Returns the number of classes written (10 or 9), or SPIN_ERR_INVALID. */
SPIN_API int spin_threshold_table(int32_t model, double beta, double J, double h, uint32_t* T, uint8_t* always);

/* Number of kernels this handle has launched since creation (for bench.py's gpu_launches). */
SPIN_API int64_t spin_kernel_launches(const spin_sim* sim);

/* Human-readable name of the sweep kernel variant the handle selects for its shape (diagnostics). */
SPIN_API const char* spin_kernel_variant(const spin_sim* sim);

/* +-J couplings (the paper writes Eq. 1 with a coupling J_ij per bond, and minimises a +-J spin glass
 * in Fig. 9).  Jh, Jv: HOST arrays, natural layout [batch][L][L], values +1 / -1:
 * Jh[b][i][j] is the sign of the bond between (i, j) and (i, (j+1) mod L), Jv[b][i][j] of the bond between (i, j) and
 * ((i+1) mod L, j).  From then on spin_sweep* use H = -J sum_bonds J_ij s_i s_j - h sum_i s_i (the local field is the
 * bond-weighted neighbour sum; thresholds, random words and acceptance are unchanged) and spin_observables* return
 * E_int = -sum_bonds J_ij s_i s_j.  Both NULL: back to uniform couplings.  The arrays are copied before return.
 * Bit-packed Ising layout: sign planes XORed into the multi-spin kernel (the fast path).  int8 layout, Ising and Potts
 * (Potts: H = -J sum_bonds J_ij delta(s_i, s_j) - h sum s_i, E_int = -sum_bonds J_ij delta): general one-thread-per-
 * group kernels.  SPIN_ERR_INVALID for a NULL handle, exactly one NULL array, a value that is not +-1, or a handle
 * with real couplings (the handle is left unchanged). */
SPIN_API int spin_set_bonds(spin_sim* sim, const int8_t* Jh, const int8_t* Jv);

/* Real-valued couplings and per-site fields (Eq. 1 as the paper writes it):
 * H = -sum_bonds J_ij s_i s_j - sum_i B_i s_i.  Jh, Jv, B: HOST double arrays, natural layout [batch][L][L] (bond
 * orientation as in spin_set_bonds), finite; copied before return.  From then on spin_sweep* ignore their J and h
 * arguments: the acceptance of each of the 32 (own spin, neighbour configuration) classes of every site is evaluated
 * on the host in IEEE double with the arithmetic of spin_threshold_table (dE = 2 s F, F = Jv[i-1][j] s_up + Jv[i][j]
 * s_down + Jh[i][j-1] s_left + Jh[i][j] s_right + B[i][j], summed in this order) whenever beta changes, uploaded
 * (132 bytes per site and replica) and looked up by the sweep kernel: bit-exact against the oracle by construction.
 * spin_observables keeps returning the uniform-model integers (E_int = -sum_bonds s_i s_j, M); the energy of the
 * general model comes from spin_energy_general.  All three NULL: back to uniform couplings.
 * Ising, int8 layout only (SPIN_ERR_UNSUPPORTED otherwise); SPIN_ERR_INVALID for a NULL handle, a partial set of
 * arrays, non-finite values, or a handle that has +-J bond signs; SPIN_ERR_NOMEM when the tables do not fit. */
SPIN_API int spin_set_couplings(spin_sim* sim, const double* Jh, const double* Jv, const double* B);

/* E[b] = -sum_bonds J_ij s_i s_j - sum_i B_i s_i of the current lattices for the couplings of spin_set_couplings, summed
 * in double on the device (agrees with a sequential double sum to ~1e-13 relative).  E: host [batch].  Synchronises. */
SPIN_API int spin_energy_general(spin_sim* sim, double* E);

/* Potts: S[b] = sum_i s_i, the sum of the state labels the field term of Eq. 5 couples to (reading P7).
 * With a field, spin_sweep samples H = J E_int - h S.  S: host [batch].  Synchronises. */
SPIN_API int spin_potts_label_sum(spin_sim* sim, int64_t* S);

/* Annealing schedule in one call (the Monte Carlo arm of the paper's Fig. 9): step k = 0 .. n_steps-1
 * runs sweeps_per_step sweeps at beta_steps[k][0..batch-1] (HOST, [n_steps][batch]), sweep indices
 * sweep_offset + k sweeps_per_step + 0 .. sweeps_per_step-1, exactly as n_steps consecutive spin_sweep calls would.
 * The tables of ALL steps are built first and uploaded in one copy; no host synchronisation between steps.
 * Asynchronous.  Class-table models only (uniform or +-J couplings; Potts without field): SPIN_ERR_UNSUPPORTED for
 * handles with real couplings or for Potts with h != 0 / bond signs.  Argument rules as for spin_sweep. */
SPIN_API int spin_sweep_schedule(spin_sim* sim, const double* beta_steps, int64_t n_steps, double J, double h,
                                 int64_t sweeps_per_step, int64_t sweep_offset);

/* Kernel selection policy (diagnostics / tests; the results never depend on it: every path computes the same
 * lattice).  A policy names a kernel family; whenever the handle's shape or couplings do not
 * qualify for it the call falls back to the streaming kernels.
 *   SPIN_POLICY_AUTO        picks per shape (rules derived from the measured grid profiles/r2_policy_grid.md).
 *   SPIN_POLICY_STREAMING   two launches per sweep (one per colour), the HBM kernels.
 *   SPIN_POLICY_RESIDENT    one CTA per replica keeps the lattice in shared memory and runs all sweeps of a call in one
 *                           launch: Ising int8 with L % 32 == 0 and L*L <= 192 KiB (E / M reductions fused for
 *                           spin_sweep_measure); bit-packed with uniform couplings and L*L/8 <= 200 KiB (plain sweeps).
 *   SPIN_POLICY_PERSISTENT  one cooperative launch for all sweeps of a call, the lattice in L2, a grid-wide barrier between
 *                           half-sweeps: Ising int8, L % 32 == 0, uniform couplings, no class whose threshold is 0.
 *                           Never picked by AUTO (the streaming kernels are faster on every measured shape).
 *   SPIN_POLICY_TILED       temporal blocking: a CTA advances a tile with a halo by 4 (small lattices: 2) sweeps per launch in
 *                           shared memory, at most one tile per SM (AUTO: up to 16 replicas and 2^21 sites); needs a second
 *                           lattice buffer (allocated by the library on first use): Ising int8, L % 8 == 0, L >= 16,
 *                           uniform couplings.
 *   SPIN_POLICY_GRAPH       the streaming kernels replayed from a CUDA graph of 64 sweeps captured once per handle (the kernels
 *                           read the sweep index from device memory): spin_sweep calls of >= 64 sweeps cost the host one
 *                           graph launch per 64 sweeps instead of 2-4 launches per sweep; the GPU-side rate is 1-5 % below
 *                           SPIN_POLICY_STREAMING.  Class-table models (uniform or +-J couplings, Potts without field),
 *                           L % 32 == 0 (bit-packed: L % 64 == 0), a handle created on a stream of its own (the legacy
 *                           default stream cannot be captured); spin_sweep only (spin_sweep_schedule and
 *                           spin_sweep_measure stream).  Never picked by AUTO.
 * Returns SPIN_OK or SPIN_ERR_INVALID (NULL handle, unknown policy). */
enum { SPIN_POLICY_AUTO = 0, SPIN_POLICY_STREAMING = 1, SPIN_POLICY_RESIDENT = 2, SPIN_POLICY_PERSISTENT = 3,
       SPIN_POLICY_TILED = 4, SPIN_POLICY_GRAPH = 5 };
SPIN_API int spin_set_policy(spin_sim* sim, int32_t policy);

/* ---------------------------------------------------------------------------------------------
 * Differentiable Monte Carlo: Algorithm 2 and Eq. 4 of the paper,
 * forward and backward, for the 2D Ising model with a coupling per bond (Eq. 1).  Stateless calls on
 * DEVICE arrays in the natural layout [batch][L][L], element type float (SPIN_DTYPE_F32) or double (SPIN_DTYPE_F64).
 * Jh[b][i][j] couples (i, j)-(i, (j+1) mod L), Jv[b][i][j] couples (i, j)-((i+1) mod L, j) (as in spin_set_bonds, but
 * real-valued); H = -sum_bonds J_ij s_i s_j - h sum_i s_i.  Per site x of the current colour (colour 0, then 1):
 *   F = sum_n J_xn s_n + h,  dE = 2 s F,  p = exp(-beta dE),  r = (w >> 8) / 2^24 with w the Philox word the Ising sweep
 *   uses for that (seed, replica, site, t, colour),  q = 1 / (1 + exp(-alpha (p - r))),  s <- q (-s) + (1 - q) s
 * (Alg. 2 lines 1-9 with the minus signs of PAPER.md:154; readings D1-D8 in DESIGN.md section 12).  alpha -> infinity
 * followed by spin_dmc_discretise reproduces spin_sweep.  beta: HOST, [batch], finite, >= 0.  alpha >= 0, h finite.
 * Inputs must keep beta |dE| below ~80 (fp32) so that p stays finite.  All work is enqueued on cuda_stream (NULL =
 * default stream); temporaries come from the stream-ordered allocator.  SPIN_ERR_INVALID: NULL pointers, bad shapes
 * (batch < 1, L odd or < 2), unknown dtype, bad sweep range; nothing is written in that case.
 * ------------------------------------------------------------------------------------------- */
enum { SPIN_DTYPE_F32 = 0, SPIN_DTYPE_F64 = 1 };

/* n_sweeps DMC sweeps t = sweep_offset .. from the lattice s0.  s_out: device, receives the final lattice (may equal s0).
 * traj: device, NULL or [(2 n_sweeps + 1)][batch][L][L]: traj[0] = s0 and traj[2k + 1 + c] = the lattice after the
 * colour-c half-sweep of sweep k (what spin_dmc_backward needs).  Asynchronous. */
SPIN_API int spin_dmc_forward(int32_t batch, int32_t L, int32_t dtype, const void* s0, const void* Jh, const void* Jv,
                              double h, const double* beta, double alpha, uint64_t seed, int64_t replica_offset,
                              int64_t n_sweeps, int64_t sweep_offset, void* s_out, void* traj, void* cuda_stream);

/* Reverse-mode derivative of a scalar loss through spin_dmc_forward (same arguments, traj as written by it).
 * grad_out: device [batch][L][L] = dLoss / d(final lattice).  Outputs, all overwritten: grad_s0, grad_Jh, grad_Jv: device
 * [batch][L][L] (same dtype); grad_beta, grad_h: HOST double [batch] (either may be NULL; per replica, h is one scalar so
 * its gradient is the sum over replicas).  Synchronises the stream when a host output is requested. */
SPIN_API int spin_dmc_backward(int32_t batch, int32_t L, int32_t dtype, const void* traj, const void* Jh, const void* Jv,
                               double h, const double* beta, double alpha, uint64_t seed, int64_t replica_offset,
                               int64_t n_sweeps, int64_t sweep_offset, const void* grad_out, void* grad_s0, void* grad_Jh,
                               void* grad_Jv, double* grad_beta, double* grad_h, void* cuda_stream);

/* Eq. 4 (Alg. 2 line 11): s <- -1 if s < 0 else +1 on n device elements.  Asynchronous. */
SPIN_API int spin_dmc_discretise(int32_t dtype, void* s, int64_t n, void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * Other lattice geometries: Algorithm 1 on the triangular lattice (Eq. 3),
 * the 3D cubic lattice and the square lattice with second neighbours ("more colors").
 * Stateless calls on a DEVICE int8 lattice of +-1 spins in the natural row-major layout, [batch][L][L] or
 * [batch][L][L][L].  H = -J1 sum_<first> s s' - J2 sum_<second> s s' - h sum s (J2 is used by SQUARE_NNN only).
 *   SPIN_STENCIL_TRIANGULAR: L % 3 == 0; neighbours (i+-1, j), (i, j+-1), (i+1, j+1), (i-1, j-1); colours (i + j) mod 3.
 *   SPIN_STENCIL_CUBIC:      L even; neighbours +-1 along each axis; colours (i + j + k) & 1.
 *   SPIN_STENCIL_SQUARE_NNN: L even; 4 first + 4 diagonal second neighbours; colours 2 (i & 1) + (j & 1).
 * A sweep visits the colours in order 0, 1, ...; the random word of a site is Philox group n >> 2, word n & 3, with n the
 * index of the site among the sites of its colour in row-major order (counter as in DESIGN.md O2, domain 3); acceptance
 * as in spin_threshold_table with dE = 2 s (J1 nn1 + J2 nn2 + h).  Readings S1-S6, DESIGN.md section 13.
 * beta: HOST [batch].  Work is enqueued on cuda_stream (NULL = default).  SPIN_ERR_INVALID for bad shapes / arguments.
 * ------------------------------------------------------------------------------------------- */
enum { SPIN_STENCIL_TRIANGULAR = 0, SPIN_STENCIL_CUBIC = 1, SPIN_STENCIL_SQUARE_NNN = 2 };

/* Sites (= bytes) per replica: L*L or L*L*L; 0 if the shape is invalid for the stencil. */
SPIN_API size_t spin_stencil_sites(int32_t stencil, int32_t L);
/* Uniform random +-1 lattice from Philox(seed): natural site index p, group p >> 2, word p & 3, +1 iff bit 31. */
SPIN_API int spin_stencil_init(int32_t stencil, int32_t batch, int32_t L, int8_t* lattice, uint64_t seed, int64_t replica_offset,
                               void* cuda_stream);
/* Sweeps t = sweep_offset .. sweep_offset + n_sweeps - 1, in place.  Asynchronous. */
SPIN_API int spin_stencil_sweep(int32_t stencil, int32_t batch, int32_t L, int8_t* lattice, const double* beta, double J1,
                                double J2, double h, uint64_t seed, int64_t replica_offset, int64_t n_sweeps,
                                int64_t sweep_offset, void* cuda_stream);
/* E1[b] = -(sum over first-neighbour bonds of s s'), E2[b] = the same over second-neighbour bonds, M[b] = sum s; every bond
 * once, with multiplicity on tiny lattices.  HOST int64 [batch], any may be NULL.  Energy = J1 E1 + J2 E2 - h M.
 * Synchronises the stream. */
SPIN_API int spin_stencil_observables(int32_t stencil, int32_t batch, int32_t L, const int8_t* lattice, int64_t* E1,
                                      int64_t* E2, int64_t* M, void* cuda_stream);
/* The same reductions for callers that may not allocate (code under CUDA graph capture, tight serving loops, harnesses
 * that forbid cudaMalloc): no cudaMalloc / cudaFree / allocating library routine, no host synchronisation.  The
 * accumulators live in a fixed device array inside the library (96 KiB per GPU that loads it, held until exit), hence
 * batch <= 4096: larger batches are rejected with SPIN_ERR_INVALID.  E1_dev, E2_dev, M_dev: DEVICE int64 [batch], any may
 * be NULL; written by work enqueued on cuda_stream (asynchronous: synchronise the stream before reading them).  The call
 * uses the CURRENT device, which must be the one holding lattice and the outputs (ordinal < 64, else
 * SPIN_ERR_UNSUPPORTED).  Every call shares the one array (cleared at the start of each call): calls that overlap on the
 * GPU - different streams, or graphs replayed concurrently - race on it; order them.  Other arguments and errors as for
 * spin_stencil_observables. */
SPIN_API int spin_stencil_observables_noalloc(int32_t stencil, int32_t batch, int32_t L, const int8_t* lattice,
                                              int64_t* E1_dev, int64_t* E2_dev, int64_t* M_dev, void* cuda_stream);

/* ---------------------------------------------------------------------------------------------
 * Cellular Potts model (Eq. 7 and Table II of the paper):
 *   H = 1/2 sum_x sum_{y in Moore(x)} J[tau(s_x)][tau(s_y)] (1 - delta(s_x, s_y)) + lambda sum_{cells s >= 1} (a_s - A_s)^2
 * on a DEVICE int8 lattice [batch][L][L] of cell identifiers 0..q-1 (0 = the medium, whose area is unconstrained), L even,
 * periodic.  tau: HOST int32 [q], type of each identifier (0..ntypes-1, ntypes <= 4); Jtab: HOST int32 [ntypes][ntypes],
 * symmetric; A: HOST int32 [q] target areas; lambda: integer >= 0 (readings C1-C9: integer
 * parameters make dH an exact integer).  A sweep = four colour passes (colour 2 (i & 1) + (j & 1)); in a pass every
 * site of the colour copies one of its eight Moore neighbours (chosen by r_prop >> 29) with the acceptance of Alg. 1
 * on dH = adhesion change + lambda [(new != 0)(2 (a_new - A_new) + 1) + (old != 0)(-2 (a_old - A_old) + 1)], the areas
 * counted at the start of the pass.  beta: HOST [batch] (= 1 / k_B T; the paper runs k_B T = 8).  Asynchronous.
 * SPIN_ERR_UNSUPPORTED when 0 < beta is so small that exp(-beta dH) 2^32 >= 1 beyond dH = 65536.
 * ------------------------------------------------------------------------------------------- */
SPIN_API int spin_cpm_sweep(int32_t batch, int32_t L, int32_t q, int8_t* lattice, const int32_t* tau, const int32_t* Jtab,
                            int32_t ntypes, int64_t lambda, const int32_t* A, const double* beta, uint64_t seed,
                            int64_t replica_offset, int64_t n_sweeps, int64_t sweep_offset, void* cuda_stream);
/* H_adh[b] = first term of Eq. 7 (every unordered Moore pair once), H_area[b] = second term, areas: [batch][q],
 * boundary: [batch][ntypes][ntypes], number of unordered Moore pairs with different identifiers and types (t, t'), stored
 * at [min][max] (the boundary lengths of the paper's Fig. 6).  HOST int64 arrays, any may be NULL.  Synchronises. */
SPIN_API int spin_cpm_observables(int32_t batch, int32_t L, int32_t q, const int8_t* lattice, const int32_t* tau,
                                  const int32_t* Jtab, int32_t ntypes, int64_t lambda, const int32_t* A, int64_t* H_adh,
                                  int64_t* H_area, int64_t* areas, int64_t* boundary, void* cuda_stream);

/* Measurement aid ("second, tighter denominator"): runs a register-only kernel on the current
 * device that does nothing but the algorithmic work of the sweep - Philox-4x32-10 calls (precomputed round keys) whose
 * four output words are each compared with a threshold - and returns the best-of-5 rate in random words per
 * nanosecond (= Ising updates/ns at one word per update; Potts uses two words per update).  Synchronous, default stream,
 * ~20 ms.  words_per_ns: host.  SPIN_ERR_INVALID for NULL, SPIN_ERR_CUDA without a device. */
SPIN_API int spin_measure_philox_compare_rate(double* words_per_ns);

#ifdef __cplusplus
}
#endif
#endif /* SPIN_H_ */
