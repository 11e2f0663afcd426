/* rfim_pt.h -- C ABI of librfimpt.so: B200-native (sm_100a) Exchange Monte Carlo (parallel
 * tempering) for the 3D Random Field Ising Model, after arxiv 1508.06268.
 *
 * Conventions
 *  - Every pointer argument is HOST memory owned by the caller unless it says "device".
 *    The library owns the handle and all device memory behind it.
 *  - Device memory comes from the allocator hook (rfim_pt_set_allocator; default cudaMalloc);
 *    kernels are enqueued on the handle's stream (rfim_pt_set_stream; default stream 0).
 *  - rfim_pt_sweep / rfim_pt_adapt_temperatures's trial enqueue work and return without
 *    synchronising where they can; every getter synchronises the handle's stream first.
 *  - Return value: 0 (RFIM_OK) or a negative code; rfim_pt_last_error gives a message.
 *    No exception crosses this boundary.  One host thread per handle at a time.
 *  - Lattice: L even, >= 2; site i = x + L*(y + L*z), x fastest; spins are int8 +1/-1 at the
 *    boundary (stored 1 byte or 1 bit per spin on the device).
 *  - R is the slot capacity; n (<= R) temperatures are active.  A "slot" is a stored lattice
 *    (lattices never move); a "rank" is a position in the ascending
 *    temperature list.  Arrays "by rank" have n entries per realisation.
 *  - A batch handle holds D independent disorder realisations ("members"), member d being
 *    exactly a single handle created with seeds[d].  Calls without a member argument act on
 *    all members; array outputs are then laid out [d][rank].
 *  - The exact arithmetic (random-number keying, thresholds, exchange rule, adaptation rule)
 *    is DESIGN.md section 3.
 */
#ifndef RFIM_PT_H
#define RFIM_PT_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct rfim_pt rfim_pt;

enum { RFIM_OK = 0, RFIM_EINVAL = -1, RFIM_ESTATE = -2, RFIM_ENOMEM = -3, RFIM_ECUDA = -4 };
enum { RFIM_FIELD_BIMODAL = 0, RFIM_FIELD_GAUSSIAN = 1 };

/* ---- the calls north_star names --------------------------------------------------------- */

/* PAPER.md:65-69 (section 3.1 steps 2-3): one random field H shared by all replicas
 * (bimodal h_i = +-1, or Gaussian N(0,1) on a 2^-20 grid), R random spin configurations.
 * H = -J sum_<ij> s_i s_j - h sum_i h_i s_i (Eq. 1).  Temperatures must be set
 * before sweeping.  EINVAL: odd or < 2 L, R < 1, bad field_kind, non-finite J or h. */
int rfim_pt_create(rfim_pt** out, int L, int R, double J, double h, int field_kind, uint64_t seed);

/* D realisations x R replicas in one handle (BASELINE.json config 5; "[..] average
 * over different disorder realizations").  seeds: D values. */
int rfim_pt_create_batch(rfim_pt** out, int L, int R, double J, double h, int field_kind,
                         int D, const uint64_t* seeds);

/* ---- replica distribution over several GPUs --------------------------
 * One realisation, R replica slots dealt to G ranks in contiguous windows of nslots = ceil(R/G) (Eq. 6:
 * m = ceil(M/D) replicas per GPU): the handle of rank g is created with slot0 = g * nslots and STORES only the
 * lattices of slots [slot0, slot0 + nslots) (slots >= R of the last window are never active).  Field, temperatures,
 * tables, the permutation t2r/r2t, exchange counters and the time series are replicated on every rank and stay
 * identical, because every rank takes the same exchange decisions from the same counter-based random stream: lattices
 * never move, only temperatures do.  The Philox counters are keyed on the global slot, so a sharded
 * run is bit-identical to the single-handle run.
 *
 * Sweeps need no communication.  Before every exchange step (and in the energy getters) each rank holds the integer
 * energy terms (Eb, Ef, Msum: 3 x int64 = 24 bytes per slot) of its own slots only; the library then calls the
 * gather function, which must complete the array on every rank -- an all-gather of local_bytes per rank:
 *   terms_device     device pointer, int64[rows][3], rows = G * nslots (padded), the same array on every call
 *   local_offset     byte offset of this rank's rows (= slot0 * 24),  local_bytes = nslots * 24
 *   total_bytes      rows * 24
 *   stream           the handle's CUDA stream (cudaStream_t): the collective must be ordered after the work already
 *                    enqueued on it and before work enqueued later (e.g. ncclAllGather on that stream, in place)
 * returning 0 on success.  The pointer stays owned by the library.  Restrictions: D = 1; slot0 a multiple of nslots;
 * the kernels that visit a slot window are the resident one (L = 32 or 64) and the small-lattice one (L % 8 == 0);
 * rfim_pt_get/set_spins_slot accept the stored slots only and rfim_pt_get/set_spins_all move the nslots stored lattices.
 *
 * rfim_pt_create_shard_rr deals the slots round-robin instead: rank g of G stores slots g, g + G, g + 2G, ...
 * (ceil(R/G) of them, padded like the windows).  This is PAPER.md:153's placement -- "new replica i goes to GPU i mod k" --
 * for every slot, so the replicas an adaptation inserts (pool slots n, n+1, ...) spread over the ranks instead of filling
 * the last window.  The gather function then receives a rank-major copy of the term array (same arguments, local_offset =
 * rank * local_bytes); everything else is as for windows.
 *
 * An adaptation step that INSERTS replicas (n < R) copies the colder neighbour's lattice into the new
 * replica's pool slot, which may live on another rank: the library then calls the broadcast function, once per inserted
 * replica and on every rank in the same order,
 *   buffer_device    device pointer, `bytes` = L^3 / 8 bytes: one lattice, bit-packed in natural site order
 *   root_rank        the rank whose buffer holds the lattice; on return every rank's buffer must hold it
 *   stream           the handle's CUDA stream (e.g. ncclBroadcast on that stream, in place)
 * returning 0 on success.  Without one, an inserting step on a shard returns RFIM_ESTATE (the fixed-count mode moves no
 * lattice and needs none). */
typedef int (*rfim_pt_gather_fn)(void* user, void* terms_device, size_t local_offset, size_t local_bytes,
                                 size_t total_bytes, void* stream);
typedef int (*rfim_pt_bcast_fn)(void* user, void* buffer_device, size_t bytes, int root_rank, void* stream);
int rfim_pt_create_shard(rfim_pt** out, int L, int R, double J, double h, int field_kind, uint64_t seed,
                         int slot0, int nslots);
int rfim_pt_create_shard_rr(rfim_pt** out, int L, int R, double J, double h, int field_kind, uint64_t seed,
                            int rank, int world);
int rfim_pt_set_gather(rfim_pt* h, rfim_pt_gather_fn fn, void* user);
int rfim_pt_set_broadcast(rfim_pt* h, rfim_pt_bcast_fn fn, void* user);
/* Native route for both collectives: the library calls NCCL itself on its stream -- ncclAllGather (in place, 24 bytes per
 * slot) before every exchange step and ncclBroadcast (L^3 / 8 bytes) per inserted replica -- so that no host callback sits
 * between the measuring kernel and the exchange kernel.  comm: an ncclComm_t whose rank / size equal this shard's;
 * all_gather_fn / broadcast_fn: the addresses of ncclAllGather and ncclBroadcast in the NCCL library that created it (the
 * library does not link NCCL).  comm = NULL switches back to the callbacks.  The communicator stays owned by the caller. */
int rfim_pt_set_nccl(rfim_pt* h, void* comm, void* all_gather_fn, void* broadcast_fn);
/* this rank, the number of ranks, first stored slot, slot stride (1: window, G: round-robin), stored slots (any may be NULL) */
int rfim_pt_get_shard_layout(rfim_pt* h, int* rank, int* world, int* first_slot, int* stride, int* nslots);
/* slot window and the energy-term array the gather function completes (any output pointer may be NULL) */
int rfim_pt_get_shard(rfim_pt* h, int* slot0, int* nslots, void** terms_device, size_t* terms_bytes);

int rfim_pt_destroy(rfim_pt* h);

/* PAPER.md:67 (step 1) + step 3's X_i <- beta_i: T[0..n) strictly ascending, > 0, 1 <= n <= R.
 * Rank t is given to slot t (identity permutation); acceptance tables are rebuilt on the host in
 * binary64 (S3); exchange statistics and the time series are reset; spins, the global
 * sweep counter and the global exchange-step counter are kept.  Applies to every member. */
int rfim_pt_set_temperatures(rfim_pt* h, const double* T, int n);

/* PAPER.md:70 (step 4): n_sweeps checkerboard Metropolis sweeps (colour (x+y+z) mod 2 = 0, then 1;
 * PAPER.md:101 Eq. 3) of every active replica; whenever the global sweep counter becomes a
 * multiple of exchange_every (> 0) an exchange step runs: per-replica energy reduction
 * (PAPER.md:220), one time-series row, then the even or odd adjacent pairs are swapped with
 * probability min(1, e^Delta) (Eq. 2) by permuting temperatures
 * (PAPER.md:131-137).  exchange_every = 0: never exchange.  Asynchronous.
 * EINVAL: negative arguments; ESTATE: temperatures not set. */
int rfim_pt_sweep(rfim_pt* h, int64_t n_sweeps, int exchange_every);

/* PAPER.md:147-153 (section 4): reset statistics, run one trial of trial_sweeps sweeps, then
 * insert midpoint temperatures where the exchange rate is lowest (growing n while n < R, else the
 * fixed-count insert-and-prune rule of DESIGN.md S8).  Synchronises.
 * ESTATE: temperatures not set, or a pair saw no exchange attempt in the trial. */
int rfim_pt_adapt_temperatures(rfim_pt* h, int64_t trial_sweeps);

/* By rank: E[t] = H of the replica now at rank t (Eq. 1), M[t] = (1/N) sum_i s_i (PAPER.md:251,
 * Eq. 11 before |.|), exchange_rate[t] = accepted/attempted swaps of pair (t,t+1) since the last
 * reset (-1 if none attempted).  Sizes D*n, D*n, D*(n-1); any pointer may be NULL.  Synchronises. */
int rfim_pt_observables(rfim_pt* h, double* E, double* M, double* exchange_rate);

/* Spins (+1/-1, L^3 bytes, x fastest) of the replica at temperature rank temp_rank of member 0. */
int rfim_pt_get_spins(rfim_pt* h, int temp_rank, int8_t* out);

/* ---- plumbing ------------------------------------------------------------------------------ */

/* cuda_stream: a cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream); NULL = default. */
int rfim_pt_set_stream(rfim_pt* h, void* cuda_stream);
/* waits for the handle's stream.  RFIM_ESTATE if a persistent sweep kernel gave up a dependency wait (it never hangs the
 * GPU: after ~2^22 polls it sets a flag and runs on; the lattices are then invalid).  rfim_pt_observables and
 * rfim_pt_get_diagnostics report the same condition. */
int rfim_pt_synchronize(rfim_pt* h);
/* Process-wide device allocator used by handles created afterwards.  alloc returns a device
 * pointer or NULL; both NULL restores cudaMalloc/cudaFree. */
typedef void* (*rfim_pt_alloc_fn)(size_t bytes);
typedef void (*rfim_pt_free_fn)(void* device_ptr);
int rfim_pt_set_allocator(rfim_pt_alloc_fn alloc, rfim_pt_free_fn release);
const char* rfim_pt_last_error(rfim_pt* h);
/* Storage of the lattices in device memory (BASELINE.json config 5 "spins bit-packed").
 * 8 = one byte per spin (default), 1 = one bit per spin (bit j & 7 of byte j >> 3, j the same colour-separated
 * site index as in the byte layout): an eighth of the footprint, every result identical to the byte layout
 * ("int8 == bit-packed").  The call converts the stored lattices (synchronises; both buffers
 * exist during the conversion).  Bit-packed lattices are read by the resident kernel only: RFIM_EINVAL unless
 * L is 32 or 64 and the kernel variant is 0 or 4; a later sweep fails with RFIM_EINVAL if the active planes do
 * not fit in shared memory.  Getters/setters keep their int8 +-1 interface in both modes. */
int rfim_pt_set_packing(rfim_pt* h, int bits);
/* which sweep implementation runs: 0 = automatic (default), 1 site, 2 word, 3 flow, 4 resident, 5 small-lattice
 * (one CTA per replica, whole lattice in shared memory). */
int rfim_pt_set_kernel_variant(rfim_pt* h, int variant);
/* tuning knobs (tests use them to force many-CTA partitions on small problems): key 0 = replicas per
 * work item of the flow kernel (1..64), key 1 = CTA limit of the resident kernel (0 = one per SM), key 2 = partition
 * of the resident kernel (0 automatic, 1 equal runs of planes, 2 whole replicas per CTA where they fit), key 3 = several
 * parallel-tempering moves per launch of the resident and small-lattice kernels (1 allowed, the default; 0 one launch per move). */
int rfim_pt_set_tuning(rfim_pt* h, int key, int value);
/* exchange period used by adapt's trial (default 10) and insertions per trial
 * (default 4, Fig. 6; the paper recommends 1-5). */
int rfim_pt_set_adapt_params(rfim_pt* h, int exchange_every, int insertions);
/* exchange rates of the adjacent pairs measured by the trial run of the LAST rfim_pt_adapt_temperatures call, i.e. the
 * rates its update was decided on (Figure 9 plots their min / avg / max per trial): rate[0 .. *n_pairs),
 * n_pairs = (replicas before that update) - 1.  RFIM_ESTATE before the first adaptation. */
int rfim_pt_get_trial_rates(rfim_pt* h, int d, double* rate, int* n_pairs);

/* ---- extensions used by tests and the benchmark (state must be observable to be compared) -- */

int rfim_pt_get_info(rfim_pt* h, int* L, int* R, int* n, int* D, int* field_kind);
int rfim_pt_get_spins_member(rfim_pt* h, int d, int temp_rank, int8_t* out);
int rfim_pt_get_spins_slot(rfim_pt* h, int d, int slot, int8_t* out);
int rfim_pt_set_spins_slot(rfim_pt* h, int d, int slot, const int8_t* in);
/* all D*R slots at once, [d][slot][L^3]; the host buffers of the end-to-end benchmark */
int rfim_pt_get_spins_all(rfim_pt* h, int8_t* out);
int rfim_pt_set_spins_all(rfim_pt* h, const int8_t* in);
/* the same with bit-packed HOST buffers (checkpoint format, an eighth of the PCIe traffic): [d][slot][L^3 / 8] bytes,
 * bit (i & 7) of byte (i >> 3) = 1 iff s_i = +1, i = x + L (y + L z).  Independent of the device storage mode
 * (rfim_pt_set_packing).  get synchronises; set is asynchronous on the handle's stream (`in` must stay valid and, for
 * true asynchrony, pinned, until the stream has consumed it). */
int rfim_pt_get_spins_all_bits(rfim_pt* h, uint8_t* out);
int rfim_pt_set_spins_all_bits(rfim_pt* h, const uint8_t* in);
/* field of member d in natural site order: bimodal +-1, Gaussian g_i in units of 2^-20 */
int rfim_pt_get_field(rfim_pt* h, int d, int32_t* out);
int rfim_pt_set_field(rfim_pt* h, int d, const int32_t* in);
int rfim_pt_get_permutation(rfim_pt* h, int d, int32_t* t2r);
int rfim_pt_set_permutation(rfim_pt* h, int d, const int32_t* t2r);
int rfim_pt_get_temperatures(rfim_pt* h, int d, double* T, int* n);
int rfim_pt_get_counters(rfim_pt* h, uint64_t* sweep_index, uint64_t* exchange_step);
int rfim_pt_set_counters(rfim_pt* h, uint64_t sweep_index, uint64_t exchange_step);
/* integer energy terms by rank: Eb = sum_bonds s_i s_j, Ef = sum h_i s_i (or sum g_i s_i), Msum */
int rfim_pt_get_energy_terms(rfim_pt* h, int d, int64_t* Eb, int64_t* Ef, int64_t* Msum);
/* one row [rank] per exchange step since the last reset */
int64_t rfim_pt_timeseries_steps(rfim_pt* h);
int rfim_pt_get_timeseries(rfim_pt* h, int d, int64_t* Eb, int64_t* Ef, int64_t* Msum);
/* thermal averages of the measurement series (one measurement per exchange step), per temperature
 * rank, over the steps [skip, steps) recorded since the last set_temperatures / adapt call.
 * rfim_pt_thermal_moments: out[n][5] = <e>, <e^2>, <|m|>, <m^2>, <m^4> of member d, e = E/N the energy per site,
 * m = (1/V) sum_i s_i.  rfim_pt_thermal_observables: the observables of Eq. 11-13 averaged over the D disorder
 * realisations of the handle, n values each (any pointer may be NULL): absM = [<|M|>] (Eq. 11),
 * C = [N/T^2 (<e^2> - <e>^2)] (Eq. 12, each realisation with its own T), g = (3 - [<M^4>]/[<M^2>]^2)/2 (Eq. 13).
 * Computed on the device from the integer series (fixed summation order: deterministic).  RFIM_ESTATE if no step has
 * been recorded after `skip`.  Host arrays are caller-owned; the calls synchronise. */
int rfim_pt_thermal_moments(rfim_pt* h, int d, int64_t skip, double* out);
int rfim_pt_thermal_observables(rfim_pt* h, int64_t skip, double* absM, double* C, double* g);
int rfim_pt_get_exchange_counts(rfim_pt* h, int d, uint64_t* attempted, uint64_t* accepted);
/* device acceptance table entry as the 33-bit threshold of DESIGN.md S3 (bimodal only) */
int rfim_pt_get_bimodal_threshold(rfim_pt* h, int d, int rank, int k, int b, uint64_t* thr);
/* The planning step of rfim_pt_adapt_temperatures alone (host only, no handle): ladder T[n] (ascending) with the trial's
 * exchange rates rate[n-1] of its adjacent pairs, capacity R, a insertions -> the new ladder in out_T (room for R values),
 * its length in *out_n.  n < R: PAPER.md:147's rule, the min(a, R-n, n-1) lowest-rate intervals (ties: lower rank) get
 * their midpoint temperature.  n == R: DESIGN.md S8's insert-and-prune.  RFIM_EINVAL on a bad argument. */
int rfim_pt_plan_adaptation(const double* T, const double* rate, int n, int R, int a, double* out_T, int* out_n);
/* The launch planning of rfim_pt_sweep alone (host only, no handle): with sweep_index sweeps done, n_sweeps >= 1 still asked for
 * and exchange steps every exchange_every sweeps (0: none), the next launch of a persistent sweep kernel covers *launch_sweeps
 * sweeps (<= 127) and holds *exchange_steps exchange steps: it stops at the first step it reaches, or, with several_moves != 0
 * (resident kernel, single unsharded handle), runs on through every whole period that fits.  RFIM_EINVAL on a bad argument. */
int rfim_pt_plan_launch(uint64_t sweep_index, int64_t n_sweeps, int exchange_every, int several_moves, int64_t* launch_sweeps,
                        int* exchange_steps);
/* diag[0] kernels launched so far, [1] Gaussian attempts decided by the exact binary64 path,
 * [2] decisions within 1e-5 of a binary64 threshold (device and host exp could disagree there;
 * expected 0), [3] exchange decisions taken with a random number */
int rfim_pt_get_diagnostics(rfim_pt* h, uint64_t diag[4]);

/* ---- an entry point that allocates nothing ---------------------------------------------------- */

/* The integer energy terms of Eq. 1 (the measurement of PAPER.md:220) for callers that may not call cudaMalloc
 * (code under CUDA graph capture, tight serving loops): no handle, no cudaMalloc / cudaFree / allocating library call.  All
 * three arrays are DEVICE memory owned by the caller:
 *   spins_device  [R][L^3] int8 +1 / -1, site i = x + L (y + L z)            (the layout of rfim_pt_get_spins_all)
 *   field_device  [L^3] int32, bimodal +-1 or Gaussian g_i in units of 2^-20 (the layout of rfim_pt_get_field)
 *   terms_device  [R][3] int64: Eb = sum_bonds s_i s_j, Ef = sum_i h_i s_i (or sum_i g_i s_i), Msum = sum_i s_i, per replica
 *                 (what rfim_pt_get_energy_terms reports by rank).
 * The kernel is enqueued on cuda_stream (NULL: stream 0) and the call returns without synchronising.  Its scratch (per-CTA
 * partial sums, one arrival counter per replica) is a static device array of RFIM_PT_NOALLOC_SCRATCH_BYTES bytes that every
 * GPU loading the library holds until exit; L <= RFIM_PT_NOALLOC_MAX_L and R <= RFIM_PT_NOALLOC_MAX_R, larger sizes return
 * RFIM_EINVAL.  All calls on a device share that array: calls that overlap on the GPU (different streams, or several host
 * threads) race and give wrong sums -- serialise them on one stream.  RFIM_EINVAL: odd or < 2 L, R < 1, bad field_kind, a
 * null pointer, a size beyond the limits; RFIM_ECUDA: a CUDA call failed.  The message is per host thread. */
#define RFIM_PT_NOALLOC_MAX_R 256
#define RFIM_PT_NOALLOC_MAX_L 128
#define RFIM_PT_NOALLOC_SCRATCH_BYTES (256 * 16 * 3 * 8 + 256 * 4)
int rfim_pt_energy_terms_noalloc(void* cuda_stream, int L, int R, int field_kind, const int8_t* spins_device,
                                 const int32_t* field_device, int64_t* terms_device);
const char* rfim_pt_noalloc_last_error(void);

/* ---- roofline microbenchmarks (bench.py measures both bounds in the same run) ------------- */

/* Philox4x32-10 only: calls_per_thread calls per thread, outputs folded; *ms = device time of one
 * launch (CUDA events), *attempts = 4 * calls issued. */
int rfim_pt_bench_philox(void* cuda_stream, int calls_per_thread, double* ms, double* attempts);
/* Issue-cost probe: the same Philox stream on one CTA of 16 warps per SM, with extra_per_call (0 or 8) extra instructions of one
 * kind per call spread between the rounds.  kind: 0 none (extra_per_call = 0), 1 LOP3, 2 PRMT, 3 I2FP (cvt.rn.f32.u32, ALU pipe),
 * 4 I2F.RM (cvt.rm.f32.u32, XU pipe), 5 FFMA, 6 FADD, 7 MUFU.EX2, 8 LDS.64.  *ms = device time of one launch, *warp_rows =
 * warp-rows (32 attempts) each SM sub-partition processed: (ms(kind) - ms(0)) * clock / warp_rows / 2 is the cost in cycles
 * of one more warp instruction of that kind next to the Philox stream. */
int rfim_pt_bench_issue(void* cuda_stream, int kind, int extra_per_call, double* ms, double* warp_rows);
/* streaming int8 read-modify-write over bytes bytes of device memory (> L2 for an HBM figure). */
int rfim_pt_bench_stream(void* cuda_stream, size_t bytes, double* ms, double* bytes_moved);

#ifdef __cplusplus
}
#endif
#endif /* RFIM_PT_H */
