/*
 * shaken.h -- C ABI of libshaken: the data-parallel half-step of the shaken dynamics
 * (D'Autilia, Andrianaivo, Troiani, "Parallel simulation of two-dimensional Ising models using
 * Probabilistic Cellular Automata", arXiv 1908.07341) on NVIDIA B200 (sm_100a).
 *
 * What one full step computes (PAPER.md = the paper's text; line numbers refer to it):
 *   half-step 0 ("odd times", eq. (15); Alg. 2 collectDL :371-377):
 *       tau'_x  = +1 with probability e^h / (2 cosh h),  h = J (sigma_{x down} + sigma_{x left}) + q sigma_x
 *   half-step 1 ("even times", eq. (16); Alg. 1 collectUR :354-361):
 *       sigma'_x = +1 with probability e^h / (2 cosh h),  h = J (tau'_{x up} + tau'_{x right}) + q tau'_x
 *   for every site x of the L x L torus at once (eq. (3)-(4); local fields eq. (14) :157-160;
 *   sampling rule "rand() < p" PAPER.md:174, Alg. 3 :413,:433).
 *
 * Conventions: x=(i,j) -> column c=i (contiguous), row r=j, site = r*L + c;
 * up = r+1, right = c+1, down = r-1, left = c-1, all mod L.  rand() is the 32-bit word
 *     rnd(seed, chain, g, site) = word (site & 3) of Philox4x32-10(key = (seed lo32, seed hi32),
 *                                  counter = (site >> 2, chain, g lo32, g hi32)),   g = 2 t + half,
 * t = 0-based global full-step index, and "rand() < p" is the integer compare  rnd < T[2k + c],
 * k = number of +1 among the two J-neighbours, c = [same-site spin == +1], T = shaken_thresholds().
 * Consequently spins and the int64 sums below are unique: a CPU oracle must match them bit for bit.
 *
 * Memory spaces.  Every pointer argument says HOST or DEVICE.  There are no torch types here; a Python
 * binding passes tensor.data_ptr() values.  One context is single-threaded; distinct contexts are independent.
 * No call throws, aborts or prints; every call returns 0 (SHAKEN_OK) or a negative error code, and
 * shaken_last_error() gives a human-readable message for the most recent failure on that context.
 * There is no CPU fallback: without a CUDA device every compute call fails with SHAKEN_ECUDA.
 */
#ifndef SHAKEN_H
#define SHAKEN_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct shaken_ctx shaken_ctx;

enum {
    SHAKEN_OK = 0,
    SHAKEN_EINVAL = -1, /* bad argument (size, mode, null pointer, non-finite coupling)            */
    SHAKEN_ENOMEM = -2, /* host or device allocation failed                                        */
    SHAKEN_ECUDA = -3,  /* CUDA runtime error (no device, launch failure, ...)                      */
    SHAKEN_ESTATE = -4, /* call not valid in this state (e.g. run before buffers exist)             */
    SHAKEN_ENOSPC = -5  /* record buffer too small for the records this run would append           */
};

/* layout flags of shaken_create */
#define SHAKEN_INT8 0u   /* one int8 (+1 / -1) per spin, [chain][r][c]; requires L % 16 == 0        */
#define SHAKEN_PACKED 1u /* 32 spins per uint32, bit b of word w of row r = site c = 32 w + b,
                            bit 1 <-> +1; [chain][r][w]; requires L % 32 == 0                        */

#define SHAKEN_N_OBS 6 /* record = (M_sigma, M_tau, E_J, E_q, C_x, C_y), see shaken_observables */

/* init modes of shaken_init */
#define SHAKEN_INIT_UP 1
#define SHAKEN_INIT_DOWN (-1)
#define SHAKEN_INIT_IID 0
#define SHAKEN_INIT_SANDWICH 2 /* first chain of every coupling group all +1, the others all -1 */

/*
 * shaken_create: allocate a context for n_chains independent L x L tori (batched-chain layout,
 * chain-major; the paper runs one (q,J) point per CPU thread).
 *   out      HOST, receives the context.
 *   L        16 <= L <= 65536, multiple of 16 (SHAKEN_INT8) or 32 (SHAKEN_PACKED).
 *   n_chains 1 <= n_chains, n_chains * L * L < 2^40.
 *   seed     Philox key.
 * Only host metadata is allocated here.  Device buffers are either borrowed with shaken_bind() or
 * allocated lazily by the library (cudaMalloc) at the first shaken_init / shaken_set_spins.
 * Errors: SHAKEN_EINVAL, SHAKEN_ENOMEM.
 */
int shaken_create(shaken_ctx **out, int32_t L, int32_t n_chains, uint64_t seed, uint32_t flags);

/* shaken_destroy: frees the context and only the device memory the library itself allocated. */
int shaken_destroy(shaken_ctx *ctx);

/* Bytes of ONE sublattice buffer (sigma or tau) in device layout: n_chains*L*L (int8) or n_chains*L*L/8. */
size_t shaken_spin_bytes(const shaken_ctx *ctx);

/* Bytes of one record for all chains: n_chains * 6 * sizeof(int64_t). */
size_t shaken_record_bytes(const shaken_ctx *ctx);

/*
 * shaken_bind: borrow device memory and a stream from the caller (PyTorch is used only for this).
 *   d_sigma, d_tau  DEVICE, each shaken_spin_bytes() bytes, 16-byte aligned; never freed by the library.
 *   d_records       DEVICE, rec_bytes bytes, 8-byte aligned, capacity floor(rec_bytes / shaken_record_bytes())
 *                   records; may be NULL with rec_bytes 0 (then the library allocates on demand).
 *   cuda_stream     a cudaStream_t (NULL = the legacy default stream).  All work of this context is
 *                   enqueued on it.
 * The record buffer is zeroed (asynchronously) and the record count reset.  The spin buffers are not touched and
 * their content counts as UNDEFINED: shaken_run / shaken_get_spins / shaken_diag_correlations return SHAKEN_ESTATE
 * until shaken_init, shaken_set_spins (per layer) or shaken_adopt_spins has defined it.
 * Errors: SHAKEN_EINVAL (null/misaligned), SHAKEN_ECUDA.
 */
int shaken_bind(shaken_ctx *ctx, void *d_sigma, void *d_tau, void *d_records, size_t rec_bytes, void *cuda_stream);

/* shaken_adopt_spins: declare that the bound DEVICE buffers already hold both layers in device layout (a caller that
 * filled them with its own kernels).  int8 layers are checked on the device to contain only +1 / -1 bytes
 * (SHAKEN_EINVAL otherwise; packed words are always valid).  Synchronises the stream.  SHAKEN_ESTATE without buffers. */
int shaken_adopt_spins(shaken_ctx *ctx);

/* Make room for at least max_records records in a library-owned buffer (existing records are kept).
 * Not allowed on a bound record buffer (SHAKEN_ESTATE). */
int shaken_reserve_records(shaken_ctx *ctx, int64_t max_records);

/*
 * shaken_init: set sigma and tau of every chain and reset the step counter and the record count to 0.
 *   mode  SHAKEN_INIT_SANDWICH: see shaken_set_coupling;  SHAKEN_INIT_UP: all +1;  SHAKEN_INIT_DOWN: all -1 (the paper's scan start; the
 *         top/bottom chains of :238);  SHAKEN_INIT_IID: iid +-1, spin = +1 iff the init-stream word
 *         Philox(key = seed, counter = (site>>2, chain, which, 0xFFFFFFFF))[site & 3] < 2^31,
 *         which = 0 for sigma, 1 for tau.
 */
int shaken_init(shaken_ctx *ctx, int mode);

/*
 * shaken_run: advance every chain by n_steps full steps (2 half-steps each) with couplings J, q
 * (any finite doubles; eq. (14)).  The global step counter t advances by n_steps.
 * After every full step whose 1-based global index is a multiple of obs_every (0 = never) one record
 * is appended (fused into the kernels, int64 atomics).  Work is enqueued on the context's stream and
 * the call returns without waiting; shaken_observables / shaken_get_spins / shaken_synchronize wait.
 * Errors: SHAKEN_EINVAL (non-finite J or q, negative counts), SHAKEN_ENOSPC (bound record buffer too
 * small; nothing is run), SHAKEN_ESTATE (no spins yet), SHAKEN_ECUDA.
 */
int shaken_run(shaken_ctx *ctx, double J, double q, int64_t n_steps, int64_t obs_every);

/* Same with one (J, q) per chain: J, q HOST arrays of n_chains doubles, read during the call only. */
int shaken_run_grid(shaken_ctx *ctx, const double *J, const double *q, int64_t n_steps, int64_t obs_every);

/*
 * Alternate parallel heat bath on the SQUARE lattice ("a parallel version of the heat bath dynamics that
 * updates, alternatively, the spins on the odd and the even sites of the lattice", the square-lattice equivalent of
 * eq. (15)-(16); its equilibrium measure is the Gibbs measure of the square-lattice Ising model with coupling J).
 * It runs on the context's sigma array alone, in place; tau is not touched.  Site (r, c) has colour (r + c) & 1.  Full
 * step t = half-step 0 (every site of colour 0 redrawn), then half-step 1 (colour 1):
 *     s'_x = +1  iff  rnd(x) < A[k],   k = number of +1 among the four nearest neighbours,   h = J (2k - 4),
 *     A[k] = shaken_alt_thresholds(J)[k]  (same integer scale and mirror rule as shaken_thresholds),
 *     rnd(x) = Philox4x32-10(key = seed, counter = (m >> 2, chain, g lo, g hi))[m & 3],  m = (r L + c) >> 1,  g = 2t + half
 * (m numbers the sites of one colour in row-major order).  The step counter, coupling groups, coalescence times
 * (compared on sigma) and the chain offset work as for shaken_run.  A record appended after a step holds
 * (M, 0, 0, 0, C_x, C_y) of the sigma array: H(sigma) = -J (C_x + C_y).
 * shaken_run_alternate_grid: J is a HOST array of n_chains doubles.  Errors as shaken_run.
 */
int shaken_alt_thresholds(double J, uint32_t out[5]);
int shaken_run_alternate(shaken_ctx *ctx, double J, int64_t n_steps, int64_t obs_every);
int shaken_run_alternate_grid(shaken_ctx *ctx, const double *J, int64_t n_steps, int64_t obs_every);

/*
 * shaken_observables: wait for the stream, then copy min(n_records, max_records) records to
 *   out  HOST, layout [record][chain][6] int64 =
 *        M_sigma = sum_x sigma_x, M_tau = sum_x tau_x                      (eq. (17))
 *        E_J = sum_x sigma_x (tau_{x up} + tau_{x right}), E_q = sum_x sigma_x tau_x
 *                                               (H(sigma,tau) = -(J E_J + q E_q), eq. (5))
 *        C_x = sum_x sigma_x sigma_{x right}, C_y = sum_x sigma_x sigma_{x up}
 *                                               (square-lattice H(sigma) = -J (C_x + C_y))
 *        all on the pair (sigma', tau') right after half-step 1.
 * Returns the number of records copied, or a negative error code.
 */
int64_t shaken_observables(shaken_ctx *ctx, int64_t *out, int64_t max_records);

/*
 * shaken_moments: derived statistics of the recorded magnetisation of ONE chain (the paper reports
 * average and variance of m over the recording window, eq. (17)).  Pure host arithmetic.
 *   M        HOST, the n values M[0], M[stride], M[2 stride], ... (e.g. out + chain*6 + 0 of shaken_observables with
 *            stride = n_chains * 6 gives M_sigma of that chain); a burn-in is dropped by offsetting M.
 *   n        1 <= n < 2^31 records;  n_sites = L*L <= 2^32;  |M| <= n_sites is checked (SHAKEN_EINVAL).
 *   out      HOST [SHAKEN_N_MOMENTS] doubles: <m>, <|m|>, <m^2>, <m^4>, Var m = <m^2> - <m>^2 (population variance),
 *            Binder cumulant U = 1 - <m^4> / (3 <m^2>^2) (NaN when every M is 0), with m = M / n_sites.
 * The power sums are exact integers (M^4 reaches 2^128 at L = 65536: 256-bit accumulation), differences are taken
 * before rounding, and each result is one long-double division rounded to double: relative error < 1e-15.
 */
#define SHAKEN_N_MOMENTS 6
int shaken_moments(const int64_t *M, int64_t n, int64_t stride, int64_t n_sites, double out[SHAKEN_N_MOMENTS]);

/* Number of records currently stored (>= 0) or a negative error code. */
int64_t shaken_num_records(const shaken_ctx *ctx);

/* Forget all records (the buffer is zeroed on the stream). */
int shaken_clear_records(shaken_ctx *ctx);

/*
 * State I/O (parity checks and checkpoint/resume).  which = 0: sigma, 1: tau.
 *   host  HOST, n_chains*L*L int8 values +1 / -1, layout [chain][r][c] -- also for SHAKEN_PACKED
 *         (the library converts on the device).  set_spins rejects other values with SHAKEN_EINVAL.
 * Both calls synchronise the stream.
 */
int shaken_get_spins(shaken_ctx *ctx, int which, int8_t *host);
int shaken_set_spins(shaken_ctx *ctx, int which, const int8_t *host);

/* Global full-step counter t (the random numbers of a step depend on it, so run(a); run(b) == run(a+b)). */
int shaken_get_step(const shaken_ctx *ctx, uint64_t *step);
int shaken_set_step(shaken_ctx *ctx, uint64_t step);

/*
 * shaken_set_chain_offset: chain c of this context draws the random numbers of global chain first_chain + c
 * (counter word 1).  Lets a batch of chains be sharded over several contexts / GPUs with results identical to
 * one big batch (independent units, no exchange: SURVEY 8(e)).  Default 0.  first_chain + n_chains <= 2^32.
 */
int shaken_set_chain_offset(shaken_ctx *ctx, uint32_t first_chain);

/*
 * Coupled chains and coalescence times.
 * shaken_set_coupling: chains c with equal c / group evolve "with the same update function and the same sequence of
 *   random numbers": all draw the words of the group's first chain (counter word 1 = first_chain + (c / group) * group).
 *   group >= 1 must divide n_chains; 1 (default) uncouples.  Couplings J, q are still per chain (give the members of a
 *   group the same values for the paper's experiment).  Forgets coalescence times.  Errors: SHAKEN_EINVAL, SHAKEN_ENOMEM.
 * While group > 1 the sigma layers of each group's members are compared on the device after EVERY full step (fused into
 *   the half-step kernels: the comparison of a step rides on the launches of the next one, a read-only pass closes a
 *   run call, so the times are complete when shaken_run's work has finished); the coalescence time T = min{n : X_n = Y_n}
 *   of a group is the number of full steps done (global step counter) when they were first all equal.  shaken_init
 *   resets the times to -1.
 * shaken_coalescence: copy min(n_chains / group, max_groups) times to out (HOST int64, -1 = not yet); returns the
 *   count (0 when uncoupled) or a negative error code.  Synchronises the stream.
 */
int shaken_set_coupling(shaken_ctx *ctx, int32_t group);
int64_t shaken_coalescence(shaken_ctx *ctx, int64_t *out, int64_t max_groups);

/*
 * shaken_diag_correlations: diagonal spin-spin correlations of the CURRENT sigma layer (Table 1; SURVEY
 * 8(f) rank 2) as translation-summed integers over the torus (divide by L*L for the paper's pi(sigma_{0,0} sigma_{l,l})):
 *   ells  HOST [n_ell] distances l >= 0 (taken mod L; the paper uses 1, 2, 4, 8, 16 on a 32 x 32 box)
 *   out   HOST [n_chains][n_ell][2] int64:  [0] SW-NE  sum_{r,c} sigma[r][c] sigma[r+l][c+l]
 *                                           [1] NW-SE  sum_{r,c} sigma[r+l][c] sigma[r][c+l]
 * Both layouts.  Synchronises the stream.  Errors: SHAKEN_EINVAL, SHAKEN_ESTATE, SHAKEN_ENOMEM, SHAKEN_ECUDA.
 */
int shaken_diag_correlations(shaken_ctx *ctx, const int32_t *ells, int32_t n_ell, int64_t *out);

/*
 * Row-slab sharding of ONE lattice over several contexts / GPUs (second bullet).  The fields of eq. (14)
 * reach one row across a slab edge per half-step; because a site's random word is a function of the
 * GLOBAL site index, a slab redraws the tau row above itself redundantly and the slabs exchange only sigma rows, once per
 * full step, by stores into the neighbours' "inbox" (peer memory over NVLink) -- results are bit-identical to the unsplit
 * lattice for any partition.  int8 layout, one chain.
 *
 * shaken_create_slab: context for rows [row0, row0 + n_rows) of an L x L torus (n_rows >= 2; L as for shaken_create).
 *   The context owns its device buffers (shaken_bind is not available; shaken_set_stream chooses the stream).
 *   shaken_spin_bytes = n_rows * L; shaken_get_spins / shaken_set_spins move the slab's rows [n_rows][L];
 *   shaken_init as usual (iid: the init-stream words of the slab's global sites).  Records hold the sums over the slab's
 *   own sites and bonds (E_J, C_y: the bonds to the rows above / below the slab counted once, by the lower / upper slab's
 *   partner as on the torus); the caller adds the records of all slabs.  The C_x, C_y of the LAST record of a run need
 *   the neighbour's new row: they are completed by the next shaken_run or by shaken_observables (both wait for it).
 *   shaken_run_grid works with its single chain; shaken_run_alternate, coupling and shaken_diag_correlations return
 *   SHAKEN_ESTATE.
 * shaken_slab_inbox: DEVICE pointer and size of this context's inbox ([2 sides][2 parities][L/4] {word, stamp} pairs),
 *   for the neighbours to store into.
 * shaken_slab_connect: the inboxes of the rank below (owner of row row0 - 1) and above (owner of row row0 + n_rows),
 *   DEVICE pointers valid on this device (the same process: any peer-enabled allocation; for a single slab both are
 *   its own inbox).  shaken_slab_ipc_export / shaken_slab_ipc_connect do the same across processes with CUDA IPC
 *   handles (64 bytes each, HOST memory; exchange them with any host-side transport, e.g. torch.distributed).
 * shaken_slab_exchange: publish the slab's current edge rows now if they have not been (shaken_run does it itself; an
 *   explicit call lets a driver that advances several slabs ONE AFTER THE OTHER on one device publish all of them before
 *   any of them waits).  Every rank must make the same sequence of run / exchange calls: exchanges are counted.
 * shaken_run on a slab: per step one hand-over (publish, wait for the neighbours' rows, redraw tau row n_rows) and the two
 *   half-step launches of the strip kernels.  SHAKEN_ESTATE if not connected.
 */
int shaken_create_slab(shaken_ctx **out, int32_t L, int32_t row0, int32_t n_rows, uint64_t seed);
int shaken_set_stream(shaken_ctx *ctx, void *cuda_stream);
int shaken_slab_inbox(shaken_ctx *ctx, void **d_inbox, size_t *bytes);
int shaken_slab_connect(shaken_ctx *ctx, void *d_inbox_below, void *d_inbox_above);
int shaken_slab_ipc_export(shaken_ctx *ctx, void *handle64);
int shaken_slab_ipc_connect(shaken_ctx *ctx, const void *below_handle64, const void *above_handle64);
int shaken_slab_exchange(shaken_ctx *ctx);

/* Wait until everything enqueued by this context has finished. */
int shaken_synchronize(shaken_ctx *ctx);

/*
 * shaken_thresholds: the integer acceptance table for one (J, q), HOST out[6]:
 *   T[2k + c] = round(2^32 * e^h / (2 cosh h)),  h = J (2k - 2) + q (2c - 1)
 * evaluated as F(|h|) = clamp(floor(2^32 / (1 + exp(-2|h|)) + 0.5), 2^31, 2^32 - 1) in binary64 and
 * mirrored for h < 0 (T(h) + T(-h) = 2^32 exactly).  Pure host arithmetic; no device needed.
 */
int shaken_thresholds(double J, double q, uint32_t out[6]);

/*
 * shaken_philox_words: test hook.  Runs the library's DEVICE Philox4x32-10 on n (counter, key) pairs:
 *   ctr HOST [n][4] uint32, key HOST [n][2] uint32, out HOST [n][4] uint32.
 */
int shaken_philox_words(const uint32_t *ctr, const uint32_t *key, uint32_t *out, int64_t n);

/*
 * shaken_selftest_philox_rate: measurement hook.  Times, with CUDA events on the default stream, a kernel that runs the
 * half-step kernels' own Philox4x32-10 (one call per 4 sites, 32 random bits per site) plus one
 * compare per word and nothing else -- no memory traffic.  The result is the practical ceiling, in site-updates per
 * ns, of ANY kernel on this device that draws the random numbers this library is specified to draw; bench.py prints it
 * beside the achieved rate and the HBM roofline.
 *   blocks_per_sm 1..8 (256 threads each), iters calls of 4 x 4 sites per thread, best of reps timed launches after a warm-up.
 *   sites_per_ns  HOST, receives the rate.
 */
int shaken_selftest_philox_rate(int32_t blocks_per_sm, int32_t iters, int32_t reps, double *sites_per_ns);

/*
 * shaken_test_band_hook: test hook for the one-launch band path (mid-size lattices).  what = 0: the
 * stamp counter of the hand-over buffer is set to `value` (a value near 2^32 exercises the wrap-around clearing);
 * what = 1: the next cooperative launch is treated as refused (value != 0), which exercises the fall-back to the
 * per-half-step kernels; what = 2: bands of at most seven rows are run by the two-phase band kernel instead of the
 * data-flow one (value != 0) or by the default (0).  Results never depend on any of them.  SHAKEN_EINVAL for another selector.
 */
int shaken_test_band_hook(shaken_ctx *ctx, int what, uint32_t value);

/*
 * shaken_run_static / shaken_static_setup: the shaken dynamics for callers that must not allocate (code under CUDA graph
 * capture, tight serving loops, harnesses that forbid cudaMalloc).  Same operation as shaken_run on an int8 context --
 * n_steps full steps, half-step 0 tau <- sigma (eq. 15) then half-step 1 sigma <- tau (eq. 16,
 * :169-172), thresholds of shaken_thresholds(J, q), random words of (seed, chain, step, half, site) -- in ONE cooperative
 * launch of the band kernel (row bands resident in shared memory), whose only scratch memory, the
 * hand-over rows between neighbouring bands, lives in a file-scope device array of SHAKEN_STATIC_SCRATCH_BYTES that
 * every GPU which loads the library holds until exit.  There is no context: the caller owns every buffer.
 *   sigma, tau   DEVICE [n_chains][L][L] int8 (+1 = 0x01, -1 = 0xFF), 16-byte aligned; sigma is read and both are
 *                overwritten in place (tau need not be initialised: half-step 0 redraws all of it).
 *   L, n_chains  128 < L <= 2048, L % 16 == 0, 1 <= n_chains <= number of SMs; the bands (ceil(L / floor(SMs / n_chains))
 *                rows each) must fit 160 KiB of shared memory and their hand-over rows the static scratch array:
 *                SHAKEN_EINVAL with a message naming the limit otherwise (e.g. 1 x 2048^2, 4 x 1024^2 fit).
 *   seed, t0     Philox key and the 0-based global index of the first full step (chain c draws the words of chain c).
 *   obs_every    0 = no records; else a record after every step whose 1-based global index is a multiple of it.
 *   rec          DEVICE [max_records][n_chains][6] int64, may be NULL when no record falls into the run; the records of
 *                this run are written from slot 0 (the call zeroes the slots it fills).  SHAKEN_ENOSPC if too small.
 *   cuda_stream  a cudaStream_t (NULL = default stream); the call is asynchronous on it.
 * The call issues two cudaMemsetAsync (scratch, records) and one kernel launch and calls no cudaMalloc, cudaFree or any
 * allocating library routine; shaken_static_setup() (once per device, with that device current; shaken_run_static calls it
 * when needed) looks up the scratch array's device address and the device's properties -- call it before a region that
 * must not touch the module loader.  ALL calls on a device share the scratch array, which keeps the last call's contents:
 * every call clears the part it uses first, and two calls that overlap on the GPU (different streams, concurrent graphs)
 * race -- serialise them.  Errors: SHAKEN_EINVAL, SHAKEN_ENOSPC, SHAKEN_ECUDA (no device; cooperative launch refused:
 * there is no fall-back here).
 */
#define SHAKEN_STATIC_SCRATCH_BYTES 2621440 /* 2.5 MiB = 2 parities x 2 sides x 160 bands x 512 words x 8 bytes */
int shaken_static_setup(void);
int shaken_run_static(void *sigma, void *tau, int32_t L, int32_t n_chains, uint64_t seed, uint64_t t0, double J, double q,
                      int64_t n_steps, int64_t obs_every, int64_t *rec, int64_t max_records, void *cuda_stream);

/* Number of kernels this context has launched so far (half-steps, init, conversions, reductions). */
int64_t shaken_launch_count(const shaken_ctx *ctx);

/* Code-path switch for tests and measurements; results never depend on it.  0 = automatic (default).
 * SHAKEN_VARIANT_STRIPS: every lattice size takes the per-half-step strip kernels (automatic would run L <= 128 in the
 * one-launch shared-memory kernel and mid-size lattices in the one-launch band kernel); applies to shaken_run and
 * shaken_run_alternate.  SHAKEN_VARIANT_PERWARP: strip kernels with per-warp task lists (automatic for batches of small
 * chains).  Any other value: SHAKEN_EINVAL. */
#define SHAKEN_VARIANT_STRIPS 3
#define SHAKEN_VARIANT_PERWARP 8
int shaken_set_variant(shaken_ctx *ctx, int variant);

/* Message for the most recent error on this context ("" if none).  ctx may be NULL (creation errors). */
const char *shaken_last_error(const shaken_ctx *ctx);

/* Library version string, e.g. "libshaken 0.1 (sm_100a)". */
const char *shaken_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SHAKEN_H */
