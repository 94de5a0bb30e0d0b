/*
 * lsm.h -- C ABI of liblsm: sublattice-parallel ("checkerboard") single-spin-flip
 * Monte Carlo sweeps of lattice spin models on one NVIDIA B200 (sm_100a).
 *
 * Method: T. Levy, G. Cohen, E. Rabani, "Simulating lattice spin models on GPUs",
 * arXiv:1209.0296.  Line references "PAPER.md:NN" are to the text of that paper;
 * "D<n>" are the readings of DESIGN.md section 3 (= SURVEY.md 8(c)) adopted where
 * the paper is silent or ambiguous.
 *
 * General rules
 *  - Every function returns an int status (LSM_OK = 0, errors < 0).  On error the
 *    out-parameters are left untouched.  Nothing is printed, nothing aborts.
 *  - The library never allocates or frees device memory and never creates streams.
 *    The caller owns the workspace, every d_* buffer and the stream (in this repo:
 *    PyTorch tensors and torch.cuda streams).  `stream` is a cudaStream_t passed as
 *    void* (NULL = the legacy default stream).  lsm_t itself lives on the host heap.
 *  - Pointers named d_* are DEVICE pointers, h_* are HOST pointers; unprefixed
 *    out-parameters (E, M, counts) are host pointers.
 *  - Calls that take a stream only enqueue work on it (asynchronous).  Calls that
 *    return values to the host synchronise the stream last given to this handle.
 *  - There is no CPU fallback: without a CUDA device every compute call returns
 *    LSM_ERR_CUDA.
 *
 * Models (argument `model`, `two_S`):
 *  LSM_ISING, two_S = 1 : s_i = +/-1,  H = -J sum_<ij> s_i s_j - h sum_i s_i
 *                         (sign convention D1); trial move s -> -s.
 *  LSM_ISING, two_S = 2 : s_i in {-1,0,+1}, same H; trial move = one of the two other
 *                         values, chosen uniformly (D5; BASELINE.json config 4).
 *  LSM_NE_HEATBATH      : North-East model, occupation n_i in {0,1},
 *                         J = 0, H = sum n_i, c = 1/(1+exp(1/T)) (D6: the paper's +/-1 spins give
 *                         c = 1/(1+exp(2/T_paper)), i.e. T_paper = 2 T here).  A site may change
 *                         only if its north (x,y+1) and east (x+1,y) neighbours are both
 *                         up (D8); then n_i is redrawn from Bernoulli(c) (D7).
 *  LSM_NE_METROPOLIS    : same constraint, Metropolis flip: 1->0 always,
 *                         0->1 with probability exp(-1/T).
 *  LSM_EA, two_S = 1     : Edwards-Anderson +/-J spin glass (Eq. 1 with discrete J_ij; D25):
 *                         H = -J sum_<ij> tau_ij s_i s_j - h sum s_i, tau_ij = +/-1 per bond, drawn from the seed
 *                         (p = 1/2) or set with lsm_set_bonds; Ising rule on the bond-weighted neighbour sum.
 *  LSM_POTTS             : q-state Potts model (D26), q = two_S + 1 in [2, 8], sigma in {0..q-1},
 *                         H = -J sum_<ij> delta(sigma_i, sigma_j), h must be 0; trial state uniform over the other
 *                         q-1 states, Metropolis acceptance.  bond_sum = bonds joining equal states, M = sites in
 *                         state 0, E = -J * bond_sum; overlap of lsm_persistence = sites in their reference state.
 *  Acceptance (P = min[1, exp(-dH/T)]) is an integer compare of a 32-bit
 *  random word w with a 33-bit threshold thr = floor(P * 2^32) in [0, 2^32]: accept iff
 *  w < thr (D3).
 *
 * Lattice: periodic, hypercubic, dims = 2 or 3, linear size L (even, >= 4; D10),
 *  N = L^dims sites, canonical site id i = x + L*(y + L*z), parity (x+y+z)&1.
 * One sweep (= one Monte Carlo step) = half-sweep over parity 0, then over
 *  parity 1 (the two kernel launches of PAPER.md:96-97; D9) = N attempted updates.
 * Random numbers: Philox4x32-10, key = seed, counter = (site group, sweep, half) (D2).
 *  The handle keeps a 64-bit sweep counter t < 2^60; sweep t uses counter fields c2 = lo32(t),
 *  c3 = tag | hi32(t) << 4, the low four bits of c3 being the stream tag alone (0/1 = half-sweep,
 *  2 = initial state, 4/5 and 8..11 = random-tile launches), so streams never alias (D2).
 *
 * Values at the boundary (int8): spin-1/2 -> {-1,+1}; spin-1 -> {-1,0,+1}; NE -> {0,1};
 *  canonical order.  The device-internal encoding (split even/odd colour arrays, flag
 *  bits) is private.
 *
 * Integer observables: M = sum_i s_i (NE: number of up sites); bond sum
 *  B = sum_<ij> s_i s_j, each bond once (NE: 0).  E = -J*B - h*M (NE: E = M) (D1, D15).
 */
#ifndef LSM_H
#define LSM_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct lsm lsm_t;             /* opaque, host heap */
typedef struct lsm_batch lsm_batch_t; /* opaque, host heap: R lattices of one shape swept together */

enum { LSM_ISING = 0, LSM_NE_HEATBATH = 1, LSM_NE_METROPOLIS = 2, LSM_EA = 3, LSM_POTTS = 4 };
enum {
    LSM_OK = 0,
    LSM_ERR_ARG = -1,         /* dims not 2|3, L odd or < 4, T <= 0 or non-finite, NULL, n < 0 */
    LSM_ERR_UNSUPPORTED = -2, /* Ising two_S not 1|2; NE with dims != 2, J != 0 or two_S != 1; EA two_S != 1; Potts q = two_S + 1
                                 outside [2, 8] or h != 0; a kernel family / tile / depth that cannot run this lattice */
    LSM_ERR_CUDA = -3,        /* a CUDA runtime call failed (text: lsm_last_cuda_error)         */
    LSM_ERR_WORKSPACE = -4,   /* workspace too small or not 256-byte aligned                   */
    LSM_ERR_STATE = -5,       /* tracking is off (lsm_persistence); replicas out of lockstep (batch) */
    LSM_ERR_LIMIT = -6        /* lsm_sweep_record_host_noalloc: n > LSM_NOALLOC_MAX_SWEEPS                 */
};
/* Kernel families (lsm_set_kernel).  AUTO picks the fastest one that supports the lattice:
 *  SMALL    one launch for all sweeps of a call: lattice slabs in the shared memory of a thread-block cluster,
 *           cluster barrier between the colours (L a power of two >= 8; other L with L % 32 == 0 up to 32 768
 *           sites); chosen below 262 144 sites (up to 256^2, 32^3);
 *  TILED    one launch per half-sweep, 16 sites per 128-bit word (L % 32 == 0, no "never" threshold);
 *  RESIDENT removed in round 3 (one cooperative launch with neighbour-flag synchronisation: measured 18 % slower than TILED,
 *           superseded by SLAB); the value stays reserved and lsm_set_kernel answers LSM_ERR_UNSUPPORTED;
 *  SLAB     one cooperative launch for all sweeps of a call with the whole lattice resident in the shared memory of
 *           one CTA per SM: slabs of march rows, boundary rows exchanged through self-validating mailbox words in L2, one per
 *           CTA, several half-sweeps per exchange (lsm_set_temporal_depth); L a multiple of 32, 512^2 ... 4096^2,
 *           64^3, 128^3 and every model (Edwards-Anderson up to 2048^2: its bond bytes are resident too), where AUTO
 *           chooses it; also from 128^2 / 32^3 where the small family has no lane kernel (Edwards-Anderson, Potts,
 *           edges that are not powers of two);
 *  BULK     the TILED half-sweep with its rows staged through shared memory by bulk asynchronous copies (TMA unit,
 *           cp.async.bulk + mbarrier; one producer thread per CTA, 4-stage ring) instead of per-thread cp.async: 2D,
 *           L a multiple of 8192, spin-1/2 and North-East.  Opt-in: measured 10 % slower than TILED on 8192^2
 *           (profiles/r2_bulk_copy_variant.md);
 *  GENERIC  one thread per site, any even L >= 4, any table.
 * All families produce bit-identical results (same random-word map D2, same thresholds D3). */
enum { LSM_KERNEL_AUTO = 0, LSM_KERNEL_GENERIC = 1, LSM_KERNEL_TILED = 2, LSM_KERNEL_RESIDENT = 3, LSM_KERNEL_SMALL = 4,
       LSM_KERNEL_SLAB = 5, LSM_KERNEL_BULK = 6 };

/* Device bytes lsm_create needs for this lattice: the two colour arrays and a few hundred bytes of state, plus, where
 * they apply, a second pair of colour arrays (North-East: the random-tile schedule), the bond bytes of both colours
 * (Edwards-Anderson) and the boundary-row mailboxes of the SLAB family (shapes it covers: up to ~10 MB, e.g. 10.5 MB for
 * 128^3, 2.6 MB for 1024^2, which for a 512^2 lattice is several times the lattice itself;
 * lsm_batch_workspace_bytes is R times this plus a descriptor array). */
int lsm_workspace_bytes(int dims, int L, int two_S, int model, size_t *bytes);

/* Build the threshold table on the host (D3), draw the initial state from `seed` on the
 * device (D4: +/-1 uniform; {-1,0,+1} uniform; Bernoulli(c)), compute (B, M), take the
 * reference snapshot (as lsm_reset_reference).  d_workspace: device, >= lsm_workspace_bytes,
 * 256-byte aligned, owned by the caller and must outlive the handle.  Asynchronous on stream. */
int lsm_create(int dims, int L, int two_S, int model, double J, double h, double T, uint64_t seed,
               void *d_workspace, size_t workspace_bytes, void *stream, lsm_t **out);
int lsm_destroy(lsm_t *);

/* n checkerboard sweeps.  Asynchronous.  Observables are evaluated for the
 * last sweep only (they feed lsm_measure). */
int lsm_sweep(lsm_t *, int64_t n, void *stream);
/* n sweeps, writing (B, M) after every sweep to d_obs[k][0..1], k = 0..n-1 (device, int64,
 * 16*n bytes, overwritten).  The sums are fused into the sweep kernels (exact integers). */
int lsm_sweep_record(lsm_t *, int64_t n, int64_t *d_obs, void *stream);
/* Same with a HOST result buffer h_obs[n][2]; the device->host copy is enqueued on stream and
 * the call returns after it completed (synchronises).  d_scratch: device, 16*n bytes. */
int lsm_sweep_record_host(lsm_t *, int64_t n, int64_t *h_obs, int64_t *d_scratch, void *stream);
/* Same without the final synchronisation: the copy into h_obs (pinned host memory) is enqueued on stream; the
 * series is valid once the caller has synchronised it.  For pipelines that keep several steps in flight. */
int lsm_sweep_record_host_async(lsm_t *, int64_t n, int64_t *h_obs, int64_t *d_scratch, void *stream);

/* lsm_sweep_record_host for callers that cannot allocate device memory and therefore cannot bring d_scratch: code that runs
 * inside a host application whose own pool owns all of the GPU's memory and exposes no allocator to plug-ins, a loop with
 * a latency budget that rules out cudaMalloc (it synchronises the whole device), a job whose memory quota is already
 * spent on the lattice.  The (B, M) series is staged in a fixed 64 KiB array that is part of the library image -- every
 * GPU the library is loaded on carries it until the process exits -- so n is limited:
 *  - n > LSM_NOALLOC_MAX_SWEEPS returns LSM_ERR_LIMIT and does nothing (split the run into several calls; the sweep
 *    counter carries on, so the series is the same as that of one long call);
 *  - the call allocates and frees no device memory: no cudaMalloc / cudaFree, no library routine that allocates;
 *  - the first call on each GPU (made with that GPU current, as for every call of this library) looks up the device address
 *    of the array once; make that first call outside any stream capture;
 *  - there is ONE array per GPU, shared by every handle and every host thread, and it still holds the previous call's
 *    series when the next call starts (the call clears the n pairs it uses, on `stream`, before the sweeps add into them).
 *    Two such calls whose GPU work overlaps -- two host threads, or two streams, on the same GPU -- race on it and both
 *    series are garbage: serialise them.  Calls on different GPUs do not interact.
 * Otherwise as lsm_sweep_record_host: h_obs[n][2] on the host (pageable or pinned), bit-identical values, the lattice,
 * workspace and stream remain the caller's, returns after the copy into h_obs completed (synchronises stream). */
enum { LSM_NOALLOC_MAX_SWEEPS = 4096 };
int lsm_sweep_record_host_noalloc(lsm_t *, int64_t n, int64_t *h_obs, void *stream);

/* North-East model only: n sweeps of the paper's "corrected algorithm" (steps 3-10) instead of
 * the checkerboard sweep, which the paper rejects for relaxation dynamics.  The lattice is
 * divided into tiles of tile_edge x tile_edge spins (P = tile_edge^2); a sweep is two launches; in each, every
 * tile is handled once: lambda threads pick lambda of its spins at random and update them (rule of the handle's
 * model), synchronise, q times with q * lambda = P/2.  Readings D17-D21: tile boundaries (upper and
 * right, Fig. 4) are those of the launch start; the picks of a sub-step read the tile as the sub-step found it;
 * on a same-site collision the highest thread wins; Philox counter (tile, sub-step * ceil(lambda/2) + thread/2,
 * sweep, 4 + launch).  d_obs: NULL, or device [n][2] receiving (0, M) after every sweep.  Asynchronous.
 * UNSUPPORTED unless tile_edge is a power of two in [8, 128] dividing L, lambda a power of two in [1, 32] and
 * 2 * lambda divides P.  tile_edge = L with lambda = 1 is the serial limit Q = lambda = 1 of PAPER.md:142 (one thread
 * updates the whole lattice: slow by construction).  Shares the sweep counter with lsm_sweep. */
int lsm_sweep_random_tile(lsm_t *, int64_t n, int tile_edge, int lambda, int64_t *d_obs, void *stream);
/* Its balance-preserving variant ("~2.5x slower"): a sub-step is lambda picks among the tile's red
 * sites, a barrier, lambda picks among its white sites, a barrier; four launches complete one MC step.  Readings
 * D22-D24: red / white = checkerboard colours (x+y)&1 = 0 / 1; q * 2 lambda = P/4 per launch, so a step attempts P
 * updates per tile; one Philox call per thread and sub-step, counter (tile, sub-step * lambda + thread, sweep,
 * 8 + launch), words 0, 1 = red pick, 2, 3 = white pick; position r = floor(w P/2 / 2^32) = r-th site of the colour
 * in row-major order.  UNSUPPORTED unless additionally 8 * lambda divides P. */
int lsm_sweep_random_tile_balanced(lsm_t *, int64_t n, int tile_edge, int lambda, int64_t *d_obs, void *stream);

/* ---- Batches: many small lattices in one launch.
 * The paper's own lattices are 32^2 ... 512^2 and it runs them one at a time -- 31 temperatures of the Fig. 6 ramp
 * (PAPER.md:196), 30 realisations per concentration for Fig. 7 -- reporting that such lattices cannot keep
 * a GPU busy ("not enough threads to execute between memory access operations").  A batch holds R independent
 * lattices of one shape (dims, L, two_S, model, J, h) with per-replica temperature T[r] and seed seeds[r] (host arrays of
 * R).  lsm_batch_sweep[_record] advances all of them by n checkerboard sweeps with ONE kernel launch per 256 replicas
 * (one thread-block cluster per replica, the lattice in shared memory for the whole call) whenever L is a power of two
 * >= 8 with at most 2^20 sites and no table has a "never" entry; otherwise the replicas are swept one after the other
 * on the same stream.  Either way replica r ends exactly as a single handle created with (T[r], seeds[r]) would: same
 * Philox key, same table, bit-identical.
 *  - workspace: device, >= lsm_batch_workspace_bytes, 256-byte aligned, owned by the caller, must outlive the batch.
 *  - d_obs: device int64 [R][n][2] = (B, M) of replica r after sweep k (overwritten).
 *  - lsm_batch_replica lends the handle of replica r (valid until lsm_batch_destroy; do NOT lsm_destroy it) for
 *    lsm_get_spins, lsm_set_spins, lsm_persistence, lsm_measure*, lsm_get_thresholds, ...  The batch sweeps in lockstep:
 *    LSM_ERR_STATE if the replicas' sweep counters differ (one of them was swept on its own).
 *  - lsm_batch_measure_int: running (B, M) of every replica into host arrays of R (either may be NULL); synchronises once.
 *  - lsm_batch_set_cluster: thread blocks per replica (power of two <= 16, 0 = automatic: about one block per SM). */
int lsm_batch_workspace_bytes(int R, int dims, int L, int two_S, int model, size_t *bytes);
int lsm_batch_create(int R, int dims, int L, int two_S, int model, double J, double h, const double *T,
                     const uint64_t *seeds, void *d_workspace, size_t workspace_bytes, void *stream, lsm_batch_t **out);
int lsm_batch_destroy(lsm_batch_t *);
int lsm_batch_size(lsm_batch_t *, int *R);
int lsm_batch_replica(lsm_batch_t *, int r, lsm_t **borrowed_handle);
int lsm_batch_sweep(lsm_batch_t *, int64_t n, void *stream);
int lsm_batch_sweep_record(lsm_batch_t *, int64_t n, int64_t *d_obs, void *stream);
/* North-East batches: n sweeps of lsm_sweep_random_tile (balanced = 0) or lsm_sweep_random_tile_balanced (balanced != 0) on
 * every replica, each launch of the schedule covering the tiles of ALL replicas -- the paper averages 30 realisations of
 * 128^2 and 512^2 lattices per concentration, and one 128^2 lattice is 16 tiles = one thread block.
 * Same arguments and restrictions as the single-lattice calls; d_obs: NULL, or device int64 [R][n][2] = (0, M) of replica r
 * after sweep k.  Replica r ends bit-identical to a single handle swept with the same call.  LSM_ERR_STATE if the replicas'
 * sweep counters or tracking states differ.  Asynchronous. */
int lsm_batch_sweep_random_tile(lsm_batch_t *, int64_t n, int tile_edge, int lambda, int balanced, int64_t *d_obs, void *stream);
int lsm_batch_set_temperatures(lsm_batch_t *, const double *T);
int lsm_batch_set_tracking(lsm_batch_t *, int on, void *stream);
int lsm_batch_set_cluster(lsm_batch_t *, int blocks_per_replica);
int lsm_batch_measure_int(lsm_batch_t *, int64_t *bond_sum, int64_t *M);
int lsm_batch_get_launch_count(lsm_batch_t *, uint64_t *kernels_launched);

/* Running observables of the current configuration (synchronises). */
int lsm_measure(lsm_t *, double *E, int64_t *M);
int lsm_measure_int(lsm_t *, int64_t *bond_sum, int64_t *M, uint64_t *sweeps_done);
/* Recompute (B, M) from scratch with the full reduction kernel (synchronises); also refreshes
 * the running values.  Must equal lsm_measure_int at any time. */
int lsm_measure_full(lsm_t *, int64_t *bond_sum, int64_t *M);

/* never_changed = #{i: the value of site i never differed from its predecessor since the
 * reference time} (persistence, D12); overlap = sum_i sigma_i(ref) sigma_i(now), sigma = s
 * (Ising) or 2n-1 (NE) (numerator of PAPER.md:120 Eq. 4, D11).  Synchronises.
 * LSM_ERR_STATE if tracking is off. */
int lsm_persistence(lsm_t *, int64_t *never_changed, int64_t *overlap);
/* Reference snapshot := current configuration, "ever changed" flags cleared, tracking on. */
int lsm_reset_reference(lsm_t *, void *stream);
/* on = 0: stop tracking (flags and snapshot dropped; sweeps get slightly cheaper);
 * on = 1: same as lsm_reset_reference.  Tracking is ON after lsm_create. */
int lsm_set_tracking(lsm_t *, int on, void *stream);

/* Configuration in canonical order, N int8 values. */
int lsm_get_spins(lsm_t *, int8_t *d_out, void *stream);
int lsm_get_spins_host(lsm_t *, int8_t *h_out, int8_t *d_scratch /* N bytes */, void *stream);
/* Replace configuration and sweep counter (LSM_ERR_ARG unless sweep_counter < 2^60), recompute (B, M);
 * snapshot and flags untouched.
 * Values outside the model's set are not an error: the conversion maps every byte into the set (Ising spin-1/2 and EA:
 * > 0 -> +1, else -1; spin-1: clamped to [-1, +1]; North-East: non-zero -> 1; Potts: clamped to [0, q-1]), so no input
 * can corrupt the packed neighbour sums or the flag bits.  LSM_ERR_ARG for NULL. */
int lsm_set_spins(lsm_t *, const int8_t *d_in, uint64_t sweep_counter, void *stream);
int lsm_set_spins_host(lsm_t *, const int8_t *h_in, int8_t *d_scratch /* N bytes */,
                       uint64_t sweep_counter, void *stream);
/* Upload only: h_in (host, N int8, pinned for a truly asynchronous copy) -> d_stage (device, N bytes) on copy_stream,
 * without touching the lattice.  Lets the upload of the next configuration overlap the sweeps of the current one:
 * stage on a copy stream, order the streams with an event, then lsm_set_spins(d_stage, ...) on the compute stream. */
int lsm_stage_spins_host(lsm_t *, const int8_t *h_in, int8_t *d_stage, void *copy_stream);

/* LSM_EA only (else UNSUPPORTED): bond signs in canonical form, d_tau int8 [dims][N] on the device, tau[a][i] = sign
 * (+1 ferro, -1 antiferro) of the bond between site i and its neighbour in direction +a (a = 0, 1, 2 = x, y, z).
 * lsm_set_bonds replaces them (values < 0 are antiferromagnetic) and recomputes (B, M). */
int lsm_set_bonds(lsm_t *, const int8_t *d_tau, void *stream);
int lsm_get_bonds(lsm_t *, int8_t *d_tau, void *stream);

int lsm_set_temperature(lsm_t *, double T); /* rebuilds the thresholds (host, D3) */
/* Host copy of the 33-bit thresholds, in the canonical order:
 *  Ising two_S=1: idx = b*(2d+1) + (nn+2d)/2, b=(s+1)/2                         [2(2d+1)]
 *  Ising two_S=2: idx = ((s+1)*2 + kk)*(4d+1) + (nn+2d), proposal (s+1+1+kk)%3  [6(4d+1)]
 *  NE: {floor(c*2^32), floor(exp(-1/T)*2^32), 2^32}                              [3]
 *  EA: as Ising two_S=1 with nn = sum_j tau_ij s_j                                [2(2d+1)]
 *  Potts: idx = (n_new - n_old) + 2d                                              [4d+1]
 * out may be NULL to query count.  out must hold 128 entries. */
int lsm_get_thresholds(lsm_t *, uint64_t *out, int *count);

int lsm_set_kernel(lsm_t *, int kernel_family);           /* LSM_KERNEL_*; UNSUPPORTED if it cannot run this lattice */
int lsm_get_kernel(lsm_t *, int *kernel_family_in_use);
/* Temporal blocking of the SLAB family (the barrier between the colours is
 * what small lattices cannot afford): `depth` half-sweeps run between two exchanges of boundary rows, each slab
 * updating depth-1-j halo rows on either side redundantly in step j (reproducible: the random words are a function
 * of (seed, sweep, colour, site), D2).  0 = the default for the shape; 1 = no redundant update; at most 4 (L <= 1024),
 * 2 (L = 2048), 1 (otherwise): UNSUPPORTED beyond.  Results do not depend on it.  get: depth in use (0 unless SLAB). */
int lsm_set_temporal_depth(lsm_t *, int depth);
int lsm_get_temporal_depth(lsm_t *, int *depth_in_use);
int lsm_get_launch_count(lsm_t *, uint64_t *kernels_launched); /* kernels this handle has enqueued */

/* Host-side derived doubles from the integer series (D11-D13), exact integer accumulation. */
int lsm_binder_u4(const int64_t *obs /* [n][2] host */, int64_t n, double *U4);   /* 1 - <M^4>/(3<M^2>^2) */
int lsm_heat_capacity(const int64_t *obs, int64_t n, int64_t N, double J, double h, double T, double *C_per_site);
/* Per-site means of a recorded series: e = <E>/N with E = -J*B - h*M (D1), abs_m = <|M|>/N (the
 * energy and magnetisation curves of Fig. 6).  Either out-pointer may be NULL. */
int lsm_series_means(const int64_t *obs, int64_t n, int64_t N, double J, double h, double *e_per_site, double *abs_m_per_site);
int lsm_phi(int64_t overlap, int64_t N, double c, double *phi);                  /* PAPER.md:120 Eq. 4, D11 */
int lsm_persistence_fraction(int64_t never_changed, int64_t N, double *P);
int lsm_energy(int model, double J, double h, int64_t bond_sum, int64_t M, double *E);

/* Test hooks.  lsm_philox_device: run the kernels' Philox4x32-10 on the device for n (counter, key)
 * pairs: d_ctr_key[n][6] -> d_out[n][4] (uint32, device).  lsm_philox_throughput: register-only
 * Philox microbenchmark (integer roofline): every thread of `blocks` x 256 runs `calls` dependent
 * calls and writes one word to d_sink[blocks*256]. */
int lsm_philox_device(const uint32_t *d_ctr_key, uint32_t *d_out, int64_t n, void *stream);
int lsm_philox_throughput(int blocks, int calls, uint32_t *d_sink, void *stream);

const char *lsm_strerror(int code);
const char *lsm_last_cuda_error(void);

#ifdef __cplusplus
}
#endif
#endif /* LSM_H */
