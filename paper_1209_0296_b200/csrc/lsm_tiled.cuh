// lsm_tiled.cuh -- the vectorised kernel family: 16 sites per 128-bit word, byte-parallel neighbour
// sums, whole Philox calls per 32-bit lane of the word, register marching along the slowest axis.
// Declarations shared with lsm_api.cu.
#pragma once
#include "lsm_internal.cuh"

namespace lsmk {

// Threshold tables in the form the vectorised kernels index.  Built on the host from the canonical
// 33-bit table (lsm_get_thresholds order), so both families accept exactly the same (w, state) pairs.
struct TiledTables {
    int usable;            // 0: this table is left to the scalar family
    int has_never;         // some entry has thr = 0: only the tiled family's two-compare (NEV) kernels can run it
    // spin-1/2 (and EA): t32[n + 8*b] = thr - 1 (accept iff w <= t32), b = (s+1)/2, n = up-neighbour count.
    //   A thr = 0 ("never") entry has no such form: t32 = 0 and y32 = 1 there (accept iff y32 <= w <= t32), else y32 = 0.
    uint32_t t32[16];
    uint32_t y32[64];      // lower bounds, indexed like t32 (spin-1/2, EA) or like s1 (spin-1)
    // NE: [0] heat-bath / init threshold, [1] Metropolis 0->1 threshold (32-bit clipped) + flag
    uint32_t ne_t32[2];
    int ne_up_always;
    int ne_all4;           // up-concentration >= 0.15: the vectorised rule runs the four Philox calls of a word together
    // spin-1: s1[16*dcode + sum] = thr - 1 (accept iff w1 <= s1), dcode = class of s' - s: 0: +1, 1: +2, 2: -1, 3: -2;
    //   sum = sum of the neighbours' a = s + 1.  The threshold depends on (s' - s, sum) only (reading D3).
    uint32_t s1[64];
};

void build_tiled_tables(int model, int dims, double J, double h, const uint64_t *thr, int nthr, TiledTables *out);
bool tiled_supported(const Lat &lat, int model, const TiledTables &t);
cudaError_t launch_sweep_tiled(const SweepArgs &a, const TiledTables &t, cudaStream_t s);
// the same half-sweep with its rows staged through shared memory by bulk copies (lsm_tiled_bulk.cu; SweepArgs::bulk)
bool tiled_bulk_supported(const Lat &lat, int model, const TiledTables &t);

// The resident family (one cooperative launch with neighbour-flag synchronisation) was removed in round 3: it measured
// 18 % slower than the tiled family and is superseded by the slab family.  Its 2048 flag words stay reserved in the state
// block of the workspace so that the layout (and lsm_workspace_bytes) does not change.
constexpr int RESIDENT_MAX_CTAS = 2048;

// Small family (lsm_small.cu): one thread block owns the whole lattice and runs `nsweeps` sweeps in one
// launch, __syncthreads() between the colours.  Chosen automatically up to LSM_SMALL_MAX_SITES sites.
struct SmallPlan { int S, threads, lane, cluster; };   // lane = 1: 32-bit lanes per thread, `cluster` thread blocks
bool small_plan(const Lat &lat, int model, const TiledTables &t, SmallPlan *out, bool ignore_size_limit);
cudaError_t launch_sweep_small(const Lat &lat, int model, int track, unsigned long long seed, unsigned long long t0,
                               int nsweeps, long long *d_obs, const SmallPlan &plan, const TiledTables &t,
                               cudaStream_t s);

// Slab family (lsm_slab.cu): one cooperative launch runs `nsweeps` whole sweeps with the lattice resident in the
// shared memory of G CTAs (one per SM); boundary rows travel through self-validating mailbox words in L2.
struct SlabPlan { int G, rows_max, threads, smem, D, dmax, early; uint32_t magic_wrow, magic_wpr; };   // D: temporal depth (half-sweeps per exchange)
constexpr int SLAB_MAX_CTAS = 160;                                   // mailbox rows reserved in the workspace
size_t slab_mailbox_bytes(int dims, int L, int model);               // internal Model id; 0: shape not covered
int slab_depth_max(int dims, int L, int model);                      // largest temporal depth of this shape
bool slab_plan(const Lat &lat, int model, const TiledTables &t, int depth, SlabPlan *out);   // depth 0: default
cudaError_t launch_sweep_slab(const Lat &lat, int model, int track, unsigned long long seed, unsigned long long t0,
                              int nsweeps, long long *d_obs, uint32_t *d_mbox, const SlabPlan &plan, const TiledTables &t,
                              cudaStream_t s);

// Batch of R same-shape lattices (lsm_batch_*): one launch of the small family's lane kernel, one cluster per replica.
struct BatchDesc {               // per replica, in device memory
    uint8_t *col[2];
    long long *run;              // the replica's running (B, M) pair
    uint32_t ne_t32;
    int ne_always;
    uint32_t tab[64];            // HalfTab (16) or OneTab (64) of the replica's temperature
};
bool small_batch_supported(const Lat &lat, int model, const TiledTables &t);
int small_batch_cluster(const Lat &lat, int R);                          // blocks per replica for R replicas
cudaError_t launch_sweep_small_batch(const Lat &lat, int model, int track, const BatchDesc *d_desc, const uint64_t *seeds,
                                     int R, int cluster, unsigned long long t0, int nsweeps, long long *d_obs,
                                     long long obs_stride, int write_run, cudaStream_t s);

}  // namespace lsmk
