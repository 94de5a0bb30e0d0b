// lsm_tiled.cuh -- the vectorised kernel family: 16 sites per 128-bit word, byte-parallel neighbour
// sums, whole Philox calls per 32-bit lane of the word, register marching along the slowest axis.
// Declarations shared with lsm_api.cu.
#pragma once
#include "lsm_internal.cuh"

namespace lsmk {

// Threshold tables in the form the vectorised kernels index.  Built on the host from the canonical
// 33-bit table (lsm_get_thresholds order), so both families accept exactly the same (w, state) pairs.
struct TiledTables {
    int usable;            // 0: this (model, J, h) combination is left to the scalar family
    int field;             // spin-1/2: h != 0, the table row depends on the spin value
    // spin-1/2: idx = a + 8*b, a = number of neighbours aligned with the spin, b = (s+1)/2.
    //   t32 = thr clipped to 32 bits; acceptance with certainty (thr = 2^32) is the byte-parallel
    //   test a < always_below[b] (dE = 4J(a-d) +- 2h is increasing in a for J > 0).
    uint32_t t32[16];
    uint32_t always_below[2];
    // NE: [0] heat-bath / init threshold, [1] Metropolis 0->1 threshold (32-bit clipped) + flag
    uint32_t ne_t32[2];
    int ne_up_always;
    // spin-1: entry[(a*2+kk)*16 + sum] = { t32, proposed a' | always << 4 }
    uint2 s1[96];
};

void build_tiled_tables(int model, int dims, double J, double h, const uint64_t *thr, int nthr, TiledTables *out);
bool tiled_supported(const Lat &lat, int model, const TiledTables &t);
cudaError_t launch_sweep_tiled(const SweepArgs &a, const TiledTables &t, cudaStream_t s);

}  // namespace lsmk
