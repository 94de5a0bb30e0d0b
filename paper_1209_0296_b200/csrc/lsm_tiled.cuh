// lsm_tiled.cuh -- the vectorised kernel family (16 sites per 128-bit word, byte-parallel neighbour
// sums, whole Philox calls per word); declarations shared with lsm_api.cu.
#pragma once
#include "lsm_internal.cuh"

namespace lsmk {

// Threshold tables in the form the tiled kernels index (built on the host from the canonical
// 33-bit table, so both families accept exactly the same (w, state) pairs).
struct TiledTables {
    int usable;                 // 0: this (model, J, h) combination is left to the generic family
    uint32_t t32[96];           // thr clipped to 32 bits (2^32 -> 0xFFFFFFFF); "always" handled apart
    uint32_t always_le[4];      // per current value: accept with certainty iff aligned count <= this
};

void build_tiled_tables(int model, int dims, double J, double h, const uint64_t *thr, int nthr, TiledTables *out);
bool tiled_supported(const Lat &lat, int model, const TiledTables &t);
cudaError_t launch_sweep_tiled(const SweepArgs &a, const TiledTables &t, cudaStream_t s);

}  // namespace lsmk
