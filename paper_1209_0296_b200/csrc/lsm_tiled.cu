// lsm_tiled.cu -- placeholder until the vectorised kernels land: reports "unsupported" so that the
// dispatcher stays on the scalar family.
#include "lsm_tiled.cuh"

namespace lsmk {
void build_tiled_tables(int, int, double, double, const uint64_t *, int, TiledTables *out) { out->usable = 0; }
bool tiled_supported(const Lat &, int, const TiledTables &) { return false; }
cudaError_t launch_sweep_tiled(const SweepArgs &, const TiledTables &, cudaStream_t) { return cudaErrorNotSupported; }
}  // namespace lsmk
