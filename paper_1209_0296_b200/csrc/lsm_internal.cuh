// lsm_internal.cuh -- shared declarations of the CUDA path (private to liblsm).
// Nothing here is shared with oracle/ (the CPU oracle has its own Philox, tables and geometry).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace lsmk {

// ------------------------------------------------------------------------------------------
// Device-internal byte encoding of one site (private; the ABI speaks int8 spin values).
//   spin-1/2 and NE : bit0 = value (b = (s+1)/2 or n), bit3 = "ever changed", bit4 = reference value
//   spin-1          : bits[1:0] = a = s+1,            bit4 = "ever changed", bits[6:5] = reference a
// With tracking off the upper bits are zero, so neighbour words can be summed without masking.
// Flag bits of spin-1/2 sit at 8/16 so that even six flagged neighbours sum without a carry into
// the next byte (6*25 = 150 < 256) and one AND with 0x07 recovers the neighbour count.
// ------------------------------------------------------------------------------------------
//   EA (+/-J bonds) : as spin-1/2; the bond signs live in two more colour arrays (Lat::bnd), one byte per site:
//                     bit k set = the bond to neighbour k is antiferromagnetic, k = 0: x-1, 1: x+1, 2: y-1, 3: y+1,
//                     4: z-1, 5: z+1 (each bond is stored at both of its ends)
//   Potts (q <= 8)  : bits[2:0] = state, bit3 = "ever changed", bits[6:4] = reference state
enum Model : int { M_ISING_HALF = 0, M_ISING_ONE = 1, M_NE_HEATBATH = 2, M_NE_METROPOLIS = 3, M_EA = 4, M_POTTS = 5 };

template <int MODEL> struct Enc {
    static constexpr uint32_t VAL = 0x01, CHG = 0x08, REF = 0x10;
    static constexpr int REF_SHIFT = 4;
};
template <> struct Enc<M_ISING_ONE> {
    static constexpr uint32_t VAL = 0x03, CHG = 0x10, REF = 0x60;
    static constexpr int REF_SHIFT = 5;
};
template <> struct Enc<M_POTTS> {
    static constexpr uint32_t VAL = 0x07, CHG = 0x08, REF = 0x70;
    static constexpr int REF_SHIFT = 4;
};

// Lattice view handed to every kernel by value.
struct Lat {
    uint8_t *col[2];     // colour (parity) arrays, N/2 bytes each, [z][y][m], x = 2m + ((y+z+colour)&1)
    int L, Lh, dims;     // Lh = L/2 bytes per compact row
    int Lz;              // L for 3D, 1 for 2D
    long long half;      // N/2
    uint8_t *bnd[2];     // M_EA: bond bytes of the two colours (same geometry as col); else nullptr
    int q;               // M_POTTS: number of states; else 0
};

// 33-bit thresholds in the canonical order of lsm_get_thresholds (include/lsm.h).
struct Thr64 { unsigned long long thr[96]; int count; };

// ------------------------------------------------------------------------------------------
// Philox4x32-10 (reading D2).  The 32x32->64 products compile to IMAD.WIDE.U32.
// ------------------------------------------------------------------------------------------
constexpr uint32_t PHILOX_M0 = 0xD2511F53u, PHILOX_M1 = 0xCD9E8D57u;
constexpr uint32_t PHILOX_W0 = 0x9E3779B9u, PHILOX_W1 = 0xBB67AE85u;

__device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                               uint32_t k0, uint32_t k1)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        unsigned long long p0 = (unsigned long long)PHILOX_M0 * c0;
        unsigned long long p1 = (unsigned long long)PHILOX_M1 * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        c1 = (uint32_t)p1;
        c3 = (uint32_t)p0;
        c0 = n0;
        c2 = n2;
        k0 += PHILOX_W0;
        k1 += PHILOX_W1;
    }
    return make_uint4(c0, c1, c2, c3);
}

// Counter fields of reading D2: c0/c1 = group, c2 = lo32(t), c3 = stream | hi32(t) << 4 (tag in the low 4 bits, t < 2^60).
struct SweepKey {
    uint32_t k0, k1;   // seed
    uint32_t c2, c3;   // sweep and stream tag of this half-sweep
};
__host__ __device__ inline SweepKey make_sweep_key(unsigned long long seed, unsigned long long t, uint32_t stream)
{
    SweepKey k;
    k.k0 = (uint32_t)seed;
    k.k1 = (uint32_t)(seed >> 32);
    k.c2 = (uint32_t)t;
    k.c3 = stream | ((uint32_t)(t >> 32) << 4);
    return k;
}

// ------------------------------------------------------------------------------------------
// Reductions: warp shuffle, then one 64-bit atomic per CTA.
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ long long warp_sum(long long v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ int warp_sum(int v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Sum two per-thread values over the CTA and add them to out[0], out[1] (either may be skipped).
__device__ __forceinline__ void block_accumulate2(long long a, long long b, long long *out, bool do_a, bool do_b)
{
    __shared__ long long red[2][32];
    a = warp_sum(a);
    b = warp_sum(b);
    int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
    if (lane == 0) { red[0][w] = a; red[1][w] = b; }
    __syncthreads();
    if (w == 0) {
        a = lane < nw ? red[0][lane] : 0;
        b = lane < nw ? red[1][lane] : 0;
        a = warp_sum(a);
        b = warp_sum(b);
        if (lane == 0) {
            if (do_a && a != 0) atomicAdd((unsigned long long *)&out[0], (unsigned long long)a);
            if (do_b && b != 0) atomicAdd((unsigned long long *)&out[1], (unsigned long long)b);
        }
    }
    __syncthreads();
}

// Same, with the caller's shared scratch (blockDim.x <= 256).
__device__ __forceinline__ void block_accumulate2_in(long long (*red)[8], long long a, long long b, long long *out,
                                                     bool do_a, bool do_b)
{
    a = warp_sum(a);
    b = warp_sum(b);
    int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
    if (lane == 0) { red[0][w] = a; red[1][w] = b; }
    __syncthreads();
    if (w == 0) {
        a = lane < nw ? red[0][lane & 7] : 0;
        b = lane < nw ? red[1][lane & 7] : 0;
        a = warp_sum(a);
        b = warp_sum(b);
        if (lane == 0) {
            if (do_a && a != 0) atomicAdd((unsigned long long *)&out[0], (unsigned long long)a);
            if (do_b && b != 0) atomicAdd((unsigned long long *)&out[1], (unsigned long long)b);
        }
    }
}

// ------------------------------------------------------------------------------------------
// Launchers implemented in the .cu files (host side, enqueue only; return cudaError_t).
// ------------------------------------------------------------------------------------------
struct SweepArgs {
    Lat lat;
    int model;             // Model
    int half;              // parity updated by this launch
    SweepKey key;
    int track;             // maintain "ever changed" bits
    long long *obs;        // device (B, M) accumulator of this sweep, or nullptr
    int want_B;            // add the bond sum (only meaningful after the second half)
    int bulk;              // tiled family: rows staged by bulk copies (lsm_tiled_bulk.cu; LSM_KERNEL_BULK)
};

cudaError_t launch_init(const Lat &lat, int model, unsigned long long seed, unsigned long long thr_c,
                        cudaStream_t s);
cudaError_t launch_sweep_generic(const SweepArgs &a, const Thr64 &thr, cudaStream_t s);
cudaError_t launch_measure_full(const Lat &lat, int model, long long *d_BM, cudaStream_t s);
cudaError_t launch_persistence(const Lat &lat, int model, long long *d_out2, cudaStream_t s);
cudaError_t launch_reset_reference(const Lat &lat, int model, int tracking_on, cudaStream_t s);
cudaError_t launch_get_spins(const Lat &lat, int model, int8_t *d_out, cudaStream_t s);
cudaError_t launch_set_spins(const Lat &lat, int model, const int8_t *d_in, cudaStream_t s);
// Edwards-Anderson bonds (reading D25; lsm_wider.cu): canonical int8 tau[dims][N] <-> the per-site bond bytes.
cudaError_t launch_ea_bonds_init(const Lat &lat, unsigned long long seed, cudaStream_t s);
cudaError_t launch_ea_set_bonds(const Lat &lat, const int8_t *d_tau, cudaStream_t s);
cudaError_t launch_ea_get_bonds(const Lat &lat, int8_t *d_tau, cudaStream_t s);
cudaError_t launch_philox_device(const uint32_t *d_ck, uint32_t *d_out, long long n, cudaStream_t s);
cudaError_t launch_philox_throughput(int blocks, int calls, uint32_t *d_sink, cudaStream_t s);

// North-East random-tile schedule (lsm_ne_tile.cu): reads lat.col, writes dst.
bool ne_tile_supported(const Lat &lat, int b, int lam, bool balanced);
cudaError_t launch_ne_random_tile(const Lat &lat, uint8_t *const dst[2], bool metropolis, bool balanced, int b, int lam,
                                  unsigned long long seed, unsigned long long t, int launch, uint32_t thr_c,
                                  uint32_t thr_up, int up_always, int track, long long *obs, cudaStream_t s);

// Batch form (lsm_batch_sweep_random_tile): one descriptor per lattice and launch direction, in device memory.
struct NeBatchDesc {
    const uint8_t *src[2];   // lattice at launch start
    uint8_t *dst[2];         // lattice after the launch
    long long *obs;          // base of the lattice's (B, M) slots (a recorded series or the running pair)
    uint32_t k0, k1;         // Philox key = the lattice's seed
    uint32_t thr_c, thr_up;  // its thresholds
    int up_always;
    int pad;
};
cudaError_t launch_ne_random_tile_batch(const Lat &lat, const NeBatchDesc *d_desc, int R, bool metropolis, bool balanced, int b,
                                        int lam, unsigned long long t, int launch, int track, long long obs_off, cudaStream_t s);

int sm_count();

}  // namespace lsmk
