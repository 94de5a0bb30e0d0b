// lsm_ne_tile.cu -- the paper's "corrected algorithm" for the North-East model (steps 3-10):
// the lattice is divided into Q tiles of P = b*b spins; in each of the two launches of a sweep every tile is
// handled once: it is copied with its upper and right boundaries (Fig. 4) into shared memory, lambda threads pick
// lambda spins of the tile at random and update them, synchronise, q times with q*lambda = P/2, and the tile is
// copied back.  Readings D17-D21 make the result unique so that it can be bit-exact against the CPU
// oracle: boundaries are those of the launch start (the kernel reads one lattice buffer and writes the other),
// the lambda picks of a sub-step read the tile as the sub-step found it, and on a same-site collision the
// highest thread wins.
//
// B200 mapping: a group of lambda lanes of a warp owns a tile (lambda = 16: two tiles per warp), so steps 6-7 --
// pick, synchronise -- are warp-level (bar.warp.sync is the barrier; collisions are found through claim bytes in
// shared memory, MATCH.ANY only when one was seen) and a CTA keeps 256/lambda tiles in flight.  The tile sits in
// shared memory in the lattice's own split-colour layout (two arrays of (b+1) rows x b/2 bytes plus the east
// boundary column), loaded with cp.async and written back in 16-byte words.
// Random words: one Philox4x32-10 call serves two picks (position and acceptance word each); over two consecutive
// sub-steps each lane of a pair computes one of the pair's two calls and hands two words to its partner by shuffle.
// The balance-preserving variant (readings D22-D24) is the BAL instantiation of the same kernel.
#include "lsm_internal.cuh"

#include <cstring>

namespace lsmk {

struct NeTileArgs {
    const uint8_t *src[2];   // lattice at launch start (colour arrays)
    uint8_t *dst[2];         // lattice after the launch
    int L, Lh;               // Lh = L/2 bytes per compact row
    int lg_b, lg_lam;        // tile edge and lambda are powers of two
    int ntx;                 // tiles per lattice row
    int ntiles;
    int gpw;                 // tile groups of a warp that hold a tile (<= 32 / lambda; fewer when tiles are large)
    uint32_t k0, k1, c2, c3; // Philox key and the (sweep, launch) fields of the counter
    uint32_t rk0[10], rk1[10];   // round keys k0 + r W0, k1 + r W1 (kernel-parameter bank: operands of the round's LOP3)
    uint32_t thr_c, thr_up;  // floor(c 2^32), floor(exp(-1/T) 2^32) clipped to 32 bits
    int up_always;           // Metropolis: exp(-1/T) rounds to 2^32
    int track;
    long long *obs;          // (B, M) slot receiving the up-count after the launch, or nullptr
    // BATCH instantiations (lsm_batch_sweep_random_tile): R lattices of this shape in one launch, tile index
    // rep * ntiles + T.  Buffers, key, thresholds and the observable slot come from desc[rep]; obs_off is the offset (in
    // int64) of this launch's (B, M) slot behind desc[rep].obs, or -1 for a launch that records nothing.
    const NeBatchDesc *desc;
    int R;
    long long obs_off;
};

__device__ __forceinline__ uint32_t lds_u8(uint32_t a)
{
    uint32_t v;
    asm volatile("ld.shared.u8 %0, [%1];" : "=r"(v) : "r"(a) : "memory");
    return v;
}
__device__ __forceinline__ void sts_u8(uint32_t a, uint32_t v)
{
    asm volatile("st.shared.u8 [%0], %1;" ::"r"(a), "r"(v) : "memory");
}

// The same with the key in registers (batch: every lattice has its own seed): two more additions per round.
__device__ __forceinline__ uint4 philox_k(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1)
{
    return philox4x32_10(c0, c1, c2, c3, k0, k1);
}

// Philox4x32-10 on counter (c0, c1, a.c2, a.c3) with the round keys read from the kernel parameters.
__device__ __forceinline__ uint4 philox_rk(uint32_t c0, uint32_t c1, const NeTileArgs &a)
{
    uint32_t c2 = a.c2, c3 = a.c3;
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const unsigned long long p0 = (unsigned long long)PHILOX_M0 * c0, p1 = (unsigned long long)PHILOX_M1 * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ a.rk0[r], n2 = (uint32_t)(p0 >> 32) ^ c3 ^ a.rk1[r];
        c1 = (uint32_t)p1;
        c3 = (uint32_t)p0;
        c0 = n0;
        c2 = n2;
    }
    return make_uint4(c0, c1, c2, c3);
}

#define LSM_NE_TILE_MINBLOCKS 4
template <bool METRO, bool BAL, bool BATCH = false>
__global__ void __launch_bounds__(256, LSM_NE_TILE_MINBLOCKS)
k_ne_random_tile(const __grid_constant__ NeTileArgs a)
{
    extern __shared__ __align__(16) uint8_t s_tiles[];
    const int b = 1 << a.lg_b, lam = 1 << a.lg_lam, P = b * b;
    const int lane = threadIdx.x & 31, j = lane & (lam - 1);          // j: thread index within the tile's group
    // A warp has 32 / lambda groups of lambda lanes; the first a.gpw of them own a tile at a time (all of them unless
    // the tiles are too large for shared memory: 128 x 128 tiles with lambda <= 4, the serial limit Q = lambda = 1 of
    // PAPER.md:142 on a 128^2 lattice).  The other groups idle: they run the same instructions on the last group's tile
    // but write nothing.
    const int grp_in_warp = lane >> a.lg_lam, grp_per_warp = a.gpw;
    const bool has_tile = grp_in_warp < grp_per_warp;
    const int warp_global = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int nwarps = (gridDim.x * blockDim.x) >> 5;
    const int rowb = b >> 1;                                          // bytes per tile row and colour
    const int col_bytes = (b + 1) * rowb;                             // rows 0..b (row b = north boundary)
    const int tile_bytes = (2 * col_bytes + b + (lam > 1 ? P : 0) + 15) & ~15;   // + east column + claim bytes
    uint8_t *const tile = s_tiles + (size_t)((threadIdx.x >> 5) * grp_per_warp + (has_tile ? grp_in_warp : grp_per_warp - 1)) * tile_bytes;
    uint8_t *const east = tile + 2 * col_bytes;
    // 32-bit shared-space addresses for the pick loop (no generic-address conversion per access)
    const uint32_t s_tile = (uint32_t)__cvta_generic_to_shared(tile), s_east = s_tile + 2u * (uint32_t)col_bytes,
                   s_claim = s_east + (uint32_t)b;
    const uint32_t chg = a.track ? 0x08u : 0u;
    uint32_t thr_c = a.thr_c, thr_up = a.thr_up;
    bool up_always = a.up_always != 0;
    const int ntiles_all = BATCH ? a.ntiles * a.R : a.ntiles;
    const uint8_t *src0 = a.src[0], *src1 = a.src[1];
    uint8_t *dst0 = a.dst[0], *dst1 = a.dst[1];
    uint32_t bk0 = 0u, bk1 = 0u;                                      // BATCH: Philox key of the tile's lattice
    long long *bobs = nullptr;
    const int q = BAL ? P >> (a.lg_lam + 3) : P >> (a.lg_lam + 1), calls = (lam + 1) >> 1;   // D23 / D17
    int ups = 0;

    for (int base = warp_global * grp_per_warp; base < ntiles_all; base += nwarps * grp_per_warp) {
        int T = base + grp_in_warp;
        const bool live = has_tile && T < ntiles_all;                  // tail groups idle but keep the warp converged
        if (BATCH) {
            const int rep = live ? T / a.ntiles : 0;
            T -= rep * a.ntiles;
            const NeBatchDesc &dsc = a.desc[rep];
            src0 = dsc.src[0]; src1 = dsc.src[1]; dst0 = dsc.dst[0]; dst1 = dsc.dst[1];
            bk0 = dsc.k0; bk1 = dsc.k1;
            thr_c = dsc.thr_c; thr_up = dsc.thr_up; up_always = dsc.up_always != 0;
            bobs = dsc.obs;
        }
        auto philox = [&](const uint32_t c0, const uint32_t c1) {
            if (BATCH) return philox_k(c0, c1, a.c2, a.c3, bk0, bk1);
            return philox_rk(c0, c1, a);
        };
        const int ty = live ? T / a.ntx : 0, tx = live ? T - ty * a.ntx : 0;   // one division per tile
        const int x0 = tx << a.lg_b, y0 = ty << a.lg_b;
        const uint32_t key_hi = ((uint32_t)grp_in_warp << 16) | (live ? 0u : 0x80000000u);
        // ---- step 5: tile + upper and right boundaries -> shared memory
        if (live) {
            // Asynchronous copies (LDGSTS) in chunks of 16 bytes (4 for tiles narrower than 32 sites): all of a lane's
            // chunks are in flight together, one round trip to L2/HBM per tile instead of one per chunk.
            // chunk i -> (row, colour, chunk in row): all powers of two, no divisions
            const int lg_cw = rowb >= 16 ? 4 : 2, lg_cr = a.lg_b - 1 - lg_cw;          // log2(chunk bytes), log2(chunks per row and colour)
            for (int i = j; i < ((b + 1) << (lg_cr + 1)); i += lam) {
                const int rr = i >> (lg_cr + 1), c = (i >> lg_cr) & 1, u = i & ((1 << lg_cr) - 1);
                int yy = y0 + rr;
                if (yy >= a.L) yy -= a.L;
                const uint8_t *g = (c ? src1 : src0) + (size_t)yy * a.Lh + (x0 >> 1) + (u << lg_cw);
                const uint32_t d = s_tile + (uint32_t)(c * col_bytes + rr * rowb + (u << lg_cw));
                if (lg_cw == 4) asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(d), "l"(g) : "memory");
                else asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(d), "l"(g) : "memory");
            }
            int xe = x0 + b;
            if (xe >= a.L) xe -= a.L;
            for (int py = j; py < b; py += lam) {
                const int yy = y0 + py;
                east[py] = (((xe + yy) & 1) ? src1 : src0)[(size_t)yy * a.Lh + (xe >> 1)];
            }
        }
        asm volatile("cp.async.commit_group;\n\tcp.async.wait_group 0;" ::: "memory");
        __syncwarp();
        // One pick: site (px, py) of colour c = (px + py) & 1 with claim index r, acceptance word w_acc.
        // Same site picked twice in one phase: the highest thread of the group wins (reading D19).  MATCH.ANY would
        // find the collisions directly but costs as much as the rest of the sub-step (measured: 100 against 186
        // Gflips/s), and collisions are rare (lambda^2 / 2P per sub-step).  So every lane writes its index into a claim
        // byte of the picked site; after the barrier a lane that reads back another index has collided, and only then
        // is MATCH used.  Stale claim bytes cannot hide a collision: every lane overwrites its byte before it reads it.
        auto pick = [&](const int r, const int px, const int py, const int c, const uint32_t w_acc) {
            if (lam > 1 && has_tile) sts_u8(s_claim + (uint32_t)r, (uint32_t)j);
            const uint32_t me = s_tile + (uint32_t)(c * col_bytes + py * rowb + (px >> 1));
            const uint32_t oth = s_tile + (uint32_t)((c ^ 1) * col_bytes + py * rowb);
            const uint32_t own = lds_u8(me);
            const uint32_t north = lds_u8(oth + (uint32_t)(rowb + (px >> 1)));
            const uint32_t est = lds_u8((px + 1 < b) ? oth + (uint32_t)((px + 1) >> 1) : s_east + (uint32_t)py);
            uint32_t n_new = own & 1u;
            if ((north & est & 1u) != 0u) {                            // facilitated
                if (METRO) {
                    if ((own & 1u) != 0u || up_always || w_acc < thr_up) n_new ^= 1u;
                } else {
                    n_new = w_acc < thr_c ? 1u : 0u;
                }
            }
            __syncwarp();                                              // all picks have read the phase's start
            bool winner = true;
            if (lam > 1 && __any_sync(0xffffffffu, has_tile && lds_u8(s_claim + (uint32_t)r) != (uint32_t)j)) {
                const uint32_t same = __match_any_sync(0xffffffffu, (uint32_t)r | key_hi);
                winner = (same >> lane) == 1u;                         // no higher lane holds the same key
            }
            if (live && winner && n_new != (own & 1u)) sts_u8(me, (own ^ 1u) | chg);
            __syncwarp();                                              // step 7
        };
        if (BAL) {
            // ---- balance-preserving variant (readings D22-D24): lambda red picks, barrier, lambda
            // white picks, barrier; one Philox call per lane and sub-step (words 0, 1: red pick; 2, 3: white pick)
            for (int k = 0; k < q; ++k) {
                const uint4 w = philox((uint32_t)T, (uint32_t)(k * lam + j));
#pragma unroll
                for (int c = 0; c < 2; ++c) {
                    const int r = (int)__umulhi(c ? w.z : w.x, (uint32_t)(P >> 1));   // r-th site of colour c, row-major
                    const int py = r >> (a.lg_b - 1), m = r & (rowb - 1);
                    pick(r, 2 * m + ((py + c) & 1), py, c, c ? w.w : w.y);
                }
            }
        } else {
            // ---- steps 6-8: q sub-steps of lambda simultaneous random picks
            auto go = [&](const uint32_t w_pos, const uint32_t w_acc) {
                const int r = (int)__umulhi(w_pos, (uint32_t)P);
                const int px = r & (b - 1), py = r >> a.lg_b;
                pick(r, px, py, (px + py) & 1, w_acc);                 // x0, y0 are even
            };
            if (lam == 1) {
                for (int k = 0; k < q; ++k) {
                    const uint4 w = philox((uint32_t)T, (uint32_t)k);
                    go(w.x, w.y);
                }
            } else {
                // One Philox call serves the two picks of a lane pair (reading D21).  Over two consecutive sub-steps the
                // even lane computes the pair's call of sub-step k and the odd lane that of sub-step k + 1, and each
                // hands two words to its partner: every lane computes one call per two sub-steps, none idles.
                for (int k = 0; k < q; k += 2) {
                    const int kk = k + (j & 1);                        // the odd lane works one sub-step ahead
                    uint4 w = make_uint4(0, 0, 0, 0);
                    if (kk < q) w = philox((uint32_t)T, (uint32_t)(kk * calls + (j >> 1)));
                    {                                                  // sub-step k: the even lane's call
                        const uint32_t pz = __shfl_xor_sync(0xffffffffu, w.z, 1), pw = __shfl_xor_sync(0xffffffffu, w.w, 1);
                        go((j & 1) ? pz : w.x, (j & 1) ? pw : w.y);
                    }
                    if (k + 1 < q) {                                   // sub-step k + 1: the odd lane's call
                        const uint32_t px_ = __shfl_xor_sync(0xffffffffu, w.x, 1), py_ = __shfl_xor_sync(0xffffffffu, w.y, 1);
                        go((j & 1) ? w.z : px_, (j & 1) ? w.w : py_);
                    }
                }
            }
        }
        // ---- step 9: copy the tile back (interior only); count the up sites for the fused observable
        if (live) {
            if (rowb >= 16) {
                const int lg_cr = a.lg_b - 5;                          // 16-byte chunks per row and colour
                for (int i = j; i < (b << (lg_cr + 1)); i += lam) {
                    const int rr = i >> (lg_cr + 1), c = (i >> lg_cr) & 1, u = i & ((1 << lg_cr) - 1);
                    const uint4 v = *reinterpret_cast<const uint4 *>((tile + c * col_bytes) + rr * rowb + 16 * u);
                    *reinterpret_cast<uint4 *>((c ? dst1 : dst0) + (size_t)(y0 + rr) * a.Lh + (x0 >> 1) + 16 * u) = v;
                    ups += (int)__dp4a((v.x & 0x01010101u) + (v.y & 0x01010101u) + (v.z & 0x01010101u) + (v.w & 0x01010101u),
                                       0x01010101u, 0u);
                }
            } else {
                const int lg_lr = a.lg_b - 3;
                for (int i = j; i < (b << (lg_lr + 1)); i += lam) {
                    const int rr = i >> (lg_lr + 1), c = (i >> lg_lr) & 1, u = i & ((1 << lg_lr) - 1);
                    const uint32_t v = *reinterpret_cast<const uint32_t *>((tile + c * col_bytes) + rr * rowb + 4 * u);
                    *reinterpret_cast<uint32_t *>((c ? dst1 : dst0) + (size_t)(y0 + rr) * a.Lh + (x0 >> 1) + 4 * u) = v;
                    ups += (int)__dp4a(v & 0x01010101u, 0x01010101u, 0u);
                }
            }
        }
        if (BATCH) {                                                   // the warp's groups may sit in different lattices
            if (live && a.obs_off >= 0 && ups != 0) atomicAdd((unsigned long long *)&bobs[a.obs_off + 1], (unsigned long long)ups);
            ups = 0;
        }
        __syncwarp();
    }
    if (!BATCH && a.obs) {
        const int s = __reduce_add_sync(0xffffffffu, ups);
        if (lane == 0 && s != 0) atomicAdd((unsigned long long *)&a.obs[1], (unsigned long long)s);
    }
}

// Shared memory of one tile (must match the kernel).
static size_t ne_tile_bytes(int b, int lam)
{
    return (size_t)((2 * (b + 1) * (b / 2) + b + (lam > 1 ? b * b : 0) + 15) & ~15);
}

bool ne_tile_supported(const Lat &lat, int b, int lam, bool balanced)
{
    if (lat.dims != 2) return false;
    if (b < 8 || b > 128 || (b & (b - 1)) != 0 || lat.L % b != 0) return false;
    if (lam < 1 || lam > 32 || (lam & (lam - 1)) != 0) return false;
    if ((b * b) % ((balanced ? 8 : 2) * lam) != 0) return false;   // q * lambda = P/2 (D17) or q * 2 lambda = P/4 (D23)
    return true;                                                   // one tile always fits: <= 33 KB
}

// Tile groups per warp that hold a tile, and threads per CTA: as many tiles as fit ~96 KB of shared memory.
static int ne_tile_gpw(int b, int lam)
{
    int gpw = 32 / lam;
    const int fit = (int)((96 * 1024) / ne_tile_bytes(b, lam));
    if (gpw > fit) gpw = fit < 1 ? 1 : fit;
    return gpw;
}
static int ne_tile_threads(int b, int lam)
{
    const int gpw = ne_tile_gpw(b, lam);
    int threads = 256;
    while (threads > 32 && (threads / 32) * gpw * ne_tile_bytes(b, lam) > 96 * 1024) threads >>= 1;
    return threads;
}

cudaError_t launch_ne_random_tile(const Lat &lat, uint8_t *const dst[2], bool metropolis, bool balanced, int b, int lam,
                                  unsigned long long seed, unsigned long long t, int launch, uint32_t thr_c,
                                  uint32_t thr_up, int up_always, int track, long long *obs, cudaStream_t s)
{
    NeTileArgs a;
    memset(&a, 0, sizeof(a));
    a.src[0] = lat.col[0];
    a.src[1] = lat.col[1];
    a.dst[0] = dst[0];
    a.dst[1] = dst[1];
    a.L = lat.L;
    a.Lh = lat.Lh;
    while ((1 << a.lg_b) < b) ++a.lg_b;
    while ((1 << a.lg_lam) < lam) ++a.lg_lam;
    a.ntx = lat.L / b;
    a.ntiles = a.ntx * a.ntx;
    a.k0 = (uint32_t)seed;
    a.k1 = (uint32_t)(seed >> 32);
    for (int r = 0; r < 10; ++r) {
        a.rk0[r] = a.k0 + (uint32_t)r * PHILOX_W0;
        a.rk1[r] = a.k1 + (uint32_t)r * PHILOX_W1;
    }
    a.c2 = (uint32_t)t;
    a.c3 = ((balanced ? 8u : 4u) + (uint32_t)launch) | ((uint32_t)(t >> 32) << 4);   // D21: tags 4, 5; D24: 8..11
    a.thr_c = thr_c;
    a.thr_up = thr_up;
    a.up_always = up_always;
    a.track = track;
    a.obs = obs;
    const int threads = ne_tile_threads(b, lam);
    a.gpw = ne_tile_gpw(b, lam);
    const int tiles_per_cta = (threads / 32) * a.gpw;
    const size_t smem = tiles_per_cta * ne_tile_bytes(b, lam);
    int grid = (a.ntiles + tiles_per_cta - 1) / tiles_per_cta;
    const int cap = sm_count() * 8;
    if (grid > cap) grid = cap;
    auto kern = balanced ? (metropolis ? k_ne_random_tile<true, true> : k_ne_random_tile<false, true>)
                         : (metropolis ? k_ne_random_tile<true, false> : k_ne_random_tile<false, false>);
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    kern<<<grid, threads, smem, s>>>(a);
    return cudaGetLastError();
}

// R lattices of one shape in one launch (lsm_batch_sweep_random_tile): d_desc[r] names lattice r's buffers of this launch.
cudaError_t launch_ne_random_tile_batch(const Lat &lat, const NeBatchDesc *d_desc, int R, bool metropolis, bool balanced, int b,
                                        int lam, unsigned long long t, int launch, int track, long long obs_off, cudaStream_t s)
{
    NeTileArgs a;
    memset(&a, 0, sizeof(a));
    a.L = lat.L;
    a.Lh = lat.Lh;
    while ((1 << a.lg_b) < b) ++a.lg_b;
    while ((1 << a.lg_lam) < lam) ++a.lg_lam;
    a.ntx = lat.L / b;
    a.ntiles = a.ntx * a.ntx;
    a.c2 = (uint32_t)t;
    a.c3 = ((balanced ? 8u : 4u) + (uint32_t)launch) | ((uint32_t)(t >> 32) << 4);
    a.track = track;
    a.desc = d_desc;
    a.R = R;
    a.obs_off = obs_off;
    const int threads = ne_tile_threads(b, lam);
    a.gpw = ne_tile_gpw(b, lam);
    const int tiles_per_cta = (threads / 32) * a.gpw;
    const size_t smem = tiles_per_cta * ne_tile_bytes(b, lam);
    const long long total = (long long)a.ntiles * R;
    if (total > 0x7fffffffLL) return cudaErrorInvalidValue;
    long long grid = (total + tiles_per_cta - 1) / tiles_per_cta;
    const int cap = sm_count() * 8;
    if (grid > cap) grid = cap;
    auto kern = balanced ? (metropolis ? k_ne_random_tile<true, true, true> : k_ne_random_tile<false, true, true>)
                         : (metropolis ? k_ne_random_tile<true, false, true> : k_ne_random_tile<false, false, true>);
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    kern<<<(unsigned)grid, threads, smem, s>>>(a);
    return cudaGetLastError();
}

}  // namespace lsmk
