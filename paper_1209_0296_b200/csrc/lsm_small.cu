// lsm_small.cu -- the single-CTA kernel family for small lattices: ONE launch runs many sweeps.
//
// The paper reports that small lattices cannot hide the cost of a kernel launch per half-sweep
// (2x at 32^2 against 150x at 512^2), and it ends the kernel only because its GPUs had
// no other barrier between the two colours.  A lattice of a few thousand sites is
// work for one SM: here one thread block owns the whole lattice, its threads take one word column
// and a short march segment each (the thread -> site map and the arithmetic are the tiled family's
// March, unchanged, so results are bit-identical), and the barrier between half-sweeps is
// __syncthreads().  The colour arrays stay in global memory; after the first touch every access is
// an L1 hit on the block's SM (bar.sync orders the block's global writes before its later reads).
// Per-sweep (B, M): per-thread sums -> warp shuffle -> shared-memory atomics -> one 16-byte store.
#include "lsm_tiled_dev.cuh"

#include <cooperative_groups.h>
#include <cstdlib>
#include <cstring>
#include <type_traits>

namespace lsmk {

struct SmallArgs {
    uint8_t *col[2];
    TiledGeom g;                 // own/oth/half/obs are set per half-sweep on the device
    unsigned long long seed, t0; // first sweep of this launch
    int nsweeps;
    long long *obs;              // [nsweeps][2] (B, M), or nullptr
};

template <int MODEL, int DIMS, bool TRACK, int OBS>
__global__ void __launch_bounds__(1024, 1)
k_sweep_small(const __grid_constant__ SmallArgs a, const __grid_constant__ PhiloxSweepConsts pk,
              const __grid_constant__ typename TabOf<MODEL>::type tab)
{
    __shared__ __align__(16) struct {
        uint32_t t[MODEL == M_ISING_ONE ? 64 : 16];
        int acc[2][2];           // (B, M) of the sweep in flight, double-buffered by sweep parity
    } sm;
    uint32_t s_t = (uint32_t)__cvta_generic_to_shared(sm.t);
    asm volatile("" : "+r"(s_t));
    if constexpr (MODEL == M_ISING_HALF) {
        if (threadIdx.x < 16) sm.t[threadIdx.x] = tab.t[threadIdx.x];
    } else if constexpr (MODEL == M_ISING_ONE) {
        for (int i = threadIdx.x; i < 64; i += blockDim.x) sm.t[i] = tab.t[i];   // blocks may have 32 threads
    }
    if (threadIdx.x < 4) sm.acc[threadIdx.x >> 1][threadIdx.x & 1] = 0;
    __syncthreads();

    constexpr bool NE = MODEL == M_NE_HEATBATH || MODEL == M_NE_METROPOLIS;
    const int nthr = a.g.ncol * a.g.S;
    const bool active = (int)threadIdx.x < nthr;
    const int seg = active ? (int)threadIdx.x / a.g.ncol : 0;
    const int col = active ? (int)threadIdx.x - seg * a.g.ncol : 0;

    const int nhalves = 2 * a.nsweeps;
#pragma unroll 1
    for (int gh = 0; gh < nhalves; ++gh) {
        const int half = gh & 1, sw = gh >> 1;
        const unsigned long long t = a.t0 + (unsigned long long)sw;
        PhiloxDyn pc = {0u, 0u, 0u, 0u, pk};
        philox_half_consts(make_sweep_key(a.seed, t, (uint32_t)half), pk.rk0, pk.rk1, pc.x1, pc.y2, pc.z2, pc.w3);

        March<MODEL, DIMS, TRACK, OBS> M;
        M.ne_t32 = 0;
        M.ne_always = 0;
        M.ne_all4 = false;
        if constexpr (NE) {
            M.ne_t32 = tab.t32;
            M.ne_always = tab.always;
            M.ne_all4 = tab.all4 != 0;
        }
        M.s_t = s_t;
        M.one = (uint32_t)a.g.one;
        M.totU = M.totBN = M.totS = 0;
        int nsites = 0;
        if (active) {
            const int n = march_init(M, a.g, a.col[half], a.col[half ^ 1], half, seg, col, true);
            nsites = 16 * n;
            M.template run<2, true>(n, pc);          // a warp spans rows of both parities: q is per thread
        }
        if (OBS >= 1) {
            long long cB, cM;
            march_observables<MODEL, DIMS>(M, nsites, half == 1, cB, cM);
            const int wB = warp_sum((int)cB), wM = warp_sum((int)cM);   // |B| <= 3N, |M| <= N: far below 2^31 here
            if ((threadIdx.x & 31) == 0) {
                if (wB != 0) atomicAdd(&sm.acc[sw & 1][0], wB);
                if (wM != 0) atomicAdd(&sm.acc[sw & 1][1], wM);
            }
        }
        __syncthreads();                              // the barrier between the two colours
        if (OBS >= 1 && half == 1 && threadIdx.x == 0) {
            // the next adds to this buffer belong to sweep sw + 2: two barriers away
            a.obs[2 * sw] = sm.acc[sw & 1][0];
            a.obs[2 * sw + 1] = sm.acc[sw & 1][1];
            sm.acc[sw & 1][0] = 0;
            sm.acc[sw & 1][1] = 0;
        }
    }
}

// Lane-granular cluster variant for power-of-two L.  A thread owns 32-bit lanes (4 sites, one Philox call)
// instead of whole words, and the lattice is cut into slabs of march rows, one slab per thread block of a
// thread-block cluster (1, 2, 4 or 8 SMs).  Each block keeps its slab of both colours in shared memory for
// the whole launch; the rows m-1 / m+1 across a slab boundary are read from the neighbour block's shared
// memory (distributed shared memory), and the barrier between the colours is the cluster barrier --
// hardware-supported, far cheaper than ending the kernel.  This is the regime of the
// paper's own lattices (32^2 ... 512^2), which a launch per half-sweep cannot serve well.
// Same rules, same (group, word) -> site map as every other family: bit-identical.
//
// The body serves two kernels: k_sweep_small_lane (one lattice = one cluster = the whole grid) and
// k_sweep_small_lane_batch (R independent lattices = R clusters of one grid, each with its own Philox key and
// threshold table: lsm_batch_sweep).  `sm_t` is the block's threshold table in shared memory (filled by the
// caller), `acc` its (B, M) scratch.  self_zero: the cluster zeroes its own obs / run slots (batch launches have no
// host memset per replica); run: where the sums of the LAST sweep are added as well (the replica's running pair).
__device__ __forceinline__ uint32_t lds_w(uint32_t a)
{
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(a) : "memory");
    return v;
}
__device__ __forceinline__ void sts_w(uint32_t a, uint32_t v) { asm volatile("st.shared.u32 [%0], %1;" ::"r"(a), "r"(v) : "memory"); }
// word of this or another block of the cluster (distributed shared memory)
__device__ __forceinline__ uint32_t ldc_w(uint32_t a)
{
    uint32_t v;
    asm volatile("ld.shared::cluster.u32 %0, [%1];" : "=r"(v) : "r"(a) : "memory");
    return v;
}
__device__ __forceinline__ uint32_t mapa_u32(uint32_t a, uint32_t rank)
{
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(a), "r"(rank));
    return r;
}

// LPT > 0: the block has exactly LPT lanes per thread and the geometry of a thread's lanes (which words hold its 2d
// neighbours, in this block's shared memory or in a neighbour block's) is computed ONCE, before the sweep loop: a
// half-sweep of a small lattice is a dependent chain per thread, and the index arithmetic was a third of it.
// LPT = 0: any number of lanes per thread, geometry recomputed in every half-sweep.
template <int MODEL, int DIMS, bool TRACK, int OBS, int LPT = 0>
__device__ __forceinline__ void small_lane_body(uint8_t *const col0, uint8_t *const col1, const PhiloxSweepConsts &pk,
                                                const unsigned long long seed, const unsigned long long t0,
                                                const int nsweeps, long long *const obs, long long *const run,
                                                const bool self_zero, uint32_t ne_t32, int ne_always, const uint32_t one,
                                                const uint32_t s_t, int (*acc)[2], const int lg_lpr, const int lg_L,
                                                const int lg_rpc)
{
    namespace cg = cooperative_groups;
    cg::cluster_group cluster = cg::this_cluster();
    const uint32_t rank = cluster.block_rank(), nrank = cluster.num_blocks();

    constexpr bool NE = MODEL == M_NE_HEATBATH || MODEL == M_NE_METROPOLIS;
    const uint32_t lpr = 1u << lg_lpr;
    const int lg_R = DIMS == 3 ? lg_L : 0;
    const uint32_t R = 1u << lg_R;
    const int lg_slab = lg_rpc + lg_R + lg_lpr;               // log2(lanes per colour in one slab)
    const uint32_t nl = 1u << lg_slab;
    const uint32_t base = rank << lg_slab;                     // first lane of this slab in the colour array
    if (!NE) { ne_t32 = 0; ne_always = 0; }

    extern __shared__ __align__(16) uint32_t s_lat[];
    uint32_t *const s_col[2] = {s_lat, s_lat + nl};
    for (uint32_t i = threadIdx.x; i < nl; i += blockDim.x) {
        s_col[0][i] = reinterpret_cast<const uint32_t *>(col0)[base + i];
        s_col[1][i] = reinterpret_cast<const uint32_t *>(col1)[base + i];
    }
    if (self_zero && rank == 0) {                              // ordered before every add by the barrier below
        if (OBS >= 1 && obs)
            for (int i = threadIdx.x; i < 2 * nsweeps; i += blockDim.x) obs[i] = 0;
        if (OBS >= 1 && run && threadIdx.x < 2) run[threadIdx.x] = 0;
    }
    // the slabs above and below (the same shared-memory offsets in the neighbour blocks)
    const uint32_t r_dn = (rank + nrank - 1) % nrank, r_up = (rank + 1) % nrank;
    const uint32_t *const dn_col[2] = {cluster.map_shared_rank(s_col[0], r_dn), cluster.map_shared_rank(s_col[1], r_dn)};
    const uint32_t *const up_col[2] = {cluster.map_shared_rank(s_col[0], r_up), cluster.map_shared_rank(s_col[1], r_up)};
    const uint32_t rpc = 1u << lg_rpc;
    if (nrank > 1) cluster.sync();
    else __syncthreads();

    // hoisted geometry (LPT > 0): shared-window addresses of the colour-0 words; colour 1 lies colB bytes behind
    constexpr int NL = LPT > 0 ? LPT : 1;
    const uint32_t colB = nl * 4u;
    uint32_t a_own[NL], a_p[NL], a_n[NL], a_cs1[NL], a_cs0[NL], a_yp[NL], a_yn[NL], g_q0[NL], g_gl[NL];
    if (LPT > 0) {
        const uint32_t s0 = (uint32_t)__cvta_generic_to_shared(s_lat);
#pragma unroll
        for (int l = 0; l < NL; ++l) {
            const uint32_t li = threadIdx.x + (uint32_t)l * blockDim.x;
            const uint32_t x = li & (lpr - 1), row = li >> lg_lpr;
            const uint32_t y = row & (R - 1), ml = row >> lg_R;
            const uint32_t m = (rank << lg_rpc) + ml;
            g_q0[l] = (m + y) & 1u;                                          // row parity bit of half 0
            g_gl[l] = base + li;
            a_own[l] = s0 + li * 4u;
            const uint32_t up_off = (rpc - 1) << (lg_R + lg_lpr);            // lanes between the first and the last row of a slab
            a_p[l] = ml > 0 ? mapa_u32(s0 + (li - (R << lg_lpr)) * 4u, rank) : mapa_u32(s0 + (li + up_off) * 4u, r_dn);
            a_n[l] = ml + 1 < rpc ? mapa_u32(s0 + (li + (R << lg_lpr)) * 4u, rank) : mapa_u32(s0 + (li - up_off) * 4u, r_up);
            a_cs1[l] = s0 + ((row << lg_lpr) + ((x + 1) & (lpr - 1))) * 4u;  // q = 1: the word to the right
            a_cs0[l] = s0 + ((row << lg_lpr) + ((x - 1) & (lpr - 1))) * 4u;  // q = 0: the word to the left
            a_yp[l] = s0 + (((ml << lg_R) + ((y - 1) & (R - 1))) * lpr + x) * 4u;
            a_yn[l] = s0 + (((ml << lg_R) + ((y + 1) & (R - 1))) * lpr + x) * 4u;
        }
    }

    int thrB = 0, thrM = 0;
    const int nhalves = 2 * nsweeps;
#pragma unroll 1
    for (int gh = 0; gh < nhalves; ++gh) {
        const int half = gh & 1, sw = gh >> 1;
        const unsigned long long t = t0 + (unsigned long long)sw;
        PhiloxDyn pc = {0u, 0u, 0u, 0u, pk};
        philox_half_consts(make_sweep_key(seed, t, (uint32_t)half), pk.rk0, pk.rk1, pc.x1, pc.y2, pc.z2, pc.w3);
        uint32_t *own = s_col[half];
        const uint32_t *oth = s_col[half ^ 1];
        int totU = 0, totBN = 0, totS = 0, nsites = 0;
        if (half == 0) thrB = thrM = 0;
        if (LPT > 0) {
            const uint32_t ownB = half ? colB : 0u, othB = half ? 0u : colB;
#pragma unroll
            for (int l = 0; l < NL; ++l) {
                const uint32_t qq = g_q0[l] ^ (uint32_t)half;
                const uint32_t c = lds_w(a_own[l] + othB), o = lds_w(a_own[l] + ownB);
                const uint32_t p = ldc_w(a_p[l] + othB), n = ldc_w(a_n[l] + othB);
                const uint32_t cs = lds_w((qq ? a_cs1[l] : a_cs0[l]) + othB);
                const uint32_t sd = qq ? __funnelshift_r(c, cs, 8) : __funnelshift_r(cs, c, 24);
                uint32_t yp = 0, yn = 0;
                if (DIMS == 3) {
                    yp = lds_w(a_yp[l] + othB);
                    yn = lds_w(a_yn[l] + othB);
                }
                const uint32_t gl = g_gl[l];
                uint32_t out;
                if (MODEL == M_ISING_HALF) {
                    uint32_t ns = p + n + c + sd;
                    if (DIMS == 3) ns += yp + yn;
                    out = rule_half<TRACK, OBS>(o, ns, philox_sweep(gl, pc), s_t, one, totU, totBN);
                } else if (MODEL == M_ISING_ONE) {
                    uint32_t ns;
                    if (TRACK) {
                        ns = ((p + n) & 0x0F0F0F0Fu) + ((c + sd) & 0x0F0F0F0Fu);
                        if (DIMS == 3) ns += (yp + yn) & 0x0F0F0F0Fu;
                    } else {
                        ns = p + n + c + sd;
                        if (DIMS == 3) ns += yp + yn;
                    }
                    out = rule_one<DIMS, TRACK, OBS>(o, ns, philox_sweep(2u * gl, pc), philox_sweep(2u * gl + 1u, pc), s_t, one,
                                                     totU, totBN, totS);
                } else {
                    uint32_t accU = 0;
                    out = rule_ne<TRACK, MODEL == M_NE_METROPOLIS, OBS>(o, n, qq ? sd : c, gl, pc, ne_t32, ne_always, accU);
                    if (OBS >= 1) totU += (int)bytesum(accU);
                }
                sts_w(a_own[l] + ownB, out);
                nsites += 4;
            }
        } else
#pragma unroll 1
        for (uint32_t li = threadIdx.x; li < nl; li += blockDim.x) {
            const uint32_t gl = base + li;                                    // lane index in the colour array
            const uint32_t x = li & (lpr - 1), row = li >> lg_lpr;           // local row = ml * R + y
            const uint32_t y = row & (R - 1), ml = row >> lg_R;
            const uint32_t m = (rank << lg_rpc) + ml;
            const uint32_t qq = (m + y + (uint32_t)half) & 1u;
            const uint32_t c = oth[li];
            const uint32_t o = own[li];
            const uint32_t p = ml > 0 ? oth[li - (R << lg_lpr)] : dn_col[half ^ 1][li + ((rpc - 1) << (lg_R + lg_lpr))];
            const uint32_t n = ml + 1 < rpc ? oth[li + (R << lg_lpr)] : up_col[half ^ 1][li - ((rpc - 1) << (lg_R + lg_lpr))];
            const uint32_t cs = oth[(row << lg_lpr) + ((qq ? x + 1 : x - 1) & (lpr - 1))];
            const uint32_t sd = qq ? __funnelshift_r(c, cs, 8) : __funnelshift_r(cs, c, 24);
            uint32_t yp = 0, yn = 0;
            if (DIMS == 3) {
                yp = oth[((ml << lg_R) + ((y - 1) & (R - 1))) * lpr + x];
                yn = oth[((ml << lg_R) + ((y + 1) & (R - 1))) * lpr + x];
            }
            uint32_t out;
            if (MODEL == M_ISING_HALF) {
                uint32_t ns = p + n + c + sd;
                if (DIMS == 3) ns += yp + yn;
                out = rule_half<TRACK, OBS>(o, ns, philox_sweep(gl, pc), s_t, one, totU, totBN);
            } else if (MODEL == M_ISING_ONE) {
                uint32_t ns;
                if (TRACK) {
                    ns = ((p + n) & 0x0F0F0F0Fu) + ((c + sd) & 0x0F0F0F0Fu);
                    if (DIMS == 3) ns += (yp + yn) & 0x0F0F0F0Fu;
                } else {
                    ns = p + n + c + sd;
                    if (DIMS == 3) ns += yp + yn;
                }
                out = rule_one<DIMS, TRACK, OBS>(o, ns, philox_sweep(2u * gl, pc), philox_sweep(2u * gl + 1u, pc), s_t, one,
                                                 totU, totBN, totS);
            } else {
                uint32_t accU = 0;
                out = rule_ne<TRACK, MODEL == M_NE_METROPOLIS, OBS>(o, n, qq ? sd : c, gl, pc, ne_t32, ne_always, accU);
                if (OBS >= 1) totU += (int)bytesum(accU);
            }
            own[li] = out;
            nsites += 4;
        }
        if (OBS >= 1) {
            March<MODEL, DIMS, TRACK, OBS> M;          // only the per-thread sums are used
            M.totU = totU;
            M.totBN = totBN;
            M.totS = totS;
            long long cB, cM;
            march_observables<MODEL, DIMS>(M, nsites, half == 1, cB, cM);
            thrB += (int)cB;                           // |B| <= 3N, |M| <= N with N <= 2^20: far below 2^31
            thrM += (int)cM;
            if (half == 1) {                           // once per sweep: warp reduce -> block-local shared atomics
                const int wB = __reduce_add_sync(0xffffffffu, thrB), wM = __reduce_add_sync(0xffffffffu, thrM);
                if ((threadIdx.x & 31) == 0) {
                    if (wB != 0) atomicAdd(&acc[sw & 1][0], wB);
                    if (wM != 0) atomicAdd(&acc[sw & 1][1], wM);
                }
            }
        }
        // the barrier between the two colours
        if (nrank > 1) cluster.sync();
        else __syncthreads();
        if (OBS >= 1 && half == 1 && threadIdx.x == 0) {
            // one fire-and-forget 64-bit add per block into the sweep's (zeroed) slot; the next adds to this
            // shared buffer belong to sweep sw + 2: two barriers away
            const int vB = acc[sw & 1][0], vM = acc[sw & 1][1];
            if (obs) {
                if (vB != 0) atomicAdd((unsigned long long *)&obs[2 * sw], (unsigned long long)(long long)vB);
                if (vM != 0) atomicAdd((unsigned long long *)&obs[2 * sw + 1], (unsigned long long)(long long)vM);
            }
            if (run && sw == nsweeps - 1) {
                if (vB != 0) atomicAdd((unsigned long long *)&run[0], (unsigned long long)(long long)vB);
                if (vM != 0) atomicAdd((unsigned long long *)&run[1], (unsigned long long)(long long)vM);
            }
            acc[sw & 1][0] = 0;
            acc[sw & 1][1] = 0;
        }
    }
    for (uint32_t i = threadIdx.x; i < nl; i += blockDim.x) {
        reinterpret_cast<uint32_t *>(col0)[base + i] = s_col[0][i];
        reinterpret_cast<uint32_t *>(col1)[base + i] = s_col[1][i];
    }
    if (nrank > 1) cluster.sync();      // no block may exit while a neighbour can still read its shared memory
}

template <int MODEL, int DIMS, bool TRACK, int OBS, int LPT>
__global__ void __launch_bounds__(1024, 1)
k_sweep_small_lane(const __grid_constant__ SmallArgs a, const __grid_constant__ PhiloxSweepConsts pk,
                   const __grid_constant__ typename TabOf<MODEL>::type tab, const int lg_lpr, const int lg_L,
                   const int lg_rpc)
{
    __shared__ __align__(16) struct {
        uint32_t t[MODEL == M_ISING_ONE ? 64 : 16];
        int acc[2][2];           // this block's share of (B, M) of the sweep in flight, double-buffered
    } sm;
    uint32_t s_t = (uint32_t)__cvta_generic_to_shared(sm.t);
    asm volatile("" : "+r"(s_t));
    uint32_t ne_t32 = 0;
    int ne_always = 0;
    if constexpr (MODEL == M_ISING_HALF) {
        if (threadIdx.x < 16) sm.t[threadIdx.x] = tab.t[threadIdx.x];
    } else if constexpr (MODEL == M_ISING_ONE) {
        for (int i = threadIdx.x; i < 64; i += blockDim.x) sm.t[i] = tab.t[i];   // blocks may have 32 threads
    } else {
        ne_t32 = tab.t32;
        ne_always = tab.always;
    }
    if (threadIdx.x < 4) sm.acc[threadIdx.x >> 1][threadIdx.x & 1] = 0;
    small_lane_body<MODEL, DIMS, TRACK, OBS, LPT>(a.col[0], a.col[1], pk, a.seed, a.t0, a.nsweeps, a.obs, nullptr, false, ne_t32,
                                             ne_always, (uint32_t)a.g.one, s_t, sm.acc, lg_lpr, lg_L, lg_rpc);
}

// R lattices in one launch: cluster c of the grid sweeps replica r0 + c.  Per replica: colour arrays, running pair,
// Philox key (seed) and the threshold table in the form the vectorised rules index -- all from the descriptor array
// in device memory (the seeds also ride in the kernel parameters so that the round keys stay warp-uniform operands).
constexpr int SMALL_BATCH_MAX = 256;              // replicas per launch (seed array in the kernel parameters)
struct SmallBatchArgs {
    const BatchDesc *desc;       // [R] device
    long long *obs;              // slot of replica 0 for the first sweep of this launch, or nullptr
    long long obs_stride;        // int64 elements between two replicas' series
    unsigned long long t0;       // first sweep of this launch (the replicas sweep in lockstep)
    int nsweeps;
    int r0;                      // replica of cluster 0
    int write_run;               // add the last sweep's sums to the replicas' running pairs
    int one;
    uint2 seed[SMALL_BATCH_MAX]; // (k0, k1) of replica r0 + i
};

template <int MODEL, int DIMS, bool TRACK, int OBS, int LPT>
__global__ void __launch_bounds__(1024, 1)
k_sweep_small_lane_batch(const __grid_constant__ SmallBatchArgs a, const int lg_lpr, const int lg_L, const int lg_rpc,
                         const int lg_clu)
{
    __shared__ __align__(16) struct {
        uint32_t t[MODEL == M_ISING_ONE ? 64 : 16];
        int acc[2][2];
    } sm;
    uint32_t s_t = (uint32_t)__cvta_generic_to_shared(sm.t);
    asm volatile("" : "+r"(s_t));
    const int ci = (int)(blockIdx.x >> lg_clu);                  // cluster index = replica of this launch
    const BatchDesc &d = a.desc[a.r0 + ci];
    constexpr int NT = MODEL == M_ISING_ONE ? 64 : MODEL == M_ISING_HALF ? 16 : 0;
    for (int i = threadIdx.x; i < NT; i += blockDim.x) sm.t[i] = d.tab[i];
    if (threadIdx.x < 4) sm.acc[threadIdx.x >> 1][threadIdx.x & 1] = 0;
    const uint2 sd = a.seed[ci];
    PhiloxSweepConsts pk;
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        pk.rk0[r] = sd.x + (uint32_t)r * PHILOX_W0;
        pk.rk1[r] = sd.y + (uint32_t)r * PHILOX_W1;
    }
    pk.x1 = pk.y2 = pk.z2 = pk.w3 = 0u;
    pk.m0 = PHILOX_M0;
    pk.m1 = PHILOX_M1;
    const unsigned long long seed = ((unsigned long long)sd.y << 32) | sd.x;
    long long *obs = (OBS >= 1 && a.obs) ? a.obs + a.obs_stride * (a.r0 + ci) : nullptr;
    small_lane_body<MODEL, DIMS, TRACK, OBS, LPT>(d.col[0], d.col[1], pk, seed, a.t0, a.nsweeps, obs,
                                             a.write_run ? d.run : nullptr, true, d.ne_t32, d.ne_always, (uint32_t)a.one,
                                             s_t, sm.acc, lg_lpr, lg_L, lg_rpc);
}

// ------------------------------------------------------------------------------------------
// Host side
// ------------------------------------------------------------------------------------------
PhiloxSweepConsts make_philox_consts(const SweepKey &k);   // lsm_tiled.cu

static int ilog2(int v)
{
    int l = 0;
    while ((1 << l) < v) ++l;
    return l;
}

template <int MODEL, int DIMS>
static cudaError_t small_launch_to(bool track, bool obs, int threads, cudaStream_t s, const SmallArgs &a,
                                   const PhiloxSweepConsts &pk, const typename TabOf<MODEL>::type &tab, int lg_lpr,
                                   int lg_L, int nclu)
{
    if (lg_L > 0) {
        const size_t smem = ((size_t)1 << (DIMS * lg_L)) / (size_t)nclu;   // N / cluster bytes: the slab of both colours
        const int lg_rpc = lg_L - ilog2(nclu);
        auto go = [&](auto kern) -> cudaError_t {
            if (smem > 48 * 1024) {
                cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
                if (e != cudaSuccess) return e;
            }
            if (nclu > 8) {
                cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
                if (e != cudaSuccess) return e;
            }
            cudaLaunchConfig_t cfg;
            memset(&cfg, 0, sizeof(cfg));
            cfg.gridDim = dim3((unsigned)nclu);
            cfg.blockDim = dim3((unsigned)threads);
            cfg.dynamicSmemBytes = smem;
            cfg.stream = s;
            cudaLaunchAttribute at[1];
            at[0].id = cudaLaunchAttributeClusterDimension;
            at[0].val.clusterDim.x = (unsigned)nclu;
            at[0].val.clusterDim.y = 1;
            at[0].val.clusterDim.z = 1;
            cfg.attrs = at;
            cfg.numAttrs = 1;
            return cudaLaunchKernelEx(&cfg, kern, a, pk, tab, lg_lpr, lg_L, lg_rpc);
        };
        // one lane per thread (every lattice up to 16 x 1024 lanes per colour): the hoisted-geometry body
        const bool one = (((size_t)1 << (DIMS * lg_L)) / 8) / (size_t)nclu == (size_t)threads;
        if (one) {
            if (track) return obs ? go(k_sweep_small_lane<MODEL, DIMS, true, 2, 1>) : go(k_sweep_small_lane<MODEL, DIMS, true, 0, 1>);
            return obs ? go(k_sweep_small_lane<MODEL, DIMS, false, 2, 1>) : go(k_sweep_small_lane<MODEL, DIMS, false, 0, 1>);
        }
        if (track) return obs ? go(k_sweep_small_lane<MODEL, DIMS, true, 2, 0>) : go(k_sweep_small_lane<MODEL, DIMS, true, 0, 0>);
        return obs ? go(k_sweep_small_lane<MODEL, DIMS, false, 2, 0>) : go(k_sweep_small_lane<MODEL, DIMS, false, 0, 0>);
    }
    if (track) {
        if (obs) k_sweep_small<MODEL, DIMS, true, 2><<<1, threads, 0, s>>>(a, pk, tab);
        else k_sweep_small<MODEL, DIMS, true, 0><<<1, threads, 0, s>>>(a, pk, tab);
    } else {
        if (obs) k_sweep_small<MODEL, DIMS, false, 2><<<1, threads, 0, s>>>(a, pk, tab);
        else k_sweep_small<MODEL, DIMS, false, 0><<<1, threads, 0, s>>>(a, pk, tab);
    }
    return cudaGetLastError();
}

// Compile-time knobs for tuning experiments; the library reads no environment variables.
#define LSM_SMALL_MAX_CLUSTER 16         // B200 schedules 16-block clusters
#define LSM_SMALL_MAX_SITES 262144       // above 512^2 / 64^3 the tiled family wins (profiles/r1_small_family.md)
static int small_max_cluster() { return LSM_SMALL_MAX_CLUSTER; }
static int small_max_sites() { return LSM_SMALL_MAX_SITES; }

// Plan: every word column gets as many march segments as 1024 threads allow.
bool small_plan(const Lat &lat, int model, const TiledTables &t, SmallPlan *out, bool ignore_size_limit)
{
    if (!t.usable) return false;
    if (model == M_EA || model == M_POTTS) return false;   // NEXT-4 models: no small-family kernels
    if (t.has_never) return false;                         // two-compare kernels exist in the tiled family only
    const bool pow2 = lat.L >= 8 && (lat.L & (lat.L - 1)) == 0;       // lane-granular kernel: whole 32-bit lanes per row
    const bool words = tiled_supported(lat, model, t);                // word-granular kernel: whole 16-byte words per row
    if (!pow2 && !words) return false;
    const long long N = 2 * lat.half;
    if (N > 1048576) return false;                    // int accumulators; beyond this the tiled family is faster anyway
    if (!ignore_size_limit && N > small_max_sites()) return false;
    const int R = lat.dims == 3 ? lat.L : 1, wpr = lat.Lh / 16;
    const long long ncol = (long long)R * wpr;
    long long S = (ncol > 1024 || ncol < 1) ? 1 : 1024 / ncol;
    if (S > lat.L) S = lat.L;
    out->S = (int)S;
    out->threads = (int)(((ncol * S + 31) / 32) * 32);
    out->lane = 0;
    out->cluster = 1;
    if (pow2) {    // power of two: lane-granular threads, index math by shifts
        const long long nlanes = lat.half / 4;
        // thread blocks of the cluster: >= 128 lanes (4 warps) each, at most 16 (B200 schedules 16-block clusters;
        // measured: profiles/r1_small_family.md) -- a half-sweep of a small lattice is bound by latency, not issue
        // ... except up to 512 lanes (64^2, 16^3): one block of <= 512 threads with bar.sync between the colours beats any
        // cluster and its barrier (64^2: 1.00 us per sweep against 1.15-1.29 for 2-16 blocks; 32^2: 0.60 against 1.16)
        int c = 1;
        if (nlanes > 512)
            while (c < small_max_cluster() && nlanes / (2 * c) >= 128 && 2 * c <= lat.L) c *= 2;
        if (N / c <= 196608) {                          // the slab must fit shared memory
            out->lane = 1;
            out->cluster = c;
            const long long per = nlanes / c;
            out->threads = (int)(per < 1024 ? ((per + 31) / 32) * 32 : 1024);
        }
    }
    if (!out->lane && (!words || ncol > 1024)) return false;
    if (!out->lane && !ignore_size_limit && N > 32768) return false;   // one SM: ~7.7 Gflips, the tiled family wins above
    return true;
}

cudaError_t launch_sweep_small(const Lat &lat, int model, int track, unsigned long long seed, unsigned long long t0,
                               int nsweeps, long long *d_obs, const SmallPlan &plan, const TiledTables &t,
                               cudaStream_t s)
{
    SmallArgs a;
    memset(&a, 0, sizeof(a));
    a.col[0] = lat.col[0];
    a.col[1] = lat.col[1];
    a.g.L = lat.L;
    a.g.R = lat.dims == 3 ? lat.L : 1;
    a.g.wpr = lat.Lh / 16;
    a.g.ncol = a.g.R * a.g.wpr;
    a.g.S = plan.S;
    a.g.one = 1;
    a.g.parity_rows = 0;                              // column_of: plain (row, word) order
    a.seed = seed;
    a.t0 = t0;
    a.nsweeps = nsweeps;
    a.obs = d_obs;
    PhiloxSweepConsts pk = make_philox_consts(make_sweep_key(seed, t0, 0u));   // only the round keys are used
    const bool obs = d_obs != nullptr, tr = track != 0;
    int lg_L = 0, lg_lpr = 0;
    if (plan.lane) {
        while ((1 << lg_L) < lat.L) ++lg_L;
        lg_lpr = lg_L - 3;                              // L/2 bytes per compact row = L/8 lanes
    }
    switch (model) {
    case M_ISING_HALF: {
        HalfTab ht;
        for (int i = 0; i < 16; ++i) ht.t[i] = t.t32[i];
        return lat.dims == 3 ? small_launch_to<M_ISING_HALF, 3>(tr, obs, plan.threads, s, a, pk, ht, lg_lpr, lg_L, plan.cluster)
                             : small_launch_to<M_ISING_HALF, 2>(tr, obs, plan.threads, s, a, pk, ht, lg_lpr, lg_L, plan.cluster);
    }
    case M_ISING_ONE: {
        OneTab ot;
        for (int i = 0; i < 64; ++i) ot.t[i] = t.s1[i];
        return lat.dims == 3 ? small_launch_to<M_ISING_ONE, 3>(tr, obs, plan.threads, s, a, pk, ot, lg_lpr, lg_L, plan.cluster)
                             : small_launch_to<M_ISING_ONE, 2>(tr, obs, plan.threads, s, a, pk, ot, lg_lpr, lg_L, plan.cluster);
    }
    case M_NE_HEATBATH: {
        NeTab nt = {t.ne_t32[0], 0, t.ne_all4};
        return small_launch_to<M_NE_HEATBATH, 2>(tr, obs, plan.threads, s, a, pk, nt, lg_lpr, lg_L, plan.cluster);
    }
    default: {
        NeTab nt = {t.ne_t32[1], t.ne_up_always, t.ne_all4};
        return small_launch_to<M_NE_METROPOLIS, 2>(tr, obs, plan.threads, s, a, pk, nt, lg_lpr, lg_L, plan.cluster);
    }
    }
}

// ------------------------------------------------------------------------------------------
// Batch: R replicas, one cluster each, one launch (lsm_batch_sweep*)
// ------------------------------------------------------------------------------------------
bool small_batch_supported(const Lat &lat, int model, const TiledTables &t)
{
    SmallPlan p;
    return small_plan(lat, model, t, &p, true) && p.lane == 1;
}

// Blocks per replica.  One lattice alone takes the largest cluster that keeps >= 4 warps per block (latency bound);
// R lattices together should fill the 148 SMs once and no more: smaller clusters mean cheaper barriers.
int small_batch_cluster(const Lat &lat, int R)
{
    const long long nlanes = lat.half / 4, N = 2 * lat.half;
    int cmax = 1;
    if (nlanes > 512)                                  // up to 512 lanes one block beats any cluster (see small_plan)
        while (cmax < small_max_cluster() && nlanes / (2 * cmax) >= 128 && 2 * cmax <= lat.L) cmax *= 2;
    int c = cmax;
    while (c > 1 && (long long)R * c > (long long)sm_count()) c >>= 1;   // measured: one block per SM beats two (32 x 128^2: c = 4)
    while (N / c > 196608 && c < 16) c <<= 1;          // the slab must fit shared memory
    while (nlanes / c > 2048 && c < 16) c <<= 1;       // at most two lanes per thread: the hoisted-geometry body
    return c;
}

template <int MODEL, int DIMS>
static cudaError_t small_batch_launch_to(bool track, bool obs, int threads, cudaStream_t s, const SmallBatchArgs &a,
                                         int nrep, int lg_lpr, int lg_L, int nclu)
{
    const size_t smem = ((size_t)1 << (DIMS * lg_L)) / (size_t)nclu;
    const int lg_rpc = lg_L - ilog2(nclu), lg_clu = ilog2(nclu);
    auto go = [&](auto kern) -> cudaError_t {
        if (smem > 48 * 1024) {
            cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (e != cudaSuccess) return e;
        }
        if (nclu > 8) {
            cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
            if (e != cudaSuccess) return e;
        }
        cudaLaunchConfig_t cfg;
        memset(&cfg, 0, sizeof(cfg));
        cfg.gridDim = dim3((unsigned)(nclu * nrep));
        cfg.blockDim = dim3((unsigned)threads);
        cfg.dynamicSmemBytes = smem;
        cfg.stream = s;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = (unsigned)nclu;
        at[0].val.clusterDim.y = 1;
        at[0].val.clusterDim.z = 1;
        cfg.attrs = at;
        cfg.numAttrs = 1;
        return cudaLaunchKernelEx(&cfg, kern, a, lg_lpr, lg_L, lg_rpc, lg_clu);
    };
    const size_t nl = (((size_t)1 << (DIMS * lg_L)) / 8) / (size_t)nclu;      // lanes per colour and block
    const int lpt = nl == (size_t)threads ? 1 : nl == 2 * (size_t)threads ? 2 : 0;
    auto pick = [&](auto T, auto O) -> cudaError_t {
        constexpr bool TR = decltype(T)::value;
        constexpr int OB = decltype(O)::value;
        if (lpt == 1) return go(k_sweep_small_lane_batch<MODEL, DIMS, TR, OB, 1>);
        if (lpt == 2) return go(k_sweep_small_lane_batch<MODEL, DIMS, TR, OB, 2>);
        return go(k_sweep_small_lane_batch<MODEL, DIMS, TR, OB, 0>);
    };
    using std::integral_constant;
    if (track) return obs ? pick(integral_constant<bool, true>{}, integral_constant<int, 2>{})
                          : pick(integral_constant<bool, true>{}, integral_constant<int, 0>{});
    return obs ? pick(integral_constant<bool, false>{}, integral_constant<int, 2>{})
               : pick(integral_constant<bool, false>{}, integral_constant<int, 0>{});
}

// d_obs: slot of replica 0 for the first sweep of this launch (replica r at d_obs + r * obs_stride) or nullptr;
// write_run: the last sweep's (B, M) also go to every replica's running pair.  Observables are formed iff d_obs or
// write_run.  Replicas beyond SMALL_BATCH_MAX take further launches.
cudaError_t launch_sweep_small_batch(const Lat &lat, int model, int track, const BatchDesc *d_desc, const uint64_t *seeds,
                                     int R, int cluster, unsigned long long t0, int nsweeps, long long *d_obs,
                                     long long obs_stride, int write_run, cudaStream_t s)
{
    int lg_L = 0;
    while ((1 << lg_L) < lat.L) ++lg_L;
    const int lg_lpr = lg_L - 3;
    const long long per = (lat.half / 4) / cluster;
    const int threads = (int)(per < 1024 ? ((per + 31) / 32) * 32 : 1024);
    const bool obs = d_obs != nullptr || write_run != 0, tr = track != 0;
    for (int r0 = 0; r0 < R; r0 += SMALL_BATCH_MAX) {
        const int nrep = R - r0 < SMALL_BATCH_MAX ? R - r0 : SMALL_BATCH_MAX;
        SmallBatchArgs a;
        memset(&a, 0, sizeof(a));
        a.desc = d_desc;
        a.obs = d_obs;
        a.obs_stride = obs_stride;
        a.t0 = t0;
        a.nsweeps = nsweeps;
        a.r0 = r0;
        a.write_run = write_run;
        a.one = 1;
        for (int i = 0; i < nrep; ++i) a.seed[i] = make_uint2((uint32_t)seeds[r0 + i], (uint32_t)(seeds[r0 + i] >> 32));
        cudaError_t e;
        switch (model) {
        case M_ISING_HALF:
            e = lat.dims == 3 ? small_batch_launch_to<M_ISING_HALF, 3>(tr, obs, threads, s, a, nrep, lg_lpr, lg_L, cluster)
                              : small_batch_launch_to<M_ISING_HALF, 2>(tr, obs, threads, s, a, nrep, lg_lpr, lg_L, cluster);
            break;
        case M_ISING_ONE:
            e = lat.dims == 3 ? small_batch_launch_to<M_ISING_ONE, 3>(tr, obs, threads, s, a, nrep, lg_lpr, lg_L, cluster)
                              : small_batch_launch_to<M_ISING_ONE, 2>(tr, obs, threads, s, a, nrep, lg_lpr, lg_L, cluster);
            break;
        case M_NE_HEATBATH:
            e = small_batch_launch_to<M_NE_HEATBATH, 2>(tr, obs, threads, s, a, nrep, lg_lpr, lg_L, cluster);
            break;
        default:
            e = small_batch_launch_to<M_NE_METROPOLIS, 2>(tr, obs, threads, s, a, nrep, lg_lpr, lg_L, cluster);
            break;
        }
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

}  // namespace lsmk
