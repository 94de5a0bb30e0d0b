// lsm_tiled_bulk.cu -- the half-sweep kernel of the tiled family with its rows staged through shared memory by bulk
// asynchronous copies (TMA unit, cp.async.bulk + mbarrier) instead of per-thread cp.async (BASELINE.json north_star:
// "neighbour rows ... of the other sublattice are staged through shared memory"; tile and boundaries to
// shared memory).  2D lattices whose compact rows are whole multiples of 256 words (L a multiple of 8192).
//
// A CTA owns 256 adjacent word columns (4 KB of a compact row) and a segment of rows; 8 consumer warps march along the
// segment exactly as in lsm_tiled.cu (one word column per thread, other-colour words of the rows below and at the
// current one in registers, March::update_word), a ninth warp is the producer: one thread issues, per row, one bulk
// copy of the other colour's 4 KB (+ the 16-byte words left and right of it: the edge lanes, periodic in x) and one
// of the own colour's 4 KB into a 4-stage ring, each stage behind a "full" mbarrier armed with the byte count; the
// consumers wait on it, read their 16-byte words with LDS.128, and one lane per warp arrives on the stage's "empty"
// mbarrier when the warp is done with it.  No per-thread address arithmetic, no LDGSTS, two rows of look-ahead.
#include "lsm_tiled_dev.cuh"

#include <cstring>

namespace lsmk {

constexpr int BULK_STAGES = 4;
struct __align__(16) BulkStage {
    uint4 lh;           // other colour: the word left of the chunk (last lane = west neighbour of the chunk's first site)
    uint4 oth[256];     // other colour, row r
    uint4 rh;           // ... the word right of the chunk
    uint4 own[256];     // own colour, row r
};

__device__ __forceinline__ uint32_t bulk_s32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "LSM_WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra LSM_DONE_%=;\n\t"
        "bra LSM_WAIT_%=;\n\t"
        "LSM_DONE_%=:\n\t}" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst), "l"(src),
                 "r"(bytes), "r"(bar) : "memory");
}

template <int MODEL, bool TRACK, int OBS, bool NEV>
__global__ void __launch_bounds__(288, 2)
k_sweep_tiled_bulk(const __grid_constant__ TiledGeom g, const __grid_constant__ PhiloxSweepConsts pc,
                   const __grid_constant__ typename TabOf<MODEL>::type tab, const __grid_constant__ NevTab ytab)
{
    __shared__ __align__(128) BulkStage st[BULK_STAGES];
    __shared__ __align__(8) unsigned long long bar_full[BULK_STAGES], bar_empty[BULK_STAGES];
    __shared__ __align__(16) struct {
        uint32_t t[16 * (NEV ? 2 : 1)];
        long long red[2][9];
    } sm;
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    const uint32_t tid = threadIdx.x, warp = tid >> 5, lane = tid & 31u;
    uint32_t s_t = bulk_s32(sm.t);
    asm volatile("" : "+r"(s_t));
    March<MODEL, 2, TRACK, OBS, NEV> M;
    M.ne_t32 = 0;
    M.ne_always = 0;
    M.ne_all4 = false;
    if constexpr (MODEL == M_ISING_HALF) {
        if (tid < 16) sm.t[tid] = tab.t[tid];
        if (NEV && tid < 16) sm.t[16 + tid] = ytab.y[tid];
    } else {
        M.ne_t32 = tab.t32;
        M.ne_always = tab.always;
        M.ne_all4 = tab.all4 != 0;
    }
    if (tid == 0) {
        for (int s = 0; s < BULK_STAGES; ++s) {
            mbar_init(bulk_s32(&bar_full[s]), 1u);         // the producer's arrive.expect_tx
            mbar_init(bulk_s32(&bar_empty[s]), 8u);        // one lane of each consumer warp
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    asm volatile("griddepcontrol.wait;" ::: "memory");   // the previous launch's spins are visible from here on

    const int nb = g.wpr >> 8;                             // 256-word chunks per compact row
    const int seg = (int)blockIdx.x / nb, cb = (int)blockIdx.x - seg * nb;
    const int m0 = (int)(((long long)g.L * seg) / g.S), m1 = (int)(((long long)g.L * (seg + 1)) / g.S);
    const int n = m1 - m0;
    long long cB = 0, cM = 0;

    if (warp == 8u) {
        // ---- producer: item k = row m0 - 1 + k, k = 0 ... n + 1 (own colour for 1 <= k <= n) -> stage k & 3
        if (lane == 0u) {
            const uint32_t wl = (uint32_t)((cb * 256 - 1 + g.wpr) % g.wpr), wr = (uint32_t)((cb * 256 + 256) % g.wpr);
            for (int k = 0; k <= n + 1; ++k) {
                const int s = k & (BULK_STAGES - 1);
                if (k >= BULK_STAGES) mbar_wait(bulk_s32(&bar_empty[s]), (uint32_t)(((k >> 2) - 1) & 1));
                int r = m0 - 1 + k;
                r = r < 0 ? r + g.L : (r >= g.L ? r - g.L : r);
                const size_t row = (size_t)r * (size_t)g.wpr;
                const bool own = k >= 1 && k <= n;
                const uint32_t bar = bulk_s32(&bar_full[s]);
                mbar_expect_tx(bar, 4096u + 32u + (own ? 4096u : 0u));
                bulk_g2s(bulk_s32(st[s].oth), g.oth + (row + (size_t)cb * 256u) * 16u, 4096u, bar);
                bulk_g2s(bulk_s32(&st[s].lh), g.oth + (row + wl) * 16u, 16u, bar);
                bulk_g2s(bulk_s32(&st[s].rh), g.oth + (row + wr) * 16u, 16u, bar);
                if (own) bulk_g2s(bulk_s32(st[s].own), g.own + (row + (size_t)cb * 256u) * 16u, 4096u, bar);
            }
        }
    } else {
        // ---- consumers
        M.s_t = s_t;
        M.one = (uint32_t)g.one;
        M.totU = M.totBN = M.totS = 0;
        M.grp = (uint32_t)(((size_t)m0 * (size_t)g.wpr + (size_t)cb * 256u + tid) * 4u);
        const uint32_t gstep = (uint32_t)g.wpr * 4u;
        uint4 *pO = reinterpret_cast<uint4 *>(g.own) + ((size_t)m0 * (size_t)g.wpr + (size_t)cb * 256u + tid);
        const uint32_t e_hi = 4u + (tid + 1u) * 4u, e_lo = 4u + tid * 4u - 1u;   // lanes of a stage: lh | oth[256] | rh
        auto release = [&](int s) {
            __syncwarp();
            if (lane == 0u) mbar_arrive(bulk_s32(&bar_empty[s]));
        };
        mbar_wait(bulk_s32(&bar_full[0]), 0u);
        M.P = st[0].oth[tid];
        release(0);
        mbar_wait(bulk_s32(&bar_full[1]), 0u);
        M.C = st[1].oth[tid];
        const uint4 Z = make_uint4(0u, 0u, 0u, 0u);
        auto step = [&](auto QC, int i) {
            constexpr int Q = decltype(QC)::value;
            const int sN = (i + 2) & (BULK_STAGES - 1), sC = (i + 1) & (BULK_STAGES - 1);
            mbar_wait(bulk_s32(&bar_full[sN]), (uint32_t)(((i + 2) >> 2) & 1));
            const uint4 N = st[sN].oth[tid];
            const uint4 O = st[sC].own[tid];
            const uint32_t e = reinterpret_cast<const uint32_t *>(&st[sC])[Q ? e_hi : e_lo];
            release(sC);
            const uint4 out = M.template update_word<Q, true>(pc, N, O, e, Z, Z);
            *pO = out;
            pO += g.wpr;
            M.P = M.C;
            M.C = N;
            M.grp += gstep;
        };
        using Q0 = std::integral_constant<int, 0>;
        using Q1 = std::integral_constant<int, 1>;
        const int q0 = (m0 + g.half) & 1;                  // 2D: the row parity bit q = (m + colour) & 1 is CTA-uniform
        int i = 0;
        if (q0) {
            for (; i + 1 < n; i += 2) { step(Q1{}, i); step(Q0{}, i + 1); }
            if (i < n) step(Q1{}, i);
        } else {
            for (; i + 1 < n; i += 2) { step(Q0{}, i); step(Q1{}, i + 1); }
            if (i < n) step(Q0{}, i);
        }
        if (OBS >= 1) march_observables(M, 16 * n, OBS >= 2, cB, cM);   // OBS = 1: first colour, 2: second colour
    }

    if (OBS >= 1) {
        cB = warp_sum(cB);
        cM = warp_sum(cM);
        if (lane == 0u) { sm.red[0][warp] = cB; sm.red[1][warp] = cM; }
        __syncthreads();
        if (tid == 0) {
            long long b = 0, m = 0;
            for (int w = 0; w < 8; ++w) { b += sm.red[0][w]; m += sm.red[1][w]; }
            if (b != 0) atomicAdd((unsigned long long *)&g.obs[0], (unsigned long long)b);
            if (m != 0) atomicAdd((unsigned long long *)&g.obs[1], (unsigned long long)m);
        }
    }
}

// ------------------------------------------------------------------------------------------
// Host side
// ------------------------------------------------------------------------------------------
bool tiled_bulk_supported(const Lat &lat, int model, const TiledTables &t)
{
    if (!t.usable || lat.dims != 2) return false;
    if (model != M_ISING_HALF && model != M_NE_HEATBATH && model != M_NE_METROPOLIS) return false;
    return (lat.Lh / 16) % 256 == 0;                       // whole 256-word chunks per compact row
}

template <int MODEL, bool TRACK, bool NEV>
static cudaError_t bulk_launch_obs(int obs_mode, dim3 grid, cudaStream_t s, const TiledGeom &g, const PhiloxSweepConsts &pc,
                                   const typename TabOf<MODEL>::type &tab, const NevTab &yt)
{
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cfg.gridDim = grid;
    cfg.blockDim = dim3(288);
    cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    if (obs_mode == 0) return cudaLaunchKernelEx(&cfg, k_sweep_tiled_bulk<MODEL, TRACK, 0, NEV>, g, pc, tab, yt);
    if (obs_mode == 1) return cudaLaunchKernelEx(&cfg, k_sweep_tiled_bulk<MODEL, TRACK, 1, NEV>, g, pc, tab, yt);
    return cudaLaunchKernelEx(&cfg, k_sweep_tiled_bulk<MODEL, TRACK, 2, NEV>, g, pc, tab, yt);
}

// g: geometry as launch_sweep_tiled fills it (own, oth, L, wpr, half, obs, one); S and the grid are chosen here.
cudaError_t launch_sweep_tiled_bulk(int model, bool track, int obs_mode, TiledGeom g, const PhiloxSweepConsts &pc,
                                    const TiledTables &t, cudaStream_t s)
{
    const int nb = g.wpr / 256;
    long long S = (long long)sm_count() * 2 / nb;          // one wave of two CTAs per SM
    if (S < 1) S = 1;
    if (S > g.L) S = g.L;
    g.S = (int)S;
    dim3 grid((unsigned)(S * nb));
    NevTab yt;
    memset(&yt, 0, sizeof(yt));
    for (int i = 0; i < 64; ++i) yt.y[i] = t.y32[i];
    switch (model) {
    case M_ISING_HALF: {
        HalfTab ht;
        for (int i = 0; i < 16; ++i) ht.t[i] = t.t32[i];
        if (t.has_never)
            return track ? bulk_launch_obs<M_ISING_HALF, true, true>(obs_mode, grid, s, g, pc, ht, yt)
                         : bulk_launch_obs<M_ISING_HALF, false, true>(obs_mode, grid, s, g, pc, ht, yt);
        return track ? bulk_launch_obs<M_ISING_HALF, true, false>(obs_mode, grid, s, g, pc, ht, yt)
                     : bulk_launch_obs<M_ISING_HALF, false, false>(obs_mode, grid, s, g, pc, ht, yt);
    }
    case M_NE_HEATBATH: {
        NeTab nt = {t.ne_t32[0], 0, t.ne_all4};
        const int om = obs_mode > 1 ? 1 : obs_mode;
        return track ? bulk_launch_obs<M_NE_HEATBATH, true, false>(om, grid, s, g, pc, nt, yt)
                     : bulk_launch_obs<M_NE_HEATBATH, false, false>(om, grid, s, g, pc, nt, yt);
    }
    default: {
        NeTab nt = {t.ne_t32[1], t.ne_up_always, t.ne_all4};
        const int om = obs_mode > 1 ? 1 : obs_mode;
        return track ? bulk_launch_obs<M_NE_METROPOLIS, true, false>(om, grid, s, g, pc, nt, yt)
                     : bulk_launch_obs<M_NE_METROPOLIS, false, false>(om, grid, s, g, pc, nt, yt);
    }
    }
}

}  // namespace lsmk
