// lsm_tiled.cu -- vectorised half-sweep kernels for sm_100a.
//
// Data layout: each colour array is [march][cross][word], one word = 16 consecutive
// bytes = 16 sites of one compact row.  2D: march = y, cross extent 1.  3D: march = z, cross = y.
// A thread owns one word column (cross row, word index) and a contiguous segment of the march axis:
// it walks that segment keeping the other colour's words at march-1, march, march+1 in registers, so
// every other-colour word along the march axis is loaded once per thread.  The remaining neighbours
// (3D: cross rows y+-1; the one byte left or right of the word) are plain loads that hit L1/L2.
// Adjacent threads own adjacent words, so all 128-bit accesses of a warp are contiguous.
//
// Per 32-bit lane of the word (4 sites) the thread makes exactly one Philox4x32-10 call (reading D2:
// group = byte offset >> 2), sums the neighbour bytes with plain 32-bit adds (no carries: a byte
// never exceeds 2d), looks the four thresholds up in shared memory and folds the four compare
// results into the lane with predicated adds.  Nothing branches on lattice data.
//
// What binds (measured): on B200 an IMAD.WIDE occupies the FMA-heavy pipe for 4 cycles
// AND one issue slot of the 16-lane ALU pipe, so a warp needs 2*(ALU instructions + wide multiplies)
// cycles per step.  The rule code is therefore written to spend as few ALU-pipe instructions as it
// can: table indexed by (spin, up-neighbour count) so no "aligned count" is formed, "w <= thr-1"
// compares so certain acceptance needs no mask, compare results merged with predicated IMAD adds
// (FMA pipe), row parity known at compile time so the side neighbour costs one funnel shift.
#include "lsm_tiled_dev.cuh"

#include <cstdlib>
#include <cstring>

// up-concentration from which the North-East rule runs the four Philox calls of a word together (see update_word)
#define LSM_NE_ALL4_C 0.25

#define LSM_TILED_THREADS 256            // threads per CTA (<= 256: the ring has 256 slots per stage)

namespace lsmk {

cudaError_t launch_sweep_tiled_bulk(int model, bool track, int obs_mode, TiledGeom g, const PhiloxSweepConsts &pc,
                                    const TiledTables &t, cudaStream_t s);

PhiloxSweepConsts make_philox_consts(const SweepKey &k)
{
    PhiloxSweepConsts c;
    for (int r = 0; r < 10; ++r) {
        c.rk0[r] = k.k0 + (uint32_t)r * PHILOX_W0;
        c.rk1[r] = k.k1 + (uint32_t)r * PHILOX_W1;
    }
    philox_half_consts(k, c.rk0, c.rk1, c.x1, c.y2, c.z2, c.w3);
    c.m0 = PHILOX_M0;
    c.m1 = PHILOX_M1;
    return c;
}

template <int MODEL, int DIMS, bool TRACK, int OBS, bool NEV>
__global__ void __launch_bounds__(LSM_TILED_THREADS, tiled_minblocks(MODEL))
k_sweep_tiled(const __grid_constant__ TiledGeom g, const __grid_constant__ PhiloxSweepConsts pc,
              const __grid_constant__ typename TabOf<MODEL>::type tab, const __grid_constant__ NevTab ytab)
{
    __shared__ __align__(16) struct {
        uint32_t t[(MODEL == M_ISING_ONE ? 64 : 16) * (NEV ? 2 : 1)];   // NEV: the y table behind the t table
        long long red[2][8];
    } sm;
    // two-stage per-thread ring of the asynchronous copies (March::step_pf): N, O [, Yp, Yn] words and the edge lane
    // (spin-1 keeps the direct loads: its rule needs the registers the copies' addresses would take)
    constexpr bool PF = MODEL != M_ISING_ONE && MODEL != M_POTTS;   // two-word rules load directly (the ring measured slower there)
    __shared__ __align__(16) uint4 ring[PF ? ((DIMS == 3 ? 8 : 4) + (MODEL == M_EA ? 2 : 0)) * 256 : 1];
    __shared__ uint32_t ringE[PF ? 2 * 256 : 1];
    // Programmatic dependent launch: the next half-sweep's CTAs may be scheduled as soon as SM resources
    // free up; they run their prologue (table, geometry) and then wait below until this grid has
    // completed and flushed -- the kernel boundary stays the barrier of PAPER.md:96,108, only the
    // launch latency and ramp are taken off the critical path.
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    uint32_t s_t = (uint32_t)__cvta_generic_to_shared(sm.t);
    asm volatile("" : "+r"(s_t));   // keep the (warp-uniform) table address out of the divergent region below
    March<MODEL, DIMS, TRACK, OBS, NEV> M;
    M.ne_t32 = 0;
    M.ne_always = 0;
    M.ne_all4 = false;
    M.potts_qm1 = (uint32_t)g.qm1;
    if constexpr (MODEL == M_ISING_HALF || MODEL == M_EA || MODEL == M_POTTS) {
        if (threadIdx.x < 16) sm.t[threadIdx.x] = tab.t[threadIdx.x];
        if (NEV && threadIdx.x < 16) sm.t[16 + threadIdx.x] = ytab.y[threadIdx.x];
    } else if constexpr (MODEL == M_ISING_ONE) {
        if (threadIdx.x < 64) sm.t[threadIdx.x] = tab.t[threadIdx.x];
        if (NEV && threadIdx.x < 64) sm.t[64 + threadIdx.x] = ytab.y[threadIdx.x];
    } else {
        M.ne_t32 = tab.t32;
        M.ne_always = tab.always;
        M.ne_all4 = tab.all4 != 0;
    }
    __syncthreads();
    asm volatile("griddepcontrol.wait;" ::: "memory");   // the previous launch's spins are visible from here on
    M.s_t = s_t;
    M.one = (uint32_t)g.one;
    M.totU = M.totBN = M.totS = 0;
    M.s_ring = (uint32_t)__cvta_generic_to_shared(ring) + threadIdx.x * 16u;
    M.s_ringE = (uint32_t)__cvta_generic_to_shared(ringE) + threadIdx.x * 4u;

    const long long gt = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    int nsites = 0;
    if (gt < (long long)g.ncol * g.S) {
        const int seg = (int)(gt / g.ncol);
        const int col = (int)(gt - (long long)seg * g.ncol);
        const int n = march_init(M, g, g.own, g.oth, g.half, seg, col, true);
        nsites = 16 * n;
        if constexpr (!PF) {
            M.template run1<true>(n, pc);
        } else
        if (g.parity_rows) {            // warp-uniform branch: q is a constant inside each loop
            if (M.q) PF ? M.template run_pf<1, true>(n, pc) : M.template run<1, true>(n, pc);
            else PF ? M.template run_pf<0, true>(n, pc) : M.template run<0, true>(n, pc);
        } else {
            PF ? M.template run_pf<2, true>(n, pc) : M.template run<2, true>(n, pc);
        }
    }

    if (OBS >= 1) {
        long long cB, cM;
        march_observables(M, nsites, OBS >= 2, cB, cM);   // OBS = 1: first colour, 2: second colour
        block_accumulate2_in(sm.red, cB, cM, g.obs, true, true);
    }
}

// ------------------------------------------------------------------------------------------
// Host side
// ------------------------------------------------------------------------------------------
void build_tiled_tables(int model, int dims, double J, double h, const uint64_t *thr, int nthr, TiledTables *out)
{
    TiledTables t;
    memset(&t, 0, sizeof(t));
    const uint64_t ALWAYS = (uint64_t)1 << 32;
    auto clip = [&](uint64_t v) { return v >= ALWAYS ? 0xFFFFFFFFu : (uint32_t)v; };
    const int d = dims;
    (void)J; (void)h; (void)nthr;
    if (model == M_POTTS) {
        // reading D26: thr[dn + 2d], 4d + 1 <= 13 entries, indexed directly
        t.usable = 1;
        for (int j = 0; j <= 4 * d; ++j) {
            const uint64_t v = thr[j];
            if (v == 0) t.has_never = 1;
            t.t32[j] = v == 0 ? 0u : (uint32_t)(v - 1);
            t.y32[j] = v == 0 ? 1u : 0u;
        }
    } else if (model == M_ISING_HALF || model == M_EA) {
        t.usable = 1;
        for (int b = 0; b < 2; ++b)
            for (int n = 0; n <= 2 * d; ++n) {
                uint64_t v = thr[b * (2 * d + 1) + n];
                if (v == 0) t.has_never = 1;               // "never" cannot be written as w <= thr-1: NEV kernels
                t.t32[n + 8 * b] = v == 0 ? 0u : (uint32_t)(v - 1);
                t.y32[n + 8 * b] = v == 0 ? 1u : 0u;
            }
    } else if (model == M_ISING_ONE) {
        t.usable = 1;
        // canonical table: idx = ((a*2 + kk) * (4d+1) + sum), a' = (a + 1 + kk) % 3.  Classes of s' - s and one
        // representative (a, kk) each; the others must carry the same thresholds.
        const int W = 4 * d + 1;
        const int rep[4][2] = {{0, 0}, {0, 1}, {1, 1}, {2, 0}};          // +1, +2, -1, -2
        const int cls[3][2] = {{0, 1}, {0, 2}, {3, 2}};                  // dcode of (a, kk)
        for (int a = 0; a < 3; ++a)
            for (int kk = 0; kk < 2; ++kk)
                for (int s = 0; s < W; ++s)
                    if (thr[(a * 2 + kk) * W + s] != thr[(rep[cls[a][kk]][0] * 2 + rep[cls[a][kk]][1]) * W + s]) t.usable = 0;
        for (int c = 0; c < 4; ++c)
            for (int s = 0; s < W; ++s) {
                uint64_t v = thr[(rep[c][0] * 2 + rep[c][1]) * W + s];
                if (v == 0) t.has_never = 1;
                t.s1[c * 16 + s] = v == 0 ? 0u : (uint32_t)(v - 1);
                t.y32[c * 16 + s] = v == 0 ? 1u : 0u;
            }
    } else {
        t.usable = 1;
        t.ne_t32[0] = clip(thr[0]);
        t.ne_t32[1] = clip(thr[1]);
        t.ne_up_always = thr[1] == ALWAYS ? 1 : 0;
        t.ne_all4 = (double)thr[0] >= LSM_NE_ALL4_C * 4294967296.0 ? 1 : 0;
        if (thr[0] == ALWAYS) t.usable = 0;
    }
    *out = t;
}

bool tiled_supported(const Lat &lat, int model, const TiledTables &t)
{
    if (!t.usable) return false;
    if (lat.Lh % 16 != 0) return false;                    // whole 16-byte words per compact row
    if (lat.half / 4 > 0xFFFFFFFFll) return false;         // Philox group must fit c0 (c1 = 0 is hoisted)
    if ((model == M_ISING_ONE || model == M_POTTS) && lat.half / 2 > 0xFFFFFFFFll) return false;
    return true;
}

// Launch shape: threads = word columns x march segments, one wave of CTAS_PER_SM resident CTAs per
// SM (finer segments do not help: measured, profiles/).  Compile-time knobs for tuning experiments
// (-DLSM_TILED_...); the library reads no environment variables.
#define LSM_TILED_CTAS_PER_SM 0          // 0: tiled_minblocks(model)
#define LSM_TILED_WAVES_X4 4             // waves in quarters
#define LSM_TILED_PDL 1                  // programmatic dependent launch
static const int g_tiled_ctas_per_sm = LSM_TILED_CTAS_PER_SM;
static const int g_tiled_waves_x4 = LSM_TILED_WAVES_X4;
static const int g_tiled_pdl = LSM_TILED_PDL;

template <int MODEL, int DIMS, bool TRACK, bool NEV>
static cudaError_t launch_obs(int obs_mode, dim3 grid, cudaStream_t s, const TiledGeom &g, const PhiloxSweepConsts &pc,
                              const typename TabOf<MODEL>::type &tab, const NevTab &yt)
{
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof(cfg));
    cfg.gridDim = grid;
    cfg.blockDim = dim3(LSM_TILED_THREADS);
    cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = g_tiled_pdl ? 1 : 0;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    if (obs_mode == 0) return cudaLaunchKernelEx(&cfg, k_sweep_tiled<MODEL, DIMS, TRACK, 0, NEV>, g, pc, tab, yt);
    if (obs_mode == 1) return cudaLaunchKernelEx(&cfg, k_sweep_tiled<MODEL, DIMS, TRACK, 1, NEV>, g, pc, tab, yt);
    return cudaLaunchKernelEx(&cfg, k_sweep_tiled<MODEL, DIMS, TRACK, 2, NEV>, g, pc, tab, yt);
}

template <int MODEL, int DIMS>
static cudaError_t launch_track(bool track, int obs_mode, dim3 grid, cudaStream_t s, const TiledGeom &g,
                                const PhiloxSweepConsts &pc, const typename TabOf<MODEL>::type &tab,
                                const TiledTables *nev = nullptr)
{
    NevTab yt;
    memset(&yt, 0, sizeof(yt));
    constexpr bool CAN_NEV = MODEL == M_ISING_HALF || MODEL == M_ISING_ONE || MODEL == M_EA || MODEL == M_POTTS;
    if constexpr (CAN_NEV) {
        if (nev && nev->has_never) {                       // a table with a "never" entry: the two-compare kernels
            for (int i = 0; i < 64; ++i) yt.y[i] = nev->y32[i];
            if (track) return launch_obs<MODEL, DIMS, true, true>(obs_mode, grid, s, g, pc, tab, yt);
            return launch_obs<MODEL, DIMS, false, true>(obs_mode, grid, s, g, pc, tab, yt);
        }
    }
    if (track) return launch_obs<MODEL, DIMS, true, false>(obs_mode, grid, s, g, pc, tab, yt);
    return launch_obs<MODEL, DIMS, false, false>(obs_mode, grid, s, g, pc, tab, yt);
}

cudaError_t launch_sweep_tiled(const SweepArgs &a, const TiledTables &t, cudaStream_t s)
{
    TiledGeom g;
    g.own = a.half ? a.lat.col[1] : a.lat.col[0];
    g.oth = a.half ? a.lat.col[0] : a.lat.col[1];
    g.L = a.lat.L;
    g.R = a.lat.dims == 3 ? a.lat.L : 1;
    g.wpr = a.lat.Lh / 16;
    g.ncol = g.R * g.wpr;
    g.half = a.half;
    g.obs = a.obs;
    g.one = 1;
    g.bnd = a.model == M_EA ? (a.half ? a.lat.bnd[1] : a.lat.bnd[0]) : nullptr;
    g.qm1 = a.model == M_POTTS ? a.lat.q - 1 : 0;
    // q = (march + y + colour) & 1 is warp-uniform if a warp sees one row parity only
    if (g.R == 1) g.parity_rows = 1;                                   // 2D: y = 0 for every thread
    else if (g.wpr % 32 == 0) g.parity_rows = 1;
    else if (g.wpr < 32 && 32 % g.wpr == 0 && g.R % (2 * (32 / g.wpr)) == 0) g.parity_rows = 1;
    else g.parity_rows = 0;
    const int per_sm = g_tiled_ctas_per_sm > 0 ? g_tiled_ctas_per_sm : tiled_minblocks(a.model);
    long long target = (long long)sm_count() * per_sm * LSM_TILED_THREADS * g_tiled_waves_x4 / 4;
    long long S = target / g.ncol;
    if (S < 1) S = 1;
    if (S > g.L) S = g.L;
    g.S = (int)S;
    long long threads = (long long)g.ncol * g.S;
    dim3 grid((unsigned)((threads + LSM_TILED_THREADS - 1) / LSM_TILED_THREADS));

    PhiloxSweepConsts pc = make_philox_consts(a.key);
    int obs_mode = a.obs ? (a.want_B ? 2 : 1) : 0;
    const bool track = a.track != 0;
    if (a.bulk && tiled_bulk_supported(a.lat, a.model, t)) return launch_sweep_tiled_bulk(a.model, track, obs_mode, g, pc, t, s);
    const bool d3 = a.lat.dims == 3;
    switch (a.model) {
    case M_ISING_HALF: {
        HalfTab ht;
        for (int i = 0; i < 16; ++i) ht.t[i] = t.t32[i];
        return d3 ? launch_track<M_ISING_HALF, 3>(track, obs_mode, grid, s, g, pc, ht, &t)
                  : launch_track<M_ISING_HALF, 2>(track, obs_mode, grid, s, g, pc, ht, &t);
    }
    case M_EA: {
        HalfTab ht;
        for (int i = 0; i < 16; ++i) ht.t[i] = t.t32[i];
        return d3 ? launch_track<M_EA, 3>(track, obs_mode, grid, s, g, pc, ht, &t)
                  : launch_track<M_EA, 2>(track, obs_mode, grid, s, g, pc, ht, &t);
    }
    case M_ISING_ONE: {
        OneTab ot;
        for (int i = 0; i < 64; ++i) ot.t[i] = t.s1[i];
        return d3 ? launch_track<M_ISING_ONE, 3>(track, obs_mode, grid, s, g, pc, ot, &t)
                  : launch_track<M_ISING_ONE, 2>(track, obs_mode, grid, s, g, pc, ot, &t);
    }
    case M_POTTS: {
        HalfTab ht;
        for (int i = 0; i < 16; ++i) ht.t[i] = t.t32[i];
        return d3 ? launch_track<M_POTTS, 3>(track, obs_mode, grid, s, g, pc, ht, &t)
                  : launch_track<M_POTTS, 2>(track, obs_mode, grid, s, g, pc, ht, &t);
    }
    case M_NE_HEATBATH: {
        NeTab nt = {t.ne_t32[0], 0, t.ne_all4};
        return launch_track<M_NE_HEATBATH, 2>(track, obs_mode > 1 ? 1 : obs_mode, grid, s, g, pc, nt);
    }
    default: {
        NeTab nt = {t.ne_t32[1], t.ne_up_always, t.ne_all4};
        return launch_track<M_NE_METROPOLIS, 2>(track, obs_mode > 1 ? 1 : obs_mode, grid, s, g, pc, nt);
    }
    }
}

}  // namespace lsmk
