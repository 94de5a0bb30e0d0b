// lsm_resident.cu -- the resident kernel family: ONE launch runs many sweeps.
//
// The paper ends the kernel after every half-sweep because its GPUs had no other grid-wide barrier
// (PAPER.md:96,108).  On B200 a 32 us half-sweep of the 8192^2 lattice loses ~13 % of its time to
// launch ramp and tail (profiles/r1_tiled_ncu_full.md), and a grid-wide barrier is more than the
// method needs: a site of one colour reads only its 2d nearest neighbours, so the thread block that
// owns a slab of the lattice depends only on the blocks that own the adjacent slabs.
//
// Every CTA stays resident (cooperative launch: all CTAs are co-scheduled) and keeps the thread ->
// (march segment, word column) map of the tiled family for the whole launch.  The march direction
// alternates: even half-sweeps of a launch walk a segment upwards, odd ones downwards.  Then the row
// a CTA needs first from the neighbour segment on its starting side is the row that neighbour wrote
// FIRST in the previous half-sweep, and the row it needs last is the one the other neighbour wrote
// LAST -- both dependencies (read-after-write on the neighbour's new spins, write-after-read on the
// colour about to be overwritten) are met almost a whole half-sweep early, so CTAs drift freely
// instead of marching in lock step.  Two progress words per CTA: first[c] = half-sweeps whose first
// row is stored, done[c] = half-sweeps completed.
//   start of half-sweep g : wait first[start-side neighbour] >= g, done[cross-axis neighbours] >= g
//   after the first row   : first[me] = g + 1
//   before the last row   : wait done[end-side neighbour] >= g
//   end                   : done[me] = g + 1
// Publishing is bar.sync -> fence.acq_rel.gpu -> st.relaxed by one thread; waiting is ld.relaxed
// polling -> fence.acq_rel.gpu -> bar.sync, so the ordinary (L1-cached) lattice loads that follow
// observe the neighbours' stores (PTX memory model: release/acquire patterns composed with the CTA
// barrier -- the protocol of a grid-wide sync, restricted to the real dependencies).
// The arithmetic of a half-sweep is the tiled family's March, unchanged (sites of one colour are
// independent, so the visiting order cannot matter): bit-identical results.
#include "lsm_tiled_dev.cuh"

#include <cstdlib>
#include <cstring>

namespace lsmk {

struct ResidentArgs {
    uint8_t *col[2];
    TiledGeom g;                 // geometry; own/oth/half/obs are set per half-sweep on the device
    unsigned long long seed, t0; // first sweep of this launch
    int nsweeps;
    int nb;                      // CTAs per march segment (= ncol / threads per CTA)
    long long *obs;              // [nsweeps][2] (B, M) slots, zeroed by the host; or nullptr
    unsigned *flags;             // first[grid] then done[grid]: progress words of every CTA
    unsigned epoch0;             // value of every flag when the launch starts
};

__device__ __forceinline__ unsigned ld_relaxed_gpu(const unsigned *p)
{
    unsigned v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_relaxed_gpu(unsigned *p, unsigned v)
{
    asm volatile("st.relaxed.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// Progress flags of one CTA's half-sweep (see the header comment).
struct ResidentHooks {
    unsigned *first_me;
    const unsigned *done_end;    // done[] word of the neighbour on the side where the march ends
    unsigned need;               // epoch0 + g
    __device__ __forceinline__ void after_first()
    {
        __syncthreads();
        if (threadIdx.x == 0) {
            __threadfence();
            st_relaxed_gpu(first_me, need + 1u);
        }
    }
    __device__ __forceinline__ void before_last()
    {
        if (threadIdx.x == 0) {
            while ((int)(ld_relaxed_gpu(done_end) - need) < 0) __nanosleep(32);
            __threadfence();
        }
        __syncthreads();
    }
};

// OBS: 0 = no observables, 2 = per-sweep (B, M) into a.obs[sweep].
template <int MODEL, int DIMS, bool TRACK, int OBS>
__global__ void __launch_bounds__(256, LSM_TILED_MINBLOCKS)
k_sweep_resident(const __grid_constant__ ResidentArgs a, const __grid_constant__ PhiloxSweepConsts pk,
                 const __grid_constant__ typename TabOf<MODEL>::type tab)
{
    __shared__ __align__(16) struct {
        uint32_t t[MODEL == M_ISING_ONE ? 64 : 16];
        long long red[2][8];
    } sm;
    uint32_t s_t = (uint32_t)__cvta_generic_to_shared(sm.t);
    asm volatile("" : "+r"(s_t));
    if constexpr (MODEL == M_ISING_HALF) {
        if (threadIdx.x < 16) sm.t[threadIdx.x] = tab.t[threadIdx.x];
    } else if constexpr (MODEL == M_ISING_ONE) {
        for (int i = threadIdx.x; i < 64; i += blockDim.x) sm.t[i] = tab.t[i];
    }
    __syncthreads();

    constexpr bool NE = MODEL == M_NE_HEATBATH || MODEL == M_NE_METROPOLIS;
    const int seg = blockIdx.x / a.nb, cb = blockIdx.x - seg * a.nb;
    const int col = cb * blockDim.x + threadIdx.x;
    const int ncta = gridDim.x;
    unsigned *const first = a.flags, *const done = a.flags + ncta;
    const int below = (seg == 0 ? a.g.S - 1 : seg - 1) * a.nb + cb;      // march-axis neighbours
    const int above = (seg + 1 == a.g.S ? 0 : seg + 1) * a.nb + cb;

    const int nhalves = 2 * a.nsweeps;
#pragma unroll 1
    for (int gh = 0; gh < nhalves; ++gh) {
        const int half = gh & 1;
        const bool up = half == 0;                  // nhalves is even: directions alternate across sweeps too
        const unsigned long long t = a.t0 + (unsigned long long)(gh >> 1);
        const unsigned need = a.epoch0 + (unsigned)gh;
        if (gh > 0) {
            if (threadIdx.x < 3) {
                const unsigned *w = first + (up ? below : above);                             // start side
                if (threadIdx.x == 1) w = done + seg * a.nb + (cb == 0 ? a.nb - 1 : cb - 1);  // cross axis
                if (threadIdx.x == 2) w = done + seg * a.nb + (cb + 1 == a.nb ? 0 : cb + 1);
                while ((int)(ld_relaxed_gpu(w) - need) < 0) __nanosleep(32);
                __threadfence();
            }
            __syncthreads();
        }
        ResidentHooks hk = {first + blockIdx.x, done + (up ? above : below), need};

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
        const int n = march_init(M, a.g, a.col[half], a.col[half ^ 1], half, seg, col, up);
        // The direction is a compile-time constant only where the rule needs it (North-East: north = y + 1).
        if (NE && !up) {
            if (a.g.parity_rows) {
                if (M.q) M.template run_hooked<1, !NE>(n, pc, hk);
                else M.template run_hooked<0, !NE>(n, pc, hk);
            } else {
                M.template run_hooked<2, !NE>(n, pc, hk);
            }
        } else {
            if (a.g.parity_rows) {
                if (M.q) M.template run_hooked<1, true>(n, pc, hk);
                else M.template run_hooked<0, true>(n, pc, hk);
            } else {
                M.template run_hooked<2, true>(n, pc, hk);
            }
        }

        if (OBS >= 1) {
            long long cB, cM;
            march_observables<MODEL, DIMS>(M, 16 * n, half == 1, cB, cM);
            block_accumulate2_in(sm.red, cB, cM, a.obs + 2 * (gh >> 1), true, true);
        }
        // publish: every thread's stores -> CTA barrier -> fence -> flag
        __syncthreads();
        if (threadIdx.x == 0) {
            __threadfence();
            st_relaxed_gpu(done + blockIdx.x, need + 1u);
        }
    }
}

// ------------------------------------------------------------------------------------------
// Host side
// ------------------------------------------------------------------------------------------
PhiloxSweepConsts make_philox_consts(const SweepKey &k);   // lsm_tiled.cu

template <int MODEL, int DIMS, bool TRACK, int OBS>
static cudaError_t launch_one(int grid, cudaStream_t s, const ResidentArgs &a, const PhiloxSweepConsts &pk,
                              const typename TabOf<MODEL>::type &tab, int *max_grid, int bs)
{
    auto kern = k_sweep_resident<MODEL, DIMS, TRACK, OBS>;
    if (max_grid) {
        int per_sm = 0;
        cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, 256, 0);
        if (e != cudaSuccess) return e;
        *max_grid = per_sm * sm_count();
        return cudaSuccess;
    }
    void *params[] = {(void *)&a, (void *)&pk, (void *)&tab};
    return cudaLaunchCooperativeKernel((const void *)kern, dim3((unsigned)grid), dim3((unsigned)bs), params, 0, s);
}

template <int MODEL, int DIMS>
static cudaError_t launch_to(bool track, int obs, int grid, cudaStream_t s, const ResidentArgs &a,
                             const PhiloxSweepConsts &pk, const typename TabOf<MODEL>::type &tab, int *max_grid, int bs)
{
    if (track) {
        if (obs) return launch_one<MODEL, DIMS, true, 2>(grid, s, a, pk, tab, max_grid, bs);
        return launch_one<MODEL, DIMS, true, 0>(grid, s, a, pk, tab, max_grid, bs);
    }
    if (obs) return launch_one<MODEL, DIMS, false, 2>(grid, s, a, pk, tab, max_grid, bs);
    return launch_one<MODEL, DIMS, false, 0>(grid, s, a, pk, tab, max_grid, bs);
}

static cudaError_t dispatch(int model, int dims, bool track, int obs, int grid, cudaStream_t s, const ResidentArgs &a,
                            const PhiloxSweepConsts &pk, const TiledTables &t, int *max_grid, int bs)
{
    switch (model) {
    case M_ISING_HALF: {
        HalfTab ht;
        for (int i = 0; i < 16; ++i) ht.t[i] = t.t32[i];
        return dims == 3 ? launch_to<M_ISING_HALF, 3>(track, obs, grid, s, a, pk, ht, max_grid, bs)
                         : launch_to<M_ISING_HALF, 2>(track, obs, grid, s, a, pk, ht, max_grid, bs);
    }
    case M_ISING_ONE: {
        OneTab ot;
        for (int i = 0; i < 64; ++i) ot.t[i] = t.s1[i];
        return dims == 3 ? launch_to<M_ISING_ONE, 3>(track, obs, grid, s, a, pk, ot, max_grid, bs)
                         : launch_to<M_ISING_ONE, 2>(track, obs, grid, s, a, pk, ot, max_grid, bs);
    }
    case M_NE_HEATBATH: {
        NeTab nt = {t.ne_t32[0], 0, t.ne_all4};
        return launch_to<M_NE_HEATBATH, 2>(track, obs, grid, s, a, pk, nt, max_grid, bs);
    }
    default: {
        NeTab nt = {t.ne_t32[1], t.ne_up_always, t.ne_all4};
        return launch_to<M_NE_METROPOLIS, 2>(track, obs, grid, s, a, pk, nt, max_grid, bs);
    }
    }
}

// Plan: word columns in whole CTAs, as many march segments as co-resident CTAs allow.
bool resident_plan(const Lat &lat, int model, int track, const TiledTables &t, ResidentPlan *out)
{
    ResidentPlan p;
    memset(&p, 0, sizeof(p));
    if (!tiled_supported(lat, model, t)) return false;
    if (model == M_EA || model == M_POTTS) return false;   // no resident instantiation for the NEXT-4 models
    if (t.has_never) return false;                         // two-compare kernels exist in the tiled family only
    int coop = 0, dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return false;
    if (cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev) != cudaSuccess || !coop) return false;
    const int R = lat.dims == 3 ? lat.L : 1, wpr = lat.Lh / 16;
    const long long ncol = (long long)R * wpr;
    int bs = 256;                       // whole CTAs of word columns; small lattices get smaller CTAs
    while (bs >= 32 && ncol % bs != 0) bs >>= 1;
    if (bs < 32) return false;
    if (R > 1 && wpr > bs) return false;   // the cross-axis neighbour row must lie in the adjacent CTA
    const long long nb = ncol / bs;
    ResidentArgs dummy;
    memset(&dummy, 0, sizeof(dummy));
    PhiloxSweepConsts pk;
    memset(&pk, 0, sizeof(pk));
    int cap = 0;
    // the four instantiations of a model share registers within a few; take the tightest
    for (int obs = 0; obs < 2; ++obs) {
        int c = 0;
        if (dispatch(model, lat.dims, track != 0, obs, 0, 0, dummy, pk, t, &c, 256) != cudaSuccess) return false;
        if (obs == 0 || c < cap) cap = c;
    }
    if (cap > RESIDENT_MAX_CTAS / 2) cap = RESIDENT_MAX_CTAS / 2;    // two flag words per CTA
    long long S = cap / nb;
    if (S > lat.L) S = lat.L;
    if (S < 1) return false;
    p.S = (int)S;
    p.nb = (int)nb;
    p.bs = bs;
    p.grid = (int)(S * nb);
    *out = p;
    return true;
}

cudaError_t launch_sweep_resident(const Lat &lat, int model, int track, unsigned long long seed, unsigned long long t0,
                                  int nsweeps, long long *d_obs, unsigned *d_flags, unsigned epoch0,
                                  const ResidentPlan &plan, const TiledTables &t, cudaStream_t s)
{
    ResidentArgs a;
    memset(&a, 0, sizeof(a));
    a.col[0] = lat.col[0];
    a.col[1] = lat.col[1];
    a.g.L = lat.L;
    a.g.R = lat.dims == 3 ? lat.L : 1;
    a.g.wpr = lat.Lh / 16;
    a.g.ncol = a.g.R * a.g.wpr;
    a.g.S = plan.S;
    a.g.one = 1;
    if (a.g.R == 1) a.g.parity_rows = 1;
    else if (a.g.wpr % 32 == 0) a.g.parity_rows = 1;
    else if (a.g.wpr < 32 && 32 % a.g.wpr == 0 && a.g.R % (2 * (32 / a.g.wpr)) == 0) a.g.parity_rows = 1;
    else a.g.parity_rows = 0;
    a.seed = seed;
    a.t0 = t0;
    a.nsweeps = nsweeps;
    a.nb = plan.nb;
    a.obs = d_obs;
    a.flags = d_flags;
    a.epoch0 = epoch0;
    SweepKey k = make_sweep_key(seed, t0, 0u);
    PhiloxSweepConsts pk = make_philox_consts(k);     // only the round keys are used by the resident kernel
    return dispatch(model, lat.dims, track != 0, d_obs != nullptr, plan.grid, s, a, pk, t, nullptr, plan.bs);
}

}  // namespace lsmk
