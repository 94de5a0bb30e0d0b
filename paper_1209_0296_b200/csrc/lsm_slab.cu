// lsm_slab.cu -- the slab family for mid-size lattices (1024^2 ... 4096^2, 128^3): ONE launch runs many sweeps and
// the whole lattice lives in the shared memory of the 148 SMs.
//
// The paper ends the kernel after every half-sweep because that was its only grid-wide barrier and
// reports what that costs on small lattices.  On B200 a dependent launch costs ~2.5-3 us, a half-sweep of
// 1024^2 is 0.45 us of work: the tiled family reaches 13 % (1024^2) to 40 % (2048^2) of its large-lattice rate there.
// A lattice of up to ~28 MB fits the shared memory of the whole GPU, and a site reads nearest neighbours only, so:
//   * the lattice is cut into G slabs of march rows (y in 2D, z planes in 3D), one per CTA, one CTA per SM, all
//     co-resident (cooperative launch); a CTA keeps its slab of BOTH colours in shared memory for the whole launch,
//     plus one halo row of each colour below and above;
//   * k sweeps = 2k half-sweeps run inside the launch.  In a half-sweep a CTA updates its two BOUNDARY rows first and
//     stores them into its mailbox in global memory (L2), then its interior rows; before the next half-sweep it
//     copies the fresh boundary rows of the two adjacent slabs from their mailboxes into its halo;
//   * the mailbox words validate themselves: bit 31 of every 32-bit lane (bit 7 of a site byte is unused by every
//     encoding, lsm_internal.cuh) carries the parity of the sweep that wrote it, the reader spins on each lane until
//     the parity is the one it expects.  No flag, no fence, no barrier beyond the CTA's own: the barrier between the
//     colours has become a point-to-point dependency on two neighbours that costs one L2 round trip.
// Same rules, same Philox counters (group = lane index in the colour array) as every other family: bit-identical.
//
// Why one mailbox row per (CTA, side, colour) is enough: a CTA rewrites its colour-c rows in half-sweep h + 2.  To
// start h + 2 it needs the neighbours' rows of half-sweep h + 1, and a neighbour computes those only after it has
// copied this CTA's rows of half-sweep h.  The host sets every mailbox lane to parity 1 before a launch; sweep k of
// the launch writes parity k & 1.
#include "lsm_tiled_dev.cuh"

#include <cstring>

namespace lsmk {

struct SlabArgs {
    uint32_t *col[2];            // colour arrays as 32-bit lanes
    unsigned long long seed, t0; // first sweep of this launch
    int nsweeps;
    int L;                       // march extent
    int lg_lpr;                  // log2(lanes per compact row) = log2(L) - 3
    int lg_R;                    // log2(cross rows per march row): 0 in 2D, log2(L) in 3D
    int rows_max;                // most march rows of any slab (shared-memory stride)
    int one;
    long long *obs;              // [nsweeps][2] (B, M) slots zeroed by the host, or nullptr
    uint32_t *mbox;              // [G][first, last][colour][lanes of a march row]; every lane 0x80808080 at launch
};

__device__ __forceinline__ uint32_t slab_ld_l2(const uint32_t *p)
{
    uint32_t v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void slab_st_l2(uint32_t *p, uint32_t v)
{
    asm volatile("st.relaxed.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
// spin until the lane carries the expected sweep parity in bit 31; returns the lane without it
__device__ __forceinline__ uint32_t slab_take(const uint32_t *p, uint32_t tag31)
{
    uint32_t v;
    do { v = slab_ld_l2(p); } while (((v ^ tag31) & 0x80000000u) != 0u);
    return v & 0x7FFFFFFFu;
}

template <int MODEL, int DIMS, bool TRACK, int OBS, bool NEV>
__global__ void __launch_bounds__(1024, 1)
k_sweep_slab(const __grid_constant__ SlabArgs a, const __grid_constant__ PhiloxSweepConsts pk,
             const __grid_constant__ typename TabOf<MODEL>::type tab, const __grid_constant__ NevTab ytab)
{
    constexpr int NT = MODEL == M_ISING_ONE ? 64 : 16;
    __shared__ __align__(16) struct {
        uint32_t t[NT * (NEV ? 2 : 1)];
        int acc[2][2];           // this CTA's share of (B, M) of the sweep in flight, double-buffered by sweep parity
    } sm;
    extern __shared__ __align__(16) uint32_t s_lat[];
    constexpr bool NE = MODEL == M_NE_HEATBATH || MODEL == M_NE_METROPOLIS;
    uint32_t s_t = (uint32_t)__cvta_generic_to_shared(sm.t);
    asm volatile("" : "+r"(s_t));
    uint32_t ne_t32 = 0;
    int ne_always = 0;
    if constexpr (MODEL == M_ISING_HALF || MODEL == M_ISING_ONE) {
        for (int i = threadIdx.x; i < NT; i += blockDim.x) {
            sm.t[i] = tab.t[i];
            if (NEV) sm.t[NT + i] = ytab.y[i];
        }
    } else {
        ne_t32 = tab.t32;
        ne_always = tab.always;
    }
    if (threadIdx.x < 4) sm.acc[threadIdx.x >> 1][threadIdx.x & 1] = 0;

    const uint32_t tid = threadIdx.x, nthr = blockDim.x;
    const int g = (int)blockIdx.x, G = (int)gridDim.x;
    const int lg_lpr = a.lg_lpr, lg_row = a.lg_lpr + a.lg_R;
    const uint32_t lpr = 1u << lg_lpr, R = 1u << a.lg_R, rowl = 1u << lg_row;   // lanes per compact row / march row
    const int m0 = (int)(((long long)a.L * g) / G), m1 = (int)(((long long)a.L * (g + 1)) / G);
    const uint32_t rows = (uint32_t)(m1 - m0);
    const uint32_t colstride = (uint32_t)(a.rows_max + 2) << lg_row;            // shared lanes per colour
    uint32_t *const s_col[2] = {s_lat, s_lat + colstride};
    // march rows of the adjacent slabs that touch this one, and their owners
    const uint32_t mb = (uint32_t)((m0 == 0 ? a.L : m0) - 1), ma = (uint32_t)(m1 == a.L ? 0 : m1);
    const int g_below = g == 0 ? G - 1 : g - 1, g_above = g + 1 == G ? 0 : g + 1;

    // the slab in shared memory: local march row 1 ... rows (rows 0 and rows + 1 of the layout are spare)
    for (uint32_t i = tid; i < (rows << lg_row); i += nthr) {
        s_col[0][rowl + i] = a.col[0][((uint32_t)m0 << lg_row) + i];
        s_col[1][rowl + i] = a.col[1][((uint32_t)m0 << lg_row) + i];
    }
    __syncthreads();

    // mailbox rows: [cta][0 = first row, 1 = last row][colour]
    auto mbox_row = [&](int cta, int which, int colour) { return a.mbox + ((size_t)((cta * 2 + which) * 2 + colour) << lg_row); };

    int thrB = 0, thrM = 0;
    const int nhalves = 2 * a.nsweeps;
    const uint32_t total = rows << lg_row, nA = (rows >= 2u ? 2u : 1u) << lg_row;
    auto flush_obs = [&](int sw) {                         // thread 0, after a barrier behind the sweep's last add
        const int vB = sm.acc[sw & 1][0], vM = sm.acc[sw & 1][1];
        if (vB != 0) atomicAdd((unsigned long long *)&a.obs[2 * sw], (unsigned long long)(long long)vB);
        if (vM != 0) atomicAdd((unsigned long long *)&a.obs[2 * sw + 1], (unsigned long long)(long long)vM);
        sm.acc[sw & 1][0] = 0;                             // next used by sweep sw + 2: several barriers away
        sm.acc[sw & 1][1] = 0;
    };
#pragma unroll 1
    for (int gh = 0; gh < nhalves; ++gh) {
        const int half = gh & 1, sw = gh >> 1;
        uint32_t *const own = s_col[half];
        uint32_t *const oth = s_col[half ^ 1];
        if (gh > 0) {
            __syncthreads();                               // the previous half-sweep's rows of this slab are complete
            if (OBS >= 1 && half == 0 && tid == 0) flush_obs(sw - 1);
        }
        // The rows of the adjacent slabs that touch this one: written by their owners in half-sweep gh - 1 (mailbox,
        // sweep parity in bit 31), or the lattice as the launch found it (gh = 0).  A boundary lane needs exactly one
        // lane of them (the same lane index), so the thread that updates it spins on that lane itself.
        const uint32_t tag31 = (uint32_t)((gh - 1) >> 1) << 31;
        const uint32_t *const below = gh ? mbox_row(g_below, 1, half ^ 1) : a.col[1] + (mb << lg_row);
        const uint32_t *const above = gh ? mbox_row(g_above, 0, half ^ 1) : a.col[1] + (ma << lg_row);
        const unsigned long long t = a.t0 + (unsigned long long)sw;
        PhiloxDyn pc = {0u, 0u, 0u, 0u, pk};
        philox_half_consts(make_sweep_key(a.seed, t, (uint32_t)half), pk.rk0, pk.rk1, pc.x1, pc.y2, pc.z2, pc.w3);
        int totU = 0, totBN = 0, totS = 0, nsites = 0;
        if (half == 0) thrB = thrM = 0;
        const uint32_t wtag = (uint32_t)(sw & 1) << 31;
        uint32_t *const mb_first = mbox_row(g, 0, half), *const mb_last = mbox_row(g, 1, half);

        // Lanes of the slab in the order boundary rows (1 and `rows`), then interior rows: the adjacent slabs wait for
        // the former, so every thread takes them first.  One lane = 4 sites, one Philox call (spin-1: two).
#pragma unroll 1
        for (uint32_t i = tid; i < total; i += nthr) {
            const bool edge = i < nA;
            const uint32_t ml = edge ? ((i >> lg_row) ? rows : 1u) : 2u + ((i - nA) >> lg_row);
            const uint32_t r = i & (rowl - 1);
            const uint32_t x = r & (lpr - 1), y = r >> lg_lpr;
            const uint32_t m = (uint32_t)m0 + ml - 1u;
            const uint32_t qq = (m + y + (uint32_t)half) & 1u;
            const uint32_t li = (ml << lg_row) + r;
            const uint32_t gl = (m << lg_row) + r;              // lane index in the colour array = Philox group (D2)
            // the random words do not depend on the neighbours: drawn before a boundary lane waits for its halo lane
            uint4 rw = make_uint4(0u, 0u, 0u, 0u), rw2 = rw;
            if (MODEL == M_ISING_HALF) rw = philox_sweep(gl, pc);
            if (MODEL == M_ISING_ONE) {
                rw = philox_sweep(2u * gl, pc);
                rw2 = philox_sweep(2u * gl + 1u, pc);
            }
            const uint32_t c = oth[li], o = own[li];
            uint32_t p, n;
            if (ml == 1u) p = gh ? slab_take(below + r, tag31) : below[r];
            else p = oth[li - rowl];
            if (ml == rows) n = gh ? slab_take(above + r, tag31) : above[r];
            else n = oth[li + rowl];
            const uint32_t cs = oth[(li - x) + ((qq ? x + 1u : x - 1u) & (lpr - 1))];
            const uint32_t sd = qq ? __funnelshift_r(c, cs, 8) : __funnelshift_r(cs, c, 24);
            uint32_t yp = 0, yn = 0;
            if (DIMS == 3) {
                yp = oth[(ml << lg_row) + (((y - 1u) & (R - 1)) << lg_lpr) + x];
                yn = oth[(ml << lg_row) + (((y + 1u) & (R - 1)) << lg_lpr) + x];
            }
            uint32_t out;
            if (MODEL == M_ISING_HALF) {
                uint32_t ns = p + n + c + sd;
                if (DIMS == 3) ns += yp + yn;
                out = rule_half<TRACK, OBS, NEV>(o, ns, rw, s_t, (uint32_t)a.one, totU, totBN);
            } else if (MODEL == M_ISING_ONE) {
                uint32_t ns;
                if (TRACK) {
                    ns = ((p + n) & 0x0F0F0F0Fu) + ((c + sd) & 0x0F0F0F0Fu);
                    if (DIMS == 3) ns += (yp + yn) & 0x0F0F0F0Fu;
                } else {
                    ns = p + n + c + sd;
                    if (DIMS == 3) ns += yp + yn;
                }
                out = rule_one<DIMS, TRACK, OBS, NEV>(o, ns, rw, rw2, s_t, (uint32_t)a.one, totU, totBN, totS);
            } else {
                uint32_t accU = 0;
                out = rule_ne<TRACK, MODEL == M_NE_METROPOLIS, OBS>(o, n, qq ? sd : c, gl, pc, ne_t32, ne_always, accU);
                if (OBS >= 1) totU += (int)bytesum(accU);
            }
            own[li] = out;
            if (edge) {
                if (ml == 1u) slab_st_l2(mb_first + r, out | wtag);
                if (ml == rows) slab_st_l2(mb_last + r, out | wtag);
            }
            nsites += 4;
        }
        if (OBS >= 1) {
            March<MODEL, DIMS, TRACK, OBS, NEV> M;         // only the per-thread sums are used
            M.totU = totU;
            M.totBN = totBN;
            M.totS = totS;
            long long cB, cM;
            march_observables<MODEL, DIMS>(M, nsites, half == 1, cB, cM);
            thrB += (int)cB;                               // one slab holds < 2^20 sites: far below 2^31
            thrM += (int)cM;
            if (half == 1) {
                const int wB = __reduce_add_sync(0xffffffffu, thrB), wM = __reduce_add_sync(0xffffffffu, thrM);
                if ((tid & 31u) == 0u) {
                    if (wB != 0) atomicAdd(&sm.acc[sw & 1][0], wB);
                    if (wM != 0) atomicAdd(&sm.acc[sw & 1][1], wM);
                }
            }
        }
    }
    __syncthreads();
    if (OBS >= 1 && nhalves > 0 && tid == 0) flush_obs(a.nsweeps - 1);
    // write the slab back
    for (uint32_t i = tid; i < total; i += nthr) {
        a.col[0][((uint32_t)m0 << lg_row) + i] = s_col[0][rowl + i];
        a.col[1][((uint32_t)m0 << lg_row) + i] = s_col[1][rowl + i];
    }
}

// ------------------------------------------------------------------------------------------
// Host side
// ------------------------------------------------------------------------------------------
PhiloxSweepConsts make_philox_consts(const SweepKey &k);   // lsm_tiled.cu

static int slab_ilog2(long long v)
{
    int l = 0;
    while ((1ll << l) < v) ++l;
    return l;
}

#ifndef LSM_SLAB_SMEM_MAX
#define LSM_SLAB_SMEM_MAX (220 * 1024)     // dynamic shared memory per CTA (227 KB opt-in minus the static part)
#endif

// Mailbox bytes reserved in the workspace for this shape (0: the slab family never runs it).  Depends on the shape
// only, so that lsm_workspace_bytes needs no device: SLAB_MAX_CTAS slabs x (first, last) x 2 colours x one march row.
size_t slab_mailbox_bytes(int dims, int L, int model)
{
    if (model != M_ISING_HALF && model != M_ISING_ONE && model != M_NE_HEATBATH && model != M_NE_METROPOLIS) return 0;
    if ((L & (L - 1)) != 0) return 0;                                 // lane index math by shifts
    if (dims == 2 ? (L < 512 || L > 4096) : (L < 64 || L > 128)) return 0;   // below: the small family; above: does not fit
    const size_t rowbytes = (size_t)(L / 2) * (dims == 3 ? (size_t)L : 1);
    return (size_t)SLAB_MAX_CTAS * 4 * rowbytes;
}

bool slab_plan(const Lat &lat, int model, const TiledTables &t, SlabPlan *out)
{
    if (!t.usable) return false;
    if (slab_mailbox_bytes(lat.dims, lat.L, model) == 0) return false;
    int coop = 0, dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return false;
    if (cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev) != cudaSuccess || !coop) return false;
    int G = sm_count();                                               // one CTA per SM, all co-resident
    if (G > SLAB_MAX_CTAS) G = SLAB_MAX_CTAS;
    if (G > lat.L) G = lat.L;
    if (G < 2) return false;
    const int rows_max = (lat.L + G - 1) / G;
    const long long rowl = (lat.dims == 3 ? (long long)lat.L : 1) * (lat.L / 8);   // lanes per march row and colour
    const long long smem = 2ll * (rows_max + 2) * rowl * 4;
    if (smem > LSM_SLAB_SMEM_MAX) return false;
    long long per = (long long)rows_max * rowl;                       // lanes per half-sweep of the largest slab
    if (2 * rowl > per) per = 2 * rowl;
    int threads = (int)(per < 1024 ? ((per + 31) / 32) * 32 : 1024);
    if (threads < 64) threads = 64;
    out->G = G;
    out->rows_max = rows_max;
    out->threads = threads;
    out->smem = (int)smem;
    return true;
}

template <int MODEL, int DIMS>
static cudaError_t slab_launch_to(bool track, bool obs, const SlabPlan &plan, cudaStream_t s, const SlabArgs &a,
                                  const PhiloxSweepConsts &pk, const typename TabOf<MODEL>::type &tab, const TiledTables &t)
{
    NevTab yt;
    memset(&yt, 0, sizeof(yt));
    for (int i = 0; i < 64; ++i) yt.y[i] = t.y32[i];
    auto go = [&](auto kern) -> cudaError_t {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, plan.smem);
        if (e != cudaSuccess) return e;
        void *params[] = {(void *)&a, (void *)&pk, (void *)&tab, (void *)&yt};
        return cudaLaunchCooperativeKernel((const void *)kern, dim3((unsigned)plan.G), dim3((unsigned)plan.threads), params,
                                           (size_t)plan.smem, s);
    };
    constexpr bool CAN_NEV = MODEL == M_ISING_HALF || MODEL == M_ISING_ONE;
    if constexpr (CAN_NEV) {
        if (t.has_never) {
            if (track) return obs ? go(k_sweep_slab<MODEL, DIMS, true, 2, true>) : go(k_sweep_slab<MODEL, DIMS, true, 0, true>);
            return obs ? go(k_sweep_slab<MODEL, DIMS, false, 2, true>) : go(k_sweep_slab<MODEL, DIMS, false, 0, true>);
        }
    }
    if (track) return obs ? go(k_sweep_slab<MODEL, DIMS, true, 2, false>) : go(k_sweep_slab<MODEL, DIMS, true, 0, false>);
    return obs ? go(k_sweep_slab<MODEL, DIMS, false, 2, false>) : go(k_sweep_slab<MODEL, DIMS, false, 0, false>);
}

// d_mbox: slab_mailbox_bytes() bytes, every byte set to 0x80 by the caller on the same stream before this launch.
cudaError_t launch_sweep_slab(const Lat &lat, int model, int track, unsigned long long seed, unsigned long long t0,
                              int nsweeps, long long *d_obs, uint32_t *d_mbox, const SlabPlan &plan, const TiledTables &t,
                              cudaStream_t s)
{
    SlabArgs a;
    memset(&a, 0, sizeof(a));
    a.col[0] = reinterpret_cast<uint32_t *>(lat.col[0]);
    a.col[1] = reinterpret_cast<uint32_t *>(lat.col[1]);
    a.seed = seed;
    a.t0 = t0;
    a.nsweeps = nsweeps;
    a.L = lat.L;
    const int lg_L = slab_ilog2(lat.L);
    a.lg_lpr = lg_L - 3;
    a.lg_R = lat.dims == 3 ? lg_L : 0;
    a.rows_max = plan.rows_max;
    a.one = 1;
    a.obs = d_obs;
    a.mbox = d_mbox;
    PhiloxSweepConsts pk = make_philox_consts(make_sweep_key(seed, t0, 0u));   // only the round keys are used
    const bool obs = d_obs != nullptr, tr = track != 0;
    switch (model) {
    case M_ISING_HALF: {
        HalfTab ht;
        for (int i = 0; i < 16; ++i) ht.t[i] = t.t32[i];
        return lat.dims == 3 ? slab_launch_to<M_ISING_HALF, 3>(tr, obs, plan, s, a, pk, ht, t)
                             : slab_launch_to<M_ISING_HALF, 2>(tr, obs, plan, s, a, pk, ht, t);
    }
    case M_ISING_ONE: {
        OneTab ot;
        for (int i = 0; i < 64; ++i) ot.t[i] = t.s1[i];
        return lat.dims == 3 ? slab_launch_to<M_ISING_ONE, 3>(tr, obs, plan, s, a, pk, ot, t)
                             : slab_launch_to<M_ISING_ONE, 2>(tr, obs, plan, s, a, pk, ot, t);
    }
    case M_NE_HEATBATH: {
        NeTab nt = {t.ne_t32[0], 0, t.ne_all4};
        return slab_launch_to<M_NE_HEATBATH, 2>(tr, obs, plan, s, a, pk, nt, t);
    }
    default: {
        NeTab nt = {t.ne_t32[1], t.ne_up_always, t.ne_all4};
        return slab_launch_to<M_NE_METROPOLIS, 2>(tr, obs, plan, s, a, pk, nt, t);
    }
    }
}

}  // namespace lsmk
