// lsm_slab.cu -- the slab family for mid-size lattices (512^2 ... 4096^2, 64^3, 128^3; from 128^2 / 32^3 for the
// Edwards-Anderson and Potts models, which have no small-family kernels): ONE launch runs many sweeps,
// the whole lattice lives in the shared memory of the SMs, and several half-sweeps run between two exchanges
// (temporal blocking with redundant halo updates).
//
// The paper ends the kernel after every half-sweep because that was its only grid-wide barrier and
// reports what that costs on small lattices.  On B200 a dependent launch costs ~2.5-3 us, a half-sweep of
// 1024^2 is 0.45 us of work: the tiled family reaches 13 % (1024^2) to 40 % (2048^2) of its large-lattice rate there.
// A lattice of up to ~28 MB fits the shared memory of the whole GPU, and a site reads nearest neighbours only, so:
//   * the lattice is cut into G slabs of march rows (y in 2D, z planes in 3D), one per CTA, one CTA per SM, all
//     co-resident (cooperative launch).  A CTA keeps its slab of BOTH colours in shared memory for the whole launch,
//     plus D halo rows of each colour below and above (D = temporal depth);
//   * time runs in epochs of D half-sweeps.  At the start of an epoch the halo holds the D adjacent rows of both
//     neighbours as of that time.  Step j of the epoch updates the slab's own rows AND the D-1-j nearest halo rows on
//     either side: a halo update is exactly the update its owner makes (same neighbours, same Philox counter =
//     lane index in the colour array, same table), so it is reproduced rather than communicated.  After D steps
//     the own rows are exact and the halo is used up;
//   * exchange: while it makes the last two steps of an epoch a CTA stores the first and the last D of its own rows
//     (of the colour updated in that step) into its mailbox in global memory (L2); the adjacent CTAs copy them into
//     their halos behind the epoch's last step.  Mailbox lanes validate themselves: bit 31 of every 32-bit lane
//     (bit 7 of a site byte is unused by every encoding, lsm_internal.cuh) carries one bit of the epoch number and the
//     reader spins on a 16-byte word until its four lanes show the expected one -- no flag, no fence.  One exchange
//     costs about one microsecond of latency on B200 whatever its size, which is why it pays to make it once per D
//     half-sweeps;
//   * D = 1 is the plain scheme (one row of the colour just updated per half-sweep, no redundant update).
// Mailboxes are double-buffered by epoch parity: a CTA rewrites buffer e & 1 in epoch e + 2, which it can only start
// after it has read the neighbours' rows of epoch e + 1, and those were computed from this CTA's rows of epoch e.
// What the reuse argument rests on (there is no fence anywhere in the protocol): a reader's load of a mailbox word has
// COMPLETED by the time the reader acts on it -- the loop in slab_take4 consumes the loaded value in its exit test, and
// the value is stored to shared memory before the CTA's bar.sync -- so once a CTA's rows of epoch e + 1 are visible to
// its neighbour (which the neighbour's tag check establishes by data dependence), every load the CTA made from the
// neighbour's buffer of epoch e is over and the neighbour may overwrite that buffer.  With the "early" exchange
// (SlabArgs::early: depth 1, long steps) the polling loads are issued before the CTA barrier instead of after it;
// the argument is the same, and that path has its own long-run cases in tests/test_gpu_parity.py
// (test_slab_long_run_against_the_tiled_family: 2048^2 and 4096^2 at depth 1).
// The host sets every mailbox lane the launch can read to 0x80808080 before a launch; epoch e writes bit 31 = (e >> 1) & 1.
// Only own rows count for the per-sweep (B, M).  Bit-identical to every other family.
#include "lsm_tiled_dev.cuh"

#include <cooperative_groups.h>
#include <cstring>
#include <type_traits>

namespace lsmk {

struct SlabArgs {
    uint32_t *col[2];            // colour arrays as 32-bit lanes
    const uint32_t *bnd[2];      // M_EA: bond bytes of the two colours (same geometry; constant during a launch)
    unsigned long long seed, t0; // first sweep of this launch
    int nsweeps;
    int L;                       // march extent
    int wpr;                     // 16-byte words per compact row = L / 32
    int R;                       // cross rows per march row: 1 in 2D, L in 3D
    uint32_t magic_wrow;         // floor(2^32 / (R * wpr)) + 1: n / (R * wpr) = umulhi(n, magic) for every n the kernel divides
    uint32_t magic_wpr;          // the same for wpr
    int lg_wpr, lg_wrow;         // POW2 instantiations (L a power of two): log2(wpr), log2(R * wpr); shifts and masks instead
    int rows_max;                // most march rows of any slab (shared-memory stride)
    int D;                       // temporal depth: half-sweeps per exchange; every slab has >= 2 D rows (3D: >= 1)
    int dmax;                    // mailbox rows reserved per slot
    int early;                   // D = 1, long steps: copy the halo behind the step instead of before the next one
    int one;
    int qm1;                     // M_POTTS: q - 1
    long long *obs;              // [nsweeps][2] (B, M) slots zeroed by the host, or nullptr
    uint32_t *mbox;              // [G][first, last][epoch parity][colour][dmax][lanes of a march row]
};

// L2-coherent 16-byte accesses to a mailbox word (relaxed, gpu scope: never served from or parked in this SM's L1)
// spin until all four lanes of the word carry the expected epoch bit in bit 31 (each lane carries its own, so a torn
// word is only retried); returns the word without the bits
__device__ __forceinline__ uint4 slab_take4(const uint32_t *p, uint32_t tag31)
{
    uint4 v;
    do {
        asm volatile("ld.relaxed.gpu.global.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p) : "memory");
    } while (((((v.x ^ tag31) | (v.y ^ tag31)) | ((v.z ^ tag31) | (v.w ^ tag31))) & 0x80000000u) != 0u);
    return make_uint4(v.x & 0x7FFFFFFFu, v.y & 0x7FFFFFFFu, v.z & 0x7FFFFFFFu, v.w & 0x7FFFFFFFu);
}
__device__ __forceinline__ void slab_st4_l2(uint32_t *p, uint4 v)
{
    asm volatile("st.relaxed.gpu.global.v4.u32 [%0], {%1,%2,%3,%4};" ::"l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}

// POW2: L is a power of two and the index arithmetic is shifts and masks (measured 7-9 % faster than the general form,
// which multiplies, divides by multiplication with a checked reciprocal and wraps by compare).
template <int MODEL, int DIMS, bool TRACK, int OBS, bool NEV, bool POW2>
__global__ void __launch_bounds__(512, 1)
k_sweep_slab(const __grid_constant__ SlabArgs a, const __grid_constant__ PhiloxSweepConsts pk,
             const __grid_constant__ typename TabOf<MODEL>::type tab, const __grid_constant__ NevTab ytab)
{
    constexpr int NT = MODEL == M_ISING_ONE ? 64 : 16;
    __shared__ __align__(16) struct {
        uint32_t t[NT * (NEV ? 2 : 1)];
        int acc[2][2];           // this CTA's share of (B, M) of the sweep in flight, double-buffered by sweep parity
    } sm;
    extern __shared__ __align__(16) uint32_t s_lat[];
    uint32_t s_t = (uint32_t)__cvta_generic_to_shared(sm.t);
    asm volatile("" : "+r"(s_t));
    uint32_t ne_t32 = 0;
    int ne_always = 0;
    bool ne_all4 = false;
    if constexpr (MODEL == M_ISING_HALF || MODEL == M_ISING_ONE || MODEL == M_EA || MODEL == M_POTTS) {
        for (int i = threadIdx.x; i < NT; i += blockDim.x) {
            sm.t[i] = tab.t[i];
            if (NEV) sm.t[NT + i] = ytab.y[i];
        }
    } else {
        ne_t32 = tab.t32;
        ne_always = tab.always;
        ne_all4 = tab.all4 != 0;
    }
    if (threadIdx.x < 4) sm.acc[threadIdx.x >> 1][threadIdx.x & 1] = 0;

    const uint32_t tid = threadIdx.x, nthr = blockDim.x;
    const int g = (int)blockIdx.x, G = (int)gridDim.x;
    const uint32_t wpr = (uint32_t)a.wpr, R = (uint32_t)a.R;                   // words per compact row; cross rows
    const uint32_t wrow = R * wpr, rowl = 4u * wrow;                            // 16-byte words / 32-bit lanes per march row
    const uint32_t mg_wrow = a.magic_wrow, mg_wpr = a.magic_wpr;
    const int lg_wpr = a.lg_wpr, lg_wrow = a.lg_wrow;
    const uint32_t Lm = (uint32_t)a.L - 1u;
    auto div_wrow = [&](uint32_t n) { return POW2 ? n >> lg_wrow : __umulhi(n, mg_wrow); };      // n / wrow
    auto mul_wrow = [&](uint32_t x) { return POW2 ? x << lg_wrow : x * wrow; };                  // x * wrow
    auto rem_wrow = [&](uint32_t n, uint32_t q) { return POW2 ? n & (wrow - 1u) : n - q * wrow; };   // n % wrow, q = n / wrow
    const uint32_t D = (uint32_t)a.D;
    const int m0 = (int)(((long long)a.L * g) / G), m1 = (int)(((long long)a.L * (g + 1)) / G);
    const uint32_t rows = (uint32_t)(m1 - m0);
    const uint32_t colstride = ((uint32_t)a.rows_max + 2u * D) * rowl;          // shared lanes per colour
    uint32_t *const s_col[2] = {s_lat, s_lat + colstride};
    uint32_t *const s_bnd[2] = {s_lat + 2u * colstride, s_lat + 3u * colstride};   // M_EA only (the launch sizes for it)
    const int g_below = g == 0 ? G - 1 : g - 1, g_above = g + 1 == G ? 0 : g + 1;
    // local march row lr <-> global march row (m0 - D + lr) mod L: 0 ... D-1 halo below, D ... D+rows-1 own rows,
    // D+rows ... rows+2D-1 halo above
    const uint32_t mbase = (uint32_t)(m0 + a.L) - D;
    auto global_row = [&](uint32_t lr) {
        if (POW2) return (mbase + lr) & Lm;
        const int m = m0 - (int)D + (int)lr;
        return (uint32_t)(m < 0 ? m + a.L : (m >= a.L ? m - a.L : m));
    };

    // the slab and its halo as the launch finds the lattice
    for (uint32_t i = tid; i < (rows + 2u * D) * wrow; i += nthr) {            // in 16-byte words
        const uint32_t lr = div_wrow(i), wr = rem_wrow(i, lr);
        const size_t src = (size_t)global_row(lr) * wrow + wr;
        reinterpret_cast<uint4 *>(s_col[0])[i] = reinterpret_cast<const uint4 *>(a.col[0])[src];
        reinterpret_cast<uint4 *>(s_col[1])[i] = reinterpret_cast<const uint4 *>(a.col[1])[src];
        if (MODEL == M_EA) {                                   // the bonds of the halo rows too: their redundant updates need them
            reinterpret_cast<uint4 *>(s_bnd[0])[i] = reinterpret_cast<const uint4 *>(a.bnd[0])[src];
            reinterpret_cast<uint4 *>(s_bnd[1])[i] = reinterpret_cast<const uint4 *>(a.bnd[1])[src];
        }
    }
    __syncthreads();
    // No CTA may write its slab back (end of the kernel) before the adjacent CTAs have read their initial halos; with
    // fewer half-sweeps than one epoch there is no exchange that would order the two.
    cooperative_groups::this_grid().sync();

    // mailbox rows
    auto mbox_row = [&](int cta, int side, uint32_t buf, int colour, uint32_t k) {
        return a.mbox + (size_t)((((uint32_t)(cta * 2 + side) * 2u + buf) * 2u + (uint32_t)colour) * (uint32_t)a.dmax + k) * rowl;
    };
    auto flush_obs = [&](int sw) {                         // thread 0, after a barrier behind the sweep's last add
        const int vB = sm.acc[sw & 1][0], vM = sm.acc[sw & 1][1];
        if (vB != 0) atomicAdd((unsigned long long *)&a.obs[2 * sw], (unsigned long long)(long long)vB);
        if (vM != 0) atomicAdd((unsigned long long *)&a.obs[2 * sw + 1], (unsigned long long)(long long)vM);
        sm.acc[sw & 1][0] = 0;                             // next used by sweep sw + 2: several barriers away
        sm.acc[sw & 1][1] = 0;
    };

    int thrB = 0, thrM = 0;
    const uint32_t H = 2u * (uint32_t)a.nsweeps;
    uint32_t e = 0;
#pragma unroll 1
    for (uint32_t h0 = 0; h0 < H; h0 += D, ++e) {
        const uint32_t De = H - h0 < D ? H - h0 : D;       // steps of this epoch (the last one may be shorter)
        const bool last = h0 + D >= H;
        // Halo copy of one colour: the rows the adjacent slabs stored during epoch pe.  Normally at the start of the next
        // epoch.  With D = 1 and long steps (a.early) right behind the step, before the CTA barrier that ends it: nobody
        // reads that colour's halo rows in the step, the load's L2 round trip overlaps the warps still updating, and one
        // barrier per step is saved (4096^2: +4 %; short steps lose: the data cannot have arrived yet and the polling
        // loads compete with the stores they wait for).
        auto halo_copy = [&](const uint32_t pe, const uint32_t c0, const uint32_t ncol) {   // colours c0 ... c0 + ncol - 1
            const uint32_t buf = pe & 1u, tag31 = ((pe >> 1) & 1u) << 31;
            const uint32_t per_side = ncol * D * wrow;              // in 16-byte words: one L2 round trip moves four lanes
#pragma unroll 1
            for (uint32_t i = tid; i < 2u * per_side; i += nthr) {
                const uint32_t above = i >= per_side ? 1u : 0u;
                const uint32_t w = i - above * per_side;
                const uint32_t kc = div_wrow(w), wr = rem_wrow(w, kc);    // kc = ci * D + k
                const uint32_t ci = kc >= D ? 1u : 0u, k = kc - ci * D;
                const int colour = (int)(c0 + ci);
                // below: the neighbour's LAST D rows -> local rows 0 ... D-1; above: its FIRST D rows -> D+rows ...
                const uint32_t *src = mbox_row(above ? g_above : g_below, above ? 0 : 1, buf, colour, k) + (wr << 2);
                const uint32_t lr = above ? D + rows + k : k;
                reinterpret_cast<uint4 *>(s_col[colour])[mul_wrow(lr) + wr] = slab_take4(src, tag31);
            }
        };
#pragma unroll 1
        for (uint32_t j = 0; j < De; ++j) {
            const uint32_t gh = h0 + j;
            const int half = (int)(gh & 1u), sw = (int)(gh >> 1);
            if (gh > 0) __syncthreads();                   // the previous step's rows (and the halo copied behind it) are complete
            if (OBS >= 1 && half == 0 && gh > 0 && tid == 0) flush_obs(sw - 1);
            uint32_t *const own = s_col[half];
            const uint32_t *const oth = s_col[half ^ 1];
            const uint32_t ext = De - 1u - j;              // halo rows updated on either side (redundant updates)
            const bool publish = !last && j + 2u >= D;     // this colour's rows are final for the coming exchange
            const unsigned long long t = a.t0 + (unsigned long long)sw;
            PhiloxDyn pc = {0u, 0u, 0u, 0u, pk};
            philox_half_consts(make_sweep_key(a.seed, t, (uint32_t)half), pk.rk0, pk.rk1, pc.x1, pc.y2, pc.z2, pc.w3);
            int totU = 0, totBN = 0, totS = 0, nsites = 0;
            if (half == 0) thrB = thrM = 0;
            const uint32_t wtag = ((e >> 1) & 1u) << 31, e_par = e & 1u;
            // Row order: the 2 D rows the neighbours wait for first (first D and last D own rows), then the others.
            // A thread takes one 16-byte word (16 sites, four independent Philox calls) at a time: the update of a
            // word is the tiled family's (March::update_word), fed from shared memory.
            // (a one-row slab -- 3D, D = 1: one plane per CTA -- has a row that is the first and the last at once and goes
            // to both mailboxes)
            const uint32_t nA = publish ? (DIMS == 3 && rows == 1u ? 1u : 2u * D) : 0u, nrows = rows + 2u * ext;
            const uint32_t total = mul_wrow(nrows);
            March<MODEL, DIMS, TRACK, OBS, NEV> W;
            W.s_t = s_t;
            W.one = (uint32_t)a.one;
            W.ne_t32 = ne_t32;
            W.ne_always = ne_always;
            W.ne_all4 = ne_all4;
            W.potts_qm1 = (uint32_t)a.qm1;
#pragma unroll 1
            for (uint32_t i = tid; i < total; i += nthr) {
                const uint32_t s = div_wrow(i), wr = rem_wrow(i, s);
                uint32_t lr;
                if (s < nA) lr = s < D ? D + s : rows + (s - D);
                else if (!publish) lr = D - ext + s;
                else {
                    const uint32_t s2 = s - nA, mid = rows - 2u * D;
                    lr = s2 < ext ? D - ext + s2 : (s2 < ext + mid ? 2u * D + (s2 - ext) : rows + D + (s2 - ext - mid));
                }
                const bool own_row = lr >= D && lr < D + rows;
                uint32_t y = 0u, xw = wr;
                if (DIMS == 3) {
                    y = POW2 ? wr >> lg_wpr : (wpr == 1u ? wr : __umulhi(wr, mg_wpr));
                    xw = POW2 ? wr & (wpr - 1u) : wr - y * wpr;
                }
                const uint32_t m = global_row(lr);
                const uint32_t qq = (m + y + (uint32_t)half) & 1u;
                const uint32_t wi = mul_wrow(lr) + wr;              // word index in the shared colour array
                const uint4 *const othw = reinterpret_cast<const uint4 *>(oth);
                W.C = othw[wi];
                W.P = othw[wi - wrow];
                const uint4 N = othw[wi + wrow];
                const uint4 O = reinterpret_cast<const uint4 *>(own)[wi];
                // the lane beyond the word's end in its compact row: first lane of the next word (q = 1) or last lane of
                // the previous one (q = 0), periodic in x
                const uint32_t xe = POW2 ? ((qq ? xw + 1u : xw - 1u) & (wpr - 1u))
                                         : (qq ? (xw + 1u == wpr ? 0u : xw + 1u) : (xw == 0u ? wpr - 1u : xw - 1u));
                const uint32_t edge = oth[(((wi - xw) + xe) << 2) + (qq ? 0u : 3u)];
                uint4 Yp = make_uint4(0u, 0u, 0u, 0u), Yn = Yp;
                if (DIMS == 3) {
                    const uint32_t ym = POW2 ? ((y - 1u) & (R - 1u)) : (y == 0u ? R - 1u : y - 1u);
                    const uint32_t yp1 = POW2 ? ((y + 1u) & (R - 1u)) : (y + 1u == R ? 0u : y + 1u);
                    Yp = othw[mul_wrow(lr) + (POW2 ? ym << lg_wpr : ym * wpr) + xw];
                    Yn = othw[mul_wrow(lr) + (POW2 ? yp1 << lg_wpr : yp1 * wpr) + xw];
                }
                W.q = (int)qq;
                W.grp = (mul_wrow(m) + wr) << 2;                    // Philox group of the word's first lane (D2)
                W.totU = W.totBN = W.totS = 0;                      // this word's sums: counted for own rows only
                uint4 BW = make_uint4(0u, 0u, 0u, 0u);
                if (MODEL == M_EA) BW = reinterpret_cast<const uint4 *>(s_bnd[half])[wi];
                const uint4 out = W.template update_word<2, true>(pc, N, O, edge, Yp, Yn, BW);
                reinterpret_cast<uint4 *>(own)[wi] = out;
                if (s < nA) {
                    const uint4 tagged = make_uint4(out.x | wtag, out.y | wtag, out.z | wtag, out.w | wtag);
                    if (DIMS == 3 && rows == 1u) {
                        slab_st4_l2(mbox_row(g, 0, e_par, half, 0u) + (wr << 2), tagged);
                        slab_st4_l2(mbox_row(g, 1, e_par, half, 0u) + (wr << 2), tagged);
                    } else {
                        slab_st4_l2(mbox_row(g, s < D ? 0 : 1, e_par, half, s < D ? s : s - D) + (wr << 2), tagged);
                    }
                }
                if (OBS >= 1 && own_row) {
                    totU += W.totU;
                    totBN += W.totBN;
                    totS += W.totS;
                    nsites += 16;
                }
            }
            if (!last && j + 1u == D) {
                // The exchange: the rows the adjacent slabs stored during this epoch -> halo.  D = 1: the colour of this
                // step; D >= 2: both colours (the next step updates its own colour in the halo rows too), in one pass so
                // that a thread waits for one L2 round trip.  a.early: before the barrier (see above), else behind it.
                if (!a.early) __syncthreads();
                halo_copy(e, D == 1u ? (uint32_t)half : 0u, D == 1u ? 1u : 2u);
            }
            if (OBS >= 1) {
                March<MODEL, DIMS, TRACK, OBS, NEV> M;     // only the per-thread sums are used
                M.totU = totU;
                M.totBN = totBN;
                M.totS = totS;
                long long cB, cM;
                march_observables<MODEL, DIMS>(M, nsites, half == 1, cB, cM);
                thrB += (int)cB;                           // one slab holds < 2^20 sites: far below 2^31
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
    }
    __syncthreads();
    if (OBS >= 1 && H > 0u && tid == 0) flush_obs(a.nsweeps - 1);
    // write the slab back
    for (uint32_t i = tid; i < rows * wrow; i += nthr) {                       // in 16-byte words
        reinterpret_cast<uint4 *>(a.col[0])[(size_t)m0 * wrow + i] = reinterpret_cast<const uint4 *>(s_col[0])[D * wrow + i];
        reinterpret_cast<uint4 *>(a.col[1])[(size_t)m0 * wrow + i] = reinterpret_cast<const uint4 *>(s_col[1])[D * wrow + i];
    }
}

// ------------------------------------------------------------------------------------------
// Host side
// ------------------------------------------------------------------------------------------
PhiloxSweepConsts make_philox_consts(const SweepKey &k);   // lsm_tiled.cu

#define LSM_SLAB_SMEM_MAX (220 * 1024)     // dynamic shared memory per CTA (227 KB opt-in minus the static part)

// Largest temporal depth the mailboxes of this shape are sized for (0: the slab family never runs it).  Deep halos pay
// where a half-sweep is shorter than an exchange (~1 us): the smaller 2D lattices.
int slab_depth_max(int dims, int L, int model)
{
    if (model != M_ISING_HALF && model != M_ISING_ONE && model != M_NE_HEATBATH && model != M_NE_METROPOLIS && model != M_EA &&
        model != M_POTTS)
        return 0;
    if (L % 32 != 0) return 0;                                        // whole 16-byte words per compact row
    // above: does not fit; below: the small family's lane kernel (cluster barrier) is faster -- for the models and the
    // power-of-two edges it covers
    const bool low = model == M_EA || model == M_POTTS || (L & (L - 1)) != 0;
    if (dims == 2 ? (L < (low ? 128 : 512) || L > 4096) : (L < (low ? 32 : 64) || L > 128)) return 0;
    if (dims == 3) return 1;
    return L <= 1024 ? 4 : L <= 2048 ? 2 : 1;
}

// Mailbox bytes reserved in the workspace for this shape.  Depends on the shape only, so that lsm_workspace_bytes
// needs no device: SLAB_MAX_CTAS slabs x (first, last) x 2 epoch parities x 2 colours x depth_max march rows.
size_t slab_mailbox_bytes(int dims, int L, int model)
{
    const size_t rowbytes = (size_t)(L / 2) * (dims == 3 ? (size_t)L : 1);
    return (size_t)SLAB_MAX_CTAS * 8 * (size_t)slab_depth_max(dims, L, model) * rowbytes;
}

// Default temporal depth (measured on B200, profiles/r2_slab_family.md): an exchange costs ~1 us, a redundant row
// 1/rows of a step; 512^2 (3-4 rows per slab) runs fastest with 3, 1024^2 and 2048^2 with 2, 4096^2 and 3D with 1.
static int slab_depth_default(int dims, int L) { return dims == 3 ? 1 : L <= 512 ? 3 : L <= 2048 ? 2 : 1; }

// depth: 0 = the default for this shape, else 1 ... slab_depth_max
bool slab_plan(const Lat &lat, int model, const TiledTables &t, int depth, SlabPlan *out)
{
    if (!t.usable) return false;
    const int dmax = slab_depth_max(lat.dims, lat.L, model);
    if (dmax == 0 || depth < 0 || depth > dmax) return false;
    int D = depth ? depth : slab_depth_default(lat.dims, lat.L);
    if (D > dmax) D = dmax;
    int coop = 0, dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return false;
    if (cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev) != cudaSuccess || !coop) return false;
    int G = sm_count();                                               // one CTA per SM, all co-resident
    if (G > SLAB_MAX_CTAS) G = SLAB_MAX_CTAS;
    // every slab: >= 2 D rows (disjoint first / last D); in 3D (D = 1) a slab may be a single plane
    const int gmax = lat.dims == 3 ? lat.L : lat.L / (2 * D);
    if (G > gmax) G = gmax;
    if (G < 2) return false;
    const int rows_max = (lat.L + G - 1) / G;
    const long long rowl = (lat.dims == 3 ? (long long)lat.L : 1) * (lat.L / 8);   // lanes per march row and colour
    const long long smem = (model == M_EA ? 4ll : 2ll) * (rows_max + 2 * D) * rowl * 4;    // EA: the bond bytes as well
    if (smem > LSM_SLAB_SMEM_MAX) return false;
    long long per = (long long)(rows_max + 2 * (D - 1)) * rowl / 4;   // words of the largest step of the largest slab
    int threads = (int)(per < 512 ? ((per + 31) / 32) * 32 : 512);
    if (threads < 64) threads = 64;
    // n / d = umulhi(n, floor(2^32 / d) + 1): checked here for every n the kernel divides (word indices of a slab
    // with its halo, of an exchange, of a march row)
    auto magic = [](long long d, long long nmax, uint32_t *m) {
        *m = (uint32_t)((1ull << 32) / (unsigned long long)d + 1ull);
        for (long long n = 0; n <= nmax; ++n)
            if ((long long)(((unsigned long long)n * *m) >> 32) != n / d) return false;
        return true;
    };
    const long long wrow_w = rowl / 4, wpr_w = lat.L / 32;
    uint32_t mg_wrow = 0, mg_wpr = 0;
    if (!magic(wrow_w, (rows_max + 2 * D + 4 * D) * wrow_w, &mg_wrow)) return false;
    if (wpr_w > 1 && !magic(wpr_w, wrow_w, &mg_wpr)) return false;    // (one word per row: the kernel does not divide)
    out->magic_wrow = mg_wrow;
    out->magic_wpr = mg_wpr;
    out->G = G;
    out->rows_max = rows_max;
    out->threads = threads;
    out->smem = (int)smem;
    out->D = D;
    out->dmax = dmax;
    out->early = (D == 1 && (long long)(lat.L / G) * rowl / 4 >= 768) ? 1 : 0;
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
    constexpr bool CAN_NEV = MODEL == M_ISING_HALF || MODEL == M_ISING_ONE || MODEL == M_EA || MODEL == M_POTTS;
    const bool pow2 = a.lg_wrow >= 0;
    auto pick = [&](auto TR, auto OB, auto NV) -> cudaError_t {
        constexpr bool T_ = decltype(TR)::value, N_ = decltype(NV)::value;
        constexpr int O_ = decltype(OB)::value;
        return pow2 ? go(k_sweep_slab<MODEL, DIMS, T_, O_, N_, true>) : go(k_sweep_slab<MODEL, DIMS, T_, O_, N_, false>);
    };
    using std::integral_constant;
    using BT = integral_constant<bool, true>;
    using BF = integral_constant<bool, false>;
    using I0 = integral_constant<int, 0>;
    using I2 = integral_constant<int, 2>;
    if constexpr (CAN_NEV) {
        if (t.has_never) {
            if (track) return obs ? pick(BT{}, I2{}, BT{}) : pick(BT{}, I0{}, BT{});
            return obs ? pick(BF{}, I2{}, BT{}) : pick(BF{}, I0{}, BT{});
        }
    }
    if (track) return obs ? pick(BT{}, I2{}, BF{}) : pick(BT{}, I0{}, BF{});
    return obs ? pick(BF{}, I2{}, BF{}) : pick(BF{}, I0{}, BF{});
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
    a.bnd[0] = reinterpret_cast<const uint32_t *>(lat.bnd[0]);
    a.bnd[1] = reinterpret_cast<const uint32_t *>(lat.bnd[1]);
    a.seed = seed;
    a.t0 = t0;
    a.nsweeps = nsweeps;
    a.L = lat.L;
    a.wpr = lat.L / 32;
    a.R = lat.dims == 3 ? lat.L : 1;
    a.magic_wrow = plan.magic_wrow;
    a.magic_wpr = plan.magic_wpr;
    a.lg_wpr = a.lg_wrow = -1;                             // L a power of two: the shift / mask instantiations
    if ((lat.L & (lat.L - 1)) == 0) {
        int lg = 0;
        while ((1 << lg) < lat.L) ++lg;
        a.lg_wpr = lg - 5;
        a.lg_wrow = a.lg_wpr + (lat.dims == 3 ? lg : 0);
    }
    a.rows_max = plan.rows_max;
    a.D = plan.D;
    a.dmax = plan.dmax;
    a.early = plan.early;
    a.one = 1;
    a.qm1 = model == M_POTTS ? lat.q - 1 : 0;
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
    case M_POTTS: {
        HalfTab ht;
        for (int i = 0; i < 16; ++i) ht.t[i] = t.t32[i];
        return lat.dims == 3 ? slab_launch_to<M_POTTS, 3>(tr, obs, plan, s, a, pk, ht, t)
                             : slab_launch_to<M_POTTS, 2>(tr, obs, plan, s, a, pk, ht, t);
    }
    case M_EA: {
        HalfTab ht;
        for (int i = 0; i < 16; ++i) ht.t[i] = t.t32[i];
        return lat.dims == 3 ? slab_launch_to<M_EA, 3>(tr, obs, plan, s, a, pk, ht, t)
                             : slab_launch_to<M_EA, 2>(tr, obs, plan, s, a, pk, ht, t);
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
