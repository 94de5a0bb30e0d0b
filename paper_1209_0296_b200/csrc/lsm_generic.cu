// lsm_generic.cu -- the scalar kernel family: one thread per site of the active colour, any even
// L >= 4, every model.  It is the first parity-checked path and the fallback for lattices the tiled
// kernels do not cover; it also holds the once-per-call kernels (initial state, full reduction,
// persistence/overlap reduction, layout conversion) and the Philox test hooks.
//
// Method: PAPER.md:88 (Metropolis), 90-98 (two launches per sweep, one per sublattice), 118 (NE
// constraint); readings D1-D12 of DESIGN.md.  No code is shared with oracle/.
#include "lsm_internal.cuh"

namespace lsmk {

int sm_count()
{
    static int n = 0;
    if (n == 0) {
        int dev = 0;
        if (cudaGetDevice(&dev) != cudaSuccess) return 148;
        if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) n = 148;
    }
    return n;
}

static inline int grid_for(long long work_items, int threads, int ctas_per_sm)
{
    long long g = (work_items + threads - 1) / threads;
    long long cap = (long long)sm_count() * ctas_per_sm;
    if (g > cap) g = cap;
    if (g < 1) g = 1;
    return (int)g;
}

// ------------------------------------------------------------------------------------------
// Geometry of the split layout.  Colour c holds the sites with (x+y+z)&1 == c; inside its array a
// site sits at k = i>>1 = m + Lh*(y + L*z) with x = 2m + q, q = (y+z+c)&1.  Its six (four)
// neighbours all have the other colour: same m in rows y+-1 and planes z+-1, and in its own row the
// bytes m and m+1 (q = 1) or m-1 and m (q = 0).
// ------------------------------------------------------------------------------------------
struct Site {
    int m, y, z, q;
    long long row;   // (z*L + y) * Lh
};
__device__ __forceinline__ Site site_of(const Lat &lat, long long k, int colour)
{
    Site s;
    long long r = k / lat.Lh;
    s.m = (int)(k - r * lat.Lh);
    s.z = (int)(r / lat.L);
    s.y = (int)(r - (long long)s.z * lat.L);
    s.q = (s.y + s.z + colour) & 1;
    s.row = r * lat.Lh;
    return s;
}

template <int MODEL>
__device__ __forceinline__ int neighbour_value_sum(const Lat &lat, const uint8_t *__restrict__ oth, const Site &s,
                                                   uint32_t &north, uint32_t &east)
{
    constexpr uint32_t VAL = Enc<MODEL>::VAL;
    const int L = lat.L, Lh = lat.Lh;
    int yu = s.y + 1 == L ? 0 : s.y + 1, yd = s.y == 0 ? L - 1 : s.y - 1;
    long long plane = (long long)s.z * L;
    uint32_t up = oth[(plane + yu) * Lh + s.m] & VAL;
    uint32_t dn = oth[(plane + yd) * Lh + s.m] & VAL;
    uint32_t ce = oth[s.row + s.m] & VAL;
    int ms = s.q ? (s.m + 1 == Lh ? 0 : s.m + 1) : (s.m == 0 ? Lh - 1 : s.m - 1);
    uint32_t sd = oth[s.row + ms] & VAL;
    int sum = (int)(up + dn + ce + sd);
    if (lat.dims == 3) {
        int zu = s.z + 1 == L ? 0 : s.z + 1, zd = s.z == 0 ? L - 1 : s.z - 1;
        sum += (int)(oth[((long long)zu * L + s.y) * Lh + s.m] & VAL);
        sum += (int)(oth[((long long)zd * L + s.y) * Lh + s.m] & VAL);
    }
    north = up;                 // (x, y+1)
    east = s.q ? sd : ce;       // (x+1, y): byte m+1 of the row when q = 1, byte m when q = 0
    return sum;
}

// ------------------------------------------------------------------------------------------
// a2-a6, scalar form.
// ------------------------------------------------------------------------------------------
template <int MODEL>
__global__ void __launch_bounds__(256) k_sweep_generic(const __grid_constant__ SweepArgs a, const __grid_constant__ Thr64 thr)
{
    constexpr uint32_t VAL = Enc<MODEL>::VAL, CHG = Enc<MODEL>::CHG;
    __shared__ unsigned long long s_thr[96];
    for (int i = threadIdx.x; i < 96; i += blockDim.x) s_thr[i] = thr.thr[i];
    __syncthreads();

    const Lat &lat = a.lat;
    uint8_t *__restrict__ own = a.half ? lat.col[1] : lat.col[0];
    const uint8_t *__restrict__ oth = a.half ? lat.col[0] : lat.col[1];
    const int d = lat.dims;
    long long accB = 0, accM = 0;

    for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < lat.half;
         k += (long long)gridDim.x * blockDim.x) {
        Site s = site_of(lat, k, a.half);
        uint32_t old = own[k], v = old & VAL, vn = v;
        uint32_t north, east;
        int sum = neighbour_value_sum<MODEL>(lat, oth, s, north, east);
        int s_new, nn;
        if (MODEL == M_ISING_HALF) {
            uint4 r = philox4x32_10((uint32_t)(k >> 2), (uint32_t)(k >> 34), a.key.c2, a.key.c3, a.key.k0, a.key.k1);
            uint32_t w = (k & 2) ? ((k & 1) ? r.w : r.z) : ((k & 1) ? r.y : r.x);
            unsigned long long t = s_thr[v * (2 * d + 1) + sum];
            if ((unsigned long long)w < t) vn = v ^ 1u;
            s_new = 2 * (int)vn - 1;
            nn = 2 * sum - 2 * d;
        } else if (MODEL == M_ISING_ONE) {
            uint4 r = philox4x32_10((uint32_t)(k >> 1), (uint32_t)(k >> 33), a.key.c2, a.key.c3, a.key.k0, a.key.k1);
            uint32_t w0 = (k & 1) ? r.z : r.x, w1 = (k & 1) ? r.w : r.y;
            uint32_t kk = w0 >> 31;
            uint32_t ap = v + 1 + kk;
            ap = ap >= 3 ? ap - 3 : ap;
            unsigned long long t = s_thr[(v * 2 + kk) * (4 * d + 1) + sum];
            if ((unsigned long long)w1 < t) vn = ap;
            s_new = (int)vn - 1;
            nn = sum - 2 * d;
        } else {
            if (north & east) {
                uint4 r = philox4x32_10((uint32_t)(k >> 2), (uint32_t)(k >> 34), a.key.c2, a.key.c3, a.key.k0, a.key.k1);
                uint32_t w = (k & 2) ? ((k & 1) ? r.w : r.z) : ((k & 1) ? r.y : r.x);
                if (MODEL == M_NE_HEATBATH) vn = ((unsigned long long)w < s_thr[0]) ? 1u : 0u;
                else if ((unsigned long long)w < s_thr[1 + v]) vn = v ^ 1u;
            }
            s_new = (int)vn;
            nn = 0;
        }
        if (vn != v) {
            uint32_t nb = (old & ~VAL) | vn;
            if (a.track) nb |= CHG;
            own[k] = (uint8_t)nb;
        }
        accM += s_new;
        accB += s_new * nn;
    }
    if (a.obs) block_accumulate2(accB, accM, a.obs, a.want_B != 0, true);
}

// The 2d neighbours' bytes in the order k = 0: x-1, 1: x+1, 2: y-1, 3: y+1, 4: z-1, 5: z+1 (the order of the bond
// bits of M_EA).  x = 2m + q: the other colour's bytes of the own row are x-1 -> m (q = 1) or m-1 (q = 0) and
// x+1 -> m+1 (q = 1) or m (q = 0).
__device__ __forceinline__ void neighbour_bytes(const Lat &lat, const uint8_t *__restrict__ oth, const Site &s, uint32_t nb[6])
{
    const int L = lat.L, Lh = lat.Lh;
    const int yu = s.y + 1 == L ? 0 : s.y + 1, yd = s.y == 0 ? L - 1 : s.y - 1;
    const long long plane = (long long)s.z * L;
    const int ml = s.m == 0 ? Lh - 1 : s.m - 1, mr = s.m + 1 == Lh ? 0 : s.m + 1;
    nb[0] = oth[s.row + (s.q ? s.m : ml)];
    nb[1] = oth[s.row + (s.q ? mr : s.m)];
    nb[2] = oth[(plane + yd) * Lh + s.m];
    nb[3] = oth[(plane + yu) * Lh + s.m];
    nb[4] = nb[5] = 0;
    if (lat.dims == 3) {
        const int zu = s.z + 1 == L ? 0 : s.z + 1, zd = s.z == 0 ? L - 1 : s.z - 1;
        nb[4] = oth[((long long)zd * L + s.y) * Lh + s.m];
        nb[5] = oth[((long long)zu * L + s.y) * Lh + s.m];
    }
}

// NEXT-4 models, scalar form (readings D25, D26).
//  M_EA   : Ising spin-1/2 rule on the bond-weighted neighbour sum: an antiferromagnetic bond turns the neighbour's
//           "up" into "down", so the up-count is sum_k (b_k xor bond bit k); same table, same word map.
//  M_POTTS: two words per site (group k>>1): w0 proposes one of the other q-1 states, w1 accepts by Metropolis on
//           dn = (neighbours equal to the new state) - (neighbours equal to the old one); table idx dn + 2d.
// Observables: M_EA  M = sum s', B += s' * nn_eff (second colour only: every bond joins the two colours);
//              M_POTTS  M = sites in state 0, B += neighbours equal to the new state (second colour only).
template <int MODEL>
__global__ void __launch_bounds__(256) k_sweep_wider(const __grid_constant__ SweepArgs a, const __grid_constant__ Thr64 thr)
{
    constexpr uint32_t VAL = Enc<MODEL>::VAL, CHG = Enc<MODEL>::CHG;
    __shared__ unsigned long long s_thr[96];
    for (int i = threadIdx.x; i < 96; i += blockDim.x) s_thr[i] = thr.thr[i];
    __syncthreads();

    const Lat &lat = a.lat;
    uint8_t *__restrict__ own = a.half ? lat.col[1] : lat.col[0];
    const uint8_t *__restrict__ oth = a.half ? lat.col[0] : lat.col[1];
    const uint8_t *__restrict__ bnd = MODEL == M_EA ? (a.half ? lat.bnd[1] : lat.bnd[0]) : nullptr;
    const int d = lat.dims, nk = 2 * d;
    const uint32_t q = (uint32_t)lat.q;
    long long accB = 0, accM = 0;

    for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < lat.half;
         k += (long long)gridDim.x * blockDim.x) {
        const Site s = site_of(lat, k, a.half);
        const uint32_t old = own[k], v = old & VAL;
        uint32_t vn = v, nb[6];
        neighbour_bytes(lat, oth, s, nb);
        if (MODEL == M_EA) {
            const uint32_t bb = bnd[k];
            int sum = 0;
            for (int j = 0; j < nk; ++j) sum += (int)((nb[j] ^ (bb >> j)) & 1u);
            uint4 r = philox4x32_10((uint32_t)(k >> 2), (uint32_t)(k >> 34), a.key.c2, a.key.c3, a.key.k0, a.key.k1);
            uint32_t w = (k & 2) ? ((k & 1) ? r.w : r.z) : ((k & 1) ? r.y : r.x);
            if ((unsigned long long)w < s_thr[v * (2 * d + 1) + sum]) vn = v ^ 1u;
            const int s_new = 2 * (int)vn - 1;
            accM += s_new;
            accB += s_new * (2 * sum - 2 * d);
        } else {
            uint4 r = philox4x32_10((uint32_t)(k >> 1), (uint32_t)(k >> 33), a.key.c2, a.key.c3, a.key.k0, a.key.k1);
            const uint32_t w0 = (k & 1) ? r.z : r.x, w1 = (k & 1) ? r.w : r.y;
            uint32_t prop = v + 1u + __umulhi(w0, q - 1u);
            prop = prop >= q ? prop - q : prop;
            int n_old = 0, n_new = 0;
            for (int j = 0; j < nk; ++j) {
                n_old += (nb[j] & VAL) == v;
                n_new += (nb[j] & VAL) == prop;
            }
            if ((unsigned long long)w1 < s_thr[n_new - n_old + 2 * d]) { vn = prop; n_old = n_new; }
            accM += vn == 0u;
            accB += n_old;                      // neighbours equal to the state the site ends up in
        }
        if (vn != v) {
            uint32_t nbyte = (old & ~VAL) | vn;
            if (a.track) nbyte |= CHG;
            own[k] = (uint8_t)nbyte;
        }
    }
    if (a.obs) block_accumulate2(accB, accM, a.obs, a.want_B != 0, true);
}

cudaError_t launch_sweep_generic(const SweepArgs &a, const Thr64 &thr, cudaStream_t s)
{
    int grid = grid_for(a.lat.half, 256, 8);
    switch (a.model) {
    case M_EA:            k_sweep_wider<M_EA><<<grid, 256, 0, s>>>(a, thr); return cudaGetLastError();
    case M_POTTS:         k_sweep_wider<M_POTTS><<<grid, 256, 0, s>>>(a, thr); return cudaGetLastError();
    default: break;
    }
    switch (a.model) {
    case M_ISING_HALF:    k_sweep_generic<M_ISING_HALF><<<grid, 256, 0, s>>>(a, thr); break;
    case M_ISING_ONE:     k_sweep_generic<M_ISING_ONE><<<grid, 256, 0, s>>>(a, thr); break;
    case M_NE_HEATBATH:   k_sweep_generic<M_NE_HEATBATH><<<grid, 256, 0, s>>>(a, thr); break;
    default:              k_sweep_generic<M_NE_METROPOLIS><<<grid, 256, 0, s>>>(a, thr); break;
    }
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------
// a1: initial state (reading D4): stream 2, t = 0, group = i>>2 over the CANONICAL id, word i&3.
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_init(Lat lat, int model, SweepKey key, unsigned long long thr_c)
{
    long long groups = (2 * lat.half + 3) >> 2;
    for (long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x; g < groups;
         g += (long long)gridDim.x * blockDim.x) {
        uint4 r = philox4x32_10((uint32_t)g, (uint32_t)(g >> 32), key.c2, key.c3, key.k0, key.k1);
        uint32_t w[4] = {r.x, r.y, r.z, r.w};
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            long long i = 4 * g + j;
            if (i >= 2 * lat.half) break;
            long long ry = i / lat.L;
            int x = (int)(i - ry * lat.L);
            int z = (int)(ry / lat.L);
            int y = (int)(ry - (long long)z * lat.L);
            uint32_t v;
            if (model == M_ISING_HALF || model == M_EA) v = w[j] >> 31;
            else if (model == M_ISING_ONE) v = __umulhi(w[j], 3u);
            else if (model == M_POTTS) v = __umulhi(w[j], (uint32_t)lat.q);       // reading D26
            else v = ((unsigned long long)w[j] < thr_c) ? 1u : 0u;
            uint8_t *dst = ((x + y + z) & 1) ? lat.col[1] : lat.col[0];
            dst[i >> 1] = (uint8_t)v;
        }
    }
}

cudaError_t launch_init(const Lat &lat, int model, unsigned long long seed, unsigned long long thr_c, cudaStream_t s)
{
    SweepKey key = make_sweep_key(seed, 0ull, 2u);
    long long groups = (2 * lat.half + 3) >> 2;
    k_init<<<grid_for(groups, 256, 8), 256, 0, s>>>(lat, model, key, thr_c);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------
// a8: full reduction.  Every bond joins a colour-0 and a colour-1 site, so
// B = sum over colour-0 sites of s_i * nn_i; M sums both colours.
// ------------------------------------------------------------------------------------------
template <int MODEL>
__global__ void __launch_bounds__(256) k_measure_full(Lat lat, long long *out)
{
    constexpr uint32_t VAL = Enc<MODEL>::VAL;
    const uint8_t *__restrict__ c0 = lat.col[0];
    const uint8_t *__restrict__ c1 = lat.col[1];
    long long accB = 0, accM = 0;
    for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < lat.half;
         k += (long long)gridDim.x * blockDim.x) {
        Site s = site_of(lat, k, 0);
        uint32_t north, east;
        int sum = neighbour_value_sum<MODEL>(lat, c1, s, north, east);
        int v0 = (int)(c0[k] & VAL), v1 = (int)(c1[k] & VAL);
        if (MODEL == M_ISING_HALF) {
            accM += 2 * (v0 + v1) - 2;
            accB += (2 * v0 - 1) * (2 * sum - 2 * lat.dims);
        } else if (MODEL == M_ISING_ONE) {
            accM += v0 + v1 - 2;
            accB += (v0 - 1) * (sum - 2 * lat.dims);
        } else {
            accM += v0 + v1;
        }
    }
    block_accumulate2(accB, accM, out, true, true);
}

// Word-granular full reduction for lattices with whole 16-byte words per compact row (L % 32 == 0): a thread
// takes words of colour 1 and the same-index words of colour 0; the neighbour sums of 16 sites are byte-parallel
// adds of the colour-0 words at march +-1, cross row +-1 (3D) and the one-byte-shifted word of the own row, as in
// the sweep kernels.  Every bond joins the two colours, so B = sum over colour-1 sites of s_i * nn_i.
template <int MODEL, int DIMS>
__global__ void __launch_bounds__(256) k_measure_words(Lat lat, long long *out)
{
    constexpr uint32_t VAL = Enc<MODEL>::VAL * 0x01010101u;
    const uint4 *__restrict__ c0 = reinterpret_cast<const uint4 *>(lat.col[0]);
    const uint4 *__restrict__ c1 = reinterpret_cast<const uint4 *>(lat.col[1]);
    const uint32_t *__restrict__ c0l = reinterpret_cast<const uint32_t *>(lat.col[0]);
    const int wpr = lat.Lh >> 4, R = DIMS == 3 ? lat.L : 1, rs = R * wpr;
    const long long nw = (long long)lat.L * rs;
    int sA0 = 0, sA1 = 0, sAS = 0, sS = 0;           // sums of values (colour 0 / 1), of value * neighbour sum, of sums
    long long nwords = 0;
    for (long long w = (long long)blockIdx.x * blockDim.x + threadIdx.x; w < nw; w += (long long)gridDim.x * blockDim.x) {
        const long long row = w / wpr;
        const int j = (int)(w - row * wpr);
        const int m = (int)(row / R), y = (int)(row - (long long)m * R);
        const int q = (m + y + 1) & 1;                // colour-1 sites of this row: x = 2k + q
        const uint4 O = c1[w], C = c0[w];
        const uint4 P = c0[m == 0 ? w + nw - rs : w - rs], N = c0[m + 1 == lat.L ? w - nw + rs : w + rs];
        const int je = q ? (j + 1 == wpr ? 0 : j + 1) : (j == 0 ? wpr - 1 : j - 1);
        const uint32_t e = c0l[(row * wpr + je) * 4 + (q ? 0 : 3)];
        uint4 Yp = make_uint4(0, 0, 0, 0), Yn = Yp;
        if (DIMS == 3) {
            Yp = c0[w + (y == 0 ? (long long)(R - 1) * wpr : -(long long)wpr)];
            Yn = c0[w + (y + 1 == R ? -(long long)(R - 1) * wpr : (long long)wpr)];
        }
        const uint32_t o[4] = {O.x, O.y, O.z, O.w}, c[4] = {C.x, C.y, C.z, C.w}, p[4] = {P.x, P.y, P.z, P.w},
                       n[4] = {N.x, N.y, N.z, N.w}, yp[4] = {Yp.x, Yp.y, Yp.z, Yp.w}, yn[4] = {Yn.x, Yn.y, Yn.z, Yn.w};
        uint32_t sd[4];
        if (q) {
            sd[0] = __funnelshift_r(c[0], c[1], 8); sd[1] = __funnelshift_r(c[1], c[2], 8);
            sd[2] = __funnelshift_r(c[2], c[3], 8); sd[3] = __funnelshift_r(c[3], e, 8);
        } else {
            sd[0] = __funnelshift_r(e, c[0], 24); sd[1] = __funnelshift_r(c[0], c[1], 24);
            sd[2] = __funnelshift_r(c[1], c[2], 24); sd[3] = __funnelshift_r(c[2], c[3], 24);
        }
#pragma unroll
        for (int d = 0; d < 4; ++d) {
            uint32_t ns = (p[d] & VAL) + (n[d] & VAL) + (c[d] & VAL) + (sd[d] & VAL);
            if (DIMS == 3) ns += (yp[d] & VAL) + (yn[d] & VAL);
            const uint32_t v1 = o[d] & VAL, v0 = c[d] & VAL;
            sA0 = (int)__dp4a(v0, 0x01010101u, (uint32_t)sA0);
            sA1 = (int)__dp4a(v1, 0x01010101u, (uint32_t)sA1);
            if (MODEL == M_ISING_HALF || MODEL == M_ISING_ONE) {
                sAS = (int)__dp4a(v1, ns, (uint32_t)sAS);
                if (MODEL == M_ISING_ONE) sS = (int)__dp4a(ns, 0x01010101u, (uint32_t)sS);
            }
        }
        ++nwords;
    }
    const long long n1 = 16 * nwords;                 // colour-1 sites (= colour-0 sites) this thread visited
    long long accB = 0, accM = 0;
    if (MODEL == M_ISING_HALF) {
        // s = 2b - 1, nn = 2n - 2d, sum over colour-1 sites of n = 2d * (ups of colour 0)
        accM = 2LL * (sA0 + sA1) - 2 * n1;
        accB = 4LL * sAS - 4LL * DIMS * sA1 - 4LL * DIMS * sA0 + 2LL * DIMS * n1;
    } else if (MODEL == M_ISING_ONE) {
        accM = (long long)sA0 + sA1 - 2 * n1;
        accB = (long long)sAS - 2LL * DIMS * sA1 - sS + 2LL * DIMS * n1;
    } else {
        accM = (long long)sA0 + sA1;
    }
    block_accumulate2(accB, accM, out, true, true);
}

// Full reduction of the NEXT-4 models: B over the colour-0 sites' bonds (every bond joins the two colours).
template <int MODEL>
__global__ void __launch_bounds__(256) k_measure_wider(Lat lat, long long *out)
{
    constexpr uint32_t VAL = Enc<MODEL>::VAL;
    long long accB = 0, accM = 0;
    const int nk = 2 * lat.dims;
    for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < lat.half;
         k += (long long)gridDim.x * blockDim.x) {
        const Site s = site_of(lat, k, 0);
        uint32_t nb[6];
        neighbour_bytes(lat, lat.col[1], s, nb);
        const uint32_t v0 = lat.col[0][k] & VAL, v1 = lat.col[1][k] & VAL;
        if (MODEL == M_EA) {
            const uint32_t bb = lat.bnd[0][k];
            int sum = 0;
            for (int j = 0; j < nk; ++j) sum += (int)((nb[j] ^ (bb >> j)) & 1u);
            accM += 2 * (int)(v0 + v1) - 2;
            accB += (2 * (int)v0 - 1) * (2 * sum - nk);
        } else {
            for (int j = 0; j < nk; ++j) accB += (nb[j] & VAL) == v0;
            accM += (v0 == 0u) + (v1 == 0u);
        }
    }
    block_accumulate2(accB, accM, out, true, true);
}

cudaError_t launch_measure_full(const Lat &lat, int model, long long *d_BM, cudaStream_t s)
{
    cudaError_t e = cudaMemsetAsync(d_BM, 0, 2 * sizeof(long long), s);
    if (e != cudaSuccess) return e;
    if (model == M_EA || model == M_POTTS) {
        const int grid = grid_for(lat.half, 256, 8);
        if (model == M_EA) k_measure_wider<M_EA><<<grid, 256, 0, s>>>(lat, d_BM);
        else k_measure_wider<M_POTTS><<<grid, 256, 0, s>>>(lat, d_BM);
        return cudaGetLastError();
    }
    if (lat.Lh % 16 == 0) {
        const int grid = grid_for(lat.half >> 4, 256, 8);
        const bool d3 = lat.dims == 3;
        if (model == M_ISING_HALF) {
            if (d3) k_measure_words<M_ISING_HALF, 3><<<grid, 256, 0, s>>>(lat, d_BM);
            else k_measure_words<M_ISING_HALF, 2><<<grid, 256, 0, s>>>(lat, d_BM);
        } else if (model == M_ISING_ONE) {
            if (d3) k_measure_words<M_ISING_ONE, 3><<<grid, 256, 0, s>>>(lat, d_BM);
            else k_measure_words<M_ISING_ONE, 2><<<grid, 256, 0, s>>>(lat, d_BM);
        } else {
            k_measure_words<M_NE_HEATBATH, 2><<<grid, 256, 0, s>>>(lat, d_BM);
        }
        return cudaGetLastError();
    }
    int grid = grid_for(lat.half, 256, 8);
    if (model == M_ISING_HALF) k_measure_full<M_ISING_HALF><<<grid, 256, 0, s>>>(lat, d_BM);
    else if (model == M_ISING_ONE) k_measure_full<M_ISING_ONE><<<grid, 256, 0, s>>>(lat, d_BM);
    else k_measure_full<M_NE_HEATBATH><<<grid, 256, 0, s>>>(lat, d_BM);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------
// a9: persistence / overlap reduction over the flag and reference bits (readings D11, D12).
// 16 sites per 128-bit load.
// ------------------------------------------------------------------------------------------
template <int MODEL>
__device__ __forceinline__ void persist_byte(uint32_t b, long long &nc, long long &ov)
{
    constexpr uint32_t VAL = Enc<MODEL>::VAL, CHG = Enc<MODEL>::CHG, REF = Enc<MODEL>::REF;
    constexpr int SH = Enc<MODEL>::REF_SHIFT;
    nc += (b & CHG) ? 0 : 1;
    int now = (int)(b & VAL), ref = (int)((b & REF) >> SH);
    if (MODEL == M_ISING_ONE) ov += (now - 1) * (ref - 1);
    else if (MODEL == M_POTTS) ov += now == ref;              // reading D26: sites in their reference state
    else ov += (2 * now - 1) * (2 * ref - 1);
}

template <int MODEL>
__global__ void __launch_bounds__(256) k_persistence(Lat lat, long long *out)
{
    long long nc = 0, ov = 0;
#pragma unroll
    for (int c = 0; c < 2; ++c) {
        const uint8_t *__restrict__ p = c ? lat.col[1] : lat.col[0];
        long long nvec = lat.half >> 4;
        const uint4 *__restrict__ pv = reinterpret_cast<const uint4 *>(p);
        for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < nvec;
             i += (long long)gridDim.x * blockDim.x) {
            uint4 v = pv[i];
            uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
            for (int j = 0; j < 4; ++j)
#pragma unroll
                for (int b = 0; b < 4; ++b) persist_byte<MODEL>((w[j] >> (8 * b)) & 0xFFu, nc, ov);
        }
        for (long long i = (nvec << 4) + (long long)blockIdx.x * blockDim.x + threadIdx.x; i < lat.half;
             i += (long long)gridDim.x * blockDim.x)
            persist_byte<MODEL>(p[i], nc, ov);
    }
    block_accumulate2(nc, ov, out, true, true);
}

cudaError_t launch_persistence(const Lat &lat, int model, long long *d_out2, cudaStream_t s)
{
    cudaError_t e = cudaMemsetAsync(d_out2, 0, 2 * sizeof(long long), s);
    if (e != cudaSuccess) return e;
    int grid = grid_for((lat.half >> 4) + 1, 256, 8);
    if (model == M_ISING_ONE) k_persistence<M_ISING_ONE><<<grid, 256, 0, s>>>(lat, d_out2);
    else if (model == M_POTTS) k_persistence<M_POTTS><<<grid, 256, 0, s>>>(lat, d_out2);
    else if (model == M_ISING_HALF || model == M_EA) k_persistence<M_ISING_HALF><<<grid, 256, 0, s>>>(lat, d_out2);
    else k_persistence<M_NE_HEATBATH><<<grid, 256, 0, s>>>(lat, d_out2);
    return cudaGetLastError();
}

// Reference snapshot := current value, flags cleared (tracking_on) / all upper bits dropped (off).
template <int MODEL>
__global__ void __launch_bounds__(256) k_reset_reference(Lat lat, int tracking_on)
{
    constexpr uint32_t VAL = Enc<MODEL>::VAL;
    constexpr int SH = Enc<MODEL>::REF_SHIFT;
#pragma unroll
    for (int c = 0; c < 2; ++c) {
        uint8_t *p = c ? lat.col[1] : lat.col[0];
        for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < lat.half;
             i += (long long)gridDim.x * blockDim.x) {
            uint32_t v = p[i] & VAL;
            p[i] = (uint8_t)(tracking_on ? (v | (v << SH)) : v);
        }
    }
}

cudaError_t launch_reset_reference(const Lat &lat, int model, int tracking_on, cudaStream_t s)
{
    int grid = grid_for(lat.half, 256, 8);
    if (model == M_ISING_ONE) k_reset_reference<M_ISING_ONE><<<grid, 256, 0, s>>>(lat, tracking_on);
    else if (model == M_POTTS) k_reset_reference<M_POTTS><<<grid, 256, 0, s>>>(lat, tracking_on);
    else k_reset_reference<M_ISING_HALF><<<grid, 256, 0, s>>>(lat, tracking_on);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------
// Canonical int8 values <-> split internal layout.
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ void canon_to_split(const Lat &lat, long long i, int &colour)
{
    long long ry = i / lat.L;
    int x = (int)(i - ry * lat.L);
    int z = (int)(ry / lat.L);
    int y = (int)(ry - (long long)z * lat.L);
    colour = (x + y + z) & 1;
}

__global__ void __launch_bounds__(256) k_get_spins(Lat lat, int model, int8_t *__restrict__ out)
{
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < 2 * lat.half;
         i += (long long)gridDim.x * blockDim.x) {
        int c;
        canon_to_split(lat, i, c);
        uint32_t b = (c ? lat.col[1] : lat.col[0])[i >> 1];
        int v;
        if (model == M_ISING_HALF || model == M_EA) v = 2 * (int)(b & 1u) - 1;
        else if (model == M_ISING_ONE) v = (int)(b & 3u) - 1;
        else if (model == M_POTTS) v = (int)(b & 7u);
        else v = (int)(b & 1u);
        out[i] = (int8_t)v;
    }
}

__global__ void __launch_bounds__(256) k_set_spins(Lat lat, int model, const int8_t *__restrict__ in)
{
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < 2 * lat.half;
         i += (long long)gridDim.x * blockDim.x) {
        int c;
        canon_to_split(lat, i, c);
        int s = in[i];
        uint32_t v, mask;
        if (model == M_ISING_HALF || model == M_EA) { v = s > 0 ? 1u : 0u; mask = 1u; }
        else if (model == M_POTTS) { v = (uint32_t)(s < 0 ? 0 : (s >= lat.q ? lat.q - 1 : s)); mask = 7u; }
        else if (model == M_ISING_ONE) { v = (uint32_t)((s < -1 ? -1 : (s > 1 ? 1 : s)) + 1); mask = 3u; }
        else { v = s != 0 ? 1u : 0u; mask = 1u; }
        uint8_t *p = &(c ? lat.col[1] : lat.col[0])[i >> 1];
        *p = (uint8_t)((*p & ~mask) | v);
    }
}

// Word-granular conversions for lattices with whole 16-byte words per compact row: a thread converts 32 consecutive
// sites of one canonical row = one word of each colour (even x -> colour (y+z)&1, odd x -> the other), de-/interleaving
// bytes with PRMT.  Same value conventions as the scalar kernels above.
__device__ __forceinline__ uint32_t prmt_b(uint32_t a, uint32_t b, uint32_t sel)
{
    uint32_t r;
    asm("prmt.b32 %0, %1, %2, %3;" : "=r"(r) : "r"(a), "r"(b), "r"(sel));
    return r;
}
__device__ __forceinline__ uint32_t encode4(uint32_t s, int model)
{
    const uint32_t nz = (((s & 0x7F7F7F7Fu) + 0x7F7F7F7Fu) | s) & 0x80808080u;     // bit 7: byte != 0
    const uint32_t pos = (nz & ~s) >> 7;                                            // int8 > 0
    if (model == M_ISING_HALF) return pos;
    if (model == M_ISING_ONE) return (pos << 1) | ((nz ^ 0x80808080u) >> 7);       // < 0: 0, == 0: 1, > 0: 2
    return nz >> 7;
}
__device__ __forceinline__ uint32_t decode4(uint32_t b, int model)
{
    if (model == M_ISING_HALF) {
        const uint32_t t = b & 0x01010101u;
        return t | ((t ^ 0x01010101u) * 0xFFu);                                     // 1 -> +1, 0 -> -1
    }
    if (model == M_ISING_ONE) {
        const uint32_t z = (b | (b >> 1)) & 0x01010101u;                            // a != 0
        return ((b & 0x02020202u) >> 1) | ((z ^ 0x01010101u) * 0xFFu);              // 2 -> +1, 1 -> 0, 0 -> -1
    }
    return b & 0x01010101u;
}

__global__ void __launch_bounds__(256) k_set_spins_words(Lat lat, int model, const int8_t *__restrict__ in)
{
    const int wpr = lat.Lh >> 4;
    const long long nw = lat.half >> 4;
    const uint32_t keep = model == M_ISING_ONE ? 0xFCFCFCFCu : 0xFEFEFEFEu;
    for (long long w = (long long)blockIdx.x * blockDim.x + threadIdx.x; w < nw; w += (long long)gridDim.x * blockDim.x) {
        const long long row = w / wpr;                                              // canonical row z*L + y
        const int ce = (int)((row % lat.L + row / lat.L) & 1);                      // colour of the even-x sites
        const uint4 *src = reinterpret_cast<const uint4 *>(in + 2 * 16 * w);
        const uint4 A = src[0], B = src[1];
        const uint32_t x[8] = {A.x, A.y, A.z, A.w, B.x, B.y, B.z, B.w};
        uint32_t ev[4], od[4];
#pragma unroll
        for (int t = 0; t < 4; ++t) {
            ev[t] = encode4(prmt_b(x[2 * t], x[2 * t + 1], 0x6420u), model);
            od[t] = encode4(prmt_b(x[2 * t], x[2 * t + 1], 0x7531u), model);
        }
        uint4 *pe = reinterpret_cast<uint4 *>(ce ? lat.col[1] : lat.col[0]) + w;
        uint4 *po = reinterpret_cast<uint4 *>(ce ? lat.col[0] : lat.col[1]) + w;
        uint4 oe = *pe, oo = *po;                                                   // flags and snapshot stay
        *pe = make_uint4((oe.x & keep) | ev[0], (oe.y & keep) | ev[1], (oe.z & keep) | ev[2], (oe.w & keep) | ev[3]);
        *po = make_uint4((oo.x & keep) | od[0], (oo.y & keep) | od[1], (oo.z & keep) | od[2], (oo.w & keep) | od[3]);
    }
}

__global__ void __launch_bounds__(256) k_get_spins_words(Lat lat, int model, int8_t *__restrict__ out)
{
    const int wpr = lat.Lh >> 4;
    const long long nw = lat.half >> 4;
    for (long long w = (long long)blockIdx.x * blockDim.x + threadIdx.x; w < nw; w += (long long)gridDim.x * blockDim.x) {
        const long long row = w / wpr;
        const int ce = (int)((row % lat.L + row / lat.L) & 1);
        const uint4 E = reinterpret_cast<const uint4 *>(ce ? lat.col[1] : lat.col[0])[w];
        const uint4 O = reinterpret_cast<const uint4 *>(ce ? lat.col[0] : lat.col[1])[w];
        const uint32_t ev[4] = {decode4(E.x, model), decode4(E.y, model), decode4(E.z, model), decode4(E.w, model)};
        const uint32_t od[4] = {decode4(O.x, model), decode4(O.y, model), decode4(O.z, model), decode4(O.w, model)};
        uint32_t x[8];
#pragma unroll
        for (int t = 0; t < 4; ++t) {
            x[2 * t] = prmt_b(ev[t], od[t], 0x5140u);                               // e0 o0 e1 o1
            x[2 * t + 1] = prmt_b(ev[t], od[t], 0x7362u);                           // e2 o2 e3 o3
        }
        uint4 *dst = reinterpret_cast<uint4 *>(out + 2 * 16 * w);
        dst[0] = make_uint4(x[0], x[1], x[2], x[3]);
        dst[1] = make_uint4(x[4], x[5], x[6], x[7]);
    }
}

cudaError_t launch_get_spins(const Lat &lat, int model, int8_t *d_out, cudaStream_t s)
{
    if (model == M_EA) model = M_ISING_HALF;          // same byte encoding of the value
    if (model != M_POTTS && lat.Lh % 16 == 0 && ((uintptr_t)d_out & 15) == 0)
        k_get_spins_words<<<grid_for(lat.half >> 4, 256, 8), 256, 0, s>>>(lat, model, d_out);
    else
        k_get_spins<<<grid_for(2 * lat.half, 256, 8), 256, 0, s>>>(lat, model, d_out);
    return cudaGetLastError();
}
cudaError_t launch_set_spins(const Lat &lat, int model, const int8_t *d_in, cudaStream_t s)
{
    if (model == M_EA) model = M_ISING_HALF;
    if (model != M_POTTS && lat.Lh % 16 == 0 && ((uintptr_t)d_in & 15) == 0)
        k_set_spins_words<<<grid_for(lat.half >> 4, 256, 8), 256, 0, s>>>(lat, model, d_in);
    else
        k_set_spins<<<grid_for(2 * lat.half, 256, 8), 256, 0, s>>>(lat, model, d_in);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------
// Edwards-Anderson bonds (reading D25).  Canonical form: int8 tau[a][i] = sign of the bond between site i and its
// neighbour in direction +a.  Device form: one byte per site, bit k = the bond to neighbour k is antiferromagnetic
// (k = 2a: towards -a, stored canonically at the neighbour; k = 2a + 1: towards +a, stored at the site itself).
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ void site_coords(const Lat &lat, long long i, int &x, int &y, int &z)
{
    long long ry = i / lat.L;
    x = (int)(i - ry * lat.L);
    z = (int)(ry / lat.L);
    y = (int)(ry - (long long)z * lat.L);
}
// canonical id of the neighbour of (x, y, z) one step back along axis a
__device__ __forceinline__ long long back_neighbour(const Lat &lat, int x, int y, int z, int a)
{
    const int L = lat.L;
    if (a == 0) x = x == 0 ? L - 1 : x - 1;
    else if (a == 1) y = y == 0 ? L - 1 : y - 1;
    else z = z == 0 ? L - 1 : z - 1;
    return x + (long long)L * (y + (long long)L * z);
}

// tau from the seed: stream tag 3, t = 0, bond id b = a*N + i, group b>>2, word b&3, tau = +1 iff the top bit is set.
__global__ void __launch_bounds__(256) k_ea_bonds_init(Lat lat, SweepKey key)
{
    const long long N = 2 * lat.half;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (long long)gridDim.x * blockDim.x) {
        int x, y, z;
        site_coords(lat, i, x, y, z);
        uint32_t bits = 0;
        for (int a = 0; a < lat.dims; ++a) {
            const long long bf = (long long)a * N + i, bb = (long long)a * N + back_neighbour(lat, x, y, z, a);
            const uint4 rf = philox4x32_10((uint32_t)(bf >> 2), (uint32_t)(bf >> 34), key.c2, key.c3, key.k0, key.k1);
            const uint4 rb = philox4x32_10((uint32_t)(bb >> 2), (uint32_t)(bb >> 34), key.c2, key.c3, key.k0, key.k1);
            const uint32_t wf = (bf & 2) ? ((bf & 1) ? rf.w : rf.z) : ((bf & 1) ? rf.y : rf.x);
            const uint32_t wb = (bb & 2) ? ((bb & 1) ? rb.w : rb.z) : ((bb & 1) ? rb.y : rb.x);
            if (!(wf >> 31)) bits |= 1u << (2 * a + 1);          // antiferromagnetic bond towards +a
            if (!(wb >> 31)) bits |= 1u << (2 * a);              // ... towards -a
        }
        (((x + y + z) & 1) ? lat.bnd[1] : lat.bnd[0])[i >> 1] = (uint8_t)bits;
    }
}
__global__ void __launch_bounds__(256) k_ea_set_bonds(Lat lat, const int8_t *__restrict__ tau)
{
    const long long N = 2 * lat.half;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (long long)gridDim.x * blockDim.x) {
        int x, y, z;
        site_coords(lat, i, x, y, z);
        uint32_t bits = 0;
        for (int a = 0; a < lat.dims; ++a) {
            if (tau[(long long)a * N + i] < 0) bits |= 1u << (2 * a + 1);
            if (tau[(long long)a * N + back_neighbour(lat, x, y, z, a)] < 0) bits |= 1u << (2 * a);
        }
        (((x + y + z) & 1) ? lat.bnd[1] : lat.bnd[0])[i >> 1] = (uint8_t)bits;
    }
}
__global__ void __launch_bounds__(256) k_ea_get_bonds(Lat lat, int8_t *__restrict__ tau)
{
    const long long N = 2 * lat.half;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (long long)gridDim.x * blockDim.x) {
        int x, y, z;
        site_coords(lat, i, x, y, z);
        const uint32_t bits = (((x + y + z) & 1) ? lat.bnd[1] : lat.bnd[0])[i >> 1];
        for (int a = 0; a < lat.dims; ++a) tau[(long long)a * N + i] = (bits >> (2 * a + 1)) & 1u ? -1 : 1;
    }
}
cudaError_t launch_ea_bonds_init(const Lat &lat, unsigned long long seed, cudaStream_t s)
{
    k_ea_bonds_init<<<grid_for(2 * lat.half, 256, 8), 256, 0, s>>>(lat, make_sweep_key(seed, 0ull, 3u));
    return cudaGetLastError();
}
cudaError_t launch_ea_set_bonds(const Lat &lat, const int8_t *d_tau, cudaStream_t s)
{
    k_ea_set_bonds<<<grid_for(2 * lat.half, 256, 8), 256, 0, s>>>(lat, d_tau);
    return cudaGetLastError();
}
cudaError_t launch_ea_get_bonds(const Lat &lat, int8_t *d_tau, cudaStream_t s)
{
    k_ea_get_bonds<<<grid_for(2 * lat.half, 256, 8), 256, 0, s>>>(lat, d_tau);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------
// Test hooks: the device Philox on arbitrary (counter, key) pairs, and a register-only Philox
// throughput loop (the integer roofline of step a4).
// ------------------------------------------------------------------------------------------
__global__ void k_philox_device(const uint32_t *__restrict__ ck, uint32_t *__restrict__ out, long long n)
{
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n;
         i += (long long)gridDim.x * blockDim.x) {
        const uint32_t *p = ck + 6 * i;
        uint4 r = philox4x32_10(p[0], p[1], p[2], p[3], p[4], p[5]);
        out[4 * i + 0] = r.x; out[4 * i + 1] = r.y; out[4 * i + 2] = r.z; out[4 * i + 3] = r.w;
    }
}
cudaError_t launch_philox_device(const uint32_t *d_ck, uint32_t *d_out, long long n, cudaStream_t s)
{
    if (n <= 0) return cudaSuccess;
    k_philox_device<<<grid_for(n, 128, 8), 128, 0, s>>>(d_ck, d_out, n);
    return cudaGetLastError();
}

__global__ void __launch_bounds__(256) k_philox_throughput(int calls, uint32_t *__restrict__ sink)
{
    uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x;
    uint32_t acc = 0;
    // independent calls (counter = loop index), as in the sweep kernels: ILP across calls
#pragma unroll 4
    for (int i = 0; i < calls; ++i) {
        uint4 r = philox4x32_10(tid, 0u, (uint32_t)i, 1u, 0x1234567u, 0x89abcdefu);
        acc ^= r.x ^ r.y ^ r.z ^ r.w;
    }
    sink[tid] = acc;
}
cudaError_t launch_philox_throughput(int blocks, int calls, uint32_t *d_sink, cudaStream_t s)
{
    k_philox_throughput<<<blocks, 256, 0, s>>>(calls, d_sink);
    return cudaGetLastError();
}

}  // namespace lsmk
