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
#include "lsm_tiled.cuh"

#include <cstdlib>
#include <cstring>

namespace lsmk {

// ------------------------------------------------------------------------------------------
// Philox4x32-10 with the warp-uniform part hoisted.  In a half-sweep the counter is
// (c0 = group, c1 = 0, c2 = sweep, c3 = stream tag): c1, c2, c3 and the key are the same for every
// site, so in round 1 the product M1*c2 and in round 2 the product M0*c0' do not depend on the
// site.  The host evaluates them once per launch; the function below is bit-identical to the plain
// ten rounds (every parity test exercises it against the oracle's plain Philox).
// 18 IMAD.WIDE.U32 + 19 LOP3 per call.
// ------------------------------------------------------------------------------------------
struct PhiloxSweepConsts {
    uint32_t x1;        // c3 ^ k1                      (round 1: n2 = hi(M0*c0) ^ x1)
    uint32_t y2;        // lo(M1*c2) ^ (k0 + W0)        (round 2: n0 = hi(M1*c2') ^ y2)
    uint32_t z2;        // hi(M0*A0) ^ (k1 + W1)        (round 2: n2 = c3' ^ z2)
    uint32_t w3;        // lo(M0*A0) ^ (k1 + 2*W1)      (round 3: n2 = hi(M0*c0'') ^ w3)
    uint32_t rk0[10];   // k0 + r*W0
    uint32_t rk1[10];   // k1 + r*W1
};

static PhiloxSweepConsts make_philox_consts(const SweepKey &k)
{
    PhiloxSweepConsts c;
    for (int r = 0; r < 10; ++r) {
        c.rk0[r] = k.k0 + (uint32_t)r * PHILOX_W0;
        c.rk1[r] = k.k1 + (uint32_t)r * PHILOX_W1;
    }
    unsigned long long p1 = (unsigned long long)PHILOX_M1 * k.c2;
    uint32_t A0 = (uint32_t)(p1 >> 32) ^ 0u ^ c.rk0[0];   // c0 after round 1 (c1 = 0)
    uint32_t A1 = (uint32_t)p1;                           // c1 after round 1
    unsigned long long p0 = (unsigned long long)PHILOX_M0 * A0;
    c.x1 = k.c3 ^ c.rk1[0];
    c.y2 = A1 ^ c.rk0[1];
    c.z2 = (uint32_t)(p0 >> 32) ^ c.rk1[1];
    c.w3 = (uint32_t)p0 ^ c.rk1[2];
    return c;
}

__device__ __forceinline__ uint4 philox_sweep(uint32_t group, const PhiloxSweepConsts &pc)
{
    // round 1 (r = 0): only M0*c0 depends on the site
    unsigned long long q0 = (unsigned long long)PHILOX_M0 * group;
    uint32_t c2 = (uint32_t)(q0 >> 32) ^ pc.x1;
    uint32_t c3 = (uint32_t)q0;
    // round 2 (r = 1): c0 = A0, c1 = A1 are uniform
    unsigned long long q1 = (unsigned long long)PHILOX_M1 * c2;
    uint32_t c0 = (uint32_t)(q1 >> 32) ^ pc.y2;
    uint32_t c1 = (uint32_t)q1;
    c2 = c3 ^ pc.z2;
    // round 3 (r = 2): c3 = lo(M0*A0) is uniform and folded into w3
    {
        unsigned long long p0 = (unsigned long long)PHILOX_M0 * c0;
        unsigned long long p1 = (unsigned long long)PHILOX_M1 * c2;
        c0 = (uint32_t)(p1 >> 32) ^ c1 ^ pc.rk0[2];
        c2 = (uint32_t)(p0 >> 32) ^ pc.w3;
        c1 = (uint32_t)p1;
        c3 = (uint32_t)p0;
    }
#pragma unroll
    for (int r = 3; r < 10; ++r) {
        unsigned long long p0 = (unsigned long long)PHILOX_M0 * c0;
        unsigned long long p1 = (unsigned long long)PHILOX_M1 * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ pc.rk0[r];
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ pc.rk1[r];
        c1 = (uint32_t)p1;
        c3 = (uint32_t)p0;
        c0 = n0;
        c2 = n2;
    }
    return make_uint4(c0, c1, c2, c3);
}

// ------------------------------------------------------------------------------------------
// Kernel arguments
// ------------------------------------------------------------------------------------------
struct TiledGeom {
    uint8_t *own;          // colour being updated
    const uint8_t *oth;    // the other colour (read only during this launch)
    int L;                 // march extent
    int R;                 // cross rows (1 in 2D, L in 3D)
    int wpr;               // 16-byte words per compact row
    int ncol;              // R * wpr word columns
    int S;                 // march segments; threads = ncol * S
    int half;              // colour
    int parity_rows;       // 1: a warp's cross rows all have the same parity (see column_of)
    int one;               // the constant 1, kept opaque to the compiler (see rule_half)
    long long *obs;        // (B, M) accumulator or nullptr
};

struct HalfTab { uint32_t t[16]; };            // spin-1/2: t[n + 8*b] = thr - 1  (accept iff w <= t)
struct NeTab { uint32_t t32; int always; };
struct OneTab { uint2 e[96]; };
template <int MODEL> struct TabOf { using type = NeTab; };
template <> struct TabOf<M_ISING_HALF> { using type = HalfTab; };
template <> struct TabOf<M_ISING_ONE> { using type = OneTab; };

__device__ __forceinline__ uint32_t bytesum(uint32_t v) { return __dp4a(v, 0x01010101u, 0u); }

// s_t: shared-state-space address of the threshold table (warp-uniform, lives in a uniform
// register).  The per-site table offset is one byte extract of the pre-scaled index word and the
// load is LDS [R + UR].
__device__ __forceinline__ uint32_t lds_u32(uint32_t s_t, uint32_t byte_off)
{
    uint32_t v;
    asm("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(s_t + byte_off));
    return v;
}

// ------------------------------------------------------------------------------------------
// Per-lane (4 sites) update rules
// ------------------------------------------------------------------------------------------
// Ising spin-1/2 (readings D1, D3).  own: 4 site bytes; nsum: byte-wise sum of the
// 2d neighbour lanes (= number of up neighbours per site); r: the four random words of the lane.
// The table holds thr-1 for every (b, n), so "w < thr" is "w <= t" and thr = 2^32 needs no special
// case (tables with a thr = 0 entry are left to the scalar family, see tiled_supported).
// t + INC if w <= thr.  `one` is a register that holds 1 but is opaque to the compiler, so the
// predicated merge stays a multiply-add (IMAD): it issues on the FMA pipe, which has slack, instead of
// the binding ALU pipe.
template <uint32_t INC>
__device__ __forceinline__ uint32_t add_if_le(uint32_t t, uint32_t w, uint32_t thr, uint32_t one)
{
    asm("{\n\t.reg .pred p;\n\tsetp.le.u32 p, %1, %2;\n\t@p mad.lo.u32 %0, %3, %4, %0;\n\t}"
        : "+r"(t) : "r"(w), "r"(thr), "r"(one), "n"(INC));
    return t;
}

template <bool TRACK, int OBS>
__device__ __forceinline__ uint32_t rule_half(uint32_t own, uint32_t nsum, uint4 r, uint32_t s_t, uint32_t one,
                                              uint32_t &accU, uint32_t &accN, uint32_t &accBN)
{
    const uint32_t b = TRACK ? (own & 0x01010101u) : own;
    const uint32_t n = TRACK ? (nsum & 0x07070707u) : nsum;
    const uint32_t adr = b * 32u + n * 4u;                 // byte offset of t[n + 8b], per site byte
    uint32_t t = b;                                        // b + accepted flips (bytes end up 0, 1 or 2)
    t = add_if_le<0x00000001u>(t, r.x, lds_u32(s_t, adr & 0xFFu), one);
    t = add_if_le<0x00000100u>(t, r.y, lds_u32(s_t, __byte_perm(adr, 0u, 0x4441)), one);
    t = add_if_le<0x00010000u>(t, r.z, lds_u32(s_t, __byte_perm(adr, 0u, 0x4442)), one);
    t = add_if_le<0x01000000u>(t, r.w, lds_u32(s_t, adr >> 24), one);
    const uint32_t b2 = t & 0x01010101u;                   // b xor flip
    if (OBS >= 1) accU += b2;
    if (OBS >= 2) {
        accN += n;
        accBN += n & (b2 * 0xFFu);
    }
    if (!TRACK) return b2;
    const uint32_t fl = b ^ b2;
    return (own ^ fl) | (fl << 3);                         // value bit, and "ever changed" (0x08) set on a flip
}

// North-East model (readings D7, D8): facilitated iff north and east are up.
template <bool TRACK, bool METRO, int OBS>
__device__ __forceinline__ uint32_t rule_ne(uint32_t own, uint32_t north, uint32_t east, uint32_t group,
                                            const PhiloxSweepConsts &pc, uint32_t t32, int always, uint32_t &accU)
{
    uint32_t n = TRACK ? (own & 0x01010101u) : own;
    uint32_t fac = north & east & 0x01010101u;
    uint32_t n2 = n;
    if (fac != 0u) {                                       // random words are needed by facilitated sites only
        uint4 r = philox_sweep(group, pc);
        uint32_t lt = always ? 0x01010101u : 0u;
        if (r.x < t32) lt |= 0x00000001u;
        if (r.y < t32) lt |= 0x00000100u;
        if (r.z < t32) lt |= 0x00010000u;
        if (r.w < t32) lt |= 0x01000000u;
        if (METRO) n2 = n ^ (fac & (n | lt));              // 1->0 always, 0->1 iff w < thr
        else n2 = (n & ~fac) | (lt & fac);                 // heat bath: redraw from Bernoulli(c)
    }
    if (OBS >= 1) accU += n2;
    if (!TRACK) return n2;
    uint32_t f = n ^ n2;
    return (own & ~0x01010101u) | n2 | (f << 3);
}

// Ising spin-1 (reading D5): two words per site, so a lane needs two Philox calls.
template <int DIMS, bool TRACK, int OBS>
__device__ __forceinline__ uint32_t rule_one(uint32_t own, uint32_t nsum, uint4 ra, uint4 rb, const uint2 *s_e,
                                             int &accB, int &accM)
{
    const uint32_t w0[4] = {ra.x, ra.z, rb.x, rb.z};
    const uint32_t w1[4] = {ra.y, ra.w, rb.y, rb.w};
    uint32_t nw = own;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        uint32_t a = (own >> (8 * k)) & 3u;
        uint32_t sum = (nsum >> (8 * k)) & 0xFu;
        uint32_t kk = w0[k] >> 31;
        uint2 e = s_e[((a * 2u + kk) << 4) | sum];
        bool acc = (w1[k] < e.x) || (e.y & 0x10u);
        uint32_t a2 = acc ? (e.y & 3u) : a;
        uint32_t x = a ^ a2;                               // change of the two value bits
        nw ^= x << (8 * k);
        if (TRACK && x != 0u) nw |= 0x10u << (8 * k);      // "ever changed"
        if (OBS >= 1) accM += (int)a2 - 1;
        if (OBS >= 2) accB += ((int)a2 - 1) * ((int)sum - 2 * DIMS);
    }
    return nw;
}

// ------------------------------------------------------------------------------------------
// One thread's march.  Q is the row parity bit q = (march + cross + colour) & 1 of the current step
// when it is known at compile time (0 / 1: the side neighbour is the byte to the left / right), or
// 2 when it has to be read from the register (warps whose lanes mix row parities).
// ------------------------------------------------------------------------------------------
template <int MODEL, int DIMS, bool TRACK, int OBS>
struct March {
    const uint4 *pC;        // other colour, word of the current step
    uint4 *pO;              // own colour, word of the current step
    const uint32_t *pE;     // other colour, start of the current compact row (32-bit lanes)
    uint4 P, C;             // other colour at march-1 and march
    uint32_t grp;           // Philox group of lane 0 of the current word
    int m, q;
    int e_hi, e_lo, dyp, dyn, rowstride, L;
    long long wrapw;
    int totU, totN, totBN;  // per-thread sums; < 2^31 for every legal lattice
    uint32_t s_t, one;
    const uint2 *s_e;
    uint32_t ne_t32;
    int ne_always;

#ifndef LSM_TILED_PREFETCH
#define LSM_TILED_PREFETCH 0
#endif
    uint4 Nn, On;           // software pipeline, distance 1: loads of the next step, issued before this step computes
    uint32_t en;
    int m_end;

    // loads of the step `ahead` march positions after the current one (row parity qa)
    __device__ __forceinline__ void fetch(int ahead, int qa)
    {
        const uint4 *pN = pC + (ahead + 1) * rowstride;
        if (m + ahead + 1 >= L) pN -= wrapw;
        Nn = *pN;
        On = pO[ahead * rowstride];
        en = pE[ahead * rowstride * 4 + (qa ? e_hi : e_lo)];
    }

    template <int Q>
    __device__ __forceinline__ void step(const PhiloxSweepConsts &pc)
    {
        const int qq = Q == 2 ? q : Q;
#if LSM_TILED_PREFETCH
        const uint4 N = Nn;
        const uint4 O = On;
        const uint32_t e = en;
        if (m + 1 < m_end) fetch(1, qq ^ 1);
#else
        const uint4 *pN = pC + rowstride;
        if (m + 1 == L) pN -= wrapw;
        const uint4 N = *pN;
        const uint4 O = *pO;
        const uint32_t e = pE[qq ? e_hi : e_lo];
#endif
        uint4 Yp, Yn;
        if (DIMS == 3) {
            Yp = pC[dyp];
            Yn = pC[dyn];
        }
        // the neighbour one byte to the right (q = 1) or left (q = 0) of every site of the word
        uint32_t sd[4];
        if (qq) {
            sd[0] = __funnelshift_r(C.x, C.y, 8);
            sd[1] = __funnelshift_r(C.y, C.z, 8);
            sd[2] = __funnelshift_r(C.z, C.w, 8);
            sd[3] = __funnelshift_r(C.w, e, 8);
        } else {
            sd[0] = __funnelshift_r(e, C.x, 24);
            sd[1] = __funnelshift_r(C.x, C.y, 24);
            sd[2] = __funnelshift_r(C.y, C.z, 24);
            sd[3] = __funnelshift_r(C.z, C.w, 24);
        }
        const uint32_t o[4] = {O.x, O.y, O.z, O.w};
        const uint32_t p[4] = {P.x, P.y, P.z, P.w};
        const uint32_t n[4] = {N.x, N.y, N.z, N.w};
        const uint32_t c[4] = {C.x, C.y, C.z, C.w};
        uint32_t yp[4] = {0, 0, 0, 0}, yn[4] = {0, 0, 0, 0};
        if (DIMS == 3) {
            yp[0] = Yp.x; yp[1] = Yp.y; yp[2] = Yp.z; yp[3] = Yp.w;
            yn[0] = Yn.x; yn[1] = Yn.y; yn[2] = Yn.z; yn[3] = Yn.w;
        }
        uint32_t out[4];

        if (MODEL == M_ISING_HALF) {
            uint32_t accU = 0, accN = 0, accBN = 0;
#pragma unroll
            for (int d = 0; d < 4; ++d) {
                uint32_t ns = p[d] + n[d] + c[d] + sd[d];
                if (DIMS == 3) ns += yp[d] + yn[d];
                uint4 r = philox_sweep(grp + d, pc);
                out[d] = rule_half<TRACK, OBS>(o[d], ns, r, s_t, one, accU, accN, accBN);
            }
            if (OBS >= 1) totU += bytesum(accU);
            if (OBS >= 2) { totN += bytesum(accN); totBN += bytesum(accBN); }
        } else if (MODEL == M_ISING_ONE) {
            int accB = 0, accM = 0;
#pragma unroll
            for (int d = 0; d < 4; ++d) {
                uint32_t ns;
                if (TRACK) {
                    // flags sit at 0x10/0x60: two flagged bytes still add without a carry
                    ns = ((p[d] + n[d]) & 0x0F0F0F0Fu) + ((c[d] + sd[d]) & 0x0F0F0F0Fu);
                    if (DIMS == 3) ns += (yp[d] + yn[d]) & 0x0F0F0F0Fu;
                } else {
                    ns = p[d] + n[d] + c[d] + sd[d];
                    if (DIMS == 3) ns += yp[d] + yn[d];
                }
                uint4 ra = philox_sweep(2u * (grp + d), pc);
                uint4 rb = philox_sweep(2u * (grp + d) + 1u, pc);
                out[d] = rule_one<DIMS, TRACK, OBS>(o[d], ns, ra, rb, s_e, accB, accM);
            }
            totU += accM;
            totBN += accB;
        } else {
            uint32_t accU = 0;
#pragma unroll
            for (int d = 0; d < 4; ++d) {
                uint32_t east = qq ? sd[d] : c[d];
                out[d] = rule_ne<TRACK, MODEL == M_NE_METROPOLIS, OBS>(o[d], n[d], east, grp + d, pc, ne_t32, ne_always, accU);
            }
            if (OBS >= 1) totU += bytesum(accU);
        }
        *pO = make_uint4(out[0], out[1], out[2], out[3]);
        P = C;
        C = N;
        pC += rowstride;
        pO += rowstride;
        pE += rowstride * 4;
        grp += (uint32_t)rowstride * 4u;
        m += 1;
        if (Q == 2) q ^= 1;
    }

    template <int Q0>
    __device__ __forceinline__ void run(int m1, const PhiloxSweepConsts &pc)
    {
        constexpr int Q1 = Q0 == 2 ? 2 : 1 - Q0;
        m_end = m1;
#if LSM_TILED_PREFETCH
        fetch(0, Q0 == 2 ? q : Q0);
#endif
        while (m + 1 < m1) {
            step<Q0>(pc);
            step<Q1>(pc);
        }
        if (m < m1) step<Q0>(pc);
    }
};

// Thread -> (cross row y, word j).  With parity_rows the 32 lanes of a warp take 32/wpr rows of the
// SAME parity (rows y0, y0+2, ...; the neighbouring warp takes the rows in between), so that q is
// warp-uniform and can be a compile-time constant of the unrolled loop; every row is still read
// as whole contiguous 16*wpr-byte pieces.
__device__ __forceinline__ void column_of(const TiledGeom &g, int col, int &y, int &j)
{
    if (g.R == 1) { y = 0; j = col; return; }
    if (g.parity_rows && g.wpr < 32) {
        const int rpw = 32 / g.wpr;
        const int wg = col >> 5, lane = col & 31;
        y = (wg >> 1) * (2 * rpw) + 2 * (lane / g.wpr) + (wg & 1);
        j = lane % g.wpr;
    } else {
        y = col / g.wpr;
        j = col - y * g.wpr;
    }
}

#ifndef LSM_TILED_MINBLOCKS
#define LSM_TILED_MINBLOCKS 4
#endif
template <int MODEL, int DIMS, bool TRACK, int OBS>
__global__ void __launch_bounds__(256, LSM_TILED_MINBLOCKS)
k_sweep_tiled(const __grid_constant__ TiledGeom g, const __grid_constant__ PhiloxSweepConsts pc,
              const __grid_constant__ typename TabOf<MODEL>::type tab)
{
    __shared__ __align__(16) struct {
        uint32_t t[16];
        long long red[2][8];
        uint2 e[MODEL == M_ISING_ONE ? 96 : 1];
    } sm;
    uint32_t s_t = (uint32_t)__cvta_generic_to_shared(sm.t);
    asm volatile("" : "+r"(s_t));   // keep the (warp-uniform) table address out of the divergent region below
    March<MODEL, DIMS, TRACK, OBS> M;
    M.ne_t32 = 0;
    M.ne_always = 0;
    if constexpr (MODEL == M_ISING_HALF) {
        if (threadIdx.x < 16) sm.t[threadIdx.x] = tab.t[threadIdx.x];
    } else if constexpr (MODEL == M_ISING_ONE) {
        if (threadIdx.x < 96) sm.e[threadIdx.x] = tab.e[threadIdx.x];
    } else {
        M.ne_t32 = tab.t32;
        M.ne_always = tab.always;
    }
    __syncthreads();
    M.s_t = s_t;
    M.one = (uint32_t)g.one;
    M.s_e = sm.e;
    M.totU = M.totN = M.totBN = 0;

    const long long gt = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    int nsites = 0;
    if (gt < (long long)g.ncol * g.S) {
        const int seg = (int)(gt / g.ncol);
        const int col = (int)(gt - (long long)seg * g.ncol);
        int y, j;
        column_of(g, col, y, j);
        const int m0 = (int)(((long long)g.L * seg) / g.S);
        const int m1 = (int)(((long long)g.L * (seg + 1)) / g.S);
        const int yu = (y + 1 == g.R) ? 0 : y + 1, yd = (y == 0) ? g.R - 1 : y - 1;
        M.e_hi = ((j + 1 == g.wpr) ? 0 : j + 1) * 4;               // first lane of the next word
        M.e_lo = ((j == 0) ? g.wpr - 1 : j - 1) * 4 + 3;           // last lane of the previous word
        M.rowstride = g.R * g.wpr;                                 // words per march step
        M.wrapw = (long long)g.L * M.rowstride;                    // words per colour array
        M.dyp = (yd - y) * g.wpr;                                  // cross-row neighbours (3D), in words
        M.dyn = (yu - y) * g.wpr;
        M.L = g.L;
        const long long w0 = (long long)m0 * M.rowstride + y * g.wpr + j;
        M.pC = reinterpret_cast<const uint4 *>(g.oth) + w0;
        M.pO = reinterpret_cast<uint4 *>(g.own) + w0;
        M.pE = reinterpret_cast<const uint32_t *>(g.oth) + ((long long)m0 * M.rowstride + y * g.wpr) * 4;
        M.grp = (uint32_t)w0 * 4u;
        M.m = m0;
        M.q = (m0 + y + g.half) & 1;
        M.P = *(m0 == 0 ? M.pC + (M.wrapw - M.rowstride) : M.pC - M.rowstride);
        M.C = *M.pC;
        nsites = 16 * (m1 - m0);
        if (g.parity_rows) {            // warp-uniform branch: q is a constant inside each loop
            if (M.q) M.template run<1>(m1, pc);
            else M.template run<0>(m1, pc);
        } else {
            M.template run<2>(m1, pc);
        }
    }

    if (OBS >= 1) {
        long long cB = 0, cM = 0;
        if (MODEL == M_ISING_HALF) {
            // sum of s' = 2b'-1 ; sum of s'*nn = sum (2b'-1)(2n-2d)
            cM = 2LL * M.totU - nsites;
            cB = 4LL * M.totBN - 2LL * M.totN - 4LL * DIMS * M.totU + 2LL * DIMS * nsites;
        } else if (MODEL == M_ISING_ONE) {
            cM = M.totU;
            cB = M.totBN;
        } else {
            cM = M.totU;
        }
        block_accumulate2_in(sm.red, cB, cM, g.obs, OBS >= 2, true);
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
    if (model == M_ISING_HALF) {
        t.usable = 1;
        for (int b = 0; b < 2; ++b)
            for (int n = 0; n <= 2 * d; ++n) {
                uint64_t v = thr[b * (2 * d + 1) + n];
                if (v == 0) t.usable = 0;                  // "never" cannot be written as w <= thr-1
                t.t32[n + 8 * b] = (uint32_t)(v - 1);
            }
    } else if (model == M_ISING_ONE) {
        t.usable = 1;
        for (int a = 0; a < 3; ++a)
            for (int kk = 0; kk < 2; ++kk)
                for (int s = 0; s <= 4 * d; ++s) {
                    uint64_t v = thr[(a * 2 + kk) * (4 * d + 1) + s];
                    uint32_t ap = (uint32_t)((a + 1 + kk) % 3);
                    t.s1[(a * 2 + kk) * 16 + s] = make_uint2(clip(v), ap | (v == ALWAYS ? 0x10u : 0u));
                }
    } else {
        t.usable = 1;
        t.ne_t32[0] = clip(thr[0]);
        t.ne_t32[1] = clip(thr[1]);
        t.ne_up_always = thr[1] == ALWAYS ? 1 : 0;
        if (thr[0] == ALWAYS) t.usable = 0;
    }
    *out = t;
}

bool tiled_supported(const Lat &lat, int model, const TiledTables &t)
{
    if (!t.usable) return false;
    if (lat.Lh % 16 != 0) return false;                    // whole 16-byte words per compact row
    if (lat.half / 4 > 0xFFFFFFFFll) return false;         // Philox group must fit c0 (c1 = 0 is hoisted)
    if (model == M_ISING_ONE && lat.half / 2 > 0xFFFFFFFFll) return false;
    return true;
}

// Launch shape: threads = word columns x march segments, one wave of CTAS_PER_SM resident CTAs per
// SM (finer segments do not help: measured, profiles/).  Overridable for tuning experiments.
static int env_int(const char *name, int dflt)
{
    const char *v = getenv(name);
    return (v && *v) ? atoi(v) : dflt;
}
static int g_tiled_ctas_per_sm = env_int("LSM_TILED_CTAS_PER_SM", 4);
static int g_tiled_waves_x4 = env_int("LSM_TILED_WAVES_X4", 4);   // waves in quarters

template <int MODEL, int DIMS, bool TRACK>
static cudaError_t launch_obs(int obs_mode, dim3 grid, cudaStream_t s, const TiledGeom &g, const PhiloxSweepConsts &pc,
                              const typename TabOf<MODEL>::type &tab)
{
    if (obs_mode == 0) k_sweep_tiled<MODEL, DIMS, TRACK, 0><<<grid, 256, 0, s>>>(g, pc, tab);
    else if (obs_mode == 1) k_sweep_tiled<MODEL, DIMS, TRACK, 1><<<grid, 256, 0, s>>>(g, pc, tab);
    else k_sweep_tiled<MODEL, DIMS, TRACK, 2><<<grid, 256, 0, s>>>(g, pc, tab);
    return cudaGetLastError();
}

template <int MODEL, int DIMS>
static cudaError_t launch_track(bool track, int obs_mode, dim3 grid, cudaStream_t s, const TiledGeom &g,
                                const PhiloxSweepConsts &pc, const typename TabOf<MODEL>::type &tab)
{
    if (track) return launch_obs<MODEL, DIMS, true>(obs_mode, grid, s, g, pc, tab);
    return launch_obs<MODEL, DIMS, false>(obs_mode, grid, s, g, pc, tab);
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
    // q = (march + y + colour) & 1 is warp-uniform if a warp sees one row parity only
    if (g.R == 1) g.parity_rows = 1;                                   // 2D: y = 0 for every thread
    else if (g.wpr % 32 == 0) g.parity_rows = 1;
    else if (g.wpr < 32 && 32 % g.wpr == 0 && g.R % (2 * (32 / g.wpr)) == 0) g.parity_rows = 1;
    else g.parity_rows = 0;
    long long target = (long long)sm_count() * g_tiled_ctas_per_sm * 256 * g_tiled_waves_x4 / 4;
    long long S = target / g.ncol;
    if (S < 1) S = 1;
    if (S > g.L) S = g.L;
    g.S = (int)S;
    long long threads = (long long)g.ncol * g.S;
    dim3 grid((unsigned)((threads + 255) / 256));

    PhiloxSweepConsts pc = make_philox_consts(a.key);
    int obs_mode = a.obs ? (a.want_B ? 2 : 1) : 0;
    const bool track = a.track != 0;
    const bool d3 = a.lat.dims == 3;
    switch (a.model) {
    case M_ISING_HALF: {
        HalfTab ht;
        for (int i = 0; i < 16; ++i) ht.t[i] = t.t32[i];
        return d3 ? launch_track<M_ISING_HALF, 3>(track, obs_mode, grid, s, g, pc, ht)
                  : launch_track<M_ISING_HALF, 2>(track, obs_mode, grid, s, g, pc, ht);
    }
    case M_ISING_ONE: {
        OneTab ot;
        for (int i = 0; i < 96; ++i) ot.e[i] = t.s1[i];
        return d3 ? launch_track<M_ISING_ONE, 3>(track, obs_mode, grid, s, g, pc, ot)
                  : launch_track<M_ISING_ONE, 2>(track, obs_mode, grid, s, g, pc, ot);
    }
    case M_NE_HEATBATH: {
        NeTab nt = {t.ne_t32[0], 0};
        return launch_track<M_NE_HEATBATH, 2>(track, obs_mode > 1 ? 1 : obs_mode, grid, s, g, pc, nt);
    }
    default: {
        NeTab nt = {t.ne_t32[1], t.ne_up_always};
        return launch_track<M_NE_METROPOLIS, 2>(track, obs_mode > 1 ? 1 : obs_mode, grid, s, g, pc, nt);
    }
    }
}

}  // namespace lsmk
