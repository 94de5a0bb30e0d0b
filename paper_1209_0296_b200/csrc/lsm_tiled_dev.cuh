// lsm_tiled_dev.cuh -- device code of the vectorised half-sweep, shared by
// the one-launch-per-half-sweep kernel (lsm_tiled.cu), its bulk-copy form and the slab / small families: hoisted Philox,
// per-lane update rules, the register march of one thread.
#pragma once
#include "lsm_tiled.cuh"

#include <type_traits>

#define LSM_TILED_MINBLOCKS 4

// spin-1 needs two Philox calls per lane; measured 2/3/4 CTAs per SM: 518/478/414 Gflips/s on cfg4
#define LSM_TILED_MINBLOCKS_ONE 2
// spin-1/2 Ising: the march is bound by pipe issue, not by latency (4 independent Philox chains per thread), and runs
// fastest with 2 CTAs per SM and up to 128 registers (measured 1/2/3/4/5/6 CTAs: 1132/1163/1141/1120/1027/970
// Gflips/s on cfg2); the North-East rule, which skips Philox for most lanes, prefers 4.
#define LSM_TILED_MINBLOCKS_HALF 2

namespace lsmk {

constexpr int tiled_minblocks(int model)
{
    return (model == M_ISING_ONE || model == M_POTTS) ? LSM_TILED_MINBLOCKS_ONE
         : (model == M_ISING_HALF || model == M_EA) ? LSM_TILED_MINBLOCKS_HALF : LSM_TILED_MINBLOCKS;
}

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
    uint32_t m0, m1;    // the multipliers M0, M1 (operands from the parameter bank instead of 32-bit immediates)
};

// The per-half-sweep part (x1..w3) as the host computes it for one launch, or as the resident kernel
// recomputes it on the device at the start of every half-sweep.
__host__ __device__ inline void philox_half_consts(const SweepKey &k, const uint32_t *rk0, const uint32_t *rk1,
                                                   uint32_t &x1, uint32_t &y2, uint32_t &z2, uint32_t &w3)
{
    unsigned long long p1 = (unsigned long long)PHILOX_M1 * k.c2;
    uint32_t A0 = (uint32_t)(p1 >> 32) ^ 0u ^ rk0[0];     // c0 after round 1 (c1 = 0)
    uint32_t A1 = (uint32_t)p1;                           // c1 after round 1
    unsigned long long p0 = (unsigned long long)PHILOX_M0 * A0;
    x1 = k.c3 ^ rk1[0];
    y2 = A1 ^ rk0[1];
    z2 = (uint32_t)(p0 >> 32) ^ rk1[1];
    w3 = (uint32_t)p0 ^ rk1[2];
}

// Resident kernel: x1..w3 live in registers, the round keys stay in the kernel-parameter bank.
struct PhiloxDyn {
    uint32_t x1, y2, z2, w3;
    const PhiloxSweepConsts &k;
};
__device__ __forceinline__ uint32_t prk0(const PhiloxSweepConsts &p, int r) { return p.rk0[r]; }
__device__ __forceinline__ uint32_t prk1(const PhiloxSweepConsts &p, int r) { return p.rk1[r]; }
__device__ __forceinline__ uint32_t prk0(const PhiloxDyn &p, int r) { return p.k.rk0[r]; }
__device__ __forceinline__ uint32_t prk1(const PhiloxDyn &p, int r) { return p.k.rk1[r]; }
// CB: the multipliers are operands from the kernel-parameter bank (uniform registers) instead of 32-bit immediates.
// Measured on one GPU (A/B, results identical): +0.6 % for the spin-1/2 rule of the tiled family (8192^2, 512^3), but
// -2.7 % for spin-1, -0.9 % for the North-East rule and -0.5 % in the slab family, so only that rule asks for it.
template <bool CB, class PC> __device__ __forceinline__ uint32_t pm0(const PC &p)
{
    if constexpr (CB && std::is_same<PC, PhiloxSweepConsts>::value) return p.m0;
    else return PHILOX_M0;
}
template <bool CB, class PC> __device__ __forceinline__ uint32_t pm1(const PC &p)
{
    if constexpr (CB && std::is_same<PC, PhiloxSweepConsts>::value) return p.m1;
    else return PHILOX_M1;
}

template <bool CB = false, class PC>
__device__ __forceinline__ uint4 philox_sweep(uint32_t group, const PC &pc)
{
    // round 1 (r = 0): only M0*c0 depends on the site
    unsigned long long q0 = (unsigned long long)pm0<CB>(pc) * group;
    uint32_t c2 = (uint32_t)(q0 >> 32) ^ pc.x1;
    uint32_t c3 = (uint32_t)q0;
    // round 2 (r = 1): c0 = A0, c1 = A1 are uniform
    unsigned long long q1 = (unsigned long long)pm1<CB>(pc) * c2;
    uint32_t c0 = (uint32_t)(q1 >> 32) ^ pc.y2;
    uint32_t c1 = (uint32_t)q1;
    c2 = c3 ^ pc.z2;
    // round 3 (r = 2): c3 = lo(M0*A0) is uniform and folded into w3
    {
        unsigned long long p0 = (unsigned long long)pm0<CB>(pc) * c0;
        unsigned long long p1 = (unsigned long long)pm1<CB>(pc) * c2;
        c0 = (uint32_t)(p1 >> 32) ^ c1 ^ prk0(pc, 2);
        c2 = (uint32_t)(p0 >> 32) ^ pc.w3;
        c1 = (uint32_t)p1;
        c3 = (uint32_t)p0;
    }
#pragma unroll
    for (int r = 3; r < 10; ++r) {
        unsigned long long p0 = (unsigned long long)pm0<CB>(pc) * c0;
        unsigned long long p1 = (unsigned long long)pm1<CB>(pc) * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ prk0(pc, r);
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ prk1(pc, r);
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
    const uint8_t *bnd;    // M_EA: bond bytes of the colour being updated (same geometry as own); else nullptr
    int qm1;               // M_POTTS: q - 1
};

struct HalfTab { uint32_t t[16]; };            // spin-1/2: t[n + 8*b] = thr - 1  (accept iff w <= t)
struct NeTab { uint32_t t32; int always; int all4; };   // all4: one Philox region per word (c >= 0.15)
struct OneTab { uint32_t t[64]; };            // spin-1: t[16*dcode + sum] = thr - 1, dcode = class of s' - s
// Tables with a "never" entry (thr = 0: exp(-dE/T) < 2^-32, any cold lattice) cannot be written as w <= thr - 1.  The
// NEV instantiations of the tiled family carry a second table y at byte offset nev_offset() behind t and accept iff
// y <= w <= t:  thr in [1, 2^32]: t = thr - 1, y = 0;  thr = 0: t = 0, y = 1 (empty interval).  One more compare per site.
struct NevTab { uint32_t y[64]; };
template <int MODEL> __host__ __device__ constexpr uint32_t nev_offset() { return MODEL == M_ISING_ONE ? 256u : 64u; }
template <int MODEL> struct TabOf { using type = NeTab; };
template <> struct TabOf<M_ISING_HALF> { using type = HalfTab; };
template <> struct TabOf<M_ISING_ONE> { using type = OneTab; };
template <> struct TabOf<M_EA> { using type = HalfTab; };     // reading D25: the Ising table on the bond-weighted up-count
template <> struct TabOf<M_POTTS> { using type = HalfTab; };  // reading D26: t[dn + 2d] = thr - 1, 4d + 1 <= 13 entries

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
// t + INC if lo <= w <= hi (the NEV form)
template <uint32_t INC>
__device__ __forceinline__ uint32_t add_if_in(uint32_t t, uint32_t w, uint32_t hi, uint32_t lo, uint32_t one)
{
    asm("{\n\t.reg .pred p;\n\tsetp.ge.u32 p, %1, %3;\n\tsetp.le.and.u32 p, %1, %2, p;\n\t@p mad.lo.u32 %0, %4, %5, %0;\n\t}"
        : "+r"(t) : "r"(w), "r"(hi), "r"(lo), "r"(one), "n"(INC));
    return t;
}
// The threshold lookup and merge of one site: table byte offset `off`, shared-space table base s_t.
template <int MODEL, bool NEV, uint32_t INC>
__device__ __forceinline__ uint32_t accept_site(uint32_t t, uint32_t w, uint32_t s_t, uint32_t off, uint32_t one)
{
    if (NEV) return add_if_in<INC>(t, w, lds_u32(s_t, off), lds_u32(s_t + nev_offset<MODEL>(), off), one);
    return add_if_le<INC>(t, w, lds_u32(s_t, off), one);
}

// Observables (a6) cost no ALU-pipe instruction: the up-count and the sum of b'*n are IDP.4A dot products
// (FMA-heavy pipe) straight into the thread's 32-bit totals.
template <bool TRACK, int OBS, bool NEV = false>
__device__ __forceinline__ uint32_t rule_half(uint32_t own, uint32_t nsum, uint4 r, uint32_t s_t, uint32_t one,
                                              int &totU, int &totBN)
{
    const uint32_t b = TRACK ? (own & 0x01010101u) : own;
    const uint32_t n = TRACK ? (nsum & 0x07070707u) : nsum;
    const uint32_t adr = b * 32u + n * 4u;                 // byte offset of t[n + 8b], per site byte
    uint32_t t = b;                                        // b + accepted flips (bytes end up 0, 1 or 2)
    t = accept_site<M_ISING_HALF, NEV, 0x00000001u>(t, r.x, s_t, adr & 0xFFu, one);
    t = accept_site<M_ISING_HALF, NEV, 0x00000100u>(t, r.y, s_t, __byte_perm(adr, 0u, 0x4441), one);
    t = accept_site<M_ISING_HALF, NEV, 0x00010000u>(t, r.z, s_t, __byte_perm(adr, 0u, 0x4442), one);
    t = accept_site<M_ISING_HALF, NEV, 0x01000000u>(t, r.w, s_t, adr >> 24, one);
    const uint32_t b2 = t & 0x01010101u;                   // b xor flip
    if (OBS >= 1) totU = (int)__dp4a(b2, 0x01010101u, (uint32_t)totU);
    if (OBS >= 2) totBN = (int)__dp4a(n, b2, (uint32_t)totBN);
    if (!TRACK) return b2;
    const uint32_t fl = b ^ b2;
    return (own ^ fl) | (fl << 3);                         // value bit, and "ever changed" (0x08) set on a flip
}

// North-East model (readings D7, D8): facilitated iff north and east are up.
template <bool TRACK, bool METRO, int OBS, class PC>
__device__ __forceinline__ uint32_t rule_ne(uint32_t own, uint32_t north, uint32_t east, uint32_t group,
                                            const PC &pc, uint32_t t32, int always, uint32_t &accU)
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

// Ising spin-1 (reading D5): two words per site, so a lane needs two Philox calls (ra: sites 0, 1; rb: sites 2, 3;
// proposal word w0 = x / z, acceptance word w1 = y / w).  Byte-parallel over the 4 sites of the lane:
//   kk = msb(w0)                      -> byte mask (PRMT with sign replication)
//   proposal a' = (a + 1 + kk) mod 3  -> x = a ^ a' is a boolean function of (a1, a0, kk): two LOP3 + one bit-select
//   threshold                         -> depends on (s' - s, sum) only (D3, no single-ion term): the four classes
//                                        d = 0: +1, 1: +2, 2: -1, 3: -2 are again boolean functions of (a1, a0, kk);
//                                        table byte offset 64 d + 4 sum <= 240 fits the per-site byte of one word
//   accept iff w1 <= thr - 1          -> per site: extract, LDS, ISETP, predicated IMAD (as in rule_half)
// Observables: raw sums SA = sum a', SAS = sum a' * sum, SS = sum of sums (IDP.4A); march_observables converts.
__device__ __forceinline__ uint32_t prmt(uint32_t a, uint32_t b, uint32_t sel)
{
    uint32_t r;
    asm("prmt.b32 %0, %1, %2, %3;" : "=r"(r) : "r"(a), "r"(b), "r"(sel));
    return r;
}
// boolean functions of (A, B, C) evaluated bitwise by one LOP3
template <int LUT> __device__ __forceinline__ uint32_t lop3(uint32_t a, uint32_t b, uint32_t c)
{
    uint32_t r;
    asm("lop3.b32 %0, %1, %2, %3, %4;" : "=r"(r) : "r"(a), "r"(b), "r"(c), "n"(LUT));
    return r;
}
// LUT of f(A, B, C): bit (4A + 2B + C) of the constant
__host__ __device__ constexpr int lut3(bool f000, bool f001, bool f010, bool f011, bool f100, bool f101, bool f110, bool f111)
{
    return (f000 ? 1 : 0) | (f001 ? 2 : 0) | (f010 ? 4 : 0) | (f011 ? 8 : 0) | (f100 ? 16 : 0) | (f101 ? 32 : 0) |
           (f110 ? 64 : 0) | (f111 ? 128 : 0);
}

template <int DIMS, bool TRACK, int OBS, bool NEV = false>
__device__ __forceinline__ uint32_t rule_one(uint32_t own, uint32_t nsum, uint4 ra, uint4 rb, uint32_t s_t, uint32_t one,
                                             int &totSA, int &totSAS, int &totSS)
{
    // kk byte mask: 0xFF where the proposal word's top bit is set
    // (inline PTX: __byte_perm() drops bit 3 of the selector nibbles, the "replicate the sign" flag)
    const uint32_t klo = prmt(ra.x, ra.z, 0x00FBu), khi = prmt(rb.x, rb.z, 0x00FBu);
    const uint32_t kk = prmt(klo, khi, 0x5410u);
    const uint32_t dn = own >> 1, up = own << 1;           // a1 at bit 0 / a0 at bit 1 of every byte
    // at bit 0: A = a0 (own), B = a1 (own >> 1), C = kk.   rows: (a0, a1, kk)
    //   x0 = bit 0 of a ^ a':  a=0: !kk ; a=1 (a0=1,a1=0): 1 ; a=2 (a0=0,a1=1): kk
    //   d0 = bit 0 of dcode :  a=0: kk  ; a=1: 0 ; a=2: !kk
    constexpr int X0 = lut3(true, false, false, true, true, true, false, false);
    constexpr int D0 = lut3(false, true, true, false, false, false, false, false);
    // at bit 1: A = a1 (own), B = a0 (own << 1), C = kk.   rows: (a1, a0, kk)
    //   x1 = bit 1 of a ^ a':  a=0: kk ; a=1 (a1=0,a0=1): !kk ; a=2 (a1=1,a0=0): 1
    //   d1 = bit 1 of dcode :  a=0: 0  ; a=1: kk ; a=2: 1
    constexpr int X1 = lut3(false, true, true, false, true, true, false, false);
    constexpr int D1 = lut3(false, false, false, true, true, true, false, false);
    const uint32_t x = lop3<0xCA>(0x01010101u, lop3<X0>(own, dn, kk), lop3<X1>(own, up, kk));   // bit 0 | bit 1 (select)
    const uint32_t d = lop3<0xCA>(0x01010101u, lop3<D0>(own, dn, kk), lop3<D1>(own, up, kk)) & 0x03030303u;
    const uint32_t adr = d * 64u + nsum * 4u;              // byte offset of t[16 d + sum], per site byte
    uint32_t acc = 0u;                                     // 0xFF in the byte of every accepted site
    acc = accept_site<M_ISING_ONE, NEV, 0x000000FFu>(acc, ra.y, s_t, adr & 0xFFu, one);
    acc = accept_site<M_ISING_ONE, NEV, 0x0000FF00u>(acc, ra.w, s_t, __byte_perm(adr, 0u, 0x4441), one);
    acc = accept_site<M_ISING_ONE, NEV, 0x00FF0000u>(acc, rb.y, s_t, __byte_perm(adr, 0u, 0x4442), one);
    acc = accept_site<M_ISING_ONE, NEV, 0xFF000000u>(acc, rb.w, s_t, adr >> 24, one);
    const uint32_t fl = x & acc & 0x03030303u;             // change of the two value bits
    uint32_t nw = own ^ fl;
    if (TRACK) nw |= ((fl | (fl >> 1)) & 0x01010101u) << 4;    // "ever changed"
    if (OBS >= 1) {
        const uint32_t a2 = TRACK ? (nw & 0x03030303u) : nw;
        totSA = (int)__dp4a(a2, 0x01010101u, (uint32_t)totSA);
        if (OBS >= 2) {
            totSAS = (int)__dp4a(a2, nsum, (uint32_t)totSAS);
            totSS = (int)__dp4a(nsum, 0x01010101u, (uint32_t)totSS);
        }
    }
    return nw;
}

// q-state Potts (reading D26), q <= 8, byte-parallel over the 4 sites of a lane.  Two words per site as for spin-1
// (ra: sites 0, 1; rb: sites 2, 3; proposal word x / z, acceptance word y / w).
//   proposal  s' = (s + 1 + mulhi32(w0, q-1)) mod q: the four r's packed into bytes, t = s + 1 + r <= 2q - 2 <= 14, and
//             t >= q  <=>  bit 4 of t + (16 - q)  (no byte reaches 32): s' = t - q * that bit
//   counts    "neighbour differs from x" = bit 3 of ((v ^ x) & 7) + 7  (a 3-bit value is non-zero iff adding 7 reaches 8);
//             summed over the 2d neighbours in units of 8 (<= 48 per byte: no carry) for x = s and x = s'
//   index     dn + 2d = (ne_old - ne_new) / 8 + 2d, so the table byte offset 4 (dn + 2d) = (ne_old + 16 d - ne_new) >> 1
//   accept    iff w1 <= t[dn + 2d] (per site: extract, LDS, ISETP, predicated IMAD, as in rule_one)
// Observables (raw sums in units of 8; march_observables converts): totNZ = sum of "final state != 0",
// totNE = sum of "neighbours different from the final state".
template <int DIMS, bool TRACK, int OBS, bool NEV = false>
__device__ __forceinline__ uint32_t rule_potts(uint32_t own, const uint32_t (&nb)[2 * DIMS], uint4 ra, uint4 rb, uint32_t qm1,
                                               uint32_t s_t, uint32_t one, int &totNZ, int &totNE)
{
    constexpr uint32_t M1 = 0x01010101u, M7 = 0x07070707u, M8 = 0x08080808u;
    const uint32_t s = TRACK ? (own & M7) : own;
    const uint32_t r = __umulhi(ra.x, qm1) | (__umulhi(ra.z, qm1) << 8) | (__umulhi(rb.x, qm1) << 16) | (__umulhi(rb.z, qm1) << 24);
    const uint32_t t = s + r + M1;
    const uint32_t ge = ((t + (15u - qm1) * M1) & 0x10101010u) >> 4;      // 16 - q = 15 - (q - 1)
    const uint32_t prop = t - ge * (qm1 + 1u);
    uint32_t ne_old = 0u, ne_new = 0u;
#pragma unroll
    for (int k = 0; k < 2 * DIMS; ++k) {
        ne_old += (lop3<0x28>(nb[k], s, M7) + M7) & M8;
        ne_new += (lop3<0x28>(nb[k], prop, M7) + M7) & M8;
    }
    const uint32_t adr = (ne_old + (uint32_t)(16 * DIMS) * M1 - ne_new) >> 1;
    uint32_t acc = 0u;                                     // 0xFF in the byte of every accepted site
    acc = accept_site<M_POTTS, NEV, 0x000000FFu>(acc, ra.y, s_t, adr & 0xFFu, one);
    acc = accept_site<M_POTTS, NEV, 0x0000FF00u>(acc, ra.w, s_t, __byte_perm(adr, 0u, 0x4441), one);
    acc = accept_site<M_POTTS, NEV, 0x00FF0000u>(acc, rb.y, s_t, __byte_perm(adr, 0u, 0x4442), one);
    acc = accept_site<M_POTTS, NEV, 0xFF000000u>(acc, rb.w, s_t, adr >> 24, one);
    const uint32_t fl = (s ^ prop) & acc;                  // change of the three state bits
    uint32_t nw = own ^ fl;
    if (TRACK) nw |= (fl + M7) & M8;                       // "ever changed" (0x08): the state bits changed
    if (OBS >= 1) {
        const uint32_t sn = s ^ fl;
        totNZ = (int)__dp4a((sn + M7) & M8, M1, (uint32_t)totNZ);
        if (OBS >= 2) totNE = (int)__dp4a(ne_old ^ ((ne_old ^ ne_new) & acc), M1, (uint32_t)totNE);
    }
    return nw;
}

// ------------------------------------------------------------------------------------------
// One thread's march.  Q is the row parity bit q = (march + cross + colour) & 1 of the current step
// when it is known at compile time (0 / 1: the side neighbour is the byte to the left / right), or
// 2 when it has to be read from the register (warps whose lanes mix row parities).
// ------------------------------------------------------------------------------------------
template <int MODEL, int DIMS, bool TRACK, int OBS, bool NEV = false>
struct March {
    const uint4 *pC;        // other colour, word of the current step
    uint4 *pO;              // own colour, word of the current step
    const uint32_t *pE;     // other colour, start of the current compact row (32-bit lanes)
    uint4 P, C;             // other colour at march-1 and march
    uint32_t grp;           // Philox group of lane 0 of the current word
    int m, q;
    int e_hi, e_lo, dyp, dyn, rowstride, m_wrap, mstep;
    long long wrapw;
    int totU, totBN, totS;  // per-thread sums; < 2^31 for every legal lattice (spin-1: sum a', sum a' * sum, sum of sums)
    uint32_t s_t, one;
    uint32_t ne_t32;
    int ne_always;
    bool ne_all4;
    uint32_t potts_qm1;     // M_POTTS: q - 1

    // One step at march position m.  The march runs upwards (rowstride > 0, the tiled family and the even
    // half-sweeps of the resident family) or downwards (rowstride < 0): P is the row the march came
    // from, N the row it goes to; `m_wrap` is the position whose successor wraps around the lattice and
    // `wrapw` the (signed) pointer correction.  UP matters to the North-East rule only (north = y + 1).
    // The update of one word (16 sites) at the current march position, given the other colour's word at the
    // next row (N), the own word (O), the edge lane of the adjacent word (e) and, in 3D, the cross rows.
    template <int Q, bool UP, class PC>
    __device__ __forceinline__ uint4 update_word(const PC &pc, const uint4 N, const uint4 O, const uint32_t e,
                                                 const uint4 Yp, const uint4 Yn, const uint4 BW = make_uint4(0, 0, 0, 0))
    {
        const int qq = Q == 2 ? q : Q;
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
#pragma unroll
            for (int d = 0; d < 4; ++d) {
                uint32_t ns = p[d] + n[d] + c[d] + sd[d];
                if (DIMS == 3) ns += yp[d] + yn[d];
                uint4 r = philox_sweep<true>(grp + d, pc);
                out[d] = rule_half<TRACK, OBS, NEV>(o[d], ns, r, s_t, one, totU, totBN);
            }
        } else if (MODEL == M_EA) {
            // Reading D25: an antiferromagnetic bond turns the neighbour's "up" into "down", so the up-count is
            // sum_k (b_k xor bond bit k), k = 0: x-1, 1: x+1, 2: y-1, 3: y+1, 4: z-1, 5: z+1 (bond byte of the site
            // being updated).  In the own row the word C holds x+1 (q = 0) or x-1 (q = 1), the shifted word sd the
            // other one; the march axis is y in 2D and z in 3D.  (a ^ b) & 0x01 also drops the flag bits.
            const uint32_t bw[4] = {BW.x, BW.y, BW.z, BW.w};
#pragma unroll
            for (int d = 0; d < 4; ++d) {
                const uint32_t xm = qq ? c[d] : sd[d], xp = qq ? sd[d] : c[d];
                const uint32_t m1 = 0x01010101u;
                uint32_t ns = lop3<0x28>(xm, bw[d], m1) + lop3<0x28>(xp, bw[d] >> 1, m1);
                if (DIMS == 3) {
                    ns += lop3<0x28>(yp[d], bw[d] >> 2, m1) + lop3<0x28>(yn[d], bw[d] >> 3, m1);
                    ns += lop3<0x28>(p[d], bw[d] >> 4, m1) + lop3<0x28>(n[d], bw[d] >> 5, m1);
                } else {
                    ns += lop3<0x28>(p[d], bw[d] >> 2, m1) + lop3<0x28>(n[d], bw[d] >> 3, m1);
                }
                uint4 r = philox_sweep(grp + d, pc);
                out[d] = rule_half<TRACK, OBS, NEV>(o[d], ns, r, s_t, one, totU, totBN);
                if (OBS >= 2) totS = (int)__dp4a(ns, m1, (uint32_t)totS);
            }
        } else if (MODEL == M_ISING_ONE) {
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
                out[d] = rule_one<DIMS, TRACK, OBS, NEV>(o[d], ns, ra, rb, s_t, one, totU, totBN, totS);
            }
        } else if (MODEL == M_POTTS) {
#pragma unroll
            for (int d = 0; d < 4; ++d) {
                uint4 ra = philox_sweep(2u * (grp + d), pc);
                uint4 rb = philox_sweep(2u * (grp + d) + 1u, pc);
                if constexpr (DIMS == 3) {
                    const uint32_t nb[6] = {p[d], n[d], c[d], sd[d], yp[d], yn[d]};
                    out[d] = rule_potts<3, TRACK, OBS, NEV>(o[d], nb, ra, rb, potts_qm1, s_t, one, totU, totBN);
                } else {
                    const uint32_t nb[4] = {p[d], n[d], c[d], sd[d]};
                    out[d] = rule_potts<2, TRACK, OBS, NEV>(o[d], nb, ra, rb, potts_qm1, s_t, one, totU, totBN);
                }
            }
        } else {
            uint32_t accU = 0;
            // Random words are needed by facilitated sites only (c^2 of them).  Two forms, chosen per launch by the
            // up-concentration c (warp-uniform flag):
            //  dense (c >= LSM_NE_ALL4_C): nearly every warp has a facilitated site in each of the four lanes, so one
            //    divergent region per WORD runs the four Philox calls together (instruction-level parallelism);
            //  sparse: every thread walks the list of ITS lanes that hold a facilitated site, one Philox call per
            //    iteration; the warp iterates max-over-threads times -- 1.3 times on average at c = 0.1 and 2.3 at
            //    c = 0.2, where a region per lane (any of 32 threads needs it: 73 % / 99 %) would run 2.9 / 4.
            uint32_t fac[4], lt[4] = {0u, 0u, 0u, 0u};
#pragma unroll
            for (int d = 0; d < 4; ++d) fac[d] = (UP ? n[d] : p[d]) & (qq ? sd[d] : c[d]) & 0x01010101u;
            auto draw = [&](const uint32_t group) {
                const uint4 r = philox_sweep(group, pc);
                uint32_t l = ne_always ? 0x01010101u : 0u;
                if (r.x < ne_t32) l |= 0x00000001u;
                if (r.y < ne_t32) l |= 0x00000100u;
                if (r.z < ne_t32) l |= 0x00010000u;
                if (r.w < ne_t32) l |= 0x01000000u;
                return l;
            };
            if (ne_all4) {
                if ((fac[0] | fac[1] | fac[2] | fac[3]) != 0u) {
#pragma unroll
                    for (int d = 0; d < 4; ++d) lt[d] = draw(grp + d);
                }
            } else {
                uint32_t rem = (fac[0] != 0u ? 1u : 0u) | (fac[1] != 0u ? 2u : 0u) | (fac[2] != 0u ? 4u : 0u) | (fac[3] != 0u ? 8u : 0u);
                while (rem != 0u) {
                    const uint32_t d = (uint32_t)__ffs((int)rem) - 1u;
                    rem &= rem - 1u;
                    const uint32_t l = draw(grp + d);
                    lt[0] = d == 0u ? l : lt[0];
                    lt[1] = d == 1u ? l : lt[1];
                    lt[2] = d == 2u ? l : lt[2];
                    lt[3] = d == 3u ? l : lt[3];
                }
            }
#pragma unroll
            for (int d = 0; d < 4; ++d) {
                const uint32_t nv = TRACK ? (o[d] & 0x01010101u) : o[d];
                uint32_t n2;
                if (MODEL == M_NE_METROPOLIS) n2 = nv ^ (fac[d] & (nv | lt[d]));
                else n2 = (nv & ~fac[d]) | (lt[d] & fac[d]);
                if (OBS >= 1) accU += n2;
                out[d] = TRACK ? ((o[d] & ~0x01010101u) | n2 | ((nv ^ n2) << 3)) : n2;
            }
            if (OBS >= 1) totU += bytesum(accU);
        }
        return make_uint4(out[0], out[1], out[2], out[3]);
    }

    // One step at march position m.  The march runs upwards (rowstride > 0, the tiled family and the even
    // half-sweeps of the resident family) or downwards (rowstride < 0): P is the row the march came
    // from, N the row it goes to; `m_wrap` is the position whose successor wraps around the lattice and
    // `wrapw` the (signed) pointer correction.  UP matters to the North-East rule only (north = y + 1).
    template <int Q, bool UP, class PC>
    __device__ __forceinline__ void step(const PC &pc)
    {
        const int qq = Q == 2 ? q : Q;
        const uint4 *pN = pC + rowstride;
        if (m == m_wrap) pN -= wrapw;
        const uint4 N = *pN;
        const uint4 O = *pO;
        const uint32_t e = pE[qq ? e_hi : e_lo];
        uint4 Yp = make_uint4(0, 0, 0, 0), Yn = Yp;
        if (DIMS == 3) {
            Yp = pC[dyp];
            Yn = pC[dyn];
        }
        uint4 BW = make_uint4(0, 0, 0, 0);
        if (MODEL == M_EA) {
            BW = *pB;
            pB += rowstride;
        }
        *pO = update_word<Q, UP>(pc, N, O, e, Yp, Yn, BW);
        P = C;
        C = N;
        pC += rowstride;
        pO += rowstride;
        pE += rowstride * 4;
        grp += (uint32_t)rowstride * 4u;
        m += mstep;
        if (Q == 2) q ^= 1;
    }

    // ---- asynchronous-copy variant of the step (tiled family) --------------------------------------
    // The words a step needs from global memory (N, O, e and the 3D cross rows) are copied one step ahead
    // into a two-stage, per-thread shared-memory ring with cp.async: the copy costs no registers and its
    // L2/HBM latency is hidden behind a whole step of arithmetic.  A thread reads back only what it copied
    // itself, so cp.async.wait_group is the only synchronisation.  Addresses are 32-bit word offsets
    // into the colour arrays (one IMAD.WIDE per address) instead of 64-bit pointer arithmetic.
    const uint8_t *b_oth;   // array bases
    uint8_t *b_own;
    const uint8_t *b_bnd;   // M_EA: bond bytes of the own colour
    const uint4 *pB;        // ... word of the current step (direct-load path)
    uint32_t offN;          // word offset of the other colour's row the NEXT step will use as N... see step_pf
    uint32_t offS;          // word offset of the own word of the current step
    uint32_t nw32;          // words per colour array
    int rs32, wrapfix;      // signed words per march step; correction applied when offN leaves [0, nw32)
    int ed_hi, ed_lo;       // byte offset from the other colour's word of this thread to the edge lane (q = 1 / 0)
    int dypb, dynb;         // byte offsets to the cross-row words (3D)
    uint32_t s_ring;        // shared address of this thread's slot in stage 0 of the N ring
    uint32_t s_ringE;       // ... of the e ring

    static constexpr uint32_t RING_STAGE = 256u * 16u;              // bytes per stage of a 16-byte ring
    static constexpr uint32_t RING_O = 2u * RING_STAGE;             // own-colour ring behind the N ring
    static constexpr uint32_t RING_YP = 4u * RING_STAGE, RING_YN = 6u * RING_STAGE;
    static constexpr uint32_t RING_BW = (DIMS == 3 ? 8u : 4u) * RING_STAGE;      // M_EA: bond words behind the others
    static constexpr uint32_t RINGE_STAGE = 256u * 4u;

    __device__ __forceinline__ static void cp16(uint32_t dst, const void *src)
    {
        asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
    }
    __device__ __forceinline__ static void cp4(uint32_t dst, const void *src)
    {
        asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(dst), "l"(src) : "memory");
    }
    __device__ __forceinline__ static uint4 lds128(uint32_t a)
    {
        uint4 v;
        asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(a) : "memory");
        return v;
    }
    __device__ __forceinline__ static uint32_t lds32v(uint32_t a)
    {
        uint32_t v;
        asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(a) : "memory");
        return v;
    }

    // Copies for the step whose current row is at word offset `cur` (own word, edge lane, cross rows) and whose
    // next row is at `nxt`, into ring stage ST; QN = row parity of that step.
    template <int QN, int ST>
    __device__ __forceinline__ void prefetch(uint32_t cur, uint32_t nxt)
    {
        const uint8_t *aC = b_oth + (size_t)cur * 16u;
        cp16(s_ring + ST * RING_STAGE, b_oth + (size_t)nxt * 16u);
        cp16(s_ring + RING_O + ST * RING_STAGE, b_own + (size_t)cur * 16u);
        const int qn = QN == 2 ? (q ^ 1) : QN;
        cp4(s_ringE + ST * RINGE_STAGE, aC + (qn ? ed_hi : ed_lo));
        if (DIMS == 3) {
            cp16(s_ring + RING_YP + ST * RING_STAGE, aC + dypb);
            cp16(s_ring + RING_YN + ST * RING_STAGE, aC + dynb);
        }
        if (MODEL == M_EA) cp16(s_ring + RING_BW + ST * RING_STAGE, b_bnd + (size_t)cur * 16u);
        asm volatile("cp.async.commit_group;" ::: "memory");
    }

    __device__ __forceinline__ uint32_t advance(uint32_t off) const
    {
        off += (uint32_t)rs32;
        if (off >= nw32) off += (uint32_t)wrapfix;    // unsigned compare: catches both directions
        return off;
    }

    // Step with ring stage ST holding this step's words; issues the copies of the next step into ST ^ 1.
    template <int Q, int ST, bool UP, class PC>
    __device__ __forceinline__ void step_pf(const PC &pc)
    {
        constexpr int QN = Q == 2 ? 2 : 1 - Q;
        const uint32_t cur = offN;                    // next step's current row = this step's N row
        offN = advance(cur);
        prefetch<QN, ST ^ 1>(cur, offN);
        asm volatile("cp.async.wait_group 1;" ::: "memory");
        const uint4 N = lds128(s_ring + ST * RING_STAGE);
        const uint4 O = lds128(s_ring + RING_O + ST * RING_STAGE);
        const uint32_t e = lds32v(s_ringE + ST * RINGE_STAGE);
        uint4 Yp = make_uint4(0, 0, 0, 0), Yn = Yp;
        if (DIMS == 3) {
            Yp = lds128(s_ring + RING_YP + ST * RING_STAGE);
            Yn = lds128(s_ring + RING_YN + ST * RING_STAGE);
        }
        uint4 BW = make_uint4(0, 0, 0, 0);
        if (MODEL == M_EA) BW = lds128(s_ring + RING_BW + ST * RING_STAGE);
        const uint4 out = update_word<Q, UP>(pc, N, O, e, Yp, Yn, BW);
        *reinterpret_cast<uint4 *>(b_own + (size_t)offS * 16u) = out;
        P = C;
        C = N;
        offS += (uint32_t)rs32;
        grp += (uint32_t)rs32 * 4u;
        if (Q == 2) q ^= 1;
    }

    template <int Q0, bool UP, class PC>
    __device__ __forceinline__ void run_pf(int n, const PC &pc)
    {
        constexpr int Q1 = Q0 == 2 ? 2 : 1 - Q0;
        // copies of the first step into stage 0
        {
            const uint32_t cur = offS;
            offN = advance(cur);
            if (Q0 == 2) q ^= 1;                      // prefetch<> takes the parity of the step AFTER q's
            prefetch<Q0, 0>(cur, offN);
            if (Q0 == 2) q ^= 1;
        }
        int k = 0;
        for (; k + 1 < n; k += 2) {
            step_pf<Q0, 0, UP>(pc);
            step_pf<Q1, 1, UP>(pc);
        }
        if (k < n) step_pf<Q0, 0, UP>(pc);
        asm volatile("cp.async.wait_group 0;" ::: "memory");
    }

    // n steps from the current position, 2x unrolled so that the row parity is a compile-time constant.
    template <int Q0, bool UP, class PC>
    __device__ __forceinline__ void run(int n, const PC &pc)
    {
        constexpr int Q1 = Q0 == 2 ? 2 : 1 - Q0;
        int k = 0;
        for (; k + 1 < n; k += 2) {
            step<Q0, UP>(pc);
            step<Q1, UP>(pc);
        }
        if (k < n) step<Q0, UP>(pc);
    }

    // One step per loop iteration, row parity read from the register (Q = 2).  For rules whose 2x-unrolled loop does not
    // fit the instruction cache (spin-1: 16 KB of code per two steps, `no_instruction` stalls 0.55 per issue).
    template <bool UP, class PC>
    __device__ __forceinline__ void run1(int n, const PC &pc)
    {
#pragma unroll 1
        for (int k = 0; k < n; ++k) step<2, UP>(pc);
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

// Geometry of one thread's march: segment `seg` of the march axis, word column `col`, colour `half`
// being updated (own) against the other colour (oth), upwards from the segment's first row or
// downwards from its last.  Returns the number of steps (rows) of the segment.
template <int MODEL, int DIMS, bool TRACK, int OBS, bool NEV>
__device__ __forceinline__ int march_init(March<MODEL, DIMS, TRACK, OBS, NEV> &M, const TiledGeom &g, uint8_t *own,
                                          const uint8_t *oth, int half, int seg, int col, bool up)
{
    int y, j;
    column_of(g, col, y, j);
    const int m0 = (int)(((long long)g.L * seg) / g.S);
    const int m1 = (int)(((long long)g.L * (seg + 1)) / g.S);
    const int yu = (y + 1 == g.R) ? 0 : y + 1, yd = (y == 0) ? g.R - 1 : y - 1;
    M.e_hi = ((j + 1 == g.wpr) ? 0 : j + 1) * 4;               // first lane of the next word
    M.e_lo = ((j == 0) ? g.wpr - 1 : j - 1) * 4 + 3;           // last lane of the previous word
    const int rs = g.R * g.wpr;                                // words per march step
    const long long nw = (long long)g.L * rs;                  // words per colour array
    M.dyp = (yd - y) * g.wpr;                                  // cross-row neighbours (3D), in words
    M.dyn = (yu - y) * g.wpr;
    const int ms = up ? m0 : m1 - 1;                           // first row of the march
    M.rowstride = up ? rs : -rs;
    M.wrapw = up ? nw : -nw;
    M.m_wrap = up ? g.L - 1 : 0;
    M.mstep = up ? 1 : -1;
    const long long w0 = (long long)ms * rs + y * g.wpr + j;
    M.pC = reinterpret_cast<const uint4 *>(oth) + w0;
    M.pO = reinterpret_cast<uint4 *>(own) + w0;
    M.pE = reinterpret_cast<const uint32_t *>(oth) + ((long long)ms * rs + y * g.wpr) * 4;
    M.grp = (uint32_t)w0 * 4u;
    M.b_oth = oth;
    M.b_own = own;
    M.b_bnd = g.bnd;
    M.pB = reinterpret_cast<const uint4 *>(g.bnd) + w0;
    M.offS = (uint32_t)w0;
    M.offN = (uint32_t)w0;
    M.nw32 = (uint32_t)nw;
    M.rs32 = M.rowstride;
    M.wrapfix = up ? -(int)nw : (int)nw;
    M.ed_hi = (M.e_hi - j * 4) * 4;
    M.ed_lo = (M.e_lo - j * 4) * 4;
    M.dypb = M.dyp * 16;
    M.dynb = M.dyn * 16;
    M.m = ms;
    M.q = (ms + y + half) & 1;
    // the row the march comes from
    const uint4 *pP = M.pC - M.rowstride;
    if (up ? ms == 0 : ms == g.L - 1) pP += M.wrapw;
    M.P = *pP;
    M.C = *M.pC;
    return m1 - m0;
}

// Per-thread sums -> the thread's contribution to (B, M) of SURVEY.md 8(a) a6.  `second` = this half-sweep
// updated the second colour of its sweep.
// Spin-1/2: s = 2b-1, nn = 2n-2d (n = up neighbours), and every bond joins the two colours, so
//   B = sum_{i in colour 1} s'_i nn_i = 4 sum b'n - 2 sum n - 4d U1 + dN   with   sum_{colour 1} n = 2d U0
// (each up site of colour 0 is a neighbour of 2d colour-1 sites).  Hence the first colour contributes
// -4d U0 and the second 4 sum b'n - 4d U1 + 2d nsites; no separate sum of n is needed.
template <int MODEL, int DIMS, bool TRACK, int OBS, bool NEV>
__device__ __forceinline__ void march_observables(const March<MODEL, DIMS, TRACK, OBS, NEV> &M, int nsites, bool second,
                                                  long long &cB, long long &cM)
{
    cB = 0;
    cM = 0;
    if (MODEL == M_ISING_HALF) {
        cM = 2LL * M.totU - nsites;
        cB = -4LL * DIMS * M.totU;
        if (second) cB += 4LL * M.totBN + 2LL * DIMS * nsites;
    } else if (MODEL == M_EA) {
        // s' = 2b' - 1, nn_eff = 2n - 2d with n the bond-weighted up-count: the sum of n over a colour is no longer
        // 2d * (ups of the other colour), so it is accumulated (totS):  B = 4 sum b'n - 2 sum n - 4d U + 2d nsites
        cM = 2LL * M.totU - nsites;
        if (second) cB = 4LL * M.totBN - 2LL * M.totS - 4LL * DIMS * M.totU + 2LL * DIMS * nsites;
    } else if (MODEL == M_ISING_ONE) {
        // s' = a' - 1, nn = sum - 2d:  M = SA - n;  B = sum s' nn = SAS - 2d SA - SS + 2d n   (second colour only)
        cM = (long long)M.totU - nsites;
        if (second) cB = (long long)M.totBN - 2LL * DIMS * M.totU - M.totS + 2LL * DIMS * nsites;
    } else if (MODEL == M_POTTS) {
        // M = sites in state 0 = n - (non-zero sites); B = sum over the second colour of the neighbours equal to the final
        // state = 2d n - (neighbours that differ); both raw sums are in units of 8
        cM = (long long)nsites - M.totU / 8;
        if (second) cB = 2LL * DIMS * nsites - M.totBN / 8;
    } else {
        cM = M.totU;
    }
}

}  // namespace lsmk
