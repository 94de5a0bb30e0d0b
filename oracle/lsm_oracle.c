/*
 * lsm_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, single-threaded CPU statement of the sublattice-parallel
 * ("checkerboard") single-spin-flip Monte Carlo sweep of Levy, Cohen and
 * Rabani, "Simulating lattice spin models on GPUs" (arXiv:1209.0296), written
 * from the paper and the readings D1-D16 of SURVEY.md section 8(c)
 * (restated in DESIGN.md).  It exists only so that tests/, bench.py's
 * cpu_baseline / --impl reference leg and __graft_entry__.smoke() can check
 * and time the CUDA path against it.  Nothing under paper_1209_0296_b200/
 * may include, link, import or call this file, and this file includes
 * nothing from there: own Philox, own threshold builder, own neighbour code.
 *
 * Parity pins (tests/test_oracle_*.py, all CPU-only):
 *   philox4x32_10 ........ Random123 known-answer vectors (tests/golden/)
 *   thresholds ........... closed-form exp(-dE/T)*2^32 values, exact 4x4
 *                          reversibility of the half-sweep kernel (P4)
 *   Ising spin-1/2 2D .... 4x4 brute force over 2^16 states (P3), exact
 *                          probability-vector transient (P15), Onsager (P5)
 *   Ising spin-1/2 3D .... high-temperature series (P6), geometry pins (P10)
 *   spin-1 ............... free-spin closed forms (P7), 4x4 brute force over
 *                          3^16 states (P8)
 *   NE ................... product measure (P11), first-sweep persistence
 *                          closed form (P12), frozen-set bound (P13)
 *   NE random tiles ...... (orc_sweep_random_tile, and its
 *                          balance-preserving variant)
 *                          dict-keyed Python restatement with its own Philox on
 *                          collision-heavy tiles, tile-order independence,
 *                          product measure, closed-form first-sweep persistence,
 *                          frozen-set bound, serial limit Q = lambda = 1
 *                          (tests/test_oracle_random_tile.py)
 *   EA +/-J bonds ........ (model ORC_EA, reading D25) Mattis gauge: bonds tau_i tau_j reproduce the
 *                          ferromagnet bit for bit; all-ferro bonds = the Ising rule; dict restatement incl. the
 *                          bond stream; 4x4 brute force over 2^16 states with a fixed random bond set
 *   Potts ................ (model ORC_POTTS, reading D26) dict restatement; q = 2 table = Ising at J/2;
 *                          4x4 brute force over 3^16 states (q = 3) and 2^16 (q = 2); J = 0 and T -> 0 closed forms
 *                          (tests/test_oracle_wider_models.py)
 *   "parity unpinned": none of the functions; the unpinned items are
 *   particular non-equilibrium VALUES, not code paths.
 *
 * Conventions (PAPER.md line refs are to /root/reference/PAPER.md):
 *   - lattice: periodic hypercubic, d = 2 or 3, linear size L (even, >= 4),
 *     canonical site id i = x + L*(y + L*z), parity (x+y+z)&1.
 *   - one sweep = half-sweep over parity 0, then over parity 1
 *     (the two kernel launches red/blue then green/white;
 *     reading D9: the parity that contains the origin goes first).
 *   - Metropolis acceptance P = min[1, exp(-dH/T)] realised as
 *     an integer compare of a 32-bit random word with a 33-bit threshold
 *     floor(P * 2^32) (reading D3).
 *   - Ising: H = -J sum_<ij> s_i s_j - h sum_i s_i (reading D1).
 *   - North-East model: a site can change only if its north (x, y+1) and east
 *     (x+1, y) neighbours are both up (reading D8); J = 0,
 *     occupation n in {0,1}, H = sum n_i, c = 1/(1+exp(1/T)) (reading D6).
 *   - random words: Philox4x32-10 keyed on (seed; site group, sweep, half)
 *     (reading D2).
 *   - Edwards-Anderson +/-J model (Eq. 1 with discrete J_ij; reading D25): spin-1/2,
 *     H = -J sum_<ij> tau_ij s_i s_j - h sum s_i, tau_ij = +/-1 per bond, drawn from the seed (stream tag 3) or
 *     set by the caller; same Metropolis rule and table as the Ising model with nn = sum_j tau_ij s_j.
 *   - q-state Potts model (reading D26): sigma in {0..q-1}, q = two_S + 1, H = -J sum_<ij>
 *     delta(sigma_i, sigma_j); trial state uniform over the other q-1 (word 0 of the site), Metropolis with word 1.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

enum { ORC_ISING = 0, ORC_NE_HEATBATH = 1, ORC_NE_METROPOLIS = 2, ORC_EA = 3, ORC_POTTS = 4 };

typedef struct orc {
    int dims, L, two_S, model;
    double J, h, T;
    uint64_t seed;
    int64_t N;
    int8_t *s;        /* current values, canonical order                   */
    int8_t *s0;       /* snapshot at the reference time                     */
    uint8_t *changed; /* 1 if the value differed from its predecessor ever  */
    uint64_t t;       /* sweeps done = Philox sweep field of the next sweep */
    uint64_t thr[128];
    int nthr;
    double c;         /* NE up-concentration recomputed from T             */
    int8_t *tau;      /* ORC_EA: bond signs, tau[a*N + i] = sign of the bond
                         between site i and its neighbour in direction +a   */
    int q;            /* ORC_POTTS: number of states (= two_S + 1)          */
} orc_t;

/* ---------------------------------------------------------------- Philox -- */
/* Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11), reading D2.
 * One round: (c0,c1,c2,c3) <- (hi(M1*c2)^c1^k0, lo(M1*c2), hi(M0*c0)^c3^k1, lo(M0*c0));
 * between rounds k0 += 0x9E3779B9, k1 += 0xBB67AE85.                          */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int r = 0; r < 10; ++r) {
        uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* Random words of one site (reading D2 detail).
 * stream: 0 = half-sweep of parity 0, 1 = parity 1, 2 = initial state.
 * group g and sweep t fill the 128-bit counter as
 *   c0 = lo32(g), c1 = hi32(g), c2 = lo32(t), c3 = stream | (hi32(t) << 4):
 * the low four bits of c3 belong to the stream tag alone (tags 0..15; t < 2^60),
 * so no two (tag, t) pairs share a counter (reading D2). */
static void words_of_group(uint64_t seed, uint64_t g, uint64_t t, uint32_t stream,
                           uint32_t out[4])
{
    uint32_t ctr[4], key[2];
    ctr[0] = (uint32_t)g;
    ctr[1] = (uint32_t)(g >> 32);
    ctr[2] = (uint32_t)t;
    ctr[3] = stream | ((uint32_t)(t >> 32) << 4);
    key[0] = (uint32_t)seed;
    key[1] = (uint32_t)(seed >> 32);
    orc_philox4x32_10(ctr, key, out);
}

/* ------------------------------------------------------------ thresholds -- */
static uint64_t thr_of_probability(double p)
{
    if (p >= 1.0) return (uint64_t)1 << 32;
    return (uint64_t)floor(ldexp(p, 32));
}

/* Reading D3: x = J*nn + h; dE = -(s'-s)*x; p = exp(-dE/T);
 * thr = 2^32 if dE <= 0 or p >= 1, else floor(p*2^32).                      */
static uint64_t thr_metropolis(double J, double h, double T, int s_old, int s_new, int nn)
{
    double x = J * (double)nn + h;
    double dE = -(double)(s_new - s_old) * x;
    if (dE <= 0.0) return (uint64_t)1 << 32;
    double p = exp(-dE / T);
    return thr_of_probability(p);
}

/* spin-1 proposal (reading D5): index a = s+1, kk in {0,1};
 * proposed index (a + 1 + kk) mod 3, i.e. uniform over the other two values. */
static int spin1_proposal(int a, int kk) { return (a + 1 + kk) % 3; }

/* Table layouts (the order lsm_get_thresholds must reproduce):
 *  Ising two_S=1: idx = b*(2d+1) + (nn+2d)/2, b = (s+1)/2          -> 2(2d+1)
 *  Ising two_S=2: idx = (a*2 + kk)*(4d+1) + (nn+2d), a = s+1        -> 6(4d+1)
 *  EA: as Ising two_S=1 with nn = sum_j tau_ij s_j (reading D25)     -> 2(2d+1)
 *  Potts: idx = (n_new - n_old) + 2d                                -> 4d+1
 *  NE (either rule): [0] = floor(c*2^32) (initial state and heat bath),
 *                    [1] = floor(exp(-1/T)*2^32) (Metropolis 0->1),
 *                    [2] = 2^32 (Metropolis 1->0, dE < 0)            -> 3    */
static void build_thresholds(orc_t *o)
{
    int d = o->dims;
    o->nthr = 0;
    if (o->model == ORC_POTTS) {
        /* reading D26: dE = -J * (n_new - n_old), idx = (n_new - n_old) + 2d */
        for (int j = 0; j <= 4 * d; ++j) {
            double x = o->J * (double)(j - 2 * d);
            double dE = -x;
            o->thr[o->nthr++] = (dE <= 0.0) ? ((uint64_t)1 << 32) : thr_of_probability(exp(-dE / o->T));
        }
    } else if ((o->model == ORC_ISING && o->two_S == 1) || o->model == ORC_EA) {
        /* ORC_EA (reading D25): the same table, indexed by the bond-weighted neighbour sum */
        for (int b = 0; b < 2; ++b)
            for (int j = 0; j <= 2 * d; ++j) {
                int s = 2 * b - 1, nn = 2 * j - 2 * d;
                o->thr[o->nthr++] = thr_metropolis(o->J, o->h, o->T, s, -s, nn);
            }
    } else if (o->model == ORC_ISING && o->two_S == 2) {
        for (int a = 0; a < 3; ++a)
            for (int kk = 0; kk < 2; ++kk)
                for (int j = 0; j <= 4 * d; ++j) {
                    int s = a - 1, sp = spin1_proposal(a, kk) - 1, nn = j - 2 * d;
                    o->thr[o->nthr++] = thr_metropolis(o->J, o->h, o->T, s, sp, nn);
                }
    } else {
        o->c = 1.0 / (1.0 + exp(1.0 / o->T));           /* reading D6 */
        o->thr[0] = thr_of_probability(o->c);
        o->thr[1] = thr_of_probability(exp(-1.0 / o->T));
        o->thr[2] = (uint64_t)1 << 32;
        o->nthr = 3;
    }
}

/* -------------------------------------------------------------- geometry -- */
static int64_t site_id(const orc_t *o, int x, int y, int z)
{
    return (int64_t)x + (int64_t)o->L * ((int64_t)y + (int64_t)o->L * (int64_t)z);
}
static int wrap(int a, int L) { return (a % L + L) % L; }

static int value_at(const orc_t *o, int x, int y, int z)
{
    int L = o->L;
    return o->s[site_id(o, wrap(x, L), wrap(y, L), o->dims == 3 ? wrap(z, L) : 0)];
}

static int neighbour_sum(const orc_t *o, int x, int y, int z)
{
    int nn = value_at(o, x - 1, y, z) + value_at(o, x + 1, y, z)
           + value_at(o, x, y - 1, z) + value_at(o, x, y + 1, z);
    if (o->dims == 3) nn += value_at(o, x, y, z - 1) + value_at(o, x, y, z + 1);
    return nn;
}

/* ORC_EA (reading D25): sum_j tau_ij s_j over the 2d neighbours.  The bond between i and i+a is stored at i,
 * the bond between i and i-a at the neighbour i-a.                                                          */
static int bond_sign(const orc_t *o, int a, int x, int y, int z)
{
    int L = o->L;
    return o->tau[(int64_t)a * o->N + site_id(o, wrap(x, L), wrap(y, L), o->dims == 3 ? wrap(z, L) : 0)];
}
static int neighbour_sum_bonds(const orc_t *o, int x, int y, int z)
{
    int nn = bond_sign(o, 0, x, y, z) * value_at(o, x + 1, y, z) + bond_sign(o, 0, x - 1, y, z) * value_at(o, x - 1, y, z)
           + bond_sign(o, 1, x, y, z) * value_at(o, x, y + 1, z) + bond_sign(o, 1, x, y - 1, z) * value_at(o, x, y - 1, z);
    if (o->dims == 3)
        nn += bond_sign(o, 2, x, y, z) * value_at(o, x, y, z + 1) + bond_sign(o, 2, x, y, z - 1) * value_at(o, x, y, z - 1);
    return nn;
}
/* ORC_POTTS: number of the 2d neighbours in state v. */
static int neighbours_equal_to(const orc_t *o, int x, int y, int z, int v)
{
    int n = (value_at(o, x - 1, y, z) == v) + (value_at(o, x + 1, y, z) == v)
          + (value_at(o, x, y - 1, z) == v) + (value_at(o, x, y + 1, z) == v);
    if (o->dims == 3) n += (value_at(o, x, y, z - 1) == v) + (value_at(o, x, y, z + 1) == v);
    return n;
}

/* ------------------------------------------------------------ initial state */
/* Reading D4: stream 2, t = 0, group = i>>2 over the canonical id, word i&3. */
static void init_from_seed(orc_t *o)
{
    for (int64_t i = 0; i < o->N; ++i) {
        uint32_t w4[4];
        words_of_group(o->seed, (uint64_t)i >> 2, 0, 2u, w4);
        uint32_t w = w4[i & 3];
        int v;
        if (o->model == ORC_POTTS)   v = (int)(((uint64_t)w * (uint64_t)o->q) >> 32);      /* reading D26 */
        else if (o->model == ORC_EA) v = (w >> 31) ? 1 : -1;
        else if (o->model != ORC_ISING) v = ((uint64_t)w < o->thr[0]) ? 1 : 0;
        else if (o->two_S == 1)    v = (w >> 31) ? 1 : -1;
        else                       v = (int)(((uint64_t)w * 3u) >> 32) - 1;
        o->s[i] = (int8_t)v;
    }
}

/* Reading D25: bond signs from stream tag 3, t = 0: bond id b = a*N + i (a = 0, 1, 2 for +x, +y, +z),
 * group b>>2, word b&3; tau = +1 if the top bit of the word is set, else -1 (the +/-J model with p = 1/2).  */
static void bonds_from_seed(orc_t *o)
{
    for (int64_t b = 0; b < (int64_t)o->dims * o->N; ++b) {
        uint32_t w4[4];
        words_of_group(o->seed, (uint64_t)b >> 2, 0, 3u, w4);
        o->tau[b] = (w4[b & 3] >> 31) ? 1 : -1;
    }
}

void orc_get_bonds(const orc_t *o, int8_t *out) { if (o->tau) memcpy(out, o->tau, (size_t)o->dims * (size_t)o->N); }
int orc_set_bonds(orc_t *o, const int8_t *in)
{
    if (!o->tau) return -1;
    memcpy(o->tau, in, (size_t)o->dims * (size_t)o->N);
    return 0;
}

void orc_reset_reference(orc_t *o)
{
    memcpy(o->s0, o->s, (size_t)o->N);
    memset(o->changed, 0, (size_t)o->N);
}

/* ------------------------------------------------------------- life cycle -- */
orc_t *orc_create(int dims, int L, int two_S, int model, double J, double h, double T,
                  uint64_t seed)
{
    if (dims != 2 && dims != 3) return NULL;
    if (L < 4 || (L & 1)) return NULL;                     /* reading D10 */
    if (!(T > 0.0) || !isfinite(T)) return NULL;
    if (model == ORC_ISING) { if (two_S != 1 && two_S != 2) return NULL; }
    else if (model == ORC_NE_HEATBATH || model == ORC_NE_METROPOLIS) {
        if (dims != 2 || J != 0.0 || two_S != 1) return NULL;
    } else if (model == ORC_EA) { if (two_S != 1) return NULL; }
    else if (model == ORC_POTTS) { if (two_S < 1 || two_S > 15 || h != 0.0) return NULL; }   /* q = two_S + 1 in [2, 16] */
    else return NULL;
    orc_t *o = (orc_t *)calloc(1, sizeof(orc_t));
    if (!o) return NULL;
    o->dims = dims; o->L = L; o->two_S = two_S; o->model = model;
    o->J = J; o->h = h; o->T = T; o->seed = seed;
    o->N = (dims == 2) ? (int64_t)L * L : (int64_t)L * L * L;
    o->s = (int8_t *)malloc((size_t)o->N);
    o->s0 = (int8_t *)malloc((size_t)o->N);
    o->changed = (uint8_t *)malloc((size_t)o->N);
    if (!o->s || !o->s0 || !o->changed) { free(o->s); free(o->s0); free(o->changed); free(o); return NULL; }
    o->q = two_S + 1;
    o->tau = NULL;
    if (model == ORC_EA) {
        o->tau = (int8_t *)malloc((size_t)dims * (size_t)o->N);
        if (!o->tau) { free(o->s); free(o->s0); free(o->changed); free(o); return NULL; }
        bonds_from_seed(o);
    }
    o->t = 0;
    build_thresholds(o);
    init_from_seed(o);
    orc_reset_reference(o);
    return o;
}

void orc_destroy(orc_t *o)
{
    if (!o) return;
    free(o->s); free(o->s0); free(o->changed); free(o->tau); free(o);
}

int orc_set_temperature(orc_t *o, double T)
{
    if (!(T > 0.0) || !isfinite(T)) return -1;
    o->T = T;
    build_thresholds(o);
    return 0;
}

int orc_get_thresholds(const orc_t *o, uint64_t *out)
{
    for (int i = 0; i < o->nthr; ++i) out[i] = o->thr[i];
    return o->nthr;
}

void orc_get_spins(const orc_t *o, int8_t *out) { memcpy(out, o->s, (size_t)o->N); }

void orc_set_spins(orc_t *o, const int8_t *in, uint64_t sweep_counter)
{
    memcpy(o->s, in, (size_t)o->N);
    o->t = sweep_counter;
}

uint64_t orc_sweeps_done(const orc_t *o) { return o->t; }
int64_t orc_num_sites(const orc_t *o) { return o->N; }
double orc_concentration(const orc_t *o) { return o->c; }

/* ------------------------------------------------------------ update rules -- */
/* One site of the active parity.  All neighbours have the other parity, so
 * they are untouched during this half-sweep.                 */
static void update_site(orc_t *o, int x, int y, int z, uint32_t half)
{
    int64_t i = site_id(o, x, y, z);
    int64_t k = i >> 1;               /* compact index inside its colour     */
    int s_old = o->s[i], s_new = s_old;
    uint32_t w4[4];

    if (o->model == ORC_ISING && o->two_S == 1) {
        /* one word per site: group k>>2, word k&3 */
        words_of_group(o->seed, (uint64_t)k >> 2, o->t, half, w4);
        uint32_t w = w4[k & 3];
        int nn = neighbour_sum(o, x, y, z);
        int b = (s_old + 1) / 2, j = (nn + 2 * o->dims) / 2;
        uint64_t thr = o->thr[b * (2 * o->dims + 1) + j];
        if ((uint64_t)w < thr) s_new = -s_old;
    } else if (o->model == ORC_EA) {
        /* reading D25: as Ising spin-1/2 with the bond-weighted neighbour sum; one word per site */
        words_of_group(o->seed, (uint64_t)k >> 2, o->t, half, w4);
        uint32_t w = w4[k & 3];
        int nn = neighbour_sum_bonds(o, x, y, z);
        int b = (s_old + 1) / 2, j = (nn + 2 * o->dims) / 2;
        if ((uint64_t)w < o->thr[b * (2 * o->dims + 1) + j]) s_new = -s_old;
    } else if (o->model == ORC_POTTS) {
        /* reading D26: two words per site (group k>>1); w0 proposes one of the other q-1 states uniformly,
         * w1 accepts by Metropolis with dE = -J (n_new - n_old) */
        words_of_group(o->seed, (uint64_t)k >> 1, o->t, half, w4);
        uint32_t w0 = w4[2 * (k & 1)], w1 = w4[2 * (k & 1) + 1];
        int r = (int)(((uint64_t)w0 * (uint64_t)(o->q - 1)) >> 32);
        int prop = (s_old + 1 + r) % o->q;
        int dn = neighbours_equal_to(o, x, y, z, prop) - neighbours_equal_to(o, x, y, z, s_old);
        if ((uint64_t)w1 < o->thr[dn + 2 * o->dims]) s_new = prop;
    } else if (o->model == ORC_ISING) {
        /* two words per site: group k>>1, words 2(k&1) and 2(k&1)+1 */
        words_of_group(o->seed, (uint64_t)k >> 1, o->t, half, w4);
        uint32_t w0 = w4[2 * (k & 1)], w1 = w4[2 * (k & 1) + 1];
        int nn = neighbour_sum(o, x, y, z);
        int a = s_old + 1;
        int kk = (int)(((uint64_t)w0 * 2u) >> 32);
        int ap = spin1_proposal(a, kk);
        uint64_t thr = o->thr[(a * 2 + kk) * (4 * o->dims + 1) + (nn + 2 * o->dims)];
        if ((uint64_t)w1 < thr) s_new = ap - 1;
    } else {
        /* North-East: facilitated iff north and east are both up */
        int north = value_at(o, x, y + 1, 0), east = value_at(o, x + 1, y, 0);
        if (north == 1 && east == 1) {
            words_of_group(o->seed, (uint64_t)k >> 2, o->t, half, w4);
            uint32_t w = w4[k & 3];
            if (o->model == ORC_NE_HEATBATH) {
                s_new = ((uint64_t)w < o->thr[0]) ? 1 : 0;       /* reading D7 */
            } else {
                uint64_t thr = (s_old == 0) ? o->thr[1] : o->thr[2];
                if ((uint64_t)w < thr) s_new = 1 - s_old;
            }
        }
    }
    if (s_new != s_old) o->changed[i] = 1;                   /* reading D12 */
    o->s[i] = (int8_t)s_new;
}

/* descending != 0 visits the sites of each half in the reverse order; the
 * result must not depend on it (pin P9).                                    */
void orc_sweep_ordered(orc_t *o, int64_t n, int descending)
{
    int L = o->L, Lz = (o->dims == 3) ? L : 1;
    for (int64_t it = 0; it < n; ++it) {
        for (uint32_t half = 0; half < 2; ++half) {
            if (!descending) {
                for (int z = 0; z < Lz; ++z)
                    for (int y = 0; y < L; ++y)
                        for (int x = 0; x < L; ++x)
                            if ((uint32_t)((x + y + z) & 1) == half) update_site(o, x, y, z, half);
            } else {
                for (int z = Lz - 1; z >= 0; --z)
                    for (int y = L - 1; y >= 0; --y)
                        for (int x = L - 1; x >= 0; --x)
                            if ((uint32_t)((x + y + z) & 1) == half) update_site(o, x, y, z, half);
            }
        }
        o->t += 1;
    }
}

void orc_sweep(orc_t *o, int64_t n) { orc_sweep_ordered(o, n, 0); }

/* ------------------------------------------- North-East, random-tile schedule -- */
/* The paper's "corrected algorithm" for the North-East model (PAPER.md:128-140,
 * steps 3-10), which it prefers to the checkerboard sweep because random picks
 * keep the relaxation dynamics of the serial code:
 *   3. the lattice is divided into Q sub-lattices ("tiles") of P = b*b spins;
 *   5. every block picks a different tile (Q blocks, Q tiles: each tile is
 *      handled exactly once per launch) and copies it "including its
 *      boundaries" -- only the upper and right ones are needed (Fig. 4);
 *   6. lambda threads concurrently pick lambda spins of the tile at random
 *      and update them;  7. synchronise;  8. repeat q times, q*lambda = P/2;
 *   9. copy the tile back;  10. relaunch and redo 5-8: one lattice sweep.
 * Readings (D17-D21), chosen so that the result is unique:
 *   D17 one sweep = 2 launches; the sweep counter t counts sweeps.
 *   D18 a tile's boundary cells are read from the lattice as it was when the
 *       launch started and never refreshed; only interior cells are written.
 *       Hence the result does not depend on which block takes which tile.
 *   D19 the lambda picks of a sub-step all read the tile as it was when the
 *       sub-step started; writes are applied in thread order, so on a
 *       same-site collision the highest thread index wins.
 *   D20 thread j picks r = floor(w_pos * P / 2^32), (px, py) = (r mod b, r div b);
 *       the update rule is that of reading D7 with acceptance word w_acc.
 *   D21 Philox counter c0 = tile id (tx + (L/b)*ty), c1 = k*ceil(lambda/2) + (j>>1)
 *       for sub-step k and thread j, c2 = lo32(t), c3 = (4 + launch) | hi32(t)<<4;
 *       w_pos = word 2(j&1), w_acc = word 2(j&1)+1.
 * tiles_descending != 0 walks the tiles in reverse order (pin: same result). */
int orc_sweep_random_tile(orc_t *o, int64_t n, int b, int lambda, int tiles_descending)
{
    if (o->model != ORC_NE_HEATBATH && o->model != ORC_NE_METROPOLIS) return -1;
    int L = o->L;
    if (b < 1 || L % b != 0 || lambda < 1) return -1;
    int P = b * b;
    if (P % (2 * lambda) != 0) return -1;
    int q = P / (2 * lambda), nt = L / b, calls = (lambda + 1) / 2;
    int8_t *start = (int8_t *)malloc((size_t)o->N);
    int *site = (int *)malloc(sizeof(int) * (size_t)lambda);
    int *val = (int *)malloc(sizeof(int) * (size_t)lambda);
    if (!start || !site || !val) { free(start); free(site); free(val); return -2; }
    uint32_t key[2] = {(uint32_t)o->seed, (uint32_t)(o->seed >> 32)};
    for (int64_t it = 0; it < n; ++it) {
        for (uint32_t launch = 0; launch < 2; ++launch) {
            memcpy(start, o->s, (size_t)o->N);                 /* D18: the lattice at launch start */
            for (int tt = 0; tt < nt * nt; ++tt) {
                int T = tiles_descending ? nt * nt - 1 - tt : tt;
                int tx = T % nt, ty = T / nt, x0 = tx * b, y0 = ty * b;
                for (int k = 0; k < q; ++k) {
                    for (int j = 0; j < lambda; ++j) {         /* decisions: all read the sub-step's start */
                        uint32_t ctr[4], w[4];
                        ctr[0] = (uint32_t)T;
                        ctr[1] = (uint32_t)(k * calls + (j >> 1));
                        ctr[2] = (uint32_t)o->t;
                        ctr[3] = (4u + launch) | ((uint32_t)(o->t >> 32) << 4);
                        orc_philox4x32_10(ctr, key, w);
                        uint32_t w_pos = w[2 * (j & 1)], w_acc = w[2 * (j & 1) + 1];
                        int r = (int)(((uint64_t)w_pos * (uint64_t)P) >> 32);
                        int px = r % b, py = r / b;
                        int x = x0 + px, y = y0 + py;
                        /* north and east: interior cells from the evolving lattice, boundary cells from `start` */
                        int xn = x, yn = y + 1, xe = x + 1, ye = y;
                        int north = (py + 1 < b) ? o->s[site_id(o, xn, yn, 0)] : start[site_id(o, xn, wrap(yn, L), 0)];
                        int east = (px + 1 < b) ? o->s[site_id(o, xe, ye, 0)] : start[site_id(o, wrap(xe, L), ye, 0)];
                        int64_t i = site_id(o, x, y, 0);
                        int s_old = o->s[i], s_new = s_old;
                        if (north == 1 && east == 1) {
                            if (o->model == ORC_NE_HEATBATH) {
                                s_new = ((uint64_t)w_acc < o->thr[0]) ? 1 : 0;
                            } else {
                                uint64_t thr = (s_old == 0) ? o->thr[1] : o->thr[2];
                                if ((uint64_t)w_acc < thr) s_new = 1 - s_old;
                            }
                        }
                        site[j] = (int)i;
                        val[j] = s_new;
                    }
                    for (int j = 0; j < lambda; ++j) {         /* D19: writes in thread order */
                        int dup = 0;
                        for (int j2 = j + 1; j2 < lambda; ++j2) dup |= (site[j2] == site[j]);
                        if (dup) continue;                     /* a higher thread wrote the same site */
                        if (val[j] != o->s[site[j]]) o->changed[site[j]] = 1;
                        o->s[site[j]] = (int8_t)val[j];
                    }
                }
            }
        }
        o->t += 1;
    }
    free(start); free(site); free(val);
    return 0;
}

/* The balance-preserving variant of the algorithm above: "The only changes are in steps 6-9:
 *   6. lambda threads concurrently pick lambda red spins from the sub-lattice randomly and update them.
 *   7. Synchronize the block and pick lambda white spins from the sub-lattice randomly and update them.
 *   8. Copy back ...  9. Relaunch ... and redo steps 6-8 three more times (this will complete one MC step)."
 * Readings (D22-D24):
 *   D22 red / white = the two checkerboard colours (x+y)&1 = 0 / 1 (Fig. 4 is absent; these are the two sets
 *       whose members never read each other under the north-east rule, which is what restores balance).
 *   D23 one MC step = 4 launches; a launch runs q sub-steps of (lambda red picks, barrier, lambda white picks,
 *       barrier) with q * 2 lambda = P/4, so that the step attempts P updates per tile like the base algorithm
 *       (twice the launches, tile copies and barriers for the same attempts: the paper's "~2.5x slower").
 *   D24 thread j of sub-step k draws ONE Philox call: counter c0 = tile id, c1 = k*lambda + j, c2 = lo32(t),
 *       c3 = (8 + launch) | hi32(t)<<4; words 0, 1 = position and acceptance of its red pick, words 2, 3 of its
 *       white pick.  Position: r = floor(w_pos * (P/2) / 2^32) is the r-th site of that colour in the tile in
 *       row-major order: py = r div (b/2), px = 2 (r mod (b/2)) + ((py + colour) & 1)   (tile origins are even).
 *   D18 (boundaries frozen at launch start), D19 (picks of a phase read the phase's start; highest thread
 *       wins a same-site collision) and the rule of D7 are unchanged.                                        */
int orc_sweep_random_tile_balanced(orc_t *o, int64_t n, int b, int lambda, int tiles_descending)
{
    if (o->model != ORC_NE_HEATBATH && o->model != ORC_NE_METROPOLIS) return -1;
    int L = o->L;
    if (b < 2 || (b & 1) || L % b != 0 || lambda < 1) return -1;
    int P = b * b;
    if (P % (8 * lambda) != 0) return -1;
    int q = P / (8 * lambda), nt = L / b, hb = b / 2;
    int8_t *start = (int8_t *)malloc((size_t)o->N);
    int *site = (int *)malloc(sizeof(int) * (size_t)lambda);
    int *val = (int *)malloc(sizeof(int) * (size_t)lambda);
    if (!start || !site || !val) { free(start); free(site); free(val); return -2; }
    uint32_t key[2] = {(uint32_t)o->seed, (uint32_t)(o->seed >> 32)};
    for (int64_t it = 0; it < n; ++it) {
        for (uint32_t launch = 0; launch < 4; ++launch) {
            memcpy(start, o->s, (size_t)o->N);
            for (int tt = 0; tt < nt * nt; ++tt) {
                int T = tiles_descending ? nt * nt - 1 - tt : tt;
                int tx = T % nt, ty = T / nt, x0 = tx * b, y0 = ty * b;
                for (int k = 0; k < q; ++k) {
                    for (int colour = 0; colour < 2; ++colour) {      /* red picks, barrier, white picks, barrier */
                        for (int j = 0; j < lambda; ++j) {
                            uint32_t ctr[4], w[4];
                            ctr[0] = (uint32_t)T;
                            ctr[1] = (uint32_t)(k * lambda + j);
                            ctr[2] = (uint32_t)o->t;
                            ctr[3] = (8u + launch) | ((uint32_t)(o->t >> 32) << 4);
                            orc_philox4x32_10(ctr, key, w);
                            uint32_t w_pos = w[2 * colour], w_acc = w[2 * colour + 1];
                            int r = (int)(((uint64_t)w_pos * (uint64_t)(P / 2)) >> 32);
                            int py = r / hb, px = 2 * (r % hb) + ((py + colour) & 1);
                            int x = x0 + px, y = y0 + py;
                            int north = (py + 1 < b) ? o->s[site_id(o, x, y + 1, 0)] : start[site_id(o, x, wrap(y + 1, L), 0)];
                            int east = (px + 1 < b) ? o->s[site_id(o, x + 1, y, 0)] : start[site_id(o, wrap(x + 1, L), y, 0)];
                            int64_t i = site_id(o, x, y, 0);
                            int s_old = o->s[i], s_new = s_old;
                            if (north == 1 && east == 1) {
                                if (o->model == ORC_NE_HEATBATH) {
                                    s_new = ((uint64_t)w_acc < o->thr[0]) ? 1 : 0;
                                } else {
                                    uint64_t thr = (s_old == 0) ? o->thr[1] : o->thr[2];
                                    if ((uint64_t)w_acc < thr) s_new = 1 - s_old;
                                }
                            }
                            site[j] = (int)i;
                            val[j] = s_new;
                        }
                        for (int j = 0; j < lambda; ++j) {
                            int dup = 0;
                            for (int j2 = j + 1; j2 < lambda; ++j2) dup |= (site[j2] == site[j]);
                            if (dup) continue;
                            if (val[j] != o->s[site[j]]) o->changed[site[j]] = 1;
                            o->s[site[j]] = (int8_t)val[j];
                        }
                    }
                }
            }
        }
        o->t += 1;
    }
    free(start); free(site); free(val);
    return 0;
}

/* obs[2*k] = B (= 0), obs[2*k+1] = M after sweep k of this call. */
void orc_measure(const orc_t *o, int64_t *B, int64_t *M);
int orc_sweep_random_tile_record(orc_t *o, int64_t n, int b, int lambda, int64_t *obs)
{
    for (int64_t k = 0; k < n; ++k) {
        int rc = orc_sweep_random_tile(o, 1, b, lambda, 0);
        if (rc != 0) return rc;
        orc_measure(o, &obs[2 * k], &obs[2 * k + 1]);
    }
    return 0;
}

/* Same for the balance-preserving variant: obs[2*k] = 0, obs[2*k+1] = M after MC step k of this call. */
int orc_sweep_random_tile_balanced_record(orc_t *o, int64_t n, int b, int lambda, int64_t *obs)
{
    for (int64_t k = 0; k < n; ++k) {
        int rc = orc_sweep_random_tile_balanced(o, 1, b, lambda, 0);
        if (rc != 0) return rc;
        orc_measure(o, &obs[2 * k], &obs[2 * k + 1]);
    }
    return 0;
}

/* ------------------------------------------------------------- observables -- */
/* M = sum s_i; B = sum over bonds of s_i s_j, each bond once (east, north, up).
 * NE (reading D15): M = number of up sites, B = 0.                          */
void orc_measure(const orc_t *o, int64_t *B, int64_t *M)
{
    int L = o->L, Lz = (o->dims == 3) ? L : 1;
    int64_t b = 0, m = 0;
    for (int z = 0; z < Lz; ++z)
        for (int y = 0; y < L; ++y)
            for (int x = 0; x < L; ++x) {
                int s = value_at(o, x, y, z);
                if (o->model == ORC_POTTS) {            /* D26: M = sites in state 0, B = bonds joining equal states */
                    m += (s == 0);
                    b += (value_at(o, x + 1, y, z) == s) + (value_at(o, x, y + 1, z) == s);
                    if (o->dims == 3) b += (value_at(o, x, y, z + 1) == s);
                    continue;
                }
                m += s;
                if (o->model == ORC_EA) {               /* D25: B = sum over bonds of tau_ij s_i s_j */
                    int f = bond_sign(o, 0, x, y, z) * value_at(o, x + 1, y, z) + bond_sign(o, 1, x, y, z) * value_at(o, x, y + 1, z);
                    if (o->dims == 3) f += bond_sign(o, 2, x, y, z) * value_at(o, x, y, z + 1);
                    b += (int64_t)s * f;
                }
                if (o->model == ORC_ISING) {
                    int f = value_at(o, x + 1, y, z) + value_at(o, x, y + 1, z);
                    if (o->dims == 3) f += value_at(o, x, y, z + 1);
                    b += (int64_t)s * f;
                }
            }
    *B = b; *M = m;
}

/* E = -J*B - h*M (Ising); E = M (NE, H = sum n_i). */
double orc_energy(const orc_t *o)
{
    int64_t B, M;
    orc_measure(o, &B, &M);
    if (o->model == ORC_ISING || o->model == ORC_EA) return -o->J * (double)B - o->h * (double)M;
    if (o->model == ORC_POTTS) return -o->J * (double)B;
    return (double)M;
}

/* obs[2*k] = B, obs[2*k+1] = M after sweep k of this call. */
void orc_sweep_record(orc_t *o, int64_t n, int64_t *obs)
{
    for (int64_t k = 0; k < n; ++k) {
        orc_sweep(o, 1);
        orc_measure(o, &obs[2 * k], &obs[2 * k + 1]);
    }
}

/* never_changed = #{i : value never differed from its predecessor since the
 * reference time}; overlap = sum_i sigma_i(ref) sigma_i(now), sigma = s for
 * Ising, 2n-1 for NE (readings D11, D12).                 */
void orc_persistence(const orc_t *o, int64_t *never_changed, int64_t *overlap)
{
    int64_t nc = 0, ov = 0;
    for (int64_t i = 0; i < o->N; ++i) {
        if (!o->changed[i]) ++nc;
        int a = o->s0[i], b = o->s[i];
        if (o->model == ORC_POTTS) { ov += (a == b); continue; }      /* D26: overlap = sites in their reference state */
        if (o->model == ORC_NE_HEATBATH || o->model == ORC_NE_METROPOLIS) { a = 2 * a - 1; b = 2 * b - 1; }
        ov += (int64_t)a * b;
    }
    *never_changed = nc; *overlap = ov;
}
