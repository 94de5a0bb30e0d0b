// lsm_api.cu -- host side of the C ABI declared in include/lsm.h.  Argument checks, the threshold
// table (reading D3), kernel-family dispatch and stream-ordered bookkeeping; every step of the hot
// path itself runs in the kernels of lsm_generic.cu / lsm_tiled.cu.
#include "../../include/lsm.h"
#include "lsm_internal.cuh"
#include "lsm_tiled.cuh"

#include <cmath>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

using namespace lsmk;

struct lsm {
    int dims, L, two_S, model_abi, model;
    double J, h, T, c;
    uint64_t seed;
    int64_t N;
    Lat lat;
    long long *d_run;   // running (B, M) of the current configuration
    long long *d_tmp;   // scratch pair for reductions
    uint64_t t;         // sweeps done
    int tracking;
    int kernel_pref, kernel_in_use;
    cudaStream_t last_stream;
    uint64_t launches;
    uint64_t thr[128];
    int nthr;
    Thr64 thr_param;
    TiledTables tiled;
    unsigned *d_flags;  // reserved words of the workspace state block (the removed resident family's progress flags)
    SmallPlan small;
    SlabPlan slab;
    uint32_t *d_mbox;   // slab family: mailbox rows at the end of the workspace (nullptr: shape not covered)
    size_t mbox_bytes;
    int slab_depth;     // requested temporal depth of the slab family (0: default)
    int slab_refused;   // a cooperative slab launch did not fit this context (SM-limited MPS / green context): AUTO avoids the family
    uint8_t *alt[2];    // NE models: second lattice buffer of the random-tile schedule (reading D18)
};

static thread_local std::string g_cuda_err;
static thread_local cudaError_t g_cuda_code = cudaSuccess;
static int cuda_fail(cudaError_t e)
{
    g_cuda_code = e;
    g_cuda_err = std::string(cudaGetErrorName(e)) + ": " + cudaGetErrorString(e);
    return LSM_ERR_CUDA;
}
#define CU(x) do { cudaError_t e__ = (x); if (e__ != cudaSuccess) return cuda_fail(e__); } while (0)

static size_t align256(size_t v) { return (v + 255) & ~(size_t)255; }
static const size_t STATE_BYTES = 256 + 4 * (size_t)RESIDENT_MAX_CTAS;   // running sums, scratch, resident-kernel flags

static int check_shape(int dims, int L, int two_S, int model)
{
    if (dims != 2 && dims != 3) return LSM_ERR_ARG;
    if (L < 4 || (L & 1)) return LSM_ERR_ARG;
    if (dims == 2 && L > 131072) return LSM_ERR_ARG;
    if (dims == 3 && L > 2048) return LSM_ERR_ARG;
    if (model == LSM_ISING) { if (two_S != 1 && two_S != 2) return LSM_ERR_UNSUPPORTED; }
    else if (model == LSM_NE_HEATBATH || model == LSM_NE_METROPOLIS) {
        if (dims != 2 || two_S != 1) return LSM_ERR_UNSUPPORTED;
    } else if (model == LSM_EA) { if (two_S != 1) return LSM_ERR_UNSUPPORTED; }          // reading D25: spin-1/2
    else if (model == LSM_POTTS) { if (two_S < 1 || two_S > 7) return LSM_ERR_UNSUPPORTED; }   // D26: q = two_S + 1 <= 8
    else return LSM_ERR_ARG;
    return LSM_OK;
}

static int internal_model(int model, int two_S)
{
    return model == LSM_ISING ? (two_S == 1 ? M_ISING_HALF : M_ISING_ONE)
         : model == LSM_EA ? M_EA : model == LSM_POTTS ? M_POTTS
         : (model == LSM_NE_HEATBATH ? M_NE_HEATBATH : M_NE_METROPOLIS);
}

extern "C" int lsm_workspace_bytes(int dims, int L, int two_S, int model, size_t *bytes)
{
    if (!bytes) return LSM_ERR_ARG;
    int rc = check_shape(dims, L, two_S, model);
    if (rc != LSM_OK) return rc;
    size_t N = (size_t)L * L * (dims == 3 ? (size_t)L : 1);
    *bytes = STATE_BYTES + 2 * align256(N / 2) + 256;
    if (model == LSM_NE_HEATBATH || model == LSM_NE_METROPOLIS) *bytes += 2 * align256(N / 2);   // second buffer of the random-tile schedule
    if (model == LSM_EA) *bytes += 2 * align256(N / 2);      // bond bytes of the two colours
    *bytes += align256(slab_mailbox_bytes(dims, L, internal_model(model, two_S)));   // slab family: boundary-row mailboxes
    return LSM_OK;
}

// ---------------------------------------------------------------------------- thresholds (a0)
// Reading D3: x = J*nn + h; dE = -(s'-s)*x; p = exp(-dE/T); thr = 2^32 if dE <= 0 or p >= 1,
// else floor(p * 2^32).  Plain IEEE double, division by T, no contraction (-ffp-contract=off).
static uint64_t thr_from_p(double p)
{
    if (p >= 1.0) return (uint64_t)1 << 32;
    return (uint64_t)std::floor(std::ldexp(p, 32));
}
static uint64_t thr_flip(double J, double h, double T, int s_old, int s_new, int nn)
{
    double x = J * (double)nn + h;
    double dE = -(double)(s_new - s_old) * x;
    if (dE <= 0.0) return (uint64_t)1 << 32;
    return thr_from_p(std::exp(-dE / T));
}

static void build_tables(lsm *o)
{
    const int d = o->dims;
    int n = 0;
    if (o->model == M_POTTS) {
        // reading D26: dE = -J * dn, dn = n_new - n_old, idx = dn + 2d
        for (int j = 0; j <= 4 * d; ++j) {
            double x = o->J * (double)(j - 2 * d);
            double dE = -x;
            o->thr[n++] = dE <= 0.0 ? ((uint64_t)1 << 32) : thr_from_p(std::exp(-dE / o->T));
        }
    } else if (o->model == M_ISING_HALF || o->model == M_EA) {
        // M_EA (reading D25): the same table, indexed by the bond-weighted up-count
        for (int b = 0; b < 2; ++b)
            for (int j = 0; j <= 2 * d; ++j) o->thr[n++] = thr_flip(o->J, o->h, o->T, 2 * b - 1, 1 - 2 * b, 2 * j - 2 * d);
    } else if (o->model == M_ISING_ONE) {
        for (int a = 0; a < 3; ++a)
            for (int kk = 0; kk < 2; ++kk)
                for (int j = 0; j <= 4 * d; ++j)
                    o->thr[n++] = thr_flip(o->J, o->h, o->T, a - 1, (a + 1 + kk) % 3 - 1, j - 2 * d);
    } else {
        o->c = 1.0 / (1.0 + std::exp(1.0 / o->T));          // reading D6
        o->thr[n++] = thr_from_p(o->c);
        o->thr[n++] = thr_from_p(std::exp(-1.0 / o->T));
        o->thr[n++] = (uint64_t)1 << 32;
    }
    o->nthr = n;
    std::memset(&o->thr_param, 0, sizeof(o->thr_param));
    for (int i = 0; i < n; ++i) o->thr_param.thr[i] = o->thr[i];
    o->thr_param.count = n;
    build_tiled_tables(o->model, d, o->J, o->h, o->thr, n, &o->tiled);
}

static void choose_kernel(lsm *o)
{
    int want = o->kernel_pref;
    bool tiled_ok = tiled_supported(o->lat, o->model, o->tiled);
    if (want == LSM_KERNEL_AUTO && o->slab_refused) {
        if (small_plan(o->lat, o->model, o->tiled, &o->small, false)) want = LSM_KERNEL_SMALL;
        else want = tiled_ok ? LSM_KERNEL_TILED : LSM_KERNEL_GENERIC;
    } else if (want == LSM_KERNEL_AUTO) {
        // 512^2 ... 4096^2, 64^3, 128^3: the lattice lives in the SMs' shared memory (profiles/r2_slab_family.md)
        // (Edwards-Anderson / Potts have no small-family kernels: the slab family from 128^2 / 32^3)
        if ((o->N >= 262144 || o->model == M_EA || o->model == M_POTTS) &&
            slab_plan(o->lat, o->model, o->tiled, o->slab_depth, &o->slab)) want = LSM_KERNEL_SLAB;
        // small lattices: the small family's lane kernel (edge a power of two); else the slab family where it runs
        // (from 128^2 / 32^3: 2 us per sweep against 5.5 for the small family's single-block word kernel); else that
        else if (small_plan(o->lat, o->model, o->tiled, &o->small, false) &&
                 (o->small.lane || !slab_plan(o->lat, o->model, o->tiled, o->slab_depth, &o->slab))) want = LSM_KERNEL_SMALL;
        else if (slab_plan(o->lat, o->model, o->tiled, o->slab_depth, &o->slab)) want = LSM_KERNEL_SLAB;
        else want = tiled_ok ? LSM_KERNEL_TILED : LSM_KERNEL_GENERIC;
    }
    if (want == LSM_KERNEL_SMALL && !small_plan(o->lat, o->model, o->tiled, &o->small, true))
        want = tiled_ok ? LSM_KERNEL_TILED : LSM_KERNEL_GENERIC;
    if (want == LSM_KERNEL_TILED && !tiled_ok) want = LSM_KERNEL_GENERIC;
    if (want == LSM_KERNEL_RESIDENT) want = tiled_ok ? LSM_KERNEL_TILED : LSM_KERNEL_GENERIC;   // family removed (lsm_set_kernel refuses it)
    if (want == LSM_KERNEL_SLAB && !slab_plan(o->lat, o->model, o->tiled, o->slab_depth, &o->slab))
        want = tiled_ok ? LSM_KERNEL_TILED : LSM_KERNEL_GENERIC;
    if (want == LSM_KERNEL_BULK && !tiled_bulk_supported(o->lat, o->model, o->tiled))
        want = tiled_ok ? LSM_KERNEL_TILED : LSM_KERNEL_GENERIC;
    o->kernel_in_use = want;
}

// ---------------------------------------------------------------------------- life cycle
static int refresh_running(lsm *o, cudaStream_t s)
{
    CU(launch_measure_full(o->lat, o->model, o->d_run, s));
    o->launches += 1;
    return LSM_OK;
}

extern "C" int lsm_create(int dims, int L, int two_S, int model, double J, double h, double T, uint64_t seed,
                          void *d_workspace, size_t workspace_bytes, void *stream, lsm_t **out)
{
    if (!out || !d_workspace) return LSM_ERR_ARG;
    int rc = check_shape(dims, L, two_S, model);
    if (rc != LSM_OK) return rc;
    if (!(T > 0.0) || !std::isfinite(T) || !std::isfinite(J) || !std::isfinite(h)) return LSM_ERR_ARG;
    if ((model == LSM_NE_HEATBATH || model == LSM_NE_METROPOLIS) && J != 0.0) return LSM_ERR_UNSUPPORTED;
    if (model == LSM_POTTS && h != 0.0) return LSM_ERR_UNSUPPORTED;        // reading D26: no field term
    size_t need = 0;
    lsm_workspace_bytes(dims, L, two_S, model, &need);
    if (workspace_bytes < need || ((uintptr_t)d_workspace & 255)) return LSM_ERR_WORKSPACE;

    lsm *o = new (std::nothrow) lsm();
    if (!o) return LSM_ERR_ARG;
    o->dims = dims; o->L = L; o->two_S = two_S; o->model_abi = model;
    o->model = internal_model(model, two_S);
    o->J = J; o->h = h; o->T = T; o->c = 0.0; o->seed = seed;
    o->N = (int64_t)L * L * (dims == 3 ? L : 1);
    uint8_t *base = (uint8_t *)d_workspace;
    o->d_run = (long long *)base;
    o->d_tmp = (long long *)(base + 64);
    o->d_flags = (unsigned *)(base + 256);
    o->lat.col[0] = base + STATE_BYTES;
    o->lat.col[1] = base + STATE_BYTES + align256((size_t)o->N / 2);
    o->alt[0] = o->alt[1] = nullptr;
    o->lat.bnd[0] = o->lat.bnd[1] = nullptr;
    o->lat.q = model == LSM_POTTS ? two_S + 1 : 0;
    if (model == LSM_NE_HEATBATH || model == LSM_NE_METROPOLIS) {
        o->alt[0] = o->lat.col[1] + align256((size_t)o->N / 2);
        o->alt[1] = o->alt[0] + align256((size_t)o->N / 2);
    }
    if (model == LSM_EA) {
        o->lat.bnd[0] = o->lat.col[1] + align256((size_t)o->N / 2);
        o->lat.bnd[1] = o->lat.bnd[0] + align256((size_t)o->N / 2);
    }
    o->mbox_bytes = slab_mailbox_bytes(dims, L, o->model);
    o->d_mbox = o->mbox_bytes ? (uint32_t *)(base + need - align256(o->mbox_bytes)) : nullptr;
    o->lat.L = L; o->lat.Lh = L / 2; o->lat.dims = dims; o->lat.Lz = dims == 3 ? L : 1;
    o->lat.half = o->N / 2;
    o->t = 0; o->tracking = 1; o->kernel_pref = LSM_KERNEL_AUTO; o->launches = 0; o->slab_depth = 0; o->slab_refused = 0;
    o->last_stream = (cudaStream_t)stream;
    build_tables(o);
    choose_kernel(o);

    cudaStream_t s = (cudaStream_t)stream;
    cudaError_t e = cudaMemsetAsync(base, 0, STATE_BYTES, s);
    if (e == cudaSuccess) e = launch_init(o->lat, o->model, seed, o->thr[0], s);
    if (e == cudaSuccess && o->model == M_EA) { e = launch_ea_bonds_init(o->lat, seed, s); o->launches += 1; }
    if (e == cudaSuccess) e = launch_reset_reference(o->lat, o->model, 1, s);
    if (e == cudaSuccess) e = launch_measure_full(o->lat, o->model, o->d_run, s);
    if (e != cudaSuccess) { delete o; return cuda_fail(e); }
    o->launches += 3;
    *out = o;
    return LSM_OK;
}

extern "C" int lsm_destroy(lsm_t *o)
{
    if (!o) return LSM_ERR_ARG;
    delete o;
    return LSM_OK;
}

// ---------------------------------------------------------------------------- sweeps (a2-a7)
static int enqueue_half(lsm *o, int family, int half, long long *obs, int want_B, cudaStream_t s)
{
    SweepArgs a;
    a.lat = o->lat; a.model = o->model; a.half = half;
    a.key = make_sweep_key(o->seed, o->t, (uint32_t)half);
    a.track = o->tracking; a.obs = obs; a.want_B = want_B;
    a.bulk = family == LSM_KERNEL_BULK ? 1 : 0;
    if (family == LSM_KERNEL_TILED || family == LSM_KERNEL_BULK) CU(launch_sweep_tiled(a, o->tiled, s));
    else CU(launch_sweep_generic(a, o->thr_param, s));
    o->launches += 1;
    return LSM_OK;
}

// Families that run whole sweeps per launch (small, slab).  Without a per-sweep record only the last sweep is
// measured (into the running pair), so it gets a launch of its own.
static int resident_launch(lsm *o, int64_t n, long long *obs, cudaStream_t s)
{
    const int64_t CHUNK = 1 << 20;
    while (n > 0) {
        int k = (int)(n < CHUNK ? n : CHUNK);
        if (o->kernel_in_use == LSM_KERNEL_SMALL) {
            CU(launch_sweep_small(o->lat, o->model, o->tracking, o->seed, o->t, k, obs, o->small, o->tiled, s));
        } else if (o->kernel_in_use == LSM_KERNEL_SLAB) {
            // every mailbox lane this launch can read: sweep parity 1 (lsm_slab.cu).  The layout puts the CTA outermost,
            // so G slabs use the first G * 8 * dmax march rows of the reservation (which is sized for SLAB_MAX_CTAS).
            const size_t rowbytes = (size_t)(o->L / 2) * (o->dims == 3 ? (size_t)o->L : 1);
            size_t used = (size_t)o->slab.G * 8 * (size_t)o->slab.dmax * rowbytes;
            if (used > o->mbox_bytes) used = o->mbox_bytes;
            CU(cudaMemsetAsync(o->d_mbox, 0x80, used, s));
            CU(launch_sweep_slab(o->lat, o->model, o->tracking, o->seed, o->t, k, obs, o->d_mbox, o->slab, o->tiled, s));
        } else {
            return LSM_ERR_UNSUPPORTED;
        }
        o->launches += 1;
        o->t += (uint64_t)k;
        if (obs) obs += 2 * (int64_t)k;
        n -= k;
    }
    return LSM_OK;
}

static int sweep_resident(lsm *o, int64_t n, long long *d_obs, cudaStream_t s)
{
    if (d_obs) {
        CU(cudaMemsetAsync(d_obs, 0, (size_t)n * 16, s));
        int rc = resident_launch(o, n, d_obs, s);
        if (rc != LSM_OK) return rc;
        CU(cudaMemcpyAsync(o->d_run, d_obs + 2 * (n - 1), 16, cudaMemcpyDeviceToDevice, s));
        return LSM_OK;
    }
    if (n > 1) {
        int rc = resident_launch(o, n - 1, nullptr, s);
        if (rc != LSM_OK) return rc;
    }
    CU(cudaMemsetAsync(o->d_run, 0, 16, s));
    return resident_launch(o, 1, o->d_run, s);
}

static int sweep_impl(lsm *o, int64_t n, long long *d_obs, cudaStream_t s)
{
    o->last_stream = s;
    if (n == 0) return LSM_OK;
    // A slab launch reads and writes the whole lattice once: on the largest slab lattices (4096^2: 2 x 16 MB, ~19 us) a
    // call of a few sweeps is cheaper as launches per half-sweep (measured: break-even at 8 sweeps; same results).
    const bool short_call = o->kernel_in_use == LSM_KERNEL_SLAB && o->kernel_pref == LSM_KERNEL_AUTO && n < 8 &&
                            o->N >= ((int64_t)1 << 24) && tiled_supported(o->lat, o->model, o->tiled);
    if (!short_call &&
        (o->kernel_in_use == LSM_KERNEL_SMALL || o->kernel_in_use == LSM_KERNEL_SLAB)) {
        const uint64_t t_before = o->t;
        const int rc = sweep_resident(o, n, d_obs, s);
        // One CTA per SM, all co-resident: under an SM-limited context (MPS active-thread percentage, green context) the
        // cooperative slab launch is refused although the launch-per-half-sweep families run the lattice.  AUTO then
        // gives the family up for this handle and finishes the call with the next best one (same results).
        if (rc == LSM_ERR_CUDA && g_cuda_code == cudaErrorCooperativeLaunchTooLarge && o->kernel_in_use == LSM_KERNEL_SLAB &&
            o->kernel_pref == LSM_KERNEL_AUTO) {
            (void)cudaGetLastError();
            o->slab_refused = 1;
            choose_kernel(o);
            const int64_t done = (int64_t)(o->t - t_before);
            return sweep_impl(o, n - done, d_obs ? d_obs + 2 * done : nullptr, s);
        }
        return rc;
    }
    const int family = short_call ? LSM_KERNEL_TILED : o->kernel_in_use;
    if (d_obs) CU(cudaMemsetAsync(d_obs, 0, (size_t)n * 16, s));
    else CU(cudaMemsetAsync(o->d_run, 0, 16, s));
    for (int64_t k = 0; k < n; ++k) {
        long long *obs = d_obs ? d_obs + 2 * k : (k == n - 1 ? o->d_run : nullptr);
        int rc = enqueue_half(o, family, 0, obs, 0, s);
        if (rc != LSM_OK) return rc;
        rc = enqueue_half(o, family, 1, obs, 1, s);
        if (rc != LSM_OK) return rc;
        o->t += 1;
    }
    if (d_obs) CU(cudaMemcpyAsync(o->d_run, d_obs + 2 * (n - 1), 16, cudaMemcpyDeviceToDevice, s));
    return LSM_OK;
}

extern "C" int lsm_sweep(lsm_t *o, int64_t n, void *stream)
{
    if (!o || n < 0) return LSM_ERR_ARG;
    return sweep_impl(o, n, nullptr, (cudaStream_t)stream);
}

extern "C" int lsm_sweep_record(lsm_t *o, int64_t n, int64_t *d_obs, void *stream)
{
    if (!o || n < 0 || (!d_obs && n > 0)) return LSM_ERR_ARG;
    return sweep_impl(o, n, (long long *)d_obs, (cudaStream_t)stream);
}

// The paper's corrected North-East algorithm: two launches per sweep, each reading one
// lattice buffer and writing the other (reading D18).
static int random_tile_impl(lsm_t *o, int64_t n, int tile_edge, int lambda, int64_t *d_obs, void *stream, bool balanced)
{
    if (!o || n < 0) return LSM_ERR_ARG;
    if (o->model != M_NE_HEATBATH && o->model != M_NE_METROPOLIS) return LSM_ERR_UNSUPPORTED;
    if (!ne_tile_supported(o->lat, tile_edge, lambda, balanced)) return LSM_ERR_UNSUPPORTED;
    cudaStream_t s = (cudaStream_t)stream;
    o->last_stream = s;
    if (n == 0) return LSM_OK;
    const uint64_t ALWAYS = (uint64_t)1 << 32;
    const uint32_t thr_c = o->thr[0] >= ALWAYS ? 0xFFFFFFFFu : (uint32_t)o->thr[0];
    const uint32_t thr_up = o->thr[1] >= ALWAYS ? 0xFFFFFFFFu : (uint32_t)o->thr[1];
    if (d_obs) CU(cudaMemsetAsync(d_obs, 0, (size_t)n * 16, s));
    else CU(cudaMemsetAsync(o->d_run, 0, 16, s));
    for (int64_t k = 0; k < n; ++k) {
        long long *obs = d_obs ? (long long *)d_obs + 2 * k : (k == n - 1 ? o->d_run : nullptr);
        const int nlaunch = balanced ? 4 : 2;                       // reading D23 / D17
        for (int launch = 0; launch < nlaunch; ++launch) {
            CU(launch_ne_random_tile(o->lat, o->alt, o->model == M_NE_METROPOLIS, balanced, tile_edge, lambda, o->seed, o->t,
                                     launch, thr_c, thr_up, o->thr[1] >= ALWAYS ? 1 : 0, o->tracking,
                                     launch == nlaunch - 1 ? obs : nullptr, s));
            o->launches += 1;
            for (int c = 0; c < 2; ++c) { uint8_t *tmp = o->lat.col[c]; o->lat.col[c] = o->alt[c]; o->alt[c] = tmp; }
        }
        o->t += 1;
    }
    if (d_obs) CU(cudaMemcpyAsync(o->d_run, (long long *)d_obs + 2 * (n - 1), 16, cudaMemcpyDeviceToDevice, s));
    return LSM_OK;
}

extern "C" int lsm_sweep_random_tile(lsm_t *o, int64_t n, int tile_edge, int lambda, int64_t *d_obs, void *stream)
{
    return random_tile_impl(o, n, tile_edge, lambda, d_obs, stream, false);
}

// The balance-preserving variant: colour-restricted picks, four launches per MC step.
extern "C" int lsm_sweep_random_tile_balanced(lsm_t *o, int64_t n, int tile_edge, int lambda, int64_t *d_obs, void *stream)
{
    return random_tile_impl(o, n, tile_edge, lambda, d_obs, stream, true);
}

// As lsm_sweep_record_host, but the device->host copy of the series is only enqueued: h_obs (pinned) is valid after
// the caller has synchronised `stream`.
extern "C" int lsm_sweep_record_host_async(lsm_t *o, int64_t n, int64_t *h_obs, int64_t *d_scratch, void *stream)
{
    if (!o || n < 0 || ((!h_obs || !d_scratch) && n > 0)) return LSM_ERR_ARG;
    cudaStream_t s = (cudaStream_t)stream;
    int rc = sweep_impl(o, n, (long long *)d_scratch, s);
    if (rc != LSM_OK) return rc;
    if (n > 0) CU(cudaMemcpyAsync(h_obs, d_scratch, (size_t)n * 16, cudaMemcpyDeviceToHost, s));
    return LSM_OK;
}

extern "C" int lsm_sweep_record_host(lsm_t *o, int64_t n, int64_t *h_obs, int64_t *d_scratch, void *stream)
{
    int rc = lsm_sweep_record_host_async(o, n, h_obs, d_scratch, stream);
    if (rc != LSM_OK) return rc;
    CU(cudaStreamSynchronize((cudaStream_t)stream));
    return LSM_OK;
}

// ---------------------------------------------------------------------------- entry point without device allocation
// lsm_sweep_record_host needs 16*n bytes of device scratch for the (B, M) series, and so far the caller had to bring
// them.  Some callers have no way to: a plug-in inside a host program that handed every byte of HBM to its own pool
// and offers no allocation hook, a control loop that may not pay cudaMalloc's device-wide synchronisation between
// two steps, a process running under a memory quota that is already spent on the lattice.  For them the scratch
// lives in the library image itself: the array below, LSM_NOALLOC_MAX_SWEEPS pairs = 64 KiB, present on every GPU
// this library is loaded on from the moment the module is loaded until the process exits.
//
// `g_noalloc_obs` is two things.  In device code it is the array.  In host code the same name is only the handle the
// runtime registered for it, NOT a device address: handing it to a kernel makes the kernel fault (or, on systems where
// the GPU can reach host memory, scribble over host memory that has nothing to do with the array).  The device address
// comes from cudaGetSymbolAddress, per device, with that device current; noalloc_scratch() asks once per device and
// keeps the answer.
static __device__ __align__(256) long long g_noalloc_obs[2 * LSM_NOALLOC_MAX_SWEEPS];

static const int NOALLOC_MAX_DEVICES = 64;
static std::mutex g_noalloc_mutex;
static long long *g_noalloc_addr[NOALLOC_MAX_DEVICES];   // device address of g_noalloc_obs on device k (nullptr: not asked yet)

static int noalloc_scratch(long long **d_ptr)
{
    int dev = -1;
    CU(cudaGetDevice(&dev));
    if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) return LSM_ERR_UNSUPPORTED;
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    if (!g_noalloc_addr[dev]) {
        void *p = nullptr;
        CU(cudaGetSymbolAddress(&p, g_noalloc_obs));     // the current device's copy of the array
        if (!p) return LSM_ERR_CUDA;
        g_noalloc_addr[dev] = (long long *)p;
    }
    *d_ptr = g_noalloc_addr[dev];
    return LSM_OK;
}

// lsm_sweep_record_host with the device scratch taken from g_noalloc_obs: the sweep kernels accumulate (B, M) of
// sweep k into pair k of the array (cleared first on `stream`, as for any d_obs: the kernels add into it), the series
// is copied to h_obs on `stream`, and the call returns once the copy has completed.  No cudaMalloc / cudaFree, no
// allocating library call.
extern "C" int lsm_sweep_record_host_noalloc(lsm_t *o, int64_t n, int64_t *h_obs, void *stream)
{
    if (!o || n < 0 || (!h_obs && n > 0)) return LSM_ERR_ARG;
    if (n > LSM_NOALLOC_MAX_SWEEPS) return LSM_ERR_LIMIT;
    long long *d_obs = nullptr;
    int rc = noalloc_scratch(&d_obs);
    if (rc != LSM_OK) return rc;
    cudaStream_t s = (cudaStream_t)stream;
    rc = sweep_impl(o, n, d_obs, s);
    if (rc != LSM_OK) return rc;
    if (n > 0) CU(cudaMemcpyAsync(h_obs, d_obs, (size_t)n * 16, cudaMemcpyDeviceToHost, s));
    CU(cudaStreamSynchronize(s));
    return LSM_OK;
}

// ---------------------------------------------------------------------------- batch of lattices (NEXT-3)
// R independent lattices of one shape, each with its own temperature and seed (the 31 temperatures of the paper's
// Fig. 6 ramp, or the 30 realisations of Fig. 7), swept by ONE kernel launch: the paper's
// small lattices cannot fill a GPU one at a time.  Every replica is a complete lsm handle on its own
// slice of the workspace (lsm_batch_replica lends it out for lsm_get_spins, lsm_persistence, ...); the batch sweep is
// the small family's lane kernel with one thread-block cluster per replica (lsm_small.cu).  Bit-identical to
// sweeping each replica on its own.
struct lsm_batch {
    int R;
    std::vector<lsm *> rep;
    std::vector<uint64_t> seeds;
    size_t rep_bytes;
    BatchDesc *d_desc;
    std::vector<BatchDesc> h_desc;   // what the device array holds
    int cluster_pref;                // 0 = auto
    uint64_t launches;               // batch launches (the replicas count their own)
};

static size_t batch_desc_bytes(int R) { return align256((size_t)R * sizeof(BatchDesc)); }

extern "C" int lsm_batch_workspace_bytes(int R, int dims, int L, int two_S, int model, size_t *bytes)
{
    if (!bytes || R < 1 || R > 65536) return LSM_ERR_ARG;
    size_t one = 0;
    int rc = lsm_workspace_bytes(dims, L, two_S, model, &one);
    if (rc != LSM_OK) return rc;
    *bytes = batch_desc_bytes(R) + (size_t)R * align256(one);
    return LSM_OK;
}

extern "C" int lsm_batch_destroy(lsm_batch_t *b)
{
    if (!b) return LSM_ERR_ARG;
    for (lsm *o : b->rep) delete o;
    delete b;
    return LSM_OK;
}

extern "C" int lsm_batch_create(int R, int dims, int L, int two_S, int model, double J, double h, const double *T,
                                const uint64_t *seeds, void *d_workspace, size_t workspace_bytes, void *stream,
                                lsm_batch_t **out)
{
    if (!out || !T || !seeds || !d_workspace) return LSM_ERR_ARG;
    size_t need = 0, one = 0;
    int rc = lsm_batch_workspace_bytes(R, dims, L, two_S, model, &need);
    if (rc != LSM_OK) return rc;
    if (workspace_bytes < need || ((uintptr_t)d_workspace & 255)) return LSM_ERR_WORKSPACE;
    lsm_workspace_bytes(dims, L, two_S, model, &one);
    lsm_batch *b = new (std::nothrow) lsm_batch();
    if (!b) return LSM_ERR_ARG;
    b->R = R;
    b->rep_bytes = align256(one);
    b->d_desc = (BatchDesc *)d_workspace;
    b->cluster_pref = 0;
    b->launches = 0;
    uint8_t *base = (uint8_t *)d_workspace + batch_desc_bytes(R);
    for (int r = 0; r < R; ++r) {
        lsm *o = nullptr;
        rc = lsm_create(dims, L, two_S, model, J, h, T[r], seeds[r], base + (size_t)r * b->rep_bytes, b->rep_bytes, stream, &o);
        if (rc != LSM_OK) { lsm_batch_destroy(b); return rc; }
        b->rep.push_back(o);
        b->seeds.push_back(seeds[r]);
    }
    *out = b;
    return LSM_OK;
}

extern "C" int lsm_batch_size(lsm_batch_t *b, int *R)
{
    if (!b || !R) return LSM_ERR_ARG;
    *R = b->R;
    return LSM_OK;
}

extern "C" int lsm_batch_replica(lsm_batch_t *b, int r, lsm_t **handle)
{
    if (!b || !handle || r < 0 || r >= b->R) return LSM_ERR_ARG;
    *handle = b->rep[r];
    return LSM_OK;
}

extern "C" int lsm_batch_set_temperatures(lsm_batch_t *b, const double *T)
{
    if (!b || !T) return LSM_ERR_ARG;
    for (int r = 0; r < b->R; ++r)
        if (!(T[r] > 0.0) || !std::isfinite(T[r])) return LSM_ERR_ARG;
    for (int r = 0; r < b->R; ++r) lsm_set_temperature(b->rep[r], T[r]);
    return LSM_OK;
}

extern "C" int lsm_batch_set_tracking(lsm_batch_t *b, int on, void *stream)
{
    if (!b) return LSM_ERR_ARG;
    for (lsm *o : b->rep) {
        int rc = lsm_set_tracking(o, on, stream);
        if (rc != LSM_OK) return rc;
    }
    return LSM_OK;
}

extern "C" int lsm_batch_set_cluster(lsm_batch_t *b, int blocks_per_replica)
{
    if (!b || blocks_per_replica < 0 || blocks_per_replica > 16 || (blocks_per_replica & (blocks_per_replica - 1))) return LSM_ERR_ARG;
    if (blocks_per_replica > 0) {
        const Lat &lat = b->rep[0]->lat;
        const long long lanes = lat.half / 4, N = 2 * lat.half;
        if (blocks_per_replica > lat.L || lanes / blocks_per_replica < 32 || N / blocks_per_replica > 196608) return LSM_ERR_UNSUPPORTED;
    }
    b->cluster_pref = blocks_per_replica;
    return LSM_OK;
}

// The one-launch path needs the lane kernel of the small family for every replica's table and one tracking state.
static bool batch_one_launch(const lsm_batch *b)
{
    for (const lsm *o : b->rep) {
        if (o->tracking != b->rep[0]->tracking) return false;
        if (!small_batch_supported(o->lat, o->model, o->tiled)) return false;
    }
    return true;
}

// Device descriptors follow the replicas' current colour arrays (the random-tile schedule swaps them) and tables.
static int batch_refresh_desc(lsm_batch *b, cudaStream_t s)
{
    std::vector<BatchDesc> now((size_t)b->R);
    for (int r = 0; r < b->R; ++r) {
        const lsm *o = b->rep[r];
        BatchDesc &d = now[r];
        std::memset(&d, 0, sizeof(d));
        d.col[0] = o->lat.col[0];
        d.col[1] = o->lat.col[1];
        d.run = o->d_run;
        if (o->model == M_ISING_HALF) for (int i = 0; i < 16; ++i) d.tab[i] = o->tiled.t32[i];
        else if (o->model == M_ISING_ONE) for (int i = 0; i < 64; ++i) d.tab[i] = o->tiled.s1[i];
        else {
            d.ne_t32 = o->tiled.ne_t32[o->model == M_NE_HEATBATH ? 0 : 1];
            d.ne_always = o->model == M_NE_HEATBATH ? 0 : o->tiled.ne_up_always;
        }
    }
    if (b->h_desc.size() == now.size() && std::memcmp(b->h_desc.data(), now.data(), now.size() * sizeof(BatchDesc)) == 0)
        return LSM_OK;
    // pageable source: the runtime stages it before returning, so `now` may go out of scope
    CU(cudaMemcpyAsync(b->d_desc, now.data(), now.size() * sizeof(BatchDesc), cudaMemcpyHostToDevice, s));
    b->h_desc.swap(now);
    return LSM_OK;
}

static int batch_sweep_impl(lsm_batch *b, int64_t n, long long *d_obs, cudaStream_t s)
{
    if (n == 0) return LSM_OK;
    if (!batch_one_launch(b)) {                       // any lattice, any table: one replica after the other
        for (int r = 0; r < b->R; ++r) {
            int rc = sweep_impl(b->rep[r], n, d_obs ? d_obs + 2 * n * r : nullptr, s);
            if (rc != LSM_OK) return rc;
        }
        return LSM_OK;
    }
    int rc = batch_refresh_desc(b, s);
    if (rc != LSM_OK) return rc;
    lsm *o0 = b->rep[0];
    const int cluster = b->cluster_pref ? b->cluster_pref : small_batch_cluster(o0->lat, b->R);
    const uint64_t t0 = o0->t;
    for (lsm *o : b->rep) {
        if (o->t != t0) return LSM_ERR_STATE;         // a replica was swept on its own: the batch sweeps in lockstep
        o->last_stream = s;
    }
    const int64_t CHUNK = 1 << 20;
    int64_t done = 0;
    if (!d_obs && n > 1) {                            // only the last sweep is measured
        for (; done < n - 1;) {
            const int k = (int)(n - 1 - done < CHUNK ? n - 1 - done : CHUNK);
            CU(launch_sweep_small_batch(o0->lat, o0->model, o0->tracking, b->d_desc, b->seeds.data(), b->R, cluster,
                                        t0 + (uint64_t)done, k, nullptr, 0, 0, s));
            b->launches += (uint64_t)((b->R + 255) / 256);
            done += k;
        }
    }
    for (; done < n;) {
        const int k = (int)(n - done < CHUNK ? n - done : CHUNK);
        const bool last = done + k == n;
        CU(launch_sweep_small_batch(o0->lat, o0->model, o0->tracking, b->d_desc, b->seeds.data(), b->R, cluster,
                                    t0 + (uint64_t)done, k, d_obs ? d_obs + 2 * done : nullptr, 2 * n, last ? 1 : 0, s));
        b->launches += (uint64_t)((b->R + 255) / 256);
        done += k;
    }
    for (lsm *o : b->rep) o->t = t0 + (uint64_t)n;
    return LSM_OK;
}

extern "C" int lsm_batch_sweep(lsm_batch_t *b, int64_t n, void *stream)
{
    if (!b || n < 0) return LSM_ERR_ARG;
    return batch_sweep_impl(b, n, nullptr, (cudaStream_t)stream);
}

extern "C" int lsm_batch_sweep_record(lsm_batch_t *b, int64_t n, int64_t *d_obs, void *stream)
{
    if (!b || n < 0 || (!d_obs && n > 0)) return LSM_ERR_ARG;
    return batch_sweep_impl(b, n, (long long *)d_obs, (cudaStream_t)stream);
}

// The random-tile schedules for a whole batch (30 realisations per concentration; a 128^2 lattice is 16
// tiles, one CTA): every launch of the schedule handles the tiles of ALL replicas, so a sweep of the batch costs the two
// (four) launches a single lattice pays.  Bit-identical to lsm_sweep_random_tile[_balanced] on every replica.
static int batch_random_tile_impl(lsm_batch *b, int64_t n, int tile_edge, int lambda, long long *d_obs, cudaStream_t s,
                                  bool balanced)
{
    lsm *o0 = b->rep[0];
    if (o0->model != M_NE_HEATBATH && o0->model != M_NE_METROPOLIS) return LSM_ERR_UNSUPPORTED;
    if (!ne_tile_supported(o0->lat, tile_edge, lambda, balanced)) return LSM_ERR_UNSUPPORTED;
    if ((size_t)b->R * 2 * sizeof(NeBatchDesc) > batch_desc_bytes(b->R)) return LSM_ERR_UNSUPPORTED;
    const uint64_t t0 = o0->t;
    for (lsm *o : b->rep) {
        if (o->t != t0 || o->tracking != o0->tracking) return LSM_ERR_STATE;
        o->last_stream = s;
    }
    if (n == 0) return LSM_OK;
    const uint64_t ALWAYS = (uint64_t)1 << 32;
    // descriptors of both launch directions (colour arrays -> second buffer and back), the checkerboard batch's
    // descriptors share the region and are uploaded again when it runs next
    std::vector<NeBatchDesc> d(2 * (size_t)b->R);
    for (int dir = 0; dir < 2; ++dir)
        for (int r = 0; r < b->R; ++r) {
            const lsm *o = b->rep[r];
            NeBatchDesc &e = d[(size_t)dir * b->R + r];
            std::memset(&e, 0, sizeof(e));
            for (int c = 0; c < 2; ++c) {
                e.src[c] = dir ? o->alt[c] : o->lat.col[c];
                e.dst[c] = dir ? o->lat.col[c] : o->alt[c];
            }
            e.obs = d_obs ? d_obs + 2 * n * r : o->d_run;
            e.k0 = (uint32_t)o->seed;
            e.k1 = (uint32_t)(o->seed >> 32);
            e.thr_c = o->thr[0] >= ALWAYS ? 0xFFFFFFFFu : (uint32_t)o->thr[0];
            e.thr_up = o->thr[1] >= ALWAYS ? 0xFFFFFFFFu : (uint32_t)o->thr[1];
            e.up_always = o->thr[1] >= ALWAYS ? 1 : 0;
        }
    NeBatchDesc *d_desc = (NeBatchDesc *)b->d_desc;
    CU(cudaMemcpyAsync(d_desc, d.data(), d.size() * sizeof(NeBatchDesc), cudaMemcpyHostToDevice, s));   // pageable: staged before return
    b->h_desc.clear();
    if (d_obs) CU(cudaMemsetAsync(d_obs, 0, (size_t)n * 16 * (size_t)b->R, s));
    else CU(cudaMemset2DAsync(o0->d_run, b->rep_bytes, 0, 16, (size_t)b->R, s));
    const int nlaunch = balanced ? 4 : 2;                           // reading D23 / D17: an even number, so the buffers end where they began
    for (int64_t k = 0; k < n; ++k) {
        for (int launch = 0; launch < nlaunch; ++launch) {
            const long long off = launch != nlaunch - 1 ? -1 : d_obs ? 2 * k : (k == n - 1 ? 0 : -1);
            CU(launch_ne_random_tile_batch(o0->lat, d_desc + (size_t)(launch & 1) * b->R, b->R, o0->model == M_NE_METROPOLIS,
                                           balanced, tile_edge, lambda, t0 + (uint64_t)k, launch, o0->tracking, off, s));
            b->launches += 1;
        }
    }
    for (lsm *o : b->rep) o->t = t0 + (uint64_t)n;
    if (d_obs)      // running pairs := last recorded pairs (rows 16 n bytes apart -> pairs rep_bytes apart)
        CU(cudaMemcpy2DAsync(o0->d_run, b->rep_bytes, d_obs + 2 * (n - 1), (size_t)n * 16, 16, (size_t)b->R, cudaMemcpyDeviceToDevice, s));
    return LSM_OK;
}

extern "C" int lsm_batch_sweep_random_tile(lsm_batch_t *b, int64_t n, int tile_edge, int lambda, int balanced, int64_t *d_obs,
                                           void *stream)
{
    if (!b || n < 0) return LSM_ERR_ARG;
    return batch_random_tile_impl(b, n, tile_edge, lambda, (long long *)d_obs, (cudaStream_t)stream, balanced != 0);
}

extern "C" int lsm_batch_measure_int(lsm_batch_t *b, int64_t *B, int64_t *M)
{
    if (!b) return LSM_ERR_ARG;
    std::vector<long long> v(2 * (size_t)b->R);
    cudaStream_t s = b->rep[0]->last_stream;
    // the replicas' running pairs sit rep_bytes apart in the batch workspace: one strided copy instead of R small ones
    if (b->R > 1 && b->rep_bytes <= ((size_t)1 << 30))
        CU(cudaMemcpy2DAsync(v.data(), 16, b->rep[0]->d_run, b->rep_bytes, 16, (size_t)b->R, cudaMemcpyDeviceToHost, s));
    else
        for (int r = 0; r < b->R; ++r) CU(cudaMemcpyAsync(&v[2 * r], b->rep[r]->d_run, 16, cudaMemcpyDeviceToHost, s));
    CU(cudaStreamSynchronize(s));
    for (int r = 0; r < b->R; ++r) {
        if (B) B[r] = v[2 * r];
        if (M) M[r] = v[2 * r + 1];
    }
    return LSM_OK;
}

extern "C" int lsm_batch_get_launch_count(lsm_batch_t *b, uint64_t *n)
{
    if (!b || !n) return LSM_ERR_ARG;
    uint64_t tot = b->launches;
    for (lsm *o : b->rep) tot += o->launches;
    *n = tot;
    return LSM_OK;
}

// ---------------------------------------------------------------------------- observables
static int read_pair(lsm *o, const long long *d, long long out[2])
{
    CU(cudaMemcpyAsync(out, d, 16, cudaMemcpyDeviceToHost, o->last_stream));
    CU(cudaStreamSynchronize(o->last_stream));
    return LSM_OK;
}

extern "C" int lsm_energy(int model, double J, double h, int64_t B, int64_t M, double *E)
{
    if (!E) return LSM_ERR_ARG;
    if (model == LSM_ISING || model == LSM_EA) *E = -J * (double)B - h * (double)M;   // D1, D25
    else if (model == LSM_POTTS) *E = -J * (double)B;                                   // D26
    else *E = (double)M;                                                                // D15
    return LSM_OK;
}

extern "C" int lsm_measure_int(lsm_t *o, int64_t *B, int64_t *M, uint64_t *sweeps_done)
{
    if (!o) return LSM_ERR_ARG;
    long long v[2];
    int rc = read_pair(o, o->d_run, v);
    if (rc != LSM_OK) return rc;
    if (B) *B = v[0];
    if (M) *M = v[1];
    if (sweeps_done) *sweeps_done = o->t;
    return LSM_OK;
}

extern "C" int lsm_measure(lsm_t *o, double *E, int64_t *M)
{
    if (!o) return LSM_ERR_ARG;
    int64_t b, m;
    int rc = lsm_measure_int(o, &b, &m, nullptr);
    if (rc != LSM_OK) return rc;
    if (E) lsm_energy(o->model_abi, o->J, o->h, b, m, E);
    if (M) *M = m;
    return LSM_OK;
}

extern "C" int lsm_measure_full(lsm_t *o, int64_t *B, int64_t *M)
{
    if (!o) return LSM_ERR_ARG;
    int rc = refresh_running(o, o->last_stream);
    if (rc != LSM_OK) return rc;
    return lsm_measure_int(o, B, M, nullptr);
}

extern "C" int lsm_persistence(lsm_t *o, int64_t *never_changed, int64_t *overlap)
{
    if (!o) return LSM_ERR_ARG;
    if (!o->tracking) return LSM_ERR_STATE;
    CU(launch_persistence(o->lat, o->model, o->d_tmp, o->last_stream));
    o->launches += 1;
    long long v[2];
    int rc = read_pair(o, o->d_tmp, v);
    if (rc != LSM_OK) return rc;
    if (never_changed) *never_changed = v[0];
    if (overlap) *overlap = v[1];
    return LSM_OK;
}

extern "C" int lsm_set_tracking(lsm_t *o, int on, void *stream)
{
    if (!o) return LSM_ERR_ARG;
    cudaStream_t s = (cudaStream_t)stream;
    o->last_stream = s;
    CU(launch_reset_reference(o->lat, o->model, on ? 1 : 0, s));
    o->launches += 1;
    o->tracking = on ? 1 : 0;
    choose_kernel(o);
    return LSM_OK;
}

extern "C" int lsm_reset_reference(lsm_t *o, void *stream) { return lsm_set_tracking(o, 1, stream); }

// ---------------------------------------------------------------------------- configuration I/O
extern "C" int lsm_get_spins(lsm_t *o, int8_t *d_out, void *stream)
{
    if (!o || !d_out) return LSM_ERR_ARG;
    o->last_stream = (cudaStream_t)stream;
    CU(launch_get_spins(o->lat, o->model, d_out, o->last_stream));
    o->launches += 1;
    return LSM_OK;
}

extern "C" int lsm_get_spins_host(lsm_t *o, int8_t *h_out, int8_t *d_scratch, void *stream)
{
    if (!o || !h_out || !d_scratch) return LSM_ERR_ARG;
    int rc = lsm_get_spins(o, d_scratch, stream);
    if (rc != LSM_OK) return rc;
    CU(cudaMemcpyAsync(h_out, d_scratch, (size_t)o->N, cudaMemcpyDeviceToHost, o->last_stream));
    CU(cudaStreamSynchronize(o->last_stream));
    return LSM_OK;
}

extern "C" int lsm_set_spins(lsm_t *o, const int8_t *d_in, uint64_t sweep_counter, void *stream)
{
    if (!o || !d_in || (sweep_counter >> 60) != 0) return LSM_ERR_ARG;   // D2: the tag owns the low 4 bits of c3
    o->last_stream = (cudaStream_t)stream;
    CU(launch_set_spins(o->lat, o->model, d_in, o->last_stream));
    o->launches += 1;
    o->t = sweep_counter;
    return refresh_running(o, o->last_stream);
}

extern "C" int lsm_set_spins_host(lsm_t *o, const int8_t *h_in, int8_t *d_scratch, uint64_t sweep_counter, void *stream)
{
    if (!o || !h_in || !d_scratch) return LSM_ERR_ARG;
    CU(cudaMemcpyAsync(d_scratch, h_in, (size_t)o->N, cudaMemcpyHostToDevice, (cudaStream_t)stream));
    return lsm_set_spins(o, d_scratch, sweep_counter, stream);
}

// Edwards-Anderson bonds (reading D25): canonical int8 tau[dims][N], tau[a][i] = sign of the bond between site i and
// its neighbour in direction +a.  Replacing the bonds changes B: the running pair is recomputed.
extern "C" int lsm_set_bonds(lsm_t *o, const int8_t *d_tau, void *stream)
{
    if (!o || !d_tau) return LSM_ERR_ARG;
    if (o->model != M_EA) return LSM_ERR_UNSUPPORTED;
    o->last_stream = (cudaStream_t)stream;
    CU(launch_ea_set_bonds(o->lat, d_tau, o->last_stream));
    o->launches += 1;
    return refresh_running(o, o->last_stream);
}

extern "C" int lsm_get_bonds(lsm_t *o, int8_t *d_tau, void *stream)
{
    if (!o || !d_tau) return LSM_ERR_ARG;
    if (o->model != M_EA) return LSM_ERR_UNSUPPORTED;
    o->last_stream = (cudaStream_t)stream;
    CU(launch_ea_get_bonds(o->lat, d_tau, o->last_stream));
    o->launches += 1;
    return LSM_OK;
}

// Pipelined host I/O: the upload of the NEXT configuration can run on a copy stream while the current one is being
// swept.  lsm_stage_spins_host only copies h_in -> d_stage (it does not touch the lattice); lsm_set_spins(d_stage, ...)
// then installs it on the compute stream once the caller has ordered the two streams (event).
extern "C" int lsm_stage_spins_host(lsm_t *o, const int8_t *h_in, int8_t *d_stage, void *copy_stream)
{
    if (!o || !h_in || !d_stage) return LSM_ERR_ARG;
    CU(cudaMemcpyAsync(d_stage, h_in, (size_t)o->N, cudaMemcpyHostToDevice, (cudaStream_t)copy_stream));
    return LSM_OK;
}

extern "C" int lsm_set_temperature(lsm_t *o, double T)
{
    if (!o || !(T > 0.0) || !std::isfinite(T)) return LSM_ERR_ARG;
    o->T = T;
    build_tables(o);
    choose_kernel(o);
    return LSM_OK;
}

extern "C" int lsm_get_thresholds(lsm_t *o, uint64_t *out, int *count)
{
    if (!o || !count) return LSM_ERR_ARG;
    if (out) for (int i = 0; i < o->nthr; ++i) out[i] = o->thr[i];
    *count = o->nthr;
    return LSM_OK;
}

extern "C" int lsm_set_kernel(lsm_t *o, int family)
{
    if (!o || family < LSM_KERNEL_AUTO || family > LSM_KERNEL_BULK) return LSM_ERR_ARG;
    if (family == LSM_KERNEL_TILED && !tiled_supported(o->lat, o->model, o->tiled)) return LSM_ERR_UNSUPPORTED;
    if (family == LSM_KERNEL_RESIDENT) return LSM_ERR_UNSUPPORTED;      // removed in round 3: superseded by the slab family
    if (family == LSM_KERNEL_SMALL && !small_plan(o->lat, o->model, o->tiled, &o->small, true)) return LSM_ERR_UNSUPPORTED;
    if (family == LSM_KERNEL_SLAB && !slab_plan(o->lat, o->model, o->tiled, o->slab_depth, &o->slab)) return LSM_ERR_UNSUPPORTED;
    if (family == LSM_KERNEL_BULK && !tiled_bulk_supported(o->lat, o->model, o->tiled)) return LSM_ERR_UNSUPPORTED;
    o->kernel_pref = family;
    choose_kernel(o);
    return LSM_OK;
}

extern "C" int lsm_set_temporal_depth(lsm_t *o, int depth)
{
    if (!o || depth < 0) return LSM_ERR_ARG;
    if (depth > slab_depth_max(o->dims, o->L, o->model)) return LSM_ERR_UNSUPPORTED;
    o->slab_depth = depth;
    choose_kernel(o);
    return LSM_OK;
}

extern "C" int lsm_get_temporal_depth(lsm_t *o, int *depth)
{
    if (!o || !depth) return LSM_ERR_ARG;
    *depth = o->kernel_in_use == LSM_KERNEL_SLAB ? o->slab.D : 0;
    return LSM_OK;
}

extern "C" int lsm_get_kernel(lsm_t *o, int *family)
{
    if (!o || !family) return LSM_ERR_ARG;
    *family = o->kernel_in_use;
    return LSM_OK;
}

extern "C" int lsm_get_launch_count(lsm_t *o, uint64_t *n)
{
    if (!o || !n) return LSM_ERR_ARG;
    *n = o->launches;
    return LSM_OK;
}

// ---------------------------------------------------------------------------- derived doubles
extern "C" int lsm_binder_u4(const int64_t *obs, int64_t n, double *U4)
{
    if (!obs || !U4 || n <= 0) return LSM_ERR_ARG;
    unsigned __int128 s2 = 0, s4 = 0;
    for (int64_t k = 0; k < n; ++k) {
        __int128 m = obs[2 * k + 1];
        unsigned __int128 m2 = (unsigned __int128)(m * m);
        s2 += m2;
        s4 += m2 * m2;
    }
    if (s2 == 0) return LSM_ERR_ARG;
    long double a = (long double)s4 * (long double)n, b = 3.0L * (long double)s2 * (long double)s2;
    *U4 = (double)(1.0L - a / b);
    return LSM_OK;
}

extern "C" int lsm_heat_capacity(const int64_t *obs, int64_t n, int64_t N, double J, double h, double T, double *C)
{
    if (!obs || !C || n <= 0 || N <= 0 || !(T > 0.0)) return LSM_ERR_ARG;
    long double mean = 0.0L;
    for (int64_t k = 0; k < n; ++k) mean += -(long double)J * obs[2 * k] - (long double)h * obs[2 * k + 1];
    mean /= (long double)n;
    long double var = 0.0L;
    for (int64_t k = 0; k < n; ++k) {
        long double e = -(long double)J * obs[2 * k] - (long double)h * obs[2 * k + 1] - mean;
        var += e * e;
    }
    var /= (long double)n;
    *C = (double)(var / ((long double)N * (long double)T * (long double)T));
    return LSM_OK;
}

extern "C" int lsm_series_means(const int64_t *obs, int64_t n, int64_t N, double J, double h, double *e, double *abs_m)
{
    if (!obs || n <= 0 || N <= 0) return LSM_ERR_ARG;
    __int128 sB = 0, sM = 0, sA = 0;
    for (int64_t k = 0; k < n; ++k) {
        sB += obs[2 * k];
        sM += obs[2 * k + 1];
        sA += obs[2 * k + 1] < 0 ? -(__int128)obs[2 * k + 1] : (__int128)obs[2 * k + 1];
    }
    const long double den = (long double)n * (long double)N;
    if (e) *e = (double)((-(long double)J * (long double)sB - (long double)h * (long double)sM) / den);
    if (abs_m) *abs_m = (double)((long double)sA / den);
    return LSM_OK;
}

extern "C" int lsm_phi(int64_t overlap, int64_t N, double c, double *phi)
{
    if (!phi || N <= 0) return LSM_ERR_ARG;
    double q = (2.0 * c - 1.0) * (2.0 * c - 1.0);
    if (q >= 1.0) return LSM_ERR_ARG;
    *phi = ((double)overlap / (double)N - q) / (1.0 - q);
    return LSM_OK;
}

extern "C" int lsm_persistence_fraction(int64_t never_changed, int64_t N, double *P)
{
    if (!P || N <= 0) return LSM_ERR_ARG;
    *P = (double)never_changed / (double)N;
    return LSM_OK;
}

// ---------------------------------------------------------------------------- test hooks
extern "C" int lsm_philox_device(const uint32_t *d_ck, uint32_t *d_out, int64_t n, void *stream)
{
    if (n < 0 || ((!d_ck || !d_out) && n > 0)) return LSM_ERR_ARG;
    CU(launch_philox_device(d_ck, d_out, n, (cudaStream_t)stream));
    return LSM_OK;
}

extern "C" int lsm_philox_throughput(int blocks, int calls, uint32_t *d_sink, void *stream)
{
    if (blocks <= 0 || calls < 0 || !d_sink) return LSM_ERR_ARG;
    CU(launch_philox_throughput(blocks, calls, d_sink, (cudaStream_t)stream));
    return LSM_OK;
}

extern "C" const char *lsm_strerror(int code)
{
    switch (code) {
    case LSM_OK: return "ok";
    case LSM_ERR_ARG: return "invalid argument";
    case LSM_ERR_UNSUPPORTED: return "unsupported model / lattice / kernel combination";
    case LSM_ERR_CUDA: return "CUDA runtime error (see lsm_last_cuda_error)";
    case LSM_ERR_WORKSPACE: return "workspace too small or misaligned";
    case LSM_ERR_STATE: return "tracking is off, or the replicas of a batch are out of lockstep";
    case LSM_ERR_LIMIT: return "n exceeds LSM_NOALLOC_MAX_SWEEPS, the capacity of the library's built-in device scratch";
    default: return "unknown error code";
    }
}

extern "C" const char *lsm_last_cuda_error(void) { return g_cuda_err.c_str(); }
