// pipe_probe.cu -- integer-pipe microbenchmarks (NOT part of liblsm.so: built as libpipe_probe.so, loaded only by
// `python bench.py --pipe-probe`).  Register-only instruction streams whose timing gives the measured integer-issue
// rate that DESIGN.md 6 uses as the "alu" roofline of the sweep kernels.
#include <cstdint>
#include <cuda_runtime.h>

namespace {

constexpr uint32_t PHILOX_M0 = 0xD2511F53u, PHILOX_M1 = 0xCD9E8D57u;
constexpr uint32_t PHILOX_W0 = 0x9E3779B9u, PHILOX_W1 = 0xBB67AE85u;

__device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        unsigned long long p0 = (unsigned long long)PHILOX_M0 * c0;
        unsigned long long p1 = (unsigned long long)PHILOX_M1 * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        c1 = (uint32_t)p1;
        c3 = (uint32_t)p0;
        c0 = n0;
        c2 = n2;
        k0 += PHILOX_W0;
        k1 += PHILOX_W1;
    }
    return make_uint4(c0, c1, c2, c3);
}

// Integer-pipe probe: register-only instruction streams whose timing shows how the ALU
// pipe (LOP3/IADD3/ISETP/PRMT) and the FMA-heavy pipe (IMAD, IMAD.WIDE) share issue on this GPU.
//   mode 0: 16 LOP3            1: 8 IMAD (32-bit)          2: 8 IMAD.WIDE.U32 (+8 adds)
//        3: 8 IMAD + 16 LOP3   4: 4 Philox calls           5/6/7: 4 Philox calls + 80/160/240 LOP3
//        8/9/10: 4 Philox calls + 80 IMAD + 0/80/160 LOP3
//        11: 8 mul.hi + 8 mul.lo (separate instructions instead of one wide multiply)
//        12/13: 4 Philox calls with every wide multiply split into mul.hi + mul.lo, + 0/80 LOP3
// per loop iteration and thread.
#define LSM_PROBE_LOP(a, b, c) a = (a ^ b) & (c | 0x55555555u);
__device__ __forceinline__ uint32_t mulhi_asm(uint32_t a, uint32_t b)
{
    uint32_t r;
    asm volatile("mul.hi.u32 %0, %1, %2;" : "=r"(r) : "r"(a), "r"(b));
    return r;
}
__device__ __forceinline__ uint32_t mullo_asm(uint32_t a, uint32_t b)
{
    uint32_t r;
    asm volatile("mul.lo.u32 %0, %1, %2;" : "=r"(r) : "r"(a), "r"(b));
    return r;
}
__device__ __forceinline__ uint4 philox4x32_10_split(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        uint32_t n0 = mulhi_asm(PHILOX_M1, c2) ^ c1 ^ k0;
        uint32_t n2 = mulhi_asm(PHILOX_M0, c0) ^ c3 ^ k1;
        c1 = mullo_asm(PHILOX_M1, c2);
        c3 = mullo_asm(PHILOX_M0, c0);
        c0 = n0;
        c2 = n2;
        k0 += PHILOX_W0;
        k1 += PHILOX_W1;
    }
    return make_uint4(c0, c1, c2, c3);
}
template <int MODE>
__global__ void __launch_bounds__(256) k_pipe_probe(int iters, uint32_t *__restrict__ sink, uint32_t k0, uint32_t k1)
{
    uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x;
    uint32_t a[8], b[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) { a[i] = (tid * (i + 1)) ^ k0; b[i] = tid + i * 77u + k1; }
    uint32_t acc = 0;
    constexpr int NLOP = MODE == 0 ? 8 : MODE == 3 ? 8 : MODE == 5 ? 40 : MODE == 6 ? 80 : MODE == 7 ? 120 : MODE == 9 ? 40 : MODE == 10 ? 80 : MODE == 13 ? 40 : 0;
    constexpr int NIMAD = (MODE >= 8 && MODE <= 10) ? 80 : 0;   // modes 8-10: 4 Philox calls + 80 IMAD (+ 80 / 160 LOP3)
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
        if (MODE == 1 || MODE == 3) {
#pragma unroll
            for (int i = 0; i < 8; ++i) a[i] = a[i] * 0x9E3779B9u + b[i];
        }
        if (MODE == 2) {
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                unsigned long long p = (unsigned long long)a[i] * PHILOX_M0;
                a[i] = (uint32_t)(p >> 32) + (uint32_t)p;
            }
        }
        if (MODE >= 4 && MODE <= 10) {
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                uint4 r = philox4x32_10(tid * 4u + c, 0u, (uint32_t)it, 1u, k0, k1);
                acc ^= r.x ^ r.y ^ r.z ^ r.w;
            }
        }
        if (MODE == 11) {
#pragma unroll
            for (int i = 0; i < 8; ++i) a[i] = mulhi_asm(a[i], PHILOX_M0) + mullo_asm(b[i], PHILOX_M1);
        }
        if (MODE >= 12) {
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                uint4 r = philox4x32_10_split(tid * 4u + c, 0u, (uint32_t)it, 1u, k0, k1);
                acc ^= r.x ^ r.y ^ r.z ^ r.w;
            }
        }
#pragma unroll
        for (int i = 0; i < NIMAD; ++i) a[i & 7] = a[i & 7] * 0x9E3779B9u + a[(i + 3) & 7];
#pragma unroll
        for (int i = 0; i < NLOP; ++i) LSM_PROBE_LOP(b[i & 7], b[(i + 1) & 7], b[(i + 3) & 7])
    }
#pragma unroll
    for (int i = 0; i < 8; ++i) acc ^= a[i] ^ b[i];
    sink[tid] = acc;
}

static cudaError_t launch_pipe_probe(int mode, int blocks, int iters, uint32_t *d_sink, cudaStream_t s)
{
    const uint32_t k0 = 0x1234567u, k1 = 0x89abcdefu;
    switch (mode) {
    case 0: k_pipe_probe<0><<<blocks, 256, 0, s>>>(iters, d_sink, k0, k1); break;
    case 1: k_pipe_probe<1><<<blocks, 256, 0, s>>>(iters, d_sink, k0, k1); break;
    case 2: k_pipe_probe<2><<<blocks, 256, 0, s>>>(iters, d_sink, k0, k1); break;
    case 3: k_pipe_probe<3><<<blocks, 256, 0, s>>>(iters, d_sink, k0, k1); break;
    case 4: k_pipe_probe<4><<<blocks, 256, 0, s>>>(iters, d_sink, k0, k1); break;
    case 5: k_pipe_probe<5><<<blocks, 256, 0, s>>>(iters, d_sink, k0, k1); break;
    case 6: k_pipe_probe<6><<<blocks, 256, 0, s>>>(iters, d_sink, k0, k1); break;
    case 7: k_pipe_probe<7><<<blocks, 256, 0, s>>>(iters, d_sink, k0, k1); break;
    case 8: k_pipe_probe<8><<<blocks, 256, 0, s>>>(iters, d_sink, k0, k1); break;
    case 9: k_pipe_probe<9><<<blocks, 256, 0, s>>>(iters, d_sink, k0, k1); break;
    case 10: k_pipe_probe<10><<<blocks, 256, 0, s>>>(iters, d_sink, k0, k1); break;
    case 11: k_pipe_probe<11><<<blocks, 256, 0, s>>>(iters, d_sink, k0, k1); break;
    case 12: k_pipe_probe<12><<<blocks, 256, 0, s>>>(iters, d_sink, k0, k1); break;
    case 13: k_pipe_probe<13><<<blocks, 256, 0, s>>>(iters, d_sink, k0, k1); break;
    default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

}  // namespace

// mode 0..13 (see above); `blocks` x 256 threads run `iters` iterations and write one word each to d_sink[blocks*256]
// (device).  Returns 0 or the cudaError_t of the launch.
extern "C" int pipe_probe_run(int mode, int blocks, int iters, uint32_t *d_sink, void *stream)
{
    if (mode < 0 || mode > 13 || blocks <= 0 || iters < 0 || !d_sink) return -1;
    return (int)launch_pipe_probe(mode, blocks, iters, d_sink, (cudaStream_t)stream);
}
