// device_common.cuh -- shared device helpers of libgcmcrt (sm_100a).
// Philox4x32-10 (A3), the zeta mapping, approximate MUFU wrappers and warp utilities.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

// Bounds and state checks of the checked build (python -m paper_2110_15640_b200.build --checked: -DGCMCRT_CHECKED, a
// library of its own, libgcmcrt_checked.so): compute-sanitizer is not available on the GPU pool this was built on, so
// the indices the kernels compute themselves -- cells, columns, shells, event slots, sort keys, list slots, bins -- are
// asserted instead; a failed check prints its source line and traps, which the host sees as GCMCRT_E_CUDA.
#ifdef GCMCRT_CHECKED
#include <cstdio>
#define GCMCRT_CHECK(c)                                                                      \
    do {                                                                                     \
        if (!(c)) { printf("GCMCRT_CHECK failed: %s  (%s:%d)\n", #c, __FILE__, __LINE__); __trap(); } \
    } while (0)
#else
#define GCMCRT_CHECK(c) ((void)0)
#endif

namespace gcmcrt {

constexpr float kPi = 3.14159265358979323846f;
#define kInf (__int_as_float(0x7f800000))
constexpr unsigned kFullMask = 0xffffffffu;

// ---- MUFU wrappers: the march loop wants single-instruction sqrt / rcp, not the IEEE sequences ----
__device__ __forceinline__ float sqrt_approx(float x)
{
    float y;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float rcp_approx(float x)
{
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

__device__ __forceinline__ void prefetch_l1(const void* p)
{
    asm volatile("prefetch.global.L1 [%0];" ::"l"(p));
}

// ---- A3: Philox4x32-10 (Salmon et al. 2011).  key = (channel, packet), counter = (event, purpose, seed) ----
struct Philox4 {
    uint32_t x, y, z, w;
};

__device__ __forceinline__ Philox4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0,
                                                 uint32_t k1)
{
#pragma unroll
    for (int round = 0; round < 10; ++round) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        const uint32_t n0 = hi1 ^ c1 ^ k0;
        const uint32_t n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    return Philox4{c0, c1, c2, c3};
}

// zeta = ((u >> 9) + 0.5) 2^-23: in (0,1), exactly representable in fp32 (2k+1 < 2^24).
__device__ __forceinline__ float u32_to_zeta(uint32_t u)
{
    return (static_cast<float>(u >> 9) + 0.5f) * (1.0f / 8388608.0f);
}

struct Zeta4 {
    float z0, z1, z2, z3;
};

__device__ __forceinline__ Zeta4 zeta_block(uint64_t seed, uint32_t chan, uint32_t pkt, uint32_t event, uint32_t purpose)
{
    const Philox4 r = philox4x32_10(event, purpose, static_cast<uint32_t>(seed), static_cast<uint32_t>(seed >> 32),
                                    chan, pkt);
    return Zeta4{u32_to_zeta(r.x), u32_to_zeta(r.y), u32_to_zeta(r.z), u32_to_zeta(r.w)};
}

// ---- exact 64-bit division by a run constant: q = floor(n / d) with m = floor(2^64 / d) computed on the host
// (m = 2^64 - 1 for d = 1).  n m / 2^64 lies in (n/d - 1, n/d], so one correction step makes it exact.
__device__ __forceinline__ unsigned long long div_magic(unsigned long long n, unsigned long long d, unsigned long long m)
{
    unsigned long long q = __umul64hi(n, m);
    if (n - q * d >= d) ++q;
    return q;
}

// ---- warp helpers ----
__device__ __forceinline__ int lane_id() { return threadIdx.x & 31; }
__device__ __forceinline__ int rank_in_mask(unsigned mask) { return __popc(mask & ((1u << lane_id()) - 1u)); }

__device__ __forceinline__ unsigned long long warp_sum_u64(unsigned long long v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(kFullMask, v, o);
    return v;
}
__device__ __forceinline__ double warp_sum_f64(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(kFullMask, v, o);
    return v;
}

}  // namespace gcmcrt
