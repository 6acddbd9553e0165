// rflbm_rng.cuh — counter-based random numbers of the step kernel (R8).
//
// "r_k is a standard normal random variable"; generator and mapping are this build's reading:
// Philox4x32-10 (Salmon et al., SC'11), key = (seed lo, seed hi), counter = (site, t>>32, t&0xffffffff, call),
// 6 calls per site and step -> 24 words -> 12 Box-Muller pairs -> the 23 normals of modes k = 4..26.
#pragma once
#include <cstdint>

#include "rflbm_fastmath.cuh"

namespace rflbm_dev {

struct PhiloxKeys {
    uint32_t k0[10];  // round keys key0 + r*0x9E3779B9 (precomputed on the host: uniform over the grid)
    uint32_t k1[10];  // key1 + r*0xBB67AE85
};

__host__ inline PhiloxKeys make_philox_keys(uint64_t seed)
{
    PhiloxKeys k;
    uint32_t a = (uint32_t)(seed & 0xFFFFFFFFu), b = (uint32_t)(seed >> 32);
    for (int r = 0; r < 10; ++r) {
        k.k0[r] = a;
        k.k1[r] = b;
        a += 0x9E3779B9u;
        b += 0xBB67AE85u;
    }
    return k;
}

// one Philox4x32-10 block; 2 IMAD.WIDE.U32 + 2 LOP3 per round
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, const PhiloxKeys& key,
                                              uint32_t (&out)[4])
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        const uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ key.k0[r];
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ key.k1[r];
        c1 = (uint32_t)p1;
        c3 = (uint32_t)p0;
        c0 = n0;
        c2 = n2;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// Box-Muller on two words.  fp64: 32-bit uniforms (x+0.5)/2^32 (exact in double, never 0 or 1); evaluated by the
// table-driven branch-free routines of rflbm_fastmath.cuh (lg/sc: the tables, staged in shared memory).
__device__ __forceinline__ void normal_pair(uint32_t xa, uint32_t xb, const f64x2* lg, const f64x2* sc, double& z0,
                                            double& z1)
{
    normal_pair_fast(xa, xb, lg, sc, z0, z1);
}

// fp32 mode (R14): 24-bit uniforms ((x>>8)+0.5)/2^24, float arithmetic, accurate (non fast-math) functions.
__device__ __forceinline__ void normal_pair(uint32_t xa, uint32_t xb, const f64x2*, const f64x2*, float& z0, float& z1)
{
    const float ua = ((float)(xa >> 8) + 0.5f) * (1.0f / 16777216.0f);
    const float two_ub = ((float)(xb >> 8) + 0.5f) * (1.0f / 8388608.0f);
    const float R = sqrtf(-2.0f * logf(ua));
    float s, c;
    sincospif(two_ub, &s, &c);
    z0 = R * c;
    z1 = R * s;
}

}  // namespace rflbm_dev
