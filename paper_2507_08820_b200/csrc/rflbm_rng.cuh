// rflbm_rng.cuh — counter-based random numbers of the step kernel (R8).
//
// "r_k is a standard normal random variable"; generator and mapping are this build's reading:
// Philox4x32-10 (Salmon et al., SC'11), key = (seed lo, seed hi), counter = (site, t>>32, t&0xffffffff, call),
// 6 calls per site and step -> 24 words -> 12 Box-Muller pairs -> the 23 normals of modes k = 4..26.
//
// The six calls of a site differ only in counter word 3, and two of the four counter words (t_hi, t_lo) and the
// key are the same for the whole grid.  Following the data flow of the first three rounds by hand:
//   round 1: M1*t_lo is grid-uniform, M0*site is shared by the six calls  -> one XOR per call
//   round 2: M0*(uniform) is grid-uniform                                  -> one IMAD.WIDE + one XOR per call (+1 shared XOR)
//   round 3: M1*(shared)  is shared by the six calls                       -> one IMAD.WIDE + two XOR per call (+1 shared IMAD)
// so the host precomputes the uniform pieces once per step (PhiloxStep) and a site spends 34 instead of 40
// integer instructions per call.  The words are bit-identical to the textbook loop (philox4x32_10 below, which
// the debug kernel cross-checks against in tests/test_gpu_parity.py).
#pragma once
#include <cstdint>

#include "rflbm_fastmath.cuh"

namespace rflbm_dev {

constexpr uint32_t PHILOX_M0 = 0xD2511F53u, PHILOX_M1 = 0xCD9E8D57u;
constexpr uint32_t PHILOX_W0 = 0x9E3779B9u, PHILOX_W1 = 0xBB67AE85u;

struct PhiloxStep {
    uint32_t k0[10];   // round keys key0 + r*W0
    uint32_t k1[10];   // key1 + r*W1
    uint32_t r1x[6];   // call ^ k1[0]                                  (round 1: n2 = hi(M0*site) ^ r1x[call])
    uint32_t r2_c0;    // round-2 c0 = hi(M1*t_lo) ^ t_hi ^ k0[0]       (only its products are used below)
    uint32_t r2_n0x;   // lo(M1*t_lo) ^ k0[1]                           (round 2: n0 = hi(M1*c2) ^ r2_n0x)
    uint32_t r2_n2x;   // hi(M0*r2_c0) ^ k1[1]                          (round 2: n2 = lo(M0*site) ^ r2_n2x)
    uint32_t r3_n2x;   // lo(M0*r2_c0) ^ k1[2]                          (round 3: n2 = hi(M0*c0) ^ r3_n2x)
};

__host__ inline PhiloxStep make_philox_step(uint64_t seed, uint64_t t)
{
    PhiloxStep s;
    uint32_t a = (uint32_t)(seed & 0xFFFFFFFFu), b = (uint32_t)(seed >> 32);
    for (int r = 0; r < 10; ++r) {
        s.k0[r] = a;
        s.k1[r] = b;
        a += PHILOX_W0;
        b += PHILOX_W1;
    }
    const uint32_t t_hi = (uint32_t)(t >> 32), t_lo = (uint32_t)(t & 0xFFFFFFFFu);
    const uint64_t p1 = (uint64_t)PHILOX_M1 * t_lo;
    for (uint32_t q = 0; q < 6; ++q) s.r1x[q] = q ^ s.k1[0];
    s.r2_c0 = (uint32_t)(p1 >> 32) ^ t_hi ^ s.k0[0];
    s.r2_n0x = (uint32_t)p1 ^ s.k0[1];
    const uint64_t p0 = (uint64_t)PHILOX_M0 * s.r2_c0;
    s.r2_n2x = (uint32_t)(p0 >> 32) ^ s.k1[1];
    s.r3_n2x = (uint32_t)p0 ^ s.k1[2];
    return s;
}

// textbook Philox4x32-10 block (test hook only): 2 IMAD.WIDE.U32 + 2 LOP3 per round
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, const PhiloxStep& key,
                                              uint32_t (&out)[4])
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)PHILOX_M0 * (uint64_t)c0;
        const uint64_t p1 = (uint64_t)PHILOX_M1 * (uint64_t)c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ key.k0[r];
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ key.k1[r];
        c1 = (uint32_t)p1;
        c3 = (uint32_t)p0;
        c0 = n0;
        c2 = n2;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// The part of the six calls that does not depend on the call index (see the header comment).
struct PhiloxSite {
    uint32_t p0_hi;    // hi(M0*site)
    uint32_t r3_c2;    // round-3 c2 = lo(M0*site) ^ r2_n2x
    uint32_t r3_p1_hi, r3_p1_lo;   // M1 * r3_c2
};

__device__ __forceinline__ PhiloxSite philox_site(uint32_t site, const PhiloxStep& S)
{
    PhiloxSite P;
    const uint64_t p0 = (uint64_t)PHILOX_M0 * (uint64_t)site;
    P.p0_hi = (uint32_t)(p0 >> 32);
    P.r3_c2 = (uint32_t)p0 ^ S.r2_n2x;
    const uint64_t p1 = (uint64_t)PHILOX_M1 * (uint64_t)P.r3_c2;
    P.r3_p1_hi = (uint32_t)(p1 >> 32);
    P.r3_p1_lo = (uint32_t)p1;
    return P;
}

// call `call` (0..5) of the site: identical words to philox4x32_10(site, t_hi, t_lo, call)
__device__ __forceinline__ void philox_call(const PhiloxSite& P, const PhiloxStep& S, int call, uint32_t (&out)[4])
{
    // round 1 -> (c0, c1, c2, c3) = (uniform, uniform, n2, lo(M0*site))
    const uint32_t r2_c2 = P.p0_hi ^ S.r1x[call];
    // round 2
    const uint64_t q1 = (uint64_t)PHILOX_M1 * (uint64_t)r2_c2;
    uint32_t c0 = (uint32_t)(q1 >> 32) ^ S.r2_n0x;
    uint32_t c1 = (uint32_t)q1;
    // round 3: c2 = P.r3_c2 (shared), c3 = lo(M0*r2_c0) (uniform, folded into r3_n2x)
    const uint64_t q0 = (uint64_t)PHILOX_M0 * (uint64_t)c0;
    c0 = P.r3_p1_hi ^ c1 ^ S.k0[2];
    uint32_t c2 = (uint32_t)(q0 >> 32) ^ S.r3_n2x;
    c1 = P.r3_p1_lo;
    uint32_t c3 = (uint32_t)q0;
#pragma unroll
    for (int r = 3; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)PHILOX_M0 * (uint64_t)c0;
        const uint64_t p1 = (uint64_t)PHILOX_M1 * (uint64_t)c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ S.k0[r];
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ S.k1[r];
        c1 = (uint32_t)p1;
        c3 = (uint32_t)p0;
        c0 = n0;
        c2 = n2;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// Box-Muller on two words, polar form: the normals are R*cs (first) and R*sn (second).  fp64: 32-bit uniforms
// (x+0.5)/2^32 (exact in double, never 0 or 1); evaluated by the table-driven branch-free routines of
// rflbm_fastmath.cuh (lg/sc: the tables, staged in shared memory).
__device__ __forceinline__ void normal_polar(uint32_t xa, uint32_t xb, const f64x2* lg, const f64x2* sc, double& R,
                                             double& sn, double& cs)
{
    normal_polar_fast(xa, xb, lg, sc, R, sn, cs);
}

// fp32 mode (R14): 24-bit uniforms ((x>>8)+0.5)/2^24, float arithmetic on the special-function unit.
// The fp32 path owes the oracle 1e-5 on the populations (BASELINE.json), i.e. ~1e-4 on a normal; the hardware
// approximations are far inside that and keep the fp32 kernel on the HBM roofline (the accurate logf / sqrtf /
// sincospif cost ~45 instructions per pair and halved the throughput, profiles/r01d):
//   -2 ln u = (-2 ln 2) lg2.approx(u)   (MUFU.LG2, abs. error < 2^-22 on lg2, u in [2^-25, 1))
//   (for u within 2^-10 of 1 the series 2v + v^2 of -2 ln(1-v), v = 1-u exact, replaces it: R error < 1e-5 everywhere)
//   R = sqrt.approx(W)                   (MUFU.SQRT, 2^-23 relative; W >= 5.9e-8 > 0)
//   sin, cos(2 pi u) = -sin, -cos(2 pi u - pi), argument in (-pi, pi) where MUFU.SIN/COS are good to 2^-21.4
__device__ __forceinline__ void normal_polar(uint32_t xa, uint32_t xb, const f64x2*, const f64x2*, float& R, float& sn,
                                             float& cs)
{
    const uint32_t k = xa >> 8;
    const float ua = fmaf((float)k, 1.0f / 16777216.0f, 1.0f / 33554432.0f);   // (k + 1/2)/2^24, one rounding; 1.0f for the last k: handled below
    float l2;
    asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(l2) : "f"(ua));        // ua is a normal number: no denormal scaling needed
    float W = -1.3862943611198906f * l2;
    if (k >= 16777216u - 16384u) {                                  // u within 2^-10 of 1 (3 % of the warps): the
        const float v = ((float)(16777216u - k) - 0.5f) * (1.0f / 16777216.0f);   // absolute error of lg2 would show,
        W = fmaf(v, v, 2.0f * v);                                   // so -2 ln(1-v) = 2v + v^2 + O(v^3 < 1e-9), v exact
    }
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(R) : "f"(W));         // MUFU.SQRT, relative error 2^-23; W >= 5.9e-8 > 0
    // 2 pi u - pi = 2 pi ((xb>>8) - 2^23 + 0.5) / 2^24, exact integer part
    constexpr float TWO_PI_24 = 6.283185307179586f / 16777216.0f;
    const float th = fmaf((float)((int)(xb >> 8) - 8388608), TWO_PI_24, 0.5f * TWO_PI_24);
    float s, c;
    __sincosf(th, &s, &c);
    sn = -s;
    cs = -c;
}

template <typename real>
__device__ __forceinline__ void normal_pair(uint32_t xa, uint32_t xb, const f64x2* lg, const f64x2* sc, real& z0, real& z1)
{
    real R, sn, cs;
    normal_polar(xa, xb, lg, sc, R, sn, cs);
    z0 = R * cs;
    z1 = R * sn;
}

}  // namespace rflbm_dev
