// rflbm_lattice.cuh — compile-time D3Q27 tables of the CUDA path.
//
// PAPER.md:70-77 (Table I) and :172-202 (Table II).  Everything here is constexpr so that, after full
// unrolling, the tables fold into immediates: nothing is read from memory at run time.
//
// Internal population order ("lex"): q = (cx+1) + 3*(cy+1) + 9*(cz+1), so opp(q) = 26 - q.
// The boundary (include/rflbm.h) uses the canonical order R1; canon_c* and lex_of map between the two.
#pragma once
#include <cstdint>

namespace rflbm_dev {

constexpr int Q = 27;

// canonical index -> velocity (R1).  Tables live inside constexpr functions (namespace-scope constexpr arrays
// cannot be referenced from device code); with constant arguments after unrolling they fold to immediates.
__host__ __device__ constexpr int canon_cx(int i)
{
    constexpr int t[Q] = {0, 1, -1, 0, 0, 0, 0, 1, 1, -1, -1, 1, 1, -1, -1, 0, 0, 0, 0, 1, 1, 1, 1, -1, -1, -1, -1};
    return t[i];
}
__host__ __device__ constexpr int canon_cy(int i)
{
    constexpr int t[Q] = {0, 0, 0, 1, -1, 0, 0, 1, -1, 1, -1, 0, 0, 0, 0, 1, 1, -1, -1, 1, 1, -1, -1, 1, 1, -1, -1};
    return t[i];
}
__host__ __device__ constexpr int canon_cz(int i)
{
    constexpr int t[Q] = {0, 0, 0, 0, 0, 1, -1, 0, 0, 0, 0, 1, -1, 1, -1, 1, -1, 1, -1, 1, -1, 1, -1, 1, -1, 1, -1};
    return t[i];
}

__host__ __device__ constexpr int lex_of(int cx, int cy, int cz) { return (cx + 1) + 3 * (cy + 1) + 9 * (cz + 1); }
__host__ __device__ constexpr int lex_of_canon(int i) { return lex_of(canon_cx(i), canon_cy(i), canon_cz(i)); }
// canonical index of the velocity with lex index q
__host__ __device__ constexpr int canon_of_lex(int q)
{
    for (int i = 0; i < Q; ++i)
        if (lex_of_canon(i) == q) return i;
    return -1;
}

// Hermite exponents (p,q,r) of mode k in the order of Table II (rows 23, 24, 26 by position, R2)
__host__ __device__ constexpr int mode_p(int k)
{
    constexpr int t[Q] = {0, 1, 0, 0, 2, 0, 0, 1, 1, 0, 2, 2, 1, 1, 0, 0, 1, 2, 2, 0, 1, 1, 2, 2, 2, 1, 2};
    return t[k];
}
__host__ __device__ constexpr int mode_q(int k)
{
    constexpr int t[Q] = {0, 0, 1, 0, 0, 2, 0, 1, 0, 1, 1, 0, 2, 0, 1, 2, 1, 2, 0, 2, 1, 2, 1, 1, 2, 2, 2};
    return t[k];
}
__host__ __device__ constexpr int mode_r(int k)
{
    constexpr int t[Q] = {0, 0, 0, 1, 0, 0, 2, 0, 1, 1, 0, 1, 0, 2, 2, 1, 1, 0, 2, 2, 2, 1, 1, 2, 1, 2, 2};
    return t[k];
}

// 1-D weights (Table I factorises: w_i = w1(cx) w1(cy) w1(cz), w1(0) = 2/3, w1(+-1) = 1/6)
// 1-D Hermite norms beta_p = sum_c w1(c) H_p(c)^2 = (1, 1/3, 2/9); b_k = beta_p beta_q beta_r (Eq.5, Eq.22)
constexpr double SQRT2 = 1.4142135623730950488016887242097;
constexpr double SQRT3 = 1.7320508075688772935274463415059;
// n_p = 1/sqrt(beta_p): (1, sqrt3, 3/sqrt2)
constexpr double NRM1 = SQRT3;
constexpr double NRM2 = 3.0 / SQRT2;

}  // namespace rflbm_dev
