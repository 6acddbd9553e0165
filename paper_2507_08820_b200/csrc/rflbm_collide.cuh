// rflbm_collide.cuh — the per-site Reg-FLBM collision, registers only (one thread = one lattice site).
//
// Implements Eq.24 with omega_g = 1 (:215):
//     f*_i = f_i^(0) + (1-omega_h) f_i^(1,h) + w_i sum_k e_ki phi_k r_k / b_k
// as ONE back-transform (Eq.10 :105) of the post-collision modes
//     M_k = rho ux^p uy^q uz^r                     (Eq.20 :160, all 27 modes)
//         + (1-omega_h) a_1,ab      for k = 4..9   (Eq.19 :153, Eq.26 :227)
//         + phi_k r_k               for k = 4..26  (Eq.8-9 :93-99)
//
// What differs from a literal reading (same real function, different operation order):
//   * D3Q27 is a tensor product, e_ki = H_p(cx) H_q(cy) H_r(cz), w_i = w1(cx) w1(cy) w1(cz), b_k = beta_p beta_q beta_r,
//     so both transforms are done separably (three passes of 3-point 1-D transforms) instead of 27x27.
//   * modes are carried SCALED, Ms[p][q][r] = M_k 2^-(number of non-zero exponents among p,q,r).  The 1-D
//     back-transform f(c) = w1(c) sum_p H_p(c) m_p / beta_p is f(0) = 2/3 m0 - m2, f(+-1) = m0/6 +- m1/2 + m2/2;
//     with m1, m2 pre-halved it costs 4 flops (e = m0/6 + m2s, f+- = e +- m1s, f0 = m0 - 2e) instead of 6, and
//     the scaling is free: the equilibrium becomes rho prod (1, u/2, u^2/2), the stress and noise coefficients
//     absorb it into constants.
//   * only the 10 moments of order <= 2 are needed from the incoming populations (ghost modes are rebuilt from
//     rho,u, not relaxed), so the forward transform is truncated.
#pragma once
#include "rflbm_lattice.cuh"
#include "rflbm_rng.cuh"

namespace rflbm_dev {

// noise amplitude classes: phi_k 2^-nnz / sqrt(rho) = sqrt(3 kT omega_k (2-omega_k)) prod_axis s_p with
// s = sqrt(beta_p) 2^-[p>0] = (1, sqrt3/6, sqrt2/6); a class is the multiset of exponents of the mode
enum { AMP_200 = 0, AMP_110, AMP_210, AMP_111, AMP_220, AMP_211, AMP_221, AMP_222, AMP_N };

__host__ __device__ constexpr int amp_class(int p, int q, int r)
{
    const int n1 = (p == 1) + (q == 1) + (r == 1), n2 = (p == 2) + (q == 2) + (r == 2);
    return (n2 == 1 && n1 == 0) ? AMP_200 : (n2 == 0 && n1 == 2) ? AMP_110 : (n2 == 1 && n1 == 1) ? AMP_210
         : (n2 == 0 && n1 == 3) ? AMP_111 : (n2 == 2 && n1 == 0) ? AMP_220 : (n2 == 1 && n1 == 2) ? AMP_211
         : (n2 == 2 && n1 == 1) ? AMP_221 : AMP_222;
}

// Geometry of one handle.  Logical lattice nx x ny x nz ("owned" layers); the internal buffers
// have a row pitch px >= nx (rows 16-byte aligned so that every lattice can take the TMA kernel) and, in slab mode
// (rflbm_set_slab), one ghost layer below and above the owned layers.  Walls and the Philox site key use GLOBAL z.
struct Geom {
    int nx, ny;             // logical extent in x, y (periodic)
    int nz;                 // owned layers
    int nzs;                // layers in storage: nz, or nz + 2 in slab mode
    int z_lo;               // storage index of the first owned layer: 0, or 1 in slab mode
    int zc;                 // first owned layer this LAUNCH works on (0 unless rflbm_run_host pipelines z-chunks), grid.z counts from it
    int zg0;                // global z of storage layer 0: 0, or z0 - 1 in slab mode
    int nzg;                // global number of layers (= nz without a slab)
    int px;                 // elements between consecutive y rows of one population (27 x the padded row length)
    long long pxy;          // px * ny: elements between consecutive z layers
    long long QS;           // elements between consecutive populations of one site (the padded row length)
    long long N;            // nx * ny * nz: length of the canonical (boundary) arrays
};

template <typename real>
struct StepParams {
    Geom G;
    real half_omc;          // (1 - omega_h)/2
    real omc_g;             // 1 - omega_g (0 in the paper's final scheme, :215)
    real amp[AMP_N];        // noise amplitude per class (times sqrt(rho) at the site), Eq.9
    real gx, gy, gz;        // acceleration (R13)
    real force_stress;      // 1 - omega_h/2
    PhiloxStep rng;         // round keys and the grid-uniform part of the first Philox rounds for this step
    const f64x2* tables;    // device: log table [LOG_TABLE_N] then sin/cos table [SC_TABLE_N] (fp64 noise only)
};

// 1/x and sqrt(x) for x of order one (the density): approximate seed + Newton, no special cases
template <typename real> __device__ __forceinline__ real rcp_pos(real x);
template <> __device__ __forceinline__ double rcp_pos<double>(double x)
{
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));       // 2^-20
    double e = fma(-x, y, 1.0);
    y = fma(y, e, y);                                            // 2^-40
    e = fma(-x, y, 1.0);
    return fma(y, e, y);                                         // < 1 ulp
}
template <> __device__ __forceinline__ float rcp_pos<float>(float x) { return 1.0f / x; }
template <typename real> __device__ __forceinline__ real sqrt_rho(real x);
template <> __device__ __forceinline__ double sqrt_rho<double>(double x) { return sqrt_pos(x); }
template <> __device__ __forceinline__ float sqrt_rho<float>(float x) { return sqrtf(x); }

// conserved moments + raw second moments of g[cz+1][cy+1][cx+1] (Eq.2-3, and sum g c_a c_b for Eq.19)
template <typename real>
struct Moments10 {
    real rho, jx, jy, jz, pxx, pyy, pzz, pxy, pxz, pyz;
};

// Packed fp32 arithmetic (sm_100: FADD2 / FMUL2 / FFMA2 work on two floats in an aligned register pair).  The fp32
// kernel is issue bound, so the two places where the same operation runs on many independent values - the separable
// transforms - are written on pairs: the same operations in the same order as the scalar code (bit-identical results).
__device__ __forceinline__ unsigned long long f2_bits(float2 a) { return *reinterpret_cast<unsigned long long*>(&a); }
__device__ __forceinline__ float2 f2_from(unsigned long long a) { return *reinterpret_cast<float2*>(&a); }
__device__ __forceinline__ float2 add2(float2 a, float2 b)
{
    unsigned long long d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(f2_bits(a)), "l"(f2_bits(b)));
    return f2_from(d);
}
__device__ __forceinline__ float2 sub2(float2 a, float2 b)
{
    unsigned long long d;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(f2_bits(a)), "l"(f2_bits(b)));
    return f2_from(d);
}
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c)
{
    unsigned long long d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(f2_bits(a)), "l"(f2_bits(b)), "l"(f2_bits(c)));
    return f2_from(d);
}

// fp32: the x and y passes run on the pair (cz = -1, cz = +1), the cz = 0 plane on scalars; same sums as below
__device__ __forceinline__ Moments10<float> forward_moments(const float (&g)[3][3][3])
{
    float2 P0[3], P1[3], P2[3];     // [cy]: pair over c = 0, 2
    float S0[3], S1[3], S2[3];      // c = 1
#pragma unroll
    for (int b = 0; b < 3; ++b) {
        const float2 g0 = make_float2(g[0][b][0], g[2][b][0]), g1 = make_float2(g[0][b][1], g[2][b][1]),
                     g2 = make_float2(g[0][b][2], g[2][b][2]);
        P2[b] = add2(g2, g0);
        P1[b] = sub2(g2, g0);
        P0[b] = add2(P2[b], g1);
        S2[b] = g[1][b][2] + g[1][b][0];
        S1[b] = g[1][b][2] - g[1][b][0];
        S0[b] = S2[b] + g[1][b][1];
    }
    const float2 Y02 = add2(P0[2], P0[0]), Y01 = sub2(P0[2], P0[0]), Y00 = add2(Y02, P0[1]);
    const float2 Y10 = add2(add2(P1[2], P1[0]), P1[1]), Y11 = sub2(P1[2], P1[0]), Y20 = add2(add2(P2[2], P2[0]), P2[1]);
    const float y02 = S0[2] + S0[0], y01 = S0[2] - S0[0], y00 = y02 + S0[1];
    const float y10 = (S1[2] + S1[0]) + S1[1], y11 = S1[2] - S1[0], y20 = (S2[2] + S2[0]) + S2[1];
    Moments10<float> m;      // .x = plane c = 0, .y = plane c = 2
    m.pzz = Y00.y + Y00.x;
    m.jz = Y00.y - Y00.x;
    m.rho = m.pzz + y00;
    m.jy = (Y01.y + Y01.x) + y01;
    m.pyz = Y01.y - Y01.x;
    m.pyy = (Y02.y + Y02.x) + y02;
    m.jx = (Y10.y + Y10.x) + y10;
    m.pxz = Y10.y - Y10.x;
    m.pxy = (Y11.y + Y11.x) + y11;
    m.pxx = (Y20.y + Y20.x) + y20;
    return m;
}

template <typename real>
__device__ __forceinline__ Moments10<real> forward_moments(const real (&g)[3][3][3])
{
    // x pass: X0 = sum, X1 = first, X2 = second raw moment along x for every (cz,cy)
    real Y00[3], Y01[3], Y02[3], Y10[3], Y11[3], Y20[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        real X0[3], X1[3], X2[3];
#pragma unroll
        for (int b = 0; b < 3; ++b) {
            X2[b] = g[c][b][2] + g[c][b][0];
            X1[b] = g[c][b][2] - g[c][b][0];
            X0[b] = X2[b] + g[c][b][1];
        }
        // y pass (only what order <= 2 needs)
        Y02[c] = X0[2] + X0[0];
        Y01[c] = X0[2] - X0[0];
        Y00[c] = Y02[c] + X0[1];
        Y10[c] = (X1[2] + X1[0]) + X1[1];
        Y11[c] = X1[2] - X1[0];
        Y20[c] = (X2[2] + X2[0]) + X2[1];
    }
    Moments10<real> m;
    m.pzz = Y00[2] + Y00[0];
    m.jz = Y00[2] - Y00[0];
    m.rho = m.pzz + Y00[1];
    m.jy = (Y01[2] + Y01[0]) + Y01[1];
    m.pyz = Y01[2] - Y01[0];
    m.pyy = (Y02[2] + Y02[0]) + Y02[1];
    m.jx = (Y10[2] + Y10[0]) + Y10[1];
    m.pxz = Y10[2] - Y10[0];
    m.pxy = (Y11[2] + Y11[0]) + Y11[1];
    m.pxx = (Y20[2] + Y20[0]) + Y20[1];
    return m;
}

// full forward transform (Eq.4, separable): m[p][q][r] = sum_i H_p(cx) H_q(cy) H_r(cz) g_i, raw (unscaled) moments.
// 1-D: m0 = f- + f0 + f+, m1 = f+ - f-, m2 = (f+ + f-) - m0/3.  Needed by BGK-FLBM only (Eq.11).
template <typename real>
__device__ __forceinline__ void fwd1d(real fm, real f0, real fp, real& m0, real& m1, real& m2)
{
    const real s = fp + fm;
    m1 = fp - fm;
    m0 = s + f0;
    m2 = fma(real(-1.0 / 3.0), m0, s);
}

template <typename real>
__device__ __forceinline__ void forward_all(const real (&g)[3][3][3], real (&m)[3][3][3])
{
    real X[3][3][3];   // [cz][cy][p]
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int b = 0; b < 3; ++b) fwd1d(g[c][b][0], g[c][b][1], g[c][b][2], X[c][b][0], X[c][b][1], X[c][b][2]);
    real Y[3][3][3];   // [cz][q][p]
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int p = 0; p < 3; ++p) fwd1d(X[c][0][p], X[c][1][p], X[c][2][p], Y[c][0][p], Y[c][1][p], Y[c][2][p]);
#pragma unroll
    for (int q = 0; q < 3; ++q)
#pragma unroll
        for (int p = 0; p < 3; ++p) fwd1d(Y[0][q][p], Y[1][q][p], Y[2][q][p], m[p][q][0], m[p][q][1], m[p][q][2]);
}

// 1-D back-transform of (m0, m1/2, m2/2) -> values at c = -1, 0, +1 (see the header comment)
template <typename real>
__device__ __forceinline__ void back1d(real m0, real m1s, real m2s, real& fm, real& f0, real& fp)
{
    const real e = fma(real(1.0 / 6.0), m0, m2s);
    fp = e + m1s;
    fm = e - m1s;
    f0 = fma(real(-2.0), e, m0);
}

// Eq.10, separable: r -> cz, then q -> cy, then p -> cx
template <typename real>
__device__ __forceinline__ void back_transform(const real (&Ms)[3][3][3], real (&g)[3][3][3])
{
    real A[3][3][3];   // [p][q][cz]
#pragma unroll
    for (int p = 0; p < 3; ++p)
#pragma unroll
        for (int q = 0; q < 3; ++q) back1d(Ms[p][q][0], Ms[p][q][1], Ms[p][q][2], A[p][q][0], A[p][q][1], A[p][q][2]);
    real B[3][3][3];   // [p][cy][cz]
#pragma unroll
    for (int p = 0; p < 3; ++p)
#pragma unroll
        for (int c = 0; c < 3; ++c) back1d(A[p][0][c], A[p][1][c], A[p][2][c], B[p][0][c], B[p][1][c], B[p][2][c]);
#pragma unroll
    for (int b = 0; b < 3; ++b)
#pragma unroll
        for (int c = 0; c < 3; ++c) back1d(B[0][b][c], B[1][b][c], B[2][b][c], g[c][b][0], g[c][b][1], g[c][b][2]);
}

// fp32: the first two passes run on the pair (p = 1, p = 2), p = 0 on scalars; the last pass mixes p and stays scalar
__device__ __forceinline__ void back1d2(float2 m0, float2 m1s, float2 m2s, float2& fm, float2& f0, float2& fp)
{
    const float2 e = fma2(make_float2(1.0f / 6.0f, 1.0f / 6.0f), m0, m2s);
    fp = add2(e, m1s);
    fm = sub2(e, m1s);
    f0 = fma2(make_float2(-2.0f, -2.0f), e, m0);
}
__device__ __forceinline__ void back_transform(const float (&Ms)[3][3][3], float (&g)[3][3][3])
{
    float A0[3][3];     // [q][cz], p = 0
    float2 A12[3][3];   // [q][cz], (p = 1, p = 2)
#pragma unroll
    for (int q = 0; q < 3; ++q) {
        back1d(Ms[0][q][0], Ms[0][q][1], Ms[0][q][2], A0[q][0], A0[q][1], A0[q][2]);
        back1d2(make_float2(Ms[1][q][0], Ms[2][q][0]), make_float2(Ms[1][q][1], Ms[2][q][1]),
                make_float2(Ms[1][q][2], Ms[2][q][2]), A12[q][0], A12[q][1], A12[q][2]);
    }
    float B0[3][3];     // [cy][cz]
    float2 B12[3][3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        back1d(A0[0][c], A0[1][c], A0[2][c], B0[0][c], B0[1][c], B0[2][c]);
        back1d2(A12[0][c], A12[1][c], A12[2][c], B12[0][c], B12[1][c], B12[2][c]);
    }
#pragma unroll
    for (int b = 0; b < 3; ++b)
#pragma unroll
        for (int c = 0; c < 3; ++c) back1d(B0[b][c], B12[b][c].x, B12[b][c].y, g[c][b][0], g[c][b][1], g[c][b][2]);
}

// In: g = pre-collision populations of the site.  Out: g = post-collision populations f*.
// BGK = false: Reg-FLBM, Eq.24 (the hot path).  BGK = true: BGK-FLBM, Eq.11 (:109-111), the paper's comparison
// model: every non-conserved mode relaxes at the one rate omega, M_k = M_k^eq + (1-omega)(m_k - M_k^eq), which
// needs all 27 moments of the incoming populations (no body force in this model).
// a1 of ghost mode (p,q,r), order >= 3: the fixed point of the recursion Eq.21 (:163-166, R20) is the sum over index
// pairs of a1^(2)[pair] times the velocities of the remaining indices.  p, q, r are compile-time after unrolling.
template <typename real>
__device__ __forceinline__ real upow(real u, real u2, int n) { return n == 0 ? real(1) : n == 1 ? u : u2; }

template <typename real>
__device__ __forceinline__ real a1_ghost(int p, int q, int r, const real (&a)[6], const real (&u)[3], const real (&u2)[3])
{
    real t = real(0);
    if (p == 2) t = fma(a[0], upow(u[1], u2[1], q) * upow(u[2], u2[2], r), t);
    if (q == 2) t = fma(a[1], upow(u[0], u2[0], p) * upow(u[2], u2[2], r), t);
    if (r == 2) t = fma(a[2], upow(u[0], u2[0], p) * upow(u[1], u2[1], q), t);
    if (p && q) t = fma(real(p * q) * a[3], upow(u[0], u2[0], p - 1) * upow(u[1], u2[1], q - 1) * upow(u[2], u2[2], r), t);
    if (p && r) t = fma(real(p * r) * a[4], upow(u[0], u2[0], p - 1) * upow(u[2], u2[2], r - 1) * upow(u[1], u2[1], q), t);
    if (q && r) t = fma(real(q * r) * a[5], upow(u[1], u2[1], q - 1) * upow(u[2], u2[2], r - 1) * upow(u[0], u2[0], p), t);
    return t;
}

// GHOST = true: general ghost rate omega_g != 1 (:211-215): adds (1-omega_g) f^(1,g) with the coefficients of Eq.21.
template <typename real, bool FORCE, bool NOISE, bool BGK = false, bool GHOST = false>
__device__ __forceinline__ void collide(real (&g)[3][3][3], const StepParams<real>& P, uint32_t site,
                                        const f64x2* lg, const f64x2* sc)
{
    static_assert(!(BGK && FORCE), "BGK-FLBM carries no body force");
    static_assert(!(GHOST && (BGK || FORCE)), "the general ghost rate is built for Reg-FLBM without body force");
    Moments10<real> m;
    real mall[3][3][3];
    if (BGK) {
        forward_all(g, mall);
        m.rho = mall[0][0][0]; m.jx = mall[1][0][0]; m.jy = mall[0][1][0]; m.jz = mall[0][0][1];
        m.pxx = m.pyy = m.pzz = m.pxy = m.pxz = m.pyz = real(0);     // unused in this branch
    } else {
        m = forward_moments(g);
    }

    // Eq.3 (with the half-force shift of R13)
    const real inv_rho = rcp_pos<real>(m.rho);
    real ux = m.jx * inv_rho, uy = m.jy * inv_rho, uz = m.jz * inv_rho;
    if (FORCE) {
        ux = fma(real(0.5), P.gx, ux); uy = fma(real(0.5), P.gy, uy); uz = fma(real(0.5), P.gz, uz);
    }

    // Eq.20, scaled: Ms[p][q][r] = rho X_p Y_q Z_r with X = (1, ux/2, ux^2/2)
    const real hx = real(0.5) * ux, hy = real(0.5) * uy, hz = real(0.5) * uz;
    const real ex[3] = {real(1.0), hx, hx * ux};
    const real ey[3] = {real(1.0), hy, hy * uy};
    const real ez[3] = {real(1.0), hz, hz * uz};
    real Ms[3][3][3];
#pragma unroll
    for (int p = 0; p < 3; ++p) {
        const real a = (p == 0) ? m.rho : m.rho * ex[p];
#pragma unroll
        for (int q = 0; q < 3; ++q) {
            const real ab = (q == 0) ? a : a * ey[q];
#pragma unroll
            for (int r = 0; r < 3; ++r) Ms[p][q][r] = (r == 0) ? ab : ab * ez[r];
        }
    }

    if (BGK) {
        // Ms_k = E_k + (1-omega)(2^-nnz m_k - E_k) = (1-omega) 2^-nnz m_k + omega E_k for k = 4..26
        const real om = real(1.0) - real(2.0) * P.half_omc;
        const real w2 = P.half_omc, w4 = real(0.5) * P.half_omc, w8 = real(0.25) * P.half_omc;
#pragma unroll
        for (int p = 0; p < 3; ++p)
#pragma unroll
            for (int q = 0; q < 3; ++q)
#pragma unroll
                for (int r = 0; r < 3; ++r) {
                    const int nnz = (p > 0) + (q > 0) + (r > 0);
                    if (p + q + r < 2) continue;                     // conserved modes keep their equilibrium value
                    const real w = (nnz == 1) ? w2 : (nnz == 2) ? w4 : w8;
                    Ms[p][q][r] = fma(w, mall[p][q][r], om * Ms[p][q][r]);
                }
    } else
    // stress modes k = 4..9: Eq.19 a_1,ab = sum_i g_i (c_a c_b - delta_ab/3) - rho u_a u_b, relaxed by (1-omega_h)
    // (Eq.26).  Scaled: diagonal E + (1-omega_h)/2 (p_aa - rho/3 - 2E), E = rho u_a^2/2;
    //           off-diagonal E + (1-omega_h)/4 (p_ab - 4E), E = rho u_a u_b/4.
    {
        const real k2 = P.half_omc, k4 = real(0.5) * P.half_omc;
        const real dxx = fma(real(-2.0), Ms[2][0][0], fma(real(-1.0 / 3.0), m.rho, m.pxx));
        const real dyy = fma(real(-2.0), Ms[0][2][0], fma(real(-1.0 / 3.0), m.rho, m.pyy));
        const real dzz = fma(real(-2.0), Ms[0][0][2], fma(real(-1.0 / 3.0), m.rho, m.pzz));
        if (GHOST) {
            // Eq.21 needs the UNRELAXED a_1^(2) = (dxx, dyy, dzz, axy, axz, ayz) and the equilibrium modes as they are now
            const real a[6] = {dxx, dyy, dzz, fma(real(-4.0), Ms[1][1][0], m.pxy), fma(real(-4.0), Ms[1][0][1], m.pxz),
                               fma(real(-4.0), Ms[0][1][1], m.pyz)};
            const real uu[3] = {ux, uy, uz}, uu2[3] = {ux * ux, uy * uy, uz * uz};
#pragma unroll
            for (int p = 0; p < 3; ++p)
#pragma unroll
                for (int q = 0; q < 3; ++q)
#pragma unroll
                    for (int r = 0; r < 3; ++r) {
                        if (p + q + r < 3) continue;
                        const int nnz = (p > 0) + (q > 0) + (r > 0);
                        const real w = P.omc_g * (nnz == 1 ? real(0.5) : nnz == 2 ? real(0.25) : real(0.125));
                        Ms[p][q][r] = fma(w, a1_ghost<real>(p, q, r, a, uu, uu2), Ms[p][q][r]);
                    }
        }
        Ms[2][0][0] = fma(k2, dxx, Ms[2][0][0]);
        Ms[0][2][0] = fma(k2, dyy, Ms[0][2][0]);
        Ms[0][0][2] = fma(k2, dzz, Ms[0][0][2]);
        Ms[1][1][0] = fma(k4, fma(real(-4.0), Ms[1][1][0], m.pxy), Ms[1][1][0]);
        Ms[1][0][1] = fma(k4, fma(real(-4.0), Ms[1][0][1], m.pxz), Ms[1][0][1]);
        Ms[0][1][1] = fma(k4, fma(real(-4.0), Ms[0][1][1], m.pyz), Ms[0][1][1]);
    }
    if (FORCE) {
        // Guo forcing in moment form (R13): post-collision momentum j + F (modes 1..3 get another F/2, scaled 1/2),
        // stress source (1-omega_h/2)(u_a F_b + u_b F_a) (scaled 1/2 diagonal, 1/4 off-diagonal)
        const real Fx = m.rho * P.gx, Fy = m.rho * P.gy, Fz = m.rho * P.gz;
        Ms[1][0][0] = fma(real(0.25), Fx, Ms[1][0][0]);
        Ms[0][1][0] = fma(real(0.25), Fy, Ms[0][1][0]);
        Ms[0][0][1] = fma(real(0.25), Fz, Ms[0][0][1]);
        const real fs = P.force_stress, fq = real(0.25) * P.force_stress;
        Ms[2][0][0] = fma(fs, ux * Fx, Ms[2][0][0]);
        Ms[0][2][0] = fma(fs, uy * Fy, Ms[0][2][0]);
        Ms[0][0][2] = fma(fs, uz * Fz, Ms[0][0][2]);
        Ms[1][1][0] = fma(fq, fma(ux, Fy, uy * Fx), Ms[1][1][0]);
        Ms[1][0][1] = fma(fq, fma(ux, Fz, uz * Fx), Ms[1][0][1]);
        Ms[0][1][1] = fma(fq, fma(uy, Fz, uz * Fy), Ms[0][1][1]);
    }

    // Eq.8-9: noise on k = 4..26, Ms_k += sqrt(rho) amp[class(k)] r_k
    if (NOISE) {
        const real sq_rho = sqrt_rho<real>(m.rho);
        real amp[AMP_N];
#pragma unroll
        for (int n = 0; n < AMP_N; ++n) amp[n] = sq_rho * P.amp[n];
        const PhiloxSite ps = philox_site(site, P.rng);
#pragma unroll
        for (int call = 0; call < 6; ++call) {
            uint32_t w[4];
            philox_call(ps, P.rng, call, w);
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                real R, sn, cs;
                normal_polar(w[2 * h], w[2 * h + 1], lg, sc, R, sn, cs);
                const int k = 4 + 4 * call + 2 * h;            // modes k (first normal R cs) and k+1 (second, R sn), R8
                const int ca = amp_class(mode_p(k), mode_q(k), mode_r(k));
                real& m0 = Ms[mode_p(k)][mode_q(k)][mode_r(k)];
                const real A0 = amp[ca] * R;                   // the FDT amplitude rides on the radius
                m0 = fma(A0, cs, m0);
                if (k + 1 < Q) {
                    const int cb = amp_class(mode_p(k + 1), mode_q(k + 1), mode_r(k + 1));
                    real& m1 = Ms[mode_p(k + 1)][mode_q(k + 1)][mode_r(k + 1)];
                    m1 = fma((cb == ca) ? A0 : amp[cb] * R, sn, m1);
                }
            }
        }
    }

    back_transform(Ms, g);
}

}  // namespace rflbm_dev
