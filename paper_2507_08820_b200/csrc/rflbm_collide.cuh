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
//   * modes are carried ORTHONORMALISED, Mt_k = M_k / sqrt(b_k): the FDT amplitude (Eq.9) becomes the same
//     sqrt(3 kT rho omega_k (2-omega_k)) for every mode, i.e. one scale for the 17 ghost modes, one for the 6
//     stress modes, and the 1-D back-transform matrix is T[c][p] = w1(c) H_p(c) / sqrt(beta_p).
//   * only the 10 moments of order <= 2 are needed from the incoming populations (ghost modes are rebuilt from
//     rho,u, not relaxed), so the forward transform is truncated.
#pragma once
#include "rflbm_lattice.cuh"
#include "rflbm_rng.cuh"

namespace rflbm_dev {

template <typename real>
struct StepParams {
    int nx, ny, nz;
    long long N;
    real one_minus_omega;   // 1 - omega_h
    real noise_ghost;       // sqrt(3 kT)                      (times sqrt(rho) at the site)
    real noise_hydro;       // sqrt(3 kT omega_h (2-omega_h))
    real gx, gy, gz;        // acceleration (R13)
    real force_stress;      // 1 - omega_h/2
    uint32_t t_hi, t_lo;    // step counter
    PhiloxKeys keys;
    const f64x2* tables;    // device: log table [256] then sin/cos table [256] (fp64 noise only)
};

template <typename real> __device__ __forceinline__ real rsqrt_real(real x);
template <> __device__ __forceinline__ double rsqrt_real<double>(double x) { return rsqrt(x); }
template <> __device__ __forceinline__ float rsqrt_real<float>(float x) { return rsqrtf(x); }

// conserved moments + raw second moments of g[cz+1][cy+1][cx+1] (Eq.2-3, and sum g c_a c_b for Eq.19)
template <typename real>
struct Moments10 {
    real rho, jx, jy, jz, pxx, pyy, pzz, pxy, pxz, pyz;
};

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

// 1-D back-transform of orthonormal modes (m0,m1,m2) -> values at c = -1, 0, +1:
//   T[c][p] = w1(c) H_p(c) / sqrt(beta_p):  c=0: (2/3, 0, -sqrt2/3);  c=+-1: (1/6, +-sqrt3/6, sqrt2/6)
template <typename real>
__device__ __forceinline__ void back1d(real m0, real m1, real m2, real& fm, real& f0, real& fp)
{
    const real t = real(SQRT2 / 6.0) * m2;
    const real e = fma(real(1.0 / 6.0), m0, t);
    f0 = fma(real(-2.0), t, real(2.0 / 3.0) * m0);
    fp = fma(real(SQRT3 / 6.0), m1, e);
    fm = fma(real(-SQRT3 / 6.0), m1, e);
}

// In: g = pre-collision populations of the site.  Out: g = post-collision populations f*.
template <typename real, bool FORCE, bool NOISE>
__device__ __forceinline__ void collide(real (&g)[3][3][3], const StepParams<real>& P, uint32_t site,
                                        const f64x2* lg, const f64x2* sc)
{
    const Moments10<real> m = forward_moments(g);

    // Eq.3 (with the half-force shift of R13)
    const real inv_rho = real(1.0) / m.rho;
    real ux = m.jx * inv_rho, uy = m.jy * inv_rho, uz = m.jz * inv_rho;
    real Fx = real(0), Fy = real(0), Fz = real(0);
    if (FORCE) {
        Fx = m.rho * P.gx; Fy = m.rho * P.gy; Fz = m.rho * P.gz;
        ux = fma(real(0.5), P.gx, ux); uy = fma(real(0.5), P.gy, uy); uz = fma(real(0.5), P.gz, uz);
    }
    const real rux = m.rho * ux, ruy = m.rho * uy, ruz = m.rho * uz;

    // Eq.19: a_1,ab = sum_i g_i (c_a c_b - delta_ab/3) - rho u_a u_b
    const real third_rho = m.rho * real(1.0 / 3.0);
    real axx = (m.pxx - third_rho) - rux * ux;
    real ayy = (m.pyy - third_rho) - ruy * uy;
    real azz = (m.pzz - third_rho) - ruz * uz;
    real axy = m.pxy - rux * uy;
    real axz = m.pxz - rux * uz;
    real ayz = m.pyz - ruy * uz;
    // relaxed: (1-omega_h) a_1 (+ Guo stress source (1-omega_h/2)(u_a F_b + u_b F_a))
    axx *= P.one_minus_omega; ayy *= P.one_minus_omega; azz *= P.one_minus_omega;
    axy *= P.one_minus_omega; axz *= P.one_minus_omega; ayz *= P.one_minus_omega;
    if (FORCE) {
        axx = fma(P.force_stress, real(2.0) * ux * Fx, axx);
        ayy = fma(P.force_stress, real(2.0) * uy * Fy, ayy);
        azz = fma(P.force_stress, real(2.0) * uz * Fz, azz);
        axy = fma(P.force_stress, ux * Fy + uy * Fx, axy);
        axz = fma(P.force_stress, ux * Fz + uz * Fx, axz);
        ayz = fma(P.force_stress, uy * Fz + uz * Fy, ayz);
    }

    // Eq.20 in orthonormal form: Mt[p][q][r] = rho * (n_p ux^p)(n_q uy^q)(n_r uz^r)
    real ex[3] = {real(1.0), real(NRM1) * ux, real(NRM2) * ux * ux};
    real ey[3] = {real(1.0), real(NRM1) * uy, real(NRM2) * uy * uy};
    real ez[3] = {real(1.0), real(NRM1) * uz, real(NRM2) * uz * uz};
    real Mt[3][3][3];
#pragma unroll
    for (int p = 0; p < 3; ++p) {
        const real a = (p == 0) ? m.rho : m.rho * ex[p];
#pragma unroll
        for (int q = 0; q < 3; ++q) {
            const real ab = (q == 0) ? a : a * ey[q];
#pragma unroll
            for (int r = 0; r < 3; ++r) Mt[p][q][r] = (r == 0) ? ab : ab * ez[r];
        }
    }
    // stress modes k = 4..9 (normalised by 1/sqrt(b_k): 3/sqrt2 for the diagonal, 3 for the off-diagonal ones)
    Mt[2][0][0] = fma(real(NRM2), axx, Mt[2][0][0]);
    Mt[0][2][0] = fma(real(NRM2), ayy, Mt[0][2][0]);
    Mt[0][0][2] = fma(real(NRM2), azz, Mt[0][0][2]);
    Mt[1][1][0] = fma(real(3.0), axy, Mt[1][1][0]);
    Mt[1][0][1] = fma(real(3.0), axz, Mt[1][0][1]);
    Mt[0][1][1] = fma(real(3.0), ayz, Mt[0][1][1]);
    if (FORCE) {   // post-collision momentum j + F: modes 1..3 get another F/2 (times n_1)
        Mt[1][0][0] = fma(real(0.5 * NRM1), Fx, Mt[1][0][0]);
        Mt[0][1][0] = fma(real(0.5 * NRM1), Fy, Mt[0][1][0]);
        Mt[0][0][1] = fma(real(0.5 * NRM1), Fz, Mt[0][0][1]);
    }

    // Eq.8-9: noise on k = 4..26, Mt_k += sqrt(3 kT rho omega_k(2-omega_k)) r_k
    if (NOISE) {
        const real sq_rho = m.rho * rsqrt_real<real>(m.rho);
        const real amp_h = sq_rho * P.noise_hydro;
        const real amp_g = sq_rho * P.noise_ghost;
#pragma unroll
        for (int call = 0; call < 6; ++call) {
            uint32_t w[4];
            philox4x32_10(site, P.t_hi, P.t_lo, (uint32_t)call, P.keys, w);
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                real z0, z1;
                normal_pair(w[2 * h], w[2 * h + 1], lg, sc, z0, z1);
                const int k = 4 + 4 * call + 2 * h;            // modes k (first) and k+1 (second), R8
                const real amp = (k <= 9) ? amp_h : amp_g;      // pairs (4,5),(6,7),(8,9) are all-stress
                real& m0 = Mt[mode_p(k)][mode_q(k)][mode_r(k)];
                m0 = fma(amp, z0, m0);
                if (k + 1 < Q) {
                    real& m1 = Mt[mode_p(k + 1)][mode_q(k + 1)][mode_r(k + 1)];
                    m1 = fma(amp, z1, m1);
                }
            }
        }
    }

    // Eq.10, separable: r -> cz, then q -> cy, then p -> cx
    real A[3][3][3];   // [p][q][cz]
#pragma unroll
    for (int p = 0; p < 3; ++p)
#pragma unroll
        for (int q = 0; q < 3; ++q) back1d(Mt[p][q][0], Mt[p][q][1], Mt[p][q][2], A[p][q][0], A[p][q][1], A[p][q][2]);
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

}  // namespace rflbm_dev
