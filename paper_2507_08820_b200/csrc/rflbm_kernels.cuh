// rflbm_kernels.cuh — CUDA kernels of the Reg-FLBM path (sm_100a).
//
// Storage: SoA buffers P[q][z][y][x] of `real` in the lex order of rflbm_lattice.cuh, the 27
// arrays QS elements apart.
//   A-B scheme: two buffers holding POST-collision, UN-streamed populations (R10).  A step PULLS
//     S_t[q](x) = P_{t-1}[q](x - c_q)  (Eq.7 :87; bounce-back: P_{t-1}[26-q](x) when x - c_q is solid, R12),
//     collides in registers and stores P_t[q](x): 27 neighbour reads (coalesced, at most one element off alignment)
//     and 27 aligned coalesced writes per site, nothing else.
//   AA scheme: one buffer updated in place, alternating an all-local step and a pull/push step (STEP_AA_EVEN/ODD).
// The observables gather the pre-collision state S_t according to scheme and phase (GATHER_*).
#pragma once
#include "rflbm_collide.cuh"

namespace rflbm_dev {

struct SiteIndex {
    int x, y, z;
    bool valid;
    long long s;        // x + nx (y + ny z)
};

// one thread per site: blockDim = (bx, by), grid = (ceil(nx/bx), ceil(ny/by), nz)
__device__ __forceinline__ SiteIndex my_site(int nx, int ny)
{
    SiteIndex i;
    i.x = blockIdx.x * blockDim.x + threadIdx.x;
    i.y = blockIdx.y * blockDim.y + threadIdx.y;
    i.z = blockIdx.z;
    i.valid = (i.x < nx) && (i.y < ny);
    i.s = (long long)i.x + (long long)nx * ((long long)i.y + (long long)ny * (long long)i.z);
    return i;
}

// Where the pre-collision population S_t[q](x) of a site sits in the buffer:
//   GATHER_AB   A-B scheme: slot q of the neighbour x - c_q   (bounce-back: slot 26-q of the site itself)
//   GATHER_AA1  AA scheme after an even (in-place) step: slot 26-q of the neighbour x - c_q (bounce-back: slot q
//               of the site itself)
//   GATHER_AA0  AA scheme after init / an odd step: slot q of the site itself (the natural layout)
enum { GATHER_AB = 0, GATHER_AA1 = 1, GATHER_AA0 = 2 };

// Gather of the 27 pre-collision populations of a site into g[cz+1][cy+1][cx+1].
template <typename real, bool WALLS, int MODE = GATHER_AB>
__device__ __forceinline__ void gather(const real* __restrict__ src, long long QS, int nx, int ny, int nz,
                                       const SiteIndex& i, real (&g)[3][3][3])
{
    if (MODE == GATHER_AA0) {
#pragma unroll
        for (int q = 0; q < Q; ++q) g[q / 9][(q / 3) % 3][q % 3] = src[(long long)q * QS + i.s];   // in-place buffer: no LDG.NC
        return;
    }
    // neighbour coordinates x - cx etc. with periodic wrap; index a = cx+1 reads from xs[a]
    const int xs[3] = {(i.x + 1 == nx) ? 0 : i.x + 1, i.x, (i.x == 0) ? nx - 1 : i.x - 1};
    const int ys[3] = {(i.y + 1 == ny) ? 0 : i.y + 1, i.y, (i.y == 0) ? ny - 1 : i.y - 1};
    const int zs[3] = {(i.z + 1 == nz) ? 0 : i.z + 1, i.z, (i.z == 0) ? nz - 1 : i.z - 1};
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        // with walls the fluid layers are z = 1..nz-2; x - c_q is solid iff (cz=+1 and z==1) or (cz=-1 and z==nz-2)
        const bool bounce = WALLS && ((c == 2 && i.z == 1) || (c == 0 && i.z == nz - 2));
#pragma unroll
        for (int b = 0; b < 3; ++b) {
            const long long row = (long long)nx * ((long long)ys[b] + (long long)ny * (long long)zs[c]);
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                const int q = a + 3 * b + 9 * c;
                const int slot_pull = (MODE == GATHER_AA1) ? 26 - q : q;
                const int slot_back = (MODE == GATHER_AA1) ? q : 26 - q;
                const long long pull = (long long)slot_pull * QS + row + xs[a];
                const long long back = (long long)slot_back * QS + i.s;
                const long long at = (WALLS && bounce) ? back : pull;
                g[c][b][a] = (MODE == GATHER_AB) ? __ldg(src + at) : src[at];     // AA: the buffer is written in place
            }
        }
    }
}

// copy the Box-Muller tables (12 KB) from global memory (L2 resident) to shared memory; ends with a barrier
__device__ __forceinline__ void stage_tables(const f64x2* __restrict__ tab, f64x2* s_tab)
{
    const int tid = threadIdx.y * blockDim.x + threadIdx.x, nt = blockDim.x * blockDim.y;
    const double2* src = reinterpret_cast<const double2*>(tab);
    double2* dst = reinterpret_cast<double2*>(s_tab);
    for (int n = tid; n < LOG_TABLE_N + SC_TABLE_N; n += nt) dst[n] = __ldg(src + n);
    __syncthreads();
}

// ---------------------------------------------------------------- the hot kernel: one time step
// PHASE selects the storage scheme:
//   STEP_AB       A-B double buffer: pull from src, store to dst at the site itself
//   STEP_AA_EVEN  AA in place (src == dst): read slot q of the site, store f*_q into slot 26-q of the site
//   STEP_AA_ODD   AA in place: read slot 26-q of x - c_q (= f*_q streamed), store f*_q into slot q of x + c_q
//                 (halfway bounce-back: read slot q / store slot 26-q of the site itself)
// Every thread writes exactly the 27 locations it has read (the AA property), so in-place is race free.
enum { STEP_AB = 0, STEP_AA_EVEN = 1, STEP_AA_ODD = 2 };

template <typename real, bool WALLS, int PHASE>
__device__ __forceinline__ void scatter(real* dst, long long QS, int nx, int ny, int nz, const SiteIndex& i,
                                        const real (&g)[3][3][3])
{
    if (PHASE != STEP_AA_ODD) {
#pragma unroll
        for (int q = 0; q < Q; ++q)
            __stcs(dst + (long long)((PHASE == STEP_AA_EVEN) ? 26 - q : q) * QS + i.s, g[q / 9][(q / 3) % 3][q % 3]);
        return;
    }
    // push: x + c_q with periodic wrap; index a = cx+1 writes to xd[a]
    const int xd[3] = {(i.x == 0) ? nx - 1 : i.x - 1, i.x, (i.x + 1 == nx) ? 0 : i.x + 1};
    const int yd[3] = {(i.y == 0) ? ny - 1 : i.y - 1, i.y, (i.y + 1 == ny) ? 0 : i.y + 1};
    const int zd[3] = {(i.z == 0) ? nz - 1 : i.z - 1, i.z, (i.z + 1 == nz) ? 0 : i.z + 1};
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        // x + c_q is solid iff (cz=-1 and z==1) or (cz=+1 and z==nz-2): the population returns to the site as 26-q
        const bool bounce = WALLS && ((c == 0 && i.z == 1) || (c == 2 && i.z == nz - 2));
#pragma unroll
        for (int b = 0; b < 3; ++b) {
            const long long row = (long long)nx * ((long long)yd[b] + (long long)ny * (long long)zd[c]);
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                const int q = a + 3 * b + 9 * c;
                const long long push = (long long)q * QS + row + xd[a];
                const long long back = (long long)(26 - q) * QS + i.s;
                __stcs(dst + ((WALLS && bounce) ? back : push), g[c][b][a]);
            }
        }
    }
}

template <typename real, bool WALLS, bool FORCE, bool NOISE, bool BGK, bool GHOST, int PHASE>
__global__ void __launch_bounds__(128)
step_kernel(const real* src, real* dst, const __grid_constant__ StepParams<real> P)
{
    constexpr bool TABLES = NOISE && sizeof(real) == 8;
    __shared__ f64x2 s_tab[TABLES ? LOG_TABLE_N + SC_TABLE_N : 1];
    if (TABLES) stage_tables(P.tables, s_tab);
    const SiteIndex i = my_site(P.nx, P.ny);
    if (!i.valid) return;
    if (WALLS && (i.z == 0 || i.z == P.nz - 1)) return;    // solid layers are never updated
    real g[3][3][3];
    gather<real, WALLS, PHASE == STEP_AB ? GATHER_AB : PHASE == STEP_AA_EVEN ? GATHER_AA0 : GATHER_AA1>(
        src, P.QS, P.nx, P.ny, P.nz, i, g);
    collide<real, FORCE, NOISE, BGK, GHOST>(g, P, (uint32_t)i.s, s_tab, s_tab + LOG_TABLE_N);
    scatter<real, WALLS, PHASE>(dst, P.QS, P.nx, P.ny, P.nz, i, g);
}

// ---------------------------------------------------------------- observables
template <typename real>
struct FieldParams {
    int nx, ny, nz;
    long long N;
    long long QS;         // elements between consecutive population arrays of the internal storage (>= N)
    real hgx, hgy, hgz;   // g/2: reported velocity u = j/rho + g/2 (R13)
    int walls;
    int aa;               // AA scheme: one buffer in the natural layout P[q](s) = S[q](s) at even phase
};

template <typename real, bool WALLS, int MODE>
__global__ void __launch_bounds__(128)
moments_kernel(const real* __restrict__ src, real* __restrict__ rho, real* __restrict__ u, const FieldParams<real> P)
{
    const SiteIndex i = my_site(P.nx, P.ny);
    if (!i.valid) return;
    if (WALLS && (i.z == 0 || i.z == P.nz - 1)) {
        rho[i.s] = real(0); u[i.s] = real(0); u[P.N + i.s] = real(0); u[2 * P.N + i.s] = real(0);
        return;
    }
    real g[3][3][3];
    gather<real, WALLS, MODE>(src, P.QS, P.nx, P.ny, P.nz, i, g);
    const Moments10<real> m = forward_moments(g);
    const real inv = real(1.0) / m.rho;
    rho[i.s] = m.rho;
    u[i.s] = fma(m.jx, inv, P.hgx);
    u[P.N + i.s] = fma(m.jy, inv, P.hgy);
    u[2 * P.N + i.s] = fma(m.jz, inv, P.hgz);
}

// Pi_ab = sum_i f_i (c_a c_b - delta_ab/3) of the current state (Eq.18 + Eq.19):
// pi[6][N] in the order xx, yy, zz, xy, xz, yz.  Solid nodes: 0.
template <typename real, bool WALLS, int MODE>
__global__ void __launch_bounds__(128)
stress_kernel(const real* __restrict__ src, real* __restrict__ pi, const FieldParams<real> P)
{
    const SiteIndex i = my_site(P.nx, P.ny);
    if (!i.valid) return;
    real v[6] = {real(0), real(0), real(0), real(0), real(0), real(0)};
    if (!(WALLS && (i.z == 0 || i.z == P.nz - 1))) {
        real g[3][3][3];
        gather<real, WALLS, MODE>(src, P.QS, P.nx, P.ny, P.nz, i, g);
        const Moments10<real> m = forward_moments(g);
        const real third = m.rho * real(1.0 / 3.0);
        v[0] = m.pxx - third; v[1] = m.pyy - third; v[2] = m.pzz - third;
        v[3] = m.pxy; v[4] = m.pxz; v[5] = m.pyz;
    }
#pragma unroll
    for (int n = 0; n < 6; ++n) pi[(long long)n * P.N + i.s] = v[n];
}

// sums over fluid sites of { rho, rho u_x,y,z, u_x,y,z, u_x^2,y^2,z^2 } -> acc[10] (fp64 atomics)
template <typename real, bool WALLS, int MODE>
__global__ void __launch_bounds__(128)
diagnostics_kernel(const real* __restrict__ src, double* __restrict__ acc, const FieldParams<real> P)
{
    const SiteIndex i = my_site(P.nx, P.ny);
    double v[10];
#pragma unroll
    for (int n = 0; n < 10; ++n) v[n] = 0.0;
    const bool fluid = i.valid && !(WALLS && (i.z == 0 || i.z == P.nz - 1));
    if (fluid) {
        real g[3][3][3];
        gather<real, WALLS, MODE>(src, P.QS, P.nx, P.ny, P.nz, i, g);
        const Moments10<real> m = forward_moments(g);
        const double rho = (double)m.rho;
        const double ux = (double)m.jx / rho + (double)P.hgx;
        const double uy = (double)m.jy / rho + (double)P.hgy;
        const double uz = (double)m.jz / rho + (double)P.hgz;
        v[0] = rho; v[1] = rho * ux; v[2] = rho * uy; v[3] = rho * uz;
        v[4] = ux; v[5] = uy; v[6] = uz; v[7] = ux * ux; v[8] = uy * uy; v[9] = uz * uz;
    }
    __shared__ double part[4][10];
    const int tid = threadIdx.y * blockDim.x + threadIdx.x;
    const int lane = tid & 31, warp = tid >> 5;
#pragma unroll
    for (int n = 0; n < 10; ++n) {
        double s = v[n];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
        if (lane == 0) part[warp][n] = s;
    }
    __syncthreads();
    const int nwarps = (blockDim.x * blockDim.y + 31) >> 5;
    if (tid < 10) {
        double s = 0.0;
        for (int w = 0; w < nwarps; ++w) s += part[w][tid];
        atomicAdd(acc + tid, s);
    }
}

// ---------------------------------------------------------------- state import / export (R10)
// out[canonical i][s] = S_t[i](s): the same gather as the step; solid nodes export their stored values.
template <typename real, bool WALLS, int MODE>
__global__ void __launch_bounds__(128)
export_kernel(const real* __restrict__ src, real* __restrict__ out, const FieldParams<real> P)
{
    const SiteIndex i = my_site(P.nx, P.ny);
    if (!i.valid) return;
    if (WALLS && (i.z == 0 || i.z == P.nz - 1)) {
#pragma unroll
        for (int n = 0; n < Q; ++n) out[(long long)n * P.N + i.s] = src[(long long)lex_of_canon(n) * P.QS + i.s];
        return;
    }
    real g[3][3][3];
    gather<real, WALLS, MODE>(src, P.QS, P.nx, P.ny, P.nz, i, g);
#pragma unroll
    for (int n = 0; n < Q; ++n)
        out[(long long)n * P.N + i.s] = g[canon_cz(n) + 1][canon_cy(n) + 1][canon_cx(n) + 1];
}

// P[q](s) = S[q](s + c_q), or S[26-q](s) when s + c_q is solid; solid nodes store S[q](s) unchanged.
// `in` is canonical; written to both A and B buffers so that the never-updated solid layers agree.
// AA scheme (P.aa): the natural layout P[q](s) = S[q](s), one buffer (bufB == nullptr).
template <typename real, bool WALLS>
__global__ void __launch_bounds__(128)
import_kernel(const real* __restrict__ in, real* __restrict__ bufA, real* __restrict__ bufB, const FieldParams<real> P)
{
    const SiteIndex i = my_site(P.nx, P.ny);
    if (!i.valid) return;
    const bool solid = WALLS && (i.z == 0 || i.z == P.nz - 1);
#pragma unroll
    for (int n = 0; n < Q; ++n) {
        const int cx = canon_cx(n), cy = canon_cy(n), cz = canon_cz(n);
        const int q = lex_of(cx, cy, cz);
        long long from = (long long)n * P.N + i.s;
        if (!solid && !P.aa) {
            const int zd = i.z + cz;
            if (WALLS && (zd == 0 || zd == P.nz - 1)) {
                // s + c_q solid: this slot is pulled back by the site itself as direction opp(q)
                const int nopp = canon_of_lex(26 - q);
                from = (long long)nopp * P.N + i.s;
            } else {
                const int xd = (i.x + cx + P.nx) % P.nx, yd = (i.y + cy + P.ny) % P.ny, zw = (zd + P.nz) % P.nz;
                from = (long long)n * P.N + (long long)xd + (long long)P.nx * ((long long)yd + (long long)P.ny * zw);
            }
        }
        const real v = in[from];
        bufA[(long long)q * P.QS + i.s] = v;
        if (bufB != nullptr) bufB[(long long)q * P.QS + i.s] = v;
    }
}

// equilibrium f^(0)_q(rho,u) in the product form of Eq.25 with Eq.20 (w_i and the Hermite sum factorise):
//   f0 = rho phi(cx,ux) phi(cy,uy) phi(cz,uz),  phi(0,u) = 2/3 - u^2,  phi(+-1,u) = 1/6 +- u/2 + u^2/2
// Written with explicit round-to-nearest intrinsics: the compiler must not contract or reassociate differently in
// the A-B and AA code paths of init_kernel (the two schemes are required to agree bit for bit).
__device__ __forceinline__ double phi1d(int c, double u)
{
    if (c == 0) return __fma_rn(-u, u, 2.0 / 3.0);
    return __fma_rn(0.5 * u, __dadd_rn(u, (double)c), 1.0 / 6.0);      // 1/6 + u (u + c) / 2
}

// init (R9, R10): P_{-1}[q](s) = f0_q(rho,u)(s + c_q), or f0_{26-q}(rho,u)(s) when s + c_q is solid.
// rho/u NULL -> uniform rho0, u = 0.
template <typename real, bool WALLS>
__global__ void __launch_bounds__(128)
init_kernel(const real* __restrict__ rho, const real* __restrict__ u, double rho0, real* __restrict__ bufA,
            real* __restrict__ bufB, const FieldParams<real> P)
{
    const SiteIndex i = my_site(P.nx, P.ny);
    if (!i.valid) return;
    const bool solid = WALLS && (i.z == 0 || i.z == P.nz - 1);
#pragma unroll 1
    for (int q = 0; q < Q; ++q) {
        int cx = q % 3 - 1, cy = (q / 3) % 3 - 1, cz = q / 9 - 1;
        long long s = i.s;
        if (!solid && !P.aa) {
            const int zd = i.z + cz;
            if (WALLS && (zd == 0 || zd == P.nz - 1)) {
                cx = -cx; cy = -cy; cz = -cz;              // f0 of the opposite direction at the site itself
            } else {
                const int xd = (i.x + cx + P.nx) % P.nx, yd = (i.y + cy + P.ny) % P.ny, zw = (zd + P.nz) % P.nz;
                s = (long long)xd + (long long)P.nx * ((long long)yd + (long long)P.ny * zw);
            }
        }
        double r = rho0, ux = 0.0, uy = 0.0, uz = 0.0;
        if (rho != nullptr) {
            r = (double)rho[s]; ux = (double)u[s]; uy = (double)u[P.N + s]; uz = (double)u[2 * P.N + s];
        }
        const real v = (real)__dmul_rn(__dmul_rn(__dmul_rn(r, phi1d(cx, ux)), phi1d(cy, uy)), phi1d(cz, uz));
        bufA[(long long)q * P.QS + i.s] = v;
        if (bufB != nullptr) bufB[(long long)q * P.QS + i.s] = v;
    }
}

// test hook: the words and normals the step kernel draws at step (t_hi,t_lo).  The words come from the
// hand-scheduled philox_call() of the step kernel; mismatch[0] counts sites where they differ from the textbook
// ten-round loop philox4x32_10() (must stay 0).
template <typename real>
__global__ void __launch_bounds__(128)
debug_rng_kernel(uint32_t* __restrict__ words, real* __restrict__ normals, unsigned long long* __restrict__ mismatch,
                 uint32_t t_hi, uint32_t t_lo, const __grid_constant__ StepParams<real> P)
{
    constexpr bool TABLES = sizeof(real) == 8;
    __shared__ f64x2 s_tab[TABLES ? LOG_TABLE_N + SC_TABLE_N : 1];
    if (TABLES) stage_tables(P.tables, s_tab);
    const SiteIndex i = my_site(P.nx, P.ny);
    if (!i.valid) return;
    const PhiloxSite ps = philox_site((uint32_t)i.s, P.rng);
    bool bad = false;
#pragma unroll
    for (int call = 0; call < 6; ++call) {
        uint32_t w[4], w_ref[4];
        philox_call(ps, P.rng, call, w);
        philox4x32_10((uint32_t)i.s, t_hi, t_lo, (uint32_t)call, P.rng, w_ref);
        bad = bad || w[0] != w_ref[0] || w[1] != w_ref[1] || w[2] != w_ref[2] || w[3] != w_ref[3];
        if (words != nullptr)
#pragma unroll
            for (int mth = 0; mth < 4; ++mth) words[(long long)(4 * call + mth) * P.N + i.s] = w[mth];
        if (normals != nullptr)
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                real z0, z1;
                normal_pair(w[2 * h], w[2 * h + 1], s_tab, s_tab + LOG_TABLE_N, z0, z1);
                const int k = 4 + 4 * call + 2 * h;
                normals[(long long)(k - 4) * P.N + i.s] = z0;
                if (k + 1 < Q) normals[(long long)(k + 1 - 4) * P.N + i.s] = z1;
            }
    }
    if (bad) atomicAdd(mismatch, 1ull);
}

}  // namespace rflbm_dev
