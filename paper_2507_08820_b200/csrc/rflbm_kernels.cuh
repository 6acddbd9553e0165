// rflbm_kernels.cuh — CUDA kernels of the Reg-FLBM path (sm_100a).
//
// Storage: buffers P[z][y][q][x] of `real`, q in the lex order of rflbm_lattice.cuh: slot stride
// Geom::QS (= the padded row length >= nx, 16-byte aligned rows whatever nx is), row stride Geom::px = 27 QS, layer
// stride Geom::pxy.  The kernels only ever use these three strides.
//   A-B scheme: two buffers holding POST-collision, UN-streamed populations (R10).  A step PULLS
//     S_t[q](x) = P_{t-1}[q](x - c_q)  (Eq.7 :87; bounce-back: P_{t-1}[26-q](x) when x - c_q is solid, R12),
//     collides in registers and stores P_t[q](x): 27 neighbour reads (coalesced, at most one element off alignment)
//     and 27 aligned coalesced writes per site, nothing else.
//   AA scheme: one buffer updated in place, alternating an all-local step and a pull/push step (STEP_AA_EVEN/ODD).
// The observables gather the pre-collision state S_t according to scheme and phase (GATHER_*).
// Slab mode (rflbm_set_slab; "linear decomposition" along z): the buffers carry one ghost layer
// below and above the owned layers, filled by the halo calls; nothing wraps in z, and the solid-layer test and the
// Philox site key use the GLOBAL z, so a slab computes exactly what the undivided lattice computes there.
#pragma once
#include "rflbm_collide.cuh"

namespace rflbm_dev {

struct SiteIndex {
    int x, y, z;        // z: storage layer
    int zg;             // global layer (walls, RNG key)
    bool valid;
    long long s;        // storage index  x + px (y + ny z)
    long long sl;       // canonical index x + nx (y + ny (z - z_lo)) of the boundary arrays
    uint32_t site;      // Philox key     x + nx (y + ny zg)  (R8; < 2^32 by rflbm_create / rflbm_set_slab)
};

// one thread per site: blockDim = (bx, by), grid = (ceil(nx/bx), ceil(ny/by), nz)
// the site of this thread in layer zrel of the launch (zrel = blockIdx.z for the one-thread-per-site kernels)
__device__ __forceinline__ SiteIndex my_site_in_layer(const Geom& G, int zrel)
{
    SiteIndex i;
    i.x = blockIdx.x * blockDim.x + threadIdx.x;
    i.y = blockIdx.y * blockDim.y + threadIdx.y;
    const int zl = zrel + G.zc;                             // owned-layer index
    i.z = zl + G.z_lo;
    i.zg = i.z + G.zg0;
    i.valid = (i.x < G.nx) && (i.y < G.ny);
    i.s = (long long)i.x + (long long)G.px * i.y + G.pxy * i.z;
    i.sl = (long long)i.x + (long long)G.nx * ((long long)i.y + (long long)G.ny * (long long)zl);
    i.site = (uint32_t)((long long)i.x + (long long)G.nx * ((long long)i.y + (long long)G.ny * (long long)i.zg));
    return i;
}

__device__ __forceinline__ SiteIndex my_site(const Geom& G) { return my_site_in_layer(G, (int)blockIdx.z); }

__device__ __forceinline__ bool solid_layer(const Geom& G, int zg) { return zg == 0 || zg == G.nzg - 1; }

// Where the pre-collision population S_t[q](x) of a site sits in the buffer:
//   GATHER_AB   A-B scheme: slot q of the neighbour x - c_q   (bounce-back: slot 26-q of the site itself)
//   GATHER_AA1  AA scheme after an even (in-place) step: slot 26-q of the neighbour x - c_q (bounce-back: slot q
//               of the site itself)
//   GATHER_AA0  AA scheme after init / an odd step: slot q of the site itself (the natural layout)
enum { GATHER_AB = 0, GATHER_AA1 = 1, GATHER_AA0 = 2 };

// Gather of the 27 pre-collision populations of a site into g[cz+1][cy+1][cx+1].
template <typename real, bool WALLS, int MODE = GATHER_AB>
__device__ __forceinline__ void gather(const real* __restrict__ src, const Geom& G, const SiteIndex& i, real (&g)[3][3][3])
{
    if (MODE == GATHER_AA0) {
#pragma unroll
        for (int q = 0; q < Q; ++q) g[q / 9][(q / 3) % 3][q % 3] = src[(long long)q * G.QS + i.s];   // in-place buffer: no LDG.NC
        return;
    }
    // neighbour coordinates x - cx etc. with periodic wrap; index a = cx+1 reads from xs[a].  In slab mode the ghost
    // layers make the z wrap unreachable (owned layers are 1..nzs-2).
    const int xs[3] = {(i.x + 1 == G.nx) ? 0 : i.x + 1, i.x, (i.x == 0) ? G.nx - 1 : i.x - 1};
    const int ys[3] = {(i.y + 1 == G.ny) ? 0 : i.y + 1, i.y, (i.y == 0) ? G.ny - 1 : i.y - 1};
    const int zs[3] = {(i.z + 1 == G.nzs) ? 0 : i.z + 1, i.z, (i.z == 0) ? G.nzs - 1 : i.z - 1};
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        // with walls the fluid layers are zg = 1..nzg-2; x - c_q is solid iff (cz=+1 and zg==1) or (cz=-1 and zg==nzg-2)
        const bool bounce = WALLS && ((c == 2 && i.zg == 1) || (c == 0 && i.zg == G.nzg - 2));
#pragma unroll
        for (int b = 0; b < 3; ++b) {
            const long long row = (long long)G.px * ys[b] + G.pxy * zs[c];
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                const int q = a + 3 * b + 9 * c;
                const int slot_pull = (MODE == GATHER_AA1) ? 26 - q : q;
                const int slot_back = (MODE == GATHER_AA1) ? q : 26 - q;
                const long long pull = (long long)slot_pull * G.QS + row + xs[a];
                const long long back = (long long)slot_back * G.QS + i.s;
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
__device__ __forceinline__ void scatter(real* dst, const Geom& G, const SiteIndex& i, const real (&g)[3][3][3])
{
    if (PHASE != STEP_AA_ODD) {
#pragma unroll
        for (int q = 0; q < Q; ++q)
            __stcs(dst + (long long)((PHASE == STEP_AA_EVEN) ? 26 - q : q) * G.QS + i.s, g[q / 9][(q / 3) % 3][q % 3]);
        return;
    }
    // push: x + c_q with periodic wrap; index a = cx+1 writes to xd[a] (slab mode: the ghost layers take the z = -1
    // and z = nz pushes, rflbm_halo_* carry them home)
    const int xd[3] = {(i.x == 0) ? G.nx - 1 : i.x - 1, i.x, (i.x + 1 == G.nx) ? 0 : i.x + 1};
    const int yd[3] = {(i.y == 0) ? G.ny - 1 : i.y - 1, i.y, (i.y + 1 == G.ny) ? 0 : i.y + 1};
    const int zd[3] = {(i.z == 0) ? G.nzs - 1 : i.z - 1, i.z, (i.z + 1 == G.nzs) ? 0 : i.z + 1};
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        // x + c_q is solid iff (cz=-1 and zg==1) or (cz=+1 and zg==nzg-2): the population returns to the site as 26-q
        const bool bounce = WALLS && ((c == 0 && i.zg == 1) || (c == 2 && i.zg == G.nzg - 2));
#pragma unroll
        for (int b = 0; b < 3; ++b) {
            const long long row = (long long)G.px * yd[b] + G.pxy * zd[c];
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                const int q = a + 3 * b + 9 * c;
                const long long push = (long long)q * G.QS + row + xd[a];
                const long long back = (long long)(26 - q) * G.QS + i.s;
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
    const SiteIndex i = my_site(P.G);
    if (!i.valid) return;
    if (WALLS && solid_layer(P.G, i.zg)) return;           // solid layers are never updated
    real g[3][3][3];
    gather<real, WALLS, PHASE == STEP_AB ? GATHER_AB : PHASE == STEP_AA_EVEN ? GATHER_AA0 : GATHER_AA1>(src, P.G, i, g);
    collide<real, FORCE, NOISE, BGK, GHOST>(g, P, i.site, s_tab, s_tab + LOG_TABLE_N);
    scatter<real, WALLS, PHASE>(dst, P.G, i, g);
}

// ---------------------------------------------------------------- observables
template <typename real>
struct FieldParams {
    Geom G;
    real hgx, hgy, hgz;   // g/2: reported velocity u = j/rho + g/2 (R13)
    int aa;               // AA scheme: one buffer in the natural layout P[q](s) = S[q](s) at even phase
    int ghost_in;         // slab mode: the fields given to init / set_populations carry one extra layer below and above
};

template <typename real, bool WALLS, int MODE>
__global__ void __launch_bounds__(128)
moments_kernel(const real* __restrict__ src, real* __restrict__ rho, real* __restrict__ u, const FieldParams<real> P)
{
    const SiteIndex i = my_site(P.G);
    if (!i.valid) return;
    const long long N = P.G.N;
    if (WALLS && solid_layer(P.G, i.zg)) {
        rho[i.sl] = real(0); u[i.sl] = real(0); u[N + i.sl] = real(0); u[2 * N + i.sl] = real(0);
        return;
    }
    real g[3][3][3];
    gather<real, WALLS, MODE>(src, P.G, i, g);
    const Moments10<real> m = forward_moments(g);
    const real inv = real(1.0) / m.rho;
    rho[i.sl] = m.rho;
    u[i.sl] = fma(m.jx, inv, P.hgx);
    u[N + i.sl] = fma(m.jy, inv, P.hgy);
    u[2 * N + i.sl] = fma(m.jz, inv, P.hgz);
}

// Pi_ab = sum_i f_i (c_a c_b - delta_ab/3) of the current state (Eq.18 + Eq.19):
// pi[6][N] in the order xx, yy, zz, xy, xz, yz.  Solid nodes: 0.
template <typename real, bool WALLS, int MODE>
__global__ void __launch_bounds__(128)
stress_kernel(const real* __restrict__ src, real* __restrict__ pi, const FieldParams<real> P)
{
    const SiteIndex i = my_site(P.G);
    if (!i.valid) return;
    real v[6] = {real(0), real(0), real(0), real(0), real(0), real(0)};
    if (!(WALLS && solid_layer(P.G, i.zg))) {
        real g[3][3][3];
        gather<real, WALLS, MODE>(src, P.G, i, g);
        const Moments10<real> m = forward_moments(g);
        const real third = m.rho * real(1.0 / 3.0);
        v[0] = m.pxx - third; v[1] = m.pyy - third; v[2] = m.pzz - third;
        v[3] = m.pxy; v[4] = m.pxz; v[5] = m.pyz;
    }
#pragma unroll
    for (int n = 0; n < 6; ++n) pi[(long long)n * P.G.N + i.sl] = v[n];
}

// rho, u and Pi_ab of the current state in ONE pass over the populations ("density rho, momentum rho u, and
// the momentum flux tensor components Pi_ab were saved every 5,000 steps"): 27 reads + 10 writes per site instead of the
// 2 x 27 reads of moments_kernel followed by stress_kernel.  Same expressions as those two kernels: the same bits.
template <typename real, bool WALLS, int MODE>
__global__ void __launch_bounds__(128)
snapshot_kernel(const real* __restrict__ src, real* __restrict__ rho, real* __restrict__ u, real* __restrict__ pi,
                const FieldParams<real> P)
{
    const SiteIndex i = my_site(P.G);
    if (!i.valid) return;
    const long long N = P.G.N;
    real r = real(0), ux = real(0), uy = real(0), uz = real(0);
    real v[6] = {real(0), real(0), real(0), real(0), real(0), real(0)};
    if (!(WALLS && solid_layer(P.G, i.zg))) {
        real g[3][3][3];
        gather<real, WALLS, MODE>(src, P.G, i, g);
        const Moments10<real> m = forward_moments(g);
        const real inv = real(1.0) / m.rho;
        r = m.rho;
        ux = fma(m.jx, inv, P.hgx);
        uy = fma(m.jy, inv, P.hgy);
        uz = fma(m.jz, inv, P.hgz);
        const real third = m.rho * real(1.0 / 3.0);
        v[0] = m.pxx - third; v[1] = m.pyy - third; v[2] = m.pzz - third;
        v[3] = m.pxy; v[4] = m.pxz; v[5] = m.pyz;
    }
    rho[i.sl] = r;
    u[i.sl] = ux; u[N + i.sl] = uy; u[2 * N + i.sl] = uz;
#pragma unroll
    for (int n = 0; n < 6; ++n) pi[(long long)n * N + i.sl] = v[n];
}

// sums over fluid sites of { rho, rho u_x,y,z, u_x,y,z, u_x^2,y^2,z^2 } -> acc[DIAG_ROWS][DIAG_PITCH] (fp64 atomics).
// One block per 128 sites would mean a million blocks at 512^3, each ending in ten atomics on the same ten addresses
// (0.84 / 0.58 of the copy rate, fp64 / fp32).  So (i) a block walks the layers blockIdx.z, blockIdx.z + gridDim.z, ...
// of its (x, y) patch and keeps its sums in registers (grid.z <= DIAG_ZBLOCKS: 32 times fewer atomics at 512 layers), and
// (ii) the 4 KiB scratch holds 32 rows of one 128-byte line each; a block adds into the row its index hashes to, and the
// host adds the rows after the read-back.
constexpr int DIAG_ROWS = 32, DIAG_PITCH = 16, DIAG_ZBLOCKS = 16;

template <typename real, bool WALLS, int MODE>
__global__ void __launch_bounds__(128)
diagnostics_kernel(const real* __restrict__ src, double* __restrict__ acc, const FieldParams<real> P, const int zn)
{
    double v[10];
#pragma unroll
    for (int n = 0; n < 10; ++n) v[n] = 0.0;
    for (int zrel = blockIdx.z; zrel < zn; zrel += gridDim.z) {
        const SiteIndex i = my_site_in_layer(P.G, zrel);
        const bool fluid = i.valid && !(WALLS && solid_layer(P.G, i.zg));
        if (fluid) {
            real g[3][3][3];
            gather<real, WALLS, MODE>(src, P.G, i, g);
            const Moments10<real> m = forward_moments(g);
            const double rho = (double)m.rho, inv = 1.0 / rho;     // one fp64 division per site, not three
            const double ux = fma((double)m.jx, inv, (double)P.hgx);
            const double uy = fma((double)m.jy, inv, (double)P.hgy);
            const double uz = fma((double)m.jz, inv, (double)P.hgz);
            v[0] += rho; v[1] += rho * ux; v[2] += rho * uy; v[3] += rho * uz;
            v[4] += ux; v[5] += uy; v[6] += uz; v[7] += ux * ux; v[8] += uy * uy; v[9] += uz * uz;
        }
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
        const unsigned row = (blockIdx.x + 5u * blockIdx.y + 11u * blockIdx.z) % DIAG_ROWS;
        atomicAdd(acc + row * DIAG_PITCH + tid, s);
    }
}

// ---------------------------------------------------------------- state import / export (R10)
// out[canonical i][sl] = S_t[i](s): the same gather as the step; solid nodes export their stored values.
template <typename real, bool WALLS, int MODE>
__global__ void __launch_bounds__(128)
export_kernel(const real* __restrict__ src, real* __restrict__ out, const FieldParams<real> P)
{
    const SiteIndex i = my_site(P.G);
    if (!i.valid) return;
    if (WALLS && solid_layer(P.G, i.zg)) {
#pragma unroll
        for (int n = 0; n < Q; ++n) out[(long long)n * P.G.N + i.sl] = src[(long long)lex_of_canon(n) * P.G.QS + i.s];
        return;
    }
    real g[3][3][3];
    gather<real, WALLS, MODE>(src, P.G, i, g);
#pragma unroll
    for (int n = 0; n < Q; ++n)
        out[(long long)n * P.G.N + i.sl] = g[canon_cz(n) + 1][canon_cy(n) + 1][canon_cx(n) + 1];
}

// Indices into a canonical INPUT field around a site: the three x, y and z coordinates of its 3 x 3 x 3 neighbourhood
// (periodic in x, y; in z periodic over the nz owned layers, or, in slab mode, plain: the input then has nz + 2 layers,
// the owned ones at 1..nz).  No integer division: the neighbours are at most one step away.
struct InputStencil {
    int xs[3], ys[3], zs[3];
};
__device__ __forceinline__ InputStencil input_stencil(const Geom& G, int ghost_in, int x, int y, int zl)
{
    InputStencil t;
    t.xs[0] = (x == 0) ? G.nx - 1 : x - 1; t.xs[1] = x; t.xs[2] = (x + 1 == G.nx) ? 0 : x + 1;
    t.ys[0] = (y == 0) ? G.ny - 1 : y - 1; t.ys[1] = y; t.ys[2] = (y + 1 == G.ny) ? 0 : y + 1;
    if (ghost_in) {
        t.zs[0] = zl; t.zs[1] = zl + 1; t.zs[2] = zl + 2;
    } else {
        t.zs[0] = (zl == 0) ? G.nz - 1 : zl - 1; t.zs[1] = zl; t.zs[2] = (zl + 1 == G.nz) ? 0 : zl + 1;
    }
    return t;
}

// P[q](s) = S[q](s + c_q), or S[26-q](s) when s + c_q is solid; solid nodes store S[q](s) unchanged.
// `in` is canonical; the never-updated solid layers are written to both A and B buffers so that they agree.
// AA scheme (P.aa): the natural layout P[q](s) = S[q](s), one buffer (bufB == nullptr).
template <typename real, bool WALLS>
__global__ void __launch_bounds__(128)
import_kernel(const real* __restrict__ in, real* __restrict__ bufA, real* __restrict__ bufB, const FieldParams<real> P)
{
    const SiteIndex i = my_site(P.G);
    if (!i.valid) return;
    const Geom& G = P.G;
    const bool solid = WALLS && solid_layer(G, i.zg);
    const bool local = solid || P.aa;                      // every slot comes from the site itself
    const int zl = (int)blockIdx.z + G.zc;
    const long long Nin = (long long)G.nx * G.ny * (G.nz + 2 * P.ghost_in);
    const InputStencil t = input_stencil(G, P.ghost_in, i.x, i.y, zl);
    const long long own = (long long)t.xs[1] + (long long)G.nx * ((long long)t.ys[1] + (long long)G.ny * t.zs[1]);
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        // s + c_q solid: the slot is pulled back by the site itself as direction opp(q)
        const bool bounce = WALLS && !local && solid_layer(G, i.zg + c - 1);
#pragma unroll
        for (int b = 0; b < 3; ++b) {
            const long long row = (long long)G.nx * ((long long)t.ys[b] + (long long)G.ny * t.zs[c]);
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                const int q = a + 3 * b + 9 * c;
                const int n = canon_of_lex(q), nopp = canon_of_lex(26 - q);
                const long long from = local ? (long long)n * Nin + own
                                             : bounce ? (long long)nopp * Nin + own : (long long)n * Nin + row + t.xs[a];
                const real v = in[from];
                bufA[(long long)q * G.QS + i.s] = v;
                // the second A-B buffer only needs the solid layers (never updated, R12): the first step overwrites every fluid site
                if (WALLS && solid && bufB != nullptr) bufB[(long long)q * G.QS + i.s] = v;
            }
        }
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
// rho/u NULL -> uniform rho0, u = 0.  Fully unrolled over the 27 neighbours (their loads are independent: the loop form
// waited for one neighbour's four loads after the other and took 22 ms at 512^3 where this takes a third of that).
template <typename real, bool WALLS>
__global__ void __launch_bounds__(128)
init_kernel(const real* __restrict__ rho, const real* __restrict__ u, double rho0, real* __restrict__ bufA,
            real* __restrict__ bufB, const FieldParams<real> P)
{
    const SiteIndex i = my_site(P.G);
    if (!i.valid) return;
    const Geom& G = P.G;
    const bool solid = WALLS && solid_layer(G, i.zg);
    const bool local = solid || P.aa;                      // every slot from the site itself, in its own direction
    const int zl = (int)blockIdx.z + G.zc;
    const long long Nin = (long long)G.nx * G.ny * (G.nz + 2 * P.ghost_in);
    const InputStencil t = input_stencil(G, P.ghost_in, i.x, i.y, zl);
    const long long own = (long long)t.xs[1] + (long long)G.nx * ((long long)t.ys[1] + (long long)G.ny * t.zs[1]);
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        // s + c_q solid: f0 of the opposite direction at the site itself
        const bool bounce = WALLS && !local && solid_layer(G, i.zg + c - 1);
        const int sg = bounce ? -1 : 1;
#pragma unroll
        for (int b = 0; b < 3; ++b) {
            const long long row = (long long)G.nx * ((long long)t.ys[b] + (long long)G.ny * t.zs[c]);
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                const int q = a + 3 * b + 9 * c;
                const long long s = (local || bounce) ? own : row + t.xs[a];
                double r = rho0, ux = 0.0, uy = 0.0, uz = 0.0;
                if (rho != nullptr) {
                    r = (double)rho[s]; ux = (double)u[s]; uy = (double)u[Nin + s]; uz = (double)u[2 * Nin + s];
                }
                const real v = (real)__dmul_rn(__dmul_rn(__dmul_rn(r, phi1d(sg * (a - 1), ux)), phi1d(sg * (b - 1), uy)),
                                               phi1d(sg * (c - 1), uz));
                bufA[(long long)q * G.QS + i.s] = v;
                // the second A-B buffer only needs the solid layers (never updated, R12): the first step overwrites every fluid site
                if (WALLS && solid && bufB != nullptr) bufB[(long long)q * G.QS + i.s] = v;
            }
        }
    }
}

// ---------------------------------------------------------------- slab faces (rflbm_halo_pack / rflbm_halo_unpack)
// One nx x ny face of 9 consecutive storage slots [slot0, slot0 + 9) of storage layer z <-> a packed buffer
// face[9][ny][nx].  Which layer and which slots depends on scheme and phase (rflbm.cu::halo_plan).
template <typename real, bool PACK>
__global__ void __launch_bounds__(128)
halo_kernel(real* __restrict__ buf, real* __restrict__ face, const Geom G, int z, int slot0)
{
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    if (x >= G.nx || y >= G.ny) return;
    const long long s = (long long)x + (long long)G.px * y + G.pxy * z;
    const long long f = (long long)x + (long long)G.nx * y;
    const long long nf = (long long)G.nx * G.ny;
#pragma unroll
    for (int n = 0; n < 9; ++n) {
        if (PACK) face[n * nf + f] = buf[(long long)(slot0 + n) * G.QS + s];
        else buf[(long long)(slot0 + n) * G.QS + s] = face[n * nf + f];
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
    const SiteIndex i = my_site(P.G);
    if (!i.valid) return;
    const long long N = P.G.N;
    const PhiloxSite ps = philox_site(i.site, P.rng);
    bool bad = false;
#pragma unroll
    for (int call = 0; call < 6; ++call) {
        uint32_t w[4], w_ref[4];
        philox_call(ps, P.rng, call, w);
        philox4x32_10(i.site, t_hi, t_lo, (uint32_t)call, P.rng, w_ref);
        bad = bad || w[0] != w_ref[0] || w[1] != w_ref[1] || w[2] != w_ref[2] || w[3] != w_ref[3];
        if (words != nullptr)
#pragma unroll
            for (int mth = 0; mth < 4; ++mth) words[(long long)(4 * call + mth) * N + i.sl] = w[mth];
        if (normals != nullptr)
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                real z0, z1;
                normal_pair(w[2 * h], w[2 * h + 1], s_tab, s_tab + LOG_TABLE_N, z0, z1);
                const int k = 4 + 4 * call + 2 * h;
                normals[(long long)(k - 4) * N + i.sl] = z0;
                if (k + 1 < Q) normals[(long long)(k + 1 - 4) * N + i.sl] = z1;
            }
    }
    if (bad) atomicAdd(mismatch, 1ull);
}

}  // namespace rflbm_dev
