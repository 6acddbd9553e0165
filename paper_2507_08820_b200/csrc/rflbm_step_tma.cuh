// rflbm_step_tma.cuh — the hot kernel, TMA-staged (sm_100a): one time step of Eq.24 on an fp64 lattice with
// nx >= 128, nx even.
//
// Why (profiles/r01a_*): in the plain one-thread-per-site kernel every one of the 27 neighbour loads costs 4-5
// integer instructions of per-thread 64-bit address arithmetic and the block's memory latency is exposed
// between its load phase and its ~1500-instruction compute phase.  Here the 27 row segments a tile of 128
// consecutive x needs are fetched by 27 `cp.async.bulk.tensor` (TMA) copies issued by one thread into shared
// memory: the TMA unit generates the addresses, applies the -c_q shift (box start x0 + c-shift, y -+ 1, z -+ 1,
// array q — or array 26-q at the same site for halfway bounce-back, R12), and the copy of tile k+1 is issued as
// soon as tile k has been moved from shared memory to registers, so it overlaps the whole collision of tile k.
// Threads read their 27 populations with LDS [reg + immediate].  A block walks `rows` consecutive y rows so the
// Box-Muller tables are staged once per block.
//
// TMA needs 16-byte aligned box starts (measured: an odd fp64 x coordinate raises "illegal instruction"), so every
// copy is a 130-element box starting at an even x: [x0, x0+130) for cx <= 0 and [x0-2, x0+128) for cx = +1, and a
// thread reads element tid + 1 of it for cx != 0 (tid for cx = 0 and for bounced-back populations).
//
// The only thing TMA cannot do is the periodic wrap in x (out-of-bounds box elements are zero-filled): the
// threads at x = 0 and x = nx-1 re-load their 9 wrapped populations directly from global memory.
#pragma once
#include <cuda.h>

#include "rflbm_kernels.cuh"

namespace rflbm_dev {

constexpr int TILE_X = 128;
constexpr int BOX_X = TILE_X + 2;      // elements per TMA box (1040 B, a multiple of 16 B)
constexpr int ROW_PITCH = 144;         // doubles per staged row: 1152 B keeps every box destination 128-byte aligned

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    uint32_t ok, spins = 0;
    do {
        if (++spins > (1u << 24)) __trap();     // a lost TMA transaction must fail loudly, never hang the GPU
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(ok)
            : "r"(bar), "r"(parity)
            : "memory");
    } while (!ok);
}
__device__ __forceinline__ void tma_load_row(uint32_t dst, const CUtensorMap* tmap, int x, int y, int z, int q, uint32_t bar)
{
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
        ::"r"(dst), "l"((unsigned long long)tmap), "r"(x), "r"(y), "r"(z), "r"(q), "r"(bar)
        : "memory");
}

// issue the 27 row copies of tile (x0, y, z); one thread
template <bool WALLS>
__device__ __forceinline__ void issue_tile(const CUtensorMap* tmap, uint32_t s_in, uint32_t bar, int x0, int y, int z,
                                           int ny, int nz)
{
    mbar_expect_tx(bar, Q * BOX_X * (uint32_t)sizeof(double));
    const int ys[3] = {(y + 1 == ny) ? 0 : y + 1, y, (y == 0) ? ny - 1 : y - 1};     // y - cy, index b = cy + 1
    const int zs[3] = {(z + 1 == nz) ? 0 : z + 1, z, (z == 0) ? nz - 1 : z - 1};
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const bool bounce = WALLS && ((c == 2 && z == 1) || (c == 0 && z == nz - 2));
#pragma unroll
        for (int b = 0; b < 3; ++b)
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                const int q = a + 3 * b + 9 * c;
                const uint32_t dst = s_in + (uint32_t)(q * ROW_PITCH * sizeof(double));
                if (WALLS && bounce) tma_load_row(dst, tmap, x0, y, z, 26 - q, bar);
                else tma_load_row(dst, tmap, (a == 2) ? x0 - 2 : x0, ys[b], zs[c], q, bar);   // even box start
            }
    }
}

template <bool WALLS, bool FORCE, bool NOISE>
__global__ void __launch_bounds__(TILE_X)
step_kernel_tma(const __grid_constant__ CUtensorMap tmap_src, const double* __restrict__ src, double* __restrict__ dst,
                const __grid_constant__ StepParams<double> P, int rows)
{
    __shared__ __align__(128) double s_in[Q][ROW_PITCH];
    __shared__ f64x2 s_tab[NOISE ? LOG_TABLE_N + SC_TABLE_N : 1];
    __shared__ __align__(8) unsigned long long s_bar;

    const int z = blockIdx.z;
    if (WALLS && (z == 0 || z == P.nz - 1)) return;            // solid layers are never updated
    const int tid = threadIdx.x;
    const int x0 = blockIdx.x * TILE_X;
    const int y_begin = blockIdx.y * rows;
    const int y_end = min(y_begin + rows, P.ny);
    const uint32_t bar = smem_u32(&s_bar), in0 = smem_u32(&s_in[0][0]);

    if (tid == 0) {
        mbar_init(bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (tid == 0) issue_tile<WALLS>(&tmap_src, in0, bar, x0, y_begin, z, P.ny, P.nz);
    if (NOISE) stage_tables(P.tables, s_tab);                   // ends with __syncthreads()

    const int x = x0 + tid;
    const bool active = x < P.nx;
    const bool wrap_lo = (x == 0), wrap_hi = (x == P.nx - 1);
    const long long nxy = (long long)P.nx * P.ny;
    uint32_t parity = 0;

    for (int y = y_begin; y < y_end; ++y) {
        const long long s = (long long)x + (long long)P.nx * y + nxy * z;
        mbar_wait(bar, parity);
        parity ^= 1u;
        double g[3][3][3];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            // x - cx sits at element tid + 1 of the box for cx != 0; bounced-back rows hold the site itself at tid
            const bool bounce = WALLS && ((c == 2 && z == 1) || (c == 0 && z == P.nz - 2));
            const int side = (WALLS && bounce) ? tid : tid + 1;
#pragma unroll
            for (int b = 0; b < 3; ++b) {
                g[c][b][0] = s_in[0 + 3 * b + 9 * c][side];
                g[c][b][1] = s_in[1 + 3 * b + 9 * c][tid];
                g[c][b][2] = s_in[2 + 3 * b + 9 * c][side];
            }
        }
        __syncthreads();                                       // the tile is in registers: the buffer is free
        if (tid == 0 && y + 1 < y_end) issue_tile<WALLS>(&tmap_src, in0, bar, x0, y + 1, z, P.ny, P.nz);

        if (wrap_lo || wrap_hi) {                              // periodic wrap in x: TMA zero-filled these
            const int ysr[3] = {(y + 1 == P.ny) ? 0 : y + 1, y, (y == 0) ? P.ny - 1 : y - 1};
            const int zsr[3] = {(z + 1 == P.nz) ? 0 : z + 1, z, (z == 0) ? P.nz - 1 : z - 1};
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const bool bounce = WALLS && ((c == 2 && z == 1) || (c == 0 && z == P.nz - 2));
                if (bounce) continue;                          // bounced populations come from the site itself
#pragma unroll
                for (int b = 0; b < 3; ++b) {
                    const long long row = (long long)P.nx * ysr[b] + nxy * zsr[c];
                    if (wrap_hi) g[c][b][0] = __ldg(src + (long long)(0 + 3 * b + 9 * c) * P.N + row);                // x+1 -> 0
                    if (wrap_lo) g[c][b][2] = __ldg(src + (long long)(2 + 3 * b + 9 * c) * P.N + row + (P.nx - 1));   // x-1 -> nx-1
                }
            }
        }
        if (active) {
            collide<double, FORCE, NOISE>(g, P, (uint32_t)s, s_tab, s_tab + LOG_TABLE_N);
            char* out = reinterpret_cast<char*>(dst + s);
            const long long qstride = P.N * (long long)sizeof(double);
#pragma unroll
            for (int c = 0; c < 3; ++c)
#pragma unroll
                for (int b = 0; b < 3; ++b)
#pragma unroll
                    for (int a = 0; a < 3; ++a)
                        __stcs(reinterpret_cast<double*>(out + (long long)(a + 3 * b + 9 * c) * qstride), g[c][b][a]);
        }
    }
}

}  // namespace rflbm_dev
